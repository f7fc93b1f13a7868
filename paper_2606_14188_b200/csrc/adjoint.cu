// ltv_scan_adjoint: lam_T = g_T; lam_t = A_t^T lam_{t+1} + g_t; grad_u[t] = B_t^T lam_{t+1}; grad_x0 = A_0^T lam_1
// (eq.(10) chained over the horizon).
//
// HBM-bound transposed-GEMV chain.  One cluster per batch item; CTA `rank` owns a band of COLUMNS of every
// A_t (so that its slice of A_t^T lam needs no cross-CTA reduction).  The band is streamed as
// [rows x <=256 columns] boxes by 2-D tensor TMA into a shared-memory ring, in reverse time order, by a
// producer thread that runs ahead of the consumers.  A consumer thread owns four adjacent columns and one
// residue class of rows, so the inner loop is one 128-bit shared load + one broadcast load + 4 FMA; the
// row classes are combined through shared memory once per (step, column slab).  The new costate is
// written into every CTA of the cluster through DSMEM (st.async + mbarrier byte count), as in the rollout.
#include <cuda.h>

#include "ltv_internal.h"
#include "ptx.cuh"

namespace ltv {

namespace {

constexpr int kAdjConsThreads = 256;   // threads of one consumer group
constexpr int kAdjGroups = 2;          // consumer groups; group g takes the ring boxes with index % kAdjGroups == g
constexpr int kAdjAllCons = kAdjConsThreads * kAdjGroups;
constexpr int kAdjThreads = kAdjAllCons + 64;  // + producer warp + helper warp
constexpr int kAdjMaxStages = 8;
constexpr int kStageVecs = 384;  // float4 of B_t the helper warp stages in shared memory per tile (6 KB)
constexpr int kMaxL = 8;         // columns of grad_u one CTA reduces on the fast path

struct AdjPlan {
  int bw;      // box width (columns), multiple of 4, <= 256
  int rcb;     // box rows
  int stages;
  int qt, rg;  // quad-threads per row, row groups
  uint32_t stage_bytes, off_lam, off_red, off_stage, off_bar, total;
};

struct AdjParams {
  const float *A, *B, *g;
  float *lam_out, *gu_out, *gx0_out;
  int batch, T, n, m;
  AdjPlan ap;
};

__host__ __device__ inline void col_band(int n, int C, int rank, int& j0, int& j1) {
  const int nq = n >> 2;
  j0 = 4 * static_cast<int>((static_cast<long long>(nq) * rank) / C);
  j1 = 4 * static_cast<int>((static_cast<long long>(nq) * (rank + 1)) / C);
}

constexpr int kLamBufs = 4;   // costate buffers / barriers: a remote CTA can be two steps ahead of this CTA's helper warp, which
                              // still reads lam_{t+1} of its step for grad_u, so the buffer written two steps ahead must differ
__device__ __forceinline__ uint32_t lam_parity(int k) {
  return static_cast<uint32_t>(k / kLamBufs - (k % kLamBufs == 0 ? 1 : 0)) & 1u;
}

__global__ void __launch_bounds__(kAdjThreads, 1)
adjoint_kernel(const AdjParams p, const __grid_constant__ CUtensorMap tmapA) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int C = static_cast<int>(cluster_nctarank());
  const int rank = static_cast<int>(cluster_ctarank());
  const int item = blockIdx.x / C;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n = p.n, T = p.T, m = p.m;
  const AdjPlan& ap = p.ap;
  int j0, j1;
  col_band(n, C, rank, j0, j1);
  const int W = j1 - j0;
  const int nslab = (W + ap.bw - 1) / ap.bw;
  const int nrb = (n + ap.rcb - 1) / ap.rcb;
  const int nstep = (T - 1) + (p.gx0_out ? 1 : 0);  // GEMV steps: A_{T-1} .. A_1 (, A_0)

  float* lambuf = reinterpret_cast<float*>(smem + ap.off_lam);  // [kLamBufs][n]
  float* red = reinterpret_cast<float*>(smem + ap.off_red);     // [rg][bw]
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + ap.off_bar);
  uint64_t* full = bars;
  uint64_t* empty = bars + kAdjMaxStages;   // kAdjConsThreads/32 arrivals
  uint64_t* lfull = bars + 2 * kAdjMaxStages;  // [kLamBufs] input costate of step k complete in lambuf[k % kLamBufs]

  if (threadIdx.x == 0) {
    for (int s = 0; s < ap.stages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], kAdjConsThreads / 32);
    }
    for (int s = 0; s < kLamBufs; ++s) mbar_init(&lfull[s], 1);
    fence_mbar_init();
    tma_prefetch_desc(&tmapA);
  }
  // lambuf[0] = lam_T = g_T
  const float* gT = p.g + (static_cast<size_t>(item) * T + (T - 1)) * n;
  for (int j = threadIdx.x; j < n; j += kAdjThreads) {
    const float v = gT[j];
    lambuf[j] = v;
    if (j >= j0 && j < j1) p.lam_out[(static_cast<size_t>(item) * T + (T - 1)) * n + j] = v;   // lam_out[T-1] = lam_T
  }
  __syncthreads();
  cluster_sync_all();

  // step k = 0 .. nstep-1 multiplies by A_t^T with t = T-1-k; its input costate lam_{t+1} is lambuf[k % kLamBufs];
  // barrier lfull[j] is used for k = j, j + kLamBufs, .. except k = 0 (local init): phase index k / kLamBufs - (k % kLamBufs == 0)
  if (warp == kAdjAllCons / 32) {
    // ------------------------------------------------------------------ producer
    if (lane == 0 && W > 0) {
      const uint64_t pol = l2_policy_evict_first();
      int st = 0;
      uint32_t eph = 1;   // parity of empty[st] (the first pass over the ring does not block)
      for (int k = 0; k < nstep; ++k) {
        const int t = T - 1 - k;
        const int row_base = (item * T + t) * n;  // validated on the host to fit in int
        for (int sl = 0; sl < nslab; ++sl) {
          for (int rb = 0; rb < nrb; ++rb) {
            mbar_wait(&empty[st], eph);
            mbar_arrive_expect_tx(&full[st], static_cast<uint32_t>(ap.bw) * ap.rcb * 4u);
            tma_load_2d(smem + static_cast<size_t>(st) * ap.stage_bytes, &tmapA, j0 + sl * ap.bw,
                        row_base + rb * ap.rcb, &full[st], pol);
            if (++st == ap.stages) { st = 0; eph ^= 1; }
          }
        }
      }
    }
  } else if (warp == kAdjAllCons / 32 + 1) {
    // ------------------------------------------------------------------ helper: barrier arming + grad_u
    // at step k (t = T-1-k): wait lam_{t+1}, arm the barrier of lam_t, grad_u[t][l] = sum_i B_t[i][l] lam_{t+1}[i]
    // for the columns l = rank, rank + C, ...  B_t is contiguous: it is read with 128-bit loads, a tile of
    // kStageVecs float4 at a time (all loads of a tile in flight together, the next tile's issued before this
    // one is reduced), staged in shared memory and reduced lane-per-row.
    float4* stB = reinterpret_cast<float4*>(smem + ap.off_stage);
    const int ncol = (p.gu_out && rank < m) ? (m - rank + C - 1) / C : 0;   // columns of grad_u this CTA owns
    const bool fast = ncol > 0 && ncol <= kMaxL && 4 * m <= kStageVecs * 4;
    const int rows_tile = fast ? ((kStageVecs * 4) / m) & ~3 : 0;           // rows of B per tile (multiple of 4: 16-byte tiles)
    const int ntile = fast ? (n + rows_tile - 1) / rows_tile : 0;
    constexpr int kVB = kStageVecs / 32;
    for (int k = 0; k < T; ++k) {
      const int t = T - 1 - k;
      const float* Bt = p.B + (static_cast<size_t>(item) * T + t) * n * m;
      float4 vb[kVB];
      auto issue = [&](int tile) {
        const float4* src = reinterpret_cast<const float4*>(Bt + static_cast<size_t>(tile) * rows_tile * m);
        const int nv = (min(rows_tile, n - tile * rows_tile) * m) >> 2;   // n % 4 == 0: whole float4
#pragma unroll
        for (int j = 0; j < kVB; ++j) vb[j] = (lane + 32 * j < nv) ? __ldg(src + lane + 32 * j) : make_float4(0.f, 0.f, 0.f, 0.f);
      };
      if (fast) issue(0);
      if (k >= 1) mbar_wait_cluster(&lfull[k % kLamBufs], lam_parity(k));
      if (k + 1 < T && lane == 0) mbar_arrive_expect_tx(&lfull[(k + 1) % kLamBufs], static_cast<uint32_t>(n) * 4u);
      const float* lam = lambuf + (k % kLamBufs) * n;
      if (fast) {
        float acc[kMaxL];
#pragma unroll
        for (int c = 0; c < kMaxL; ++c) acc[c] = 0.f;
        for (int tile = 0; tile < ntile; ++tile) {
          const int rt = min(rows_tile, n - tile * rows_tile);
          const int nv = (rt * m) >> 2;
          __syncwarp();   // the previous tile has been reduced
#pragma unroll
          for (int j = 0; j < kVB; ++j)
            if (lane + 32 * j < nv) stB[lane + 32 * j] = vb[j];
          __syncwarp();
          if (tile + 1 < ntile) issue(tile + 1);
          const float* sB = reinterpret_cast<const float*>(stB);
          for (int i = lane; i < rt; i += 32) {
            const float li = lam[tile * rows_tile + i];
#pragma unroll
            for (int c = 0; c < kMaxL; ++c)
              if (c < ncol) acc[c] = fmaf(sB[i * m + rank + c * C], li, acc[c]);
          }
        }
#pragma unroll
        for (int c = 0; c < kMaxL; ++c) {
          if (c < ncol) {
            float a = acc[c];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
            if (lane == 0) p.gu_out[(static_cast<size_t>(item) * T + t) * m + rank + c * C] = a;
          }
        }
      } else if (p.gu_out) {
        for (int l = rank; l < m; l += C) {
          float acc = 0.f;
          for (int i = lane; i < n; i += 32) acc = fmaf(__ldg(Bt + static_cast<size_t>(i) * m + l), lam[i], acc);
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
          if (lane == 0) p.gu_out[(static_cast<size_t>(item) * T + t) * m + l] = acc;
        }
      }
    }
  } else {
    // ------------------------------------------------------------------ consumers
    // Two groups of 256 threads take alternate ring boxes (one group's shared loads run under the other
    // group's barrier waits and loop overheads); a thread keeps one accumulator quad per slab over its group's
    // boxes, and the row classes of BOTH groups are combined in fixed order at the end of the slab.
    const int grp = threadIdx.x / kAdjConsThreads;
    const int tid = threadIdx.x % kAdjConsThreads;
    const int q = tid % ap.qt, rgi = tid / ap.qt;
    const bool active = rgi < ap.rg;
    uint32_t it = 0;
    int st = 0;
    uint32_t fph = 0;
    for (int k = 0; k < nstep; ++k) {
      const int t = T - 1 - k;
      if (k >= 1) mbar_wait_cluster(&lfull[k % kLamBufs], lam_parity(k));
      const float* lam = lambuf + (k % kLamBufs) * n;
      float* lnext = lambuf + ((k + 1) % kLamBufs) * n;
      uint64_t* lbar = &lfull[(k + 1) % kLamBufs];
      const float* gt = (t >= 1) ? p.g + (static_cast<size_t>(item) * T + (t - 1)) * n : nullptr;
      for (int sl = 0; sl < nslab; ++sl) {
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int rb = 0; rb < nrb; ++rb, ++it) {
          if (static_cast<int>(it % kAdjGroups) == grp) {
            mbar_wait(&full[st], fph);
            const float* tile = reinterpret_cast<const float*>(smem + static_cast<size_t>(st) * ap.stage_bytes);
            const int i0 = rb * ap.rcb;
            const int rk = min(ap.rcb, n - i0);
            if (active) {
#pragma unroll 8
              for (int i = rgi; i < rk; i += ap.rg) {
                const float4 a = *reinterpret_cast<const float4*>(tile + static_cast<size_t>(i) * ap.bw + 4 * q);
                const float l = lam[i0 + i];
                acc.x = fmaf(a.x, l, acc.x);
                acc.y = fmaf(a.y, l, acc.y);
                acc.z = fmaf(a.z, l, acc.z);
                acc.w = fmaf(a.w, l, acc.w);
              }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]);
          }
          if (++st == ap.stages) { st = 0; fph ^= 1; }
        }
        // combine the row classes (fixed order => deterministic) and publish this slab of the costate
        if (active) *reinterpret_cast<float4*>(red + static_cast<size_t>(grp * ap.rg + rgi) * ap.bw + 4 * q) = acc;
        named_bar_sync(1, kAdjAllCons);
        // thread (column quad, destination CTA): one 16-byte remote store per pair instead of 4 x C 4-byte ones
        const int nquad = ap.bw >> 2;
        for (int idx = threadIdx.x; idx < nquad * C; idx += kAdjAllCons) {
          const int jq = idx / C, cta = idx - jq * C;
          const int col = j0 + sl * ap.bw + 4 * jq;
          if (col < j1) {   // bands and boxes are whole quads
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int r = 0; r < kAdjGroups * ap.rg; ++r) {
              const float4 pr = *reinterpret_cast<const float4*>(red + static_cast<size_t>(r) * ap.bw + 4 * jq);
              v.x += pr.x; v.y += pr.y; v.z += pr.z; v.w += pr.w;
            }
            if (t >= 1) {
              const float4 gq = __ldg(reinterpret_cast<const float4*>(gt + col));
              v.x += gq.x; v.y += gq.y; v.z += gq.z; v.w += gq.w;
              st_async_remote_f32x4(lnext + col, v, lbar, cta);
              if (cta == 0)   // lam_out[t-1] = lam_t
                *reinterpret_cast<float4*>(p.lam_out + (static_cast<size_t>(item) * T + (t - 1)) * n + col) = v;
            } else if (cta == 0) {
              *reinterpret_cast<float4*>(p.gx0_out + static_cast<size_t>(item) * n + col) = v;
            }
          }
        }
        named_bar_sync(1, kAdjAllCons);
      }
    }
  }
  __syncthreads();
  cluster_sync_all();
}

AdjPlan plan_adjoint(int n, int C) {
  AdjPlan ap{};
  const int nq = n >> 2;
  const int wmax = 4 * ((nq + C - 1) / C);
  ap.bw = wmax < 256 ? wmax : 256;
  if (ap.bw < 4) ap.bw = 4;
  ap.qt = ap.bw / 4;
  ap.rg = kAdjConsThreads / ap.qt;
  if (ap.rg > 32) ap.rg = 32;
  const uint32_t lam_bytes = static_cast<uint32_t>(align_up(static_cast<size_t>(kLamBufs) * n * 4u, 128));
  const uint32_t red_bytes = static_cast<uint32_t>(align_up(static_cast<size_t>(kAdjGroups) * ap.rg * ap.bw * 4, 128));
  const uint32_t budget = 227u * 1024u - lam_bytes - red_bytes - kStageVecs * 16u - 256u;
  // The ring must have an EVEN number of stages.  The two consumer groups take alternate boxes and never look at the other
  // group's: with an odd ring a stage changes hands every pass, so a group sees only every other phase of that stage's `full`
  // barrier and its parity test cannot tell "my box has landed" from "the other group's box of the pass before is still in
  // flight" (bulk copies of different boxes may complete out of order).  A group that runs into this reads a stale box and
  // arrives on `empty` out of turn - an mbarrier arrival-count underflow, i.e. the sporadic "unspecified launch failure"s
  // (and, rarely, dead locks) that matrices of n >= 1536 on >= ~100 CTAs raised in round 2 with a ring of 5.  With an even ring
  // every stage belongs to one group, which then observes every phase.
  // Boxes of ~32 KB, shrunk so that an even number of them fills the budget, the row blocks of a step equal.
  int st = static_cast<int>(budget / (32u * 1024u));
  if (st > kAdjMaxStages) st = kAdjMaxStages;
  if (st & 1) st += 1;                     // e.g. 5 boxes of 32 KB -> 6 of ~27 KB
  if (st < 2) st = 2;
  uint32_t box = budget / static_cast<uint32_t>(st);
  if (box > 32u * 1024u) box = 32u * 1024u;
  int rcb = static_cast<int>(box / (ap.bw * 4u));
  if (rcb > 256) rcb = 256;
  if (rcb > n) rcb = n;
  if (rcb < 1) rcb = 1;
  rcb = (n + (n + rcb - 1) / rcb - 1) / ((n + rcb - 1) / rcb);   // equal row blocks: no rows of the next matrix are fetched
  ap.rcb = rcb;
  ap.stage_bytes = static_cast<uint32_t>(align_up(static_cast<size_t>(ap.bw) * rcb * 4, 128));
  st = static_cast<int>(budget / ap.stage_bytes);
  if (st > kAdjMaxStages) st = kAdjMaxStages;
  st &= ~1;
  if (env_int("ADJ_ODD_RING", 0) && st > 3) st -= 1;   // developer builds: bring the ring bug back (to check the regression test)
  ap.stages = st;
  ap.off_lam = ap.stage_bytes * st;
  ap.off_red = ap.off_lam + lam_bytes;
  ap.off_stage = ap.off_red + red_bytes;
  ap.off_bar = ap.off_stage + kStageVecs * 16u;
  ap.total = ap.off_bar + (2 * kAdjMaxStages + kLamBufs) * 8;
  return ap;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

// shared with phi.cu
void* get_encode_tiled() {
  static void* fn = nullptr;
  if (!fn) {
    cudaDriverEntryPointQueryResult q;
    void* f = nullptr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = f;
  }
  return fn;
}

static const int* adjoint_max_active() {
  static int max_active[17];
  static bool have = false;
  if (!have) {
    query_max_active_clusters(reinterpret_cast<const void*>(adjoint_kernel), kAdjThreads, 200 * 1024, max_active);
    have = true;
  }
  return max_active;
}

int adjoint_cluster_choice(const AdjointArgs& a) { return pick_cluster_model(a.batch, a.n, adjoint_max_active(), a.sm_budget); }

int adjoint_clusters_resident(const AdjointArgs& a, int cluster) {
  return (cluster >= 1 && cluster <= 16) ? adjoint_max_active()[cluster] : 0;
}

cudaError_t launch_adjoint(const AdjointArgs& a, int cluster, cudaStream_t stream, unsigned long long* launches) {
  AdjParams p{};
  p.A = a.A; p.B = a.B; p.g = a.g;
  p.lam_out = a.lambda_out; p.gu_out = (a.m > 0) ? a.grad_u_out : nullptr; p.gx0_out = a.grad_x0_out;
  p.batch = a.batch; p.T = a.T; p.n = a.n; p.m = a.m;
  if (cluster <= 0) cluster = pick_cluster_model(a.batch, a.n, adjoint_max_active(), a.sm_budget);
  p.ap = plan_adjoint(a.n, cluster);
  if (p.ap.stages < 2) return cudaErrorInvalidConfiguration;

  EncodeTiledFn enc = reinterpret_cast<EncodeTiledFn>(get_encode_tiled());
  if (!enc) return cudaErrorNotSupported;
  CUtensorMap tmap;
  const cuuint64_t dims[2] = {static_cast<cuuint64_t>(a.n), static_cast<cuuint64_t>(a.batch) * a.T * a.n};
  const cuuint64_t strides[1] = {static_cast<cuuint64_t>(a.n) * 4};
  const cuuint32_t box[2] = {static_cast<cuuint32_t>(p.ap.bw), static_cast<cuuint32_t>(p.ap.rcb)};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(a.A), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;

  cudaError_t e = cudaFuncSetAttribute(adjoint_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, p.ap.total);
  if (e != cudaSuccess) return e;
  if (cluster > 8) {
    e = cudaFuncSetAttribute(adjoint_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
  }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>(a.batch) * cluster);
  cfg.blockDim = dim3(kAdjThreads);
  cfg.dynamicSmemBytes = p.ap.total;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = cluster;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  LTV_DBG_INSTALL();
  {
    ProfScope prof(kProfAdjoint, stream);
    e = cudaLaunchKernelEx(&cfg, adjoint_kernel, p, tmap);
  }
  if (e == cudaSuccess) ++*launches;
  return e;
}

}  // namespace ltv
