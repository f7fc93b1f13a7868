// ltv_scan_rollout: x_{t+1} = A_t x_t + B_t u_t + c_t   (eq.(2), :139 eq.(12b))
//
// HBM-bound GEMV chain.  One thread-block cluster per batch item; CTA `rank` of the cluster owns a
// contiguous band of rows of every A_t.  A dedicated producer thread streams that band through a
// shared-memory ring with 1-D bulk TMA copies (the band of one step is contiguous in memory), running
// ahead of the consumers across step boundaries, so the only thing on the sequential critical path is the
// shared-memory GEMV and the exchange of the new state: the consumer warps write their rows of x_{t+1}
// straight into the x buffer of EVERY CTA of the cluster (st.async through DSMEM) and the byte count of an
// mbarrier in each CTA tells that CTA when x_{t+1} is complete.  The affine term b_t = B_t u_t + c_t is
// formed one step ahead by a helper warp and never touches global memory.
//
// GEMV inner loop (the measured limiter of the first version, which reduced every row with a 5-level shuffle
// tree: 63 % of the HBM peak at C2 against 95 % with the arithmetic knocked out).  A lane owns column quads
// and keeps its slice of x_t in registers for the whole step; a warp walks FOUR rows at a time, so a pass is
// 4 x QL independent 128-bit shared loads feeding 4 accumulators, and the four row sums are finished with a
// transpose-reduce (6 shuffles for 4 rows instead of 20).
//   mode A (n <= 640): a ring chunk holds rc = 8 * rpw rows, warp w owns rows [w rpw, (w+1) rpw) of it and
//                      all columns (QL <= 5 quads per lane);
//   mode B (n  > 640): a chunk holds <= 4 rows, warp w owns an eighth of the columns of every row (QL <= 8),
//                      the eight partial sums per row meet in shared memory behind one named barrier.
#include "ltv_internal.h"
#include "ptx.cuh"

#ifndef LTV_ROLL_DBG
#define LTV_ROLL_DBG 0
#endif

namespace ltv {

namespace {

constexpr int kConsWarps = 8;
constexpr int kRollThreads = (kConsWarps + 2) * 32;  // + producer warp + affine warp
constexpr int kMaxStages = 8;
constexpr int kModeAMaxN = 640;

struct RollSmemPlan {
  int rc;              // rows per ring chunk
  int rpw;             // mode A: rows per warp per chunk (rc = 8 rpw)
  int wide;            // 0 = mode A, 1 = mode B
  int stages;
  uint32_t stage_bytes;
  uint32_t off_x, off_b, off_part, off_bar, total;
  int rows_max;        // max rows owned by one CTA
};

__host__ __device__ inline void band(int n, int C, int rank, int& r0, int& r1) {
  r0 = static_cast<int>((static_cast<long long>(n) * rank) / C);
  r1 = static_cast<int>((static_cast<long long>(n) * (rank + 1)) / C);
}

struct RollParams {
  const float *A, *B, *c, *x0, *u;
  float* x_out;
  int batch, T, n, m;
  RollSmemPlan sp;
};

// Four per-lane partial sums (one per row) -> every lane of lane group g = lane / 8 holds the complete sum of
// row g.  Two exchange levels halve the values per lane, three butterfly levels finish: 6 shuffles.
__device__ __forceinline__ float reduce4_rows(const float (&a)[4], int lane) {
  const bool hi16 = (lane & 16) != 0;
  const float k0 = hi16 ? a[2] : a[0], k1 = hi16 ? a[3] : a[1];
  const float s0 = hi16 ? a[0] : a[2], s1 = hi16 ? a[1] : a[3];
  const float b0 = k0 + __shfl_xor_sync(0xffffffffu, s0, 16);
  const float b1 = k1 + __shfl_xor_sync(0xffffffffu, s1, 16);
  const bool hi8 = (lane & 8) != 0;
  float v = (hi8 ? b1 : b0) + __shfl_xor_sync(0xffffffffu, hi8 ? b0 : b1, 8);
  v += __shfl_xor_sync(0xffffffffu, v, 4);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  return v;
}

__device__ __forceinline__ float dot4(const float4 a, const float4 x, float acc) {
  return fmaf(a.x, x.x, fmaf(a.y, x.y, fmaf(a.z, x.z, fmaf(a.w, x.w, acc))));
}

// acc[r] += sum_j A[row_r][q0 + 32 j] . xq[j] for four rows of a shared-memory tile (row stride n floats);
// quads at or beyond q_end are skipped, rows flagged invalid contribute nothing (their address is clamped by
// the caller so that the loads stay inside the stage)
template <int QLMAX>
__device__ __forceinline__ void rows4_dot(const float* tile, int n, const int (&rowi)[4], int q0, int q_end, int ql,
                                          const float4 (&xq)[QLMAX], float (&acc)[4]) {
#pragma unroll
  for (int j = 0; j < QLMAX; ++j) {
    if (j < ql) {
      const int q = q0 + 32 * j;
      if (q < q_end) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          const float4 a = *reinterpret_cast<const float4*>(tile + static_cast<size_t>(rowi[r]) * n + 4 * q);
          acc[r] = dot4(a, xq[j], acc[r]);
        }
      }
    }
  }
}

template <bool WIDE>
__global__ void __launch_bounds__(kRollThreads, 1) rollout_kernel(const RollParams p) {
  constexpr int QLMAX = WIDE ? 8 : 5;
  extern __shared__ __align__(128) uint8_t smem[];
  const int C = static_cast<int>(cluster_nctarank());
  const int rank = static_cast<int>(cluster_ctarank());
  const int item = blockIdx.x / C;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n = p.n, T = p.T, m = p.m;
  int r0, r1;
  band(n, C, rank, r0, r1);
  const int rows = r1 - r0;
  const int rc = p.sp.rc, stages = p.sp.stages;
  const int nchunks = (rows + rc - 1) / rc;

  float* ring = reinterpret_cast<float*>(smem);
  float* xbuf = reinterpret_cast<float*>(smem + p.sp.off_x);   // [2][n]
  float* bvec = reinterpret_cast<float*>(smem + p.sp.off_b);   // [2][rows_max]
  float* part = reinterpret_cast<float*>(smem + p.sp.off_part);  // mode B: [2][kConsWarps][4]
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + p.sp.off_bar);
  uint64_t* full = bars;                    // [stages]  producer -> consumers (tx bytes)
  uint64_t* empty = bars + kMaxStages;      // [stages]  consumers -> producer (kConsWarps arrivals)
  uint64_t* xfull = bars + 2 * kMaxStages;  // [2]       x_{t} complete in xbuf[t&1] (n*4 tx bytes + 1 arrival)
  uint64_t* bfull = xfull + 2;              // [2]       b_t complete in bvec[t&1]

  if (threadIdx.x == 0) {
    for (int s = 0; s < stages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], kConsWarps);
    }
    mbar_init(&xfull[0], 1);
    mbar_init(&xfull[1], 1);
    mbar_init(&bfull[0], 1);
    mbar_init(&bfull[1], 1);
    fence_mbar_init();
  }
  for (int j = threadIdx.x; j < n; j += kRollThreads) xbuf[j] = p.x0[static_cast<size_t>(item) * n + j];
  __syncthreads();
  cluster_sync_all();  // every CTA's barriers are initialised before any remote st.async can target them

  const size_t itemA = static_cast<size_t>(item) * T * n * n;

  if (warp == kConsWarps) {
    // ------------------------------------------------------------------ producer (one thread)
    if (lane == 0 && rows > 0) {
      const uint64_t pol = l2_policy_evict_first();
      int st = 0;
      uint32_t eph = 1;   // parity of empty[st] to wait for (the first pass over the ring does not block)
      for (int t = 0; t < T; ++t) {
        const float* At = p.A + itemA + (static_cast<size_t>(t) * n + r0) * n;
        for (int k = 0; k < nchunks; ++k) {
          mbar_wait(&empty[st], eph);
          const int rk = min(rc, rows - k * rc);
          const uint32_t bytes = static_cast<uint32_t>(rk) * n * 4u;
          mbar_arrive_expect_tx(&full[st], bytes);
          bulk_g2s(reinterpret_cast<uint8_t*>(ring) + static_cast<size_t>(st) * p.sp.stage_bytes,
                   At + static_cast<size_t>(k) * rc * n, bytes, &full[st], pol);
          if (++st == stages) { st = 0; eph ^= 1; }
        }
      }
    }
  } else if (warp == kConsWarps + 1) {
    // ------------------------------------------------------------------ affine / output warp
    // step t: wait x_t, arm the barrier of x_{t+1}, write x_t to global, form b_{t+1}
    auto form_b = [&](int t) {
      float* bv = bvec + (t & 1) * p.sp.rows_max;
      const size_t bt = static_cast<size_t>(item) * T + t;
      for (int i = lane; i < rows; i += 32) {
        float acc = p.c ? p.c[bt * n + r0 + i] : 0.f;
        if (p.B && p.u) {
          const float* Brow = p.B + (bt * n + r0 + i) * m;
          const float* ut = p.u + bt * m;
          for (int l = 0; l < m; ++l) acc = fmaf(__ldg(Brow + l), __ldg(ut + l), acc);
        }
        bv[i] = acc;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&bfull[t & 1]);
    };
    form_b(0);
    for (int t = 0; t <= T; ++t) {
      if (t >= 1) {
        mbar_wait_cluster(&xfull[t & 1], (((t + 1) >> 1) - 1) & 1);
        const float* xt = xbuf + (t & 1) * n;
        float* dst = p.x_out + (static_cast<size_t>(item) * T + (t - 1)) * n;
        for (int i = r0 + lane; i < r1; i += 32) dst[i] = xt[i];
      }
      if (t < T) {
        if (lane == 0) mbar_arrive_expect_tx(&xfull[(t + 1) & 1], static_cast<uint32_t>(n) * 4u);
        if (t + 1 < T) form_b(t + 1);
      }
    }
  } else {
    // ------------------------------------------------------------------ consumers: shared-memory GEMV
    const int n4 = n >> 2;
    const int sl = WIDE ? (n4 + kConsWarps - 1) / kConsWarps : n4;   // quads in this warp's column slice
    const int q0 = (WIDE ? warp * sl : 0) + lane;
    const int q_end = WIDE ? min(n4, (warp + 1) * sl) : n4;
    const int ql = (sl + 31) / 32;
    const int rpw = p.sp.rpw;
    const int grp = lane >> 3, sub = lane & 7;   // after reduce4_rows lane group `grp` holds row `grp` of the pass
    int st = 0;
    uint32_t fph = 0, cidx = 0;
    for (int t = 0; t < T; ++t) {
      if (t >= 1 && !(LTV_ROLL_DBG & 2)) mbar_wait_cluster(&xfull[t & 1], (((t + 1) >> 1) - 1) & 1);
      const float4* x4 = reinterpret_cast<const float4*>(xbuf + (t & 1) * n);
      float4 xq[QLMAX];
#pragma unroll
      for (int j = 0; j < QLMAX; ++j) {
        const int q = q0 + 32 * j;
        xq[j] = (j < ql && q < q_end) ? x4[q] : make_float4(0.f, 0.f, 0.f, 0.f);
      }
      mbar_wait(&bfull[t & 1], (t >> 1) & 1);
      float* xn = xbuf + ((t + 1) & 1) * n;
      const float* bv = bvec + (t & 1) * p.sp.rows_max;
      uint64_t* xbar = &xfull[(t + 1) & 1];
      for (int k = 0; k < nchunks; ++k, ++cidx) {
        mbar_wait(&full[st], fph);
        const float* tile = reinterpret_cast<const float*>(reinterpret_cast<uint8_t*>(ring) +
                                                            static_cast<size_t>(st) * p.sp.stage_bytes);
        const int rk = min(rc, rows - k * rc);
        if (!WIDE) {
          // warp w: rows [w rpw, (w+1) rpw) of the chunk, four per pass
          for (int b0 = 0; b0 < rpw; b0 += 4) {
            const int base = warp * rpw + b0;
            if (base >= rk) break;
            int rowi[4];
            const int nval = min(min(4, rpw - b0), rk - base);
#pragma unroll
            for (int r = 0; r < 4; ++r) rowi[r] = base + (r < nval ? r : 0);
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
            if (!(LTV_ROLL_DBG & 1)) rows4_dot<QLMAX>(tile, n, rowi, q0, q_end, ql, xq, acc);
            const float v = (LTV_ROLL_DBG & 4) ? acc[0] : reduce4_rows(acc, lane);
            if (grp < nval) {
              const int li = k * rc + base + grp;
              const float y = v + bv[li];
              for (int cta = sub; cta < C; cta += 8) st_async_remote_f32(xn + r0 + li, y, xbar, cta);
            }
          }
        } else {
          // warp w: its eighth of the columns of all (<= 4) rows of the chunk; partial sums meet in shared memory
          int rowi[4];
#pragma unroll
          for (int r = 0; r < 4; ++r) rowi[r] = r < rk ? r : 0;
          float acc[4] = {0.f, 0.f, 0.f, 0.f};
          rows4_dot<QLMAX>(tile, n, rowi, q0, q_end, ql, xq, acc);
          const float v = reduce4_rows(acc, lane);
          float* pb = part + (cidx & 1) * (kConsWarps * 4);
          if (sub == 0) pb[warp * 4 + grp] = v;
          named_bar_sync(1, kConsWarps * 32);
          const int tid = threadIdx.x;   // consumers are threads 0 .. 255
          if (tid < rk * C) {
            const int row = tid / C, cta = tid - row * C;
            float y = bv[k * rc + row];
#pragma unroll
            for (int w = 0; w < kConsWarps; ++w) y += pb[w * 4 + row];
            st_async_remote_f32(xn + r0 + k * rc + row, y, xbar, cta);
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);
        if (++st == stages) { st = 0; fph ^= 1; }
      }
    }
  }
  __syncthreads();
  cluster_sync_all();  // no CTA may exit while a peer can still write into its shared memory
}

RollSmemPlan plan_rollout(int n, int C) {
  RollSmemPlan sp{};
  sp.rows_max = (n + C - 1) / C + 1;
  sp.wide = n > kModeAMaxN ? 1 : 0;
  const uint32_t row_bytes = static_cast<uint32_t>(n) * 4u;
  const uint32_t vec_bytes = static_cast<uint32_t>(align_up(2 * row_bytes, 128) + align_up(2u * sp.rows_max * 4u, 128)) +
                             256u /* part */;
  const uint32_t budget = 227u * 1024u - vec_bytes - 256u;
  const uint32_t target = 32u * 1024u;
  int rc;
  if (sp.wide) {
    rc = static_cast<int>(target / row_bytes);
    if (rc < 1) rc = 1;
    if (rc > 4) rc = 4;
    sp.rpw = 0;
  } else {
    // a multiple of 8 rows near the 32 KB target, at most 64 (8 per warp) and no more than the band needs
    rc = static_cast<int>((target + row_bytes * 4) / (row_bytes * 8)) * 8;
    if (rc < 8) rc = 8;
    if (rc > 64) rc = 64;
    const int need = (sp.rows_max - 1 + 7) / 8 * 8;
    if (rc > need) rc = need;
    sp.rpw = rc / 8;
  }
  sp.rc = rc;
  sp.stage_bytes = static_cast<uint32_t>(align_up(static_cast<size_t>(rc) * row_bytes, 128));
  int st = static_cast<int>(budget / sp.stage_bytes);
  if (st > kMaxStages) st = kMaxStages;
  sp.stages = st;
  sp.off_x = sp.stage_bytes * st;
  sp.off_b = sp.off_x + static_cast<uint32_t>(align_up(2 * row_bytes, 128));
  sp.off_part = sp.off_b + static_cast<uint32_t>(align_up(2u * sp.rows_max * 4u, 128));
  sp.off_bar = sp.off_part + 256u;
  sp.total = sp.off_bar + (2 * kMaxStages + 4) * 8;
  return sp;
}

}  // namespace

cudaError_t launch_rollout(const RolloutArgs& a, int cluster, cudaStream_t stream, unsigned long long* launches) {
  RollParams p{};
  p.A = a.A; p.B = (a.m > 0) ? a.B : nullptr; p.c = a.c; p.x0 = a.x0; p.u = a.u; p.x_out = a.x_out;
  p.batch = a.batch; p.T = a.T; p.n = a.n; p.m = a.m;
  p.sp = plan_rollout(a.n, cluster);
  if (p.sp.stages < 2) return cudaErrorInvalidConfiguration;

  auto kern = p.sp.wide ? rollout_kernel<true> : rollout_kernel<false>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, p.sp.total);
  if (e != cudaSuccess) return e;
  if (cluster > 8) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
  }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>(a.batch) * cluster);
  cfg.blockDim = dim3(kRollThreads);
  cfg.dynamicSmemBytes = p.sp.total;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = cluster;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  {
    ProfScope prof(kProfRollout, stream);
    e = cudaLaunchKernelEx(&cfg, kern, p);
  }
  if (e == cudaSuccess) ++*launches;
  return e;
}

}  // namespace ltv
