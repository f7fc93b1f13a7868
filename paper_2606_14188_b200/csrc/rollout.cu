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

namespace ltv {

namespace {

constexpr int kConsWarps = 8;    // warps of one consumer group
constexpr int kGroups = 2;       // consumer groups; group g takes the ring chunks with index % kGroups == g
constexpr int kAllCons = kConsWarps * kGroups;
constexpr int kAffWarps = 2;      // affine warps; warp a forms the terms of the steps with number % kAffWarps == a
constexpr int kRollThreads = (kAllCons + 1 + kAffWarps) * 32;  // + producer warp + affine warps
constexpr int kMaxStages = 8;
constexpr int kBStages = 4;     // affine terms formed ahead of the consumers
constexpr int kStageVecs = 384; // float4 of the B band the affine warp stages in shared memory (6 KB)
constexpr int kModeAMaxN = 640;

struct RollSmemPlan {
  int rc;              // rows per ring chunk
  int rpw;             // mode A: rows per warp per chunk (rc = 8 rpw)
  int wide;            // 0 = mode A, 1 = mode B
  int stages;
  uint32_t stage_bytes;
  uint32_t off_x, off_b, off_part, off_stage, off_bar, total;
  int rows_max;        // max rows owned by one CTA
};

// rows [r0, r1) of CTA `rank`: multiples of 4 rows (n % 4 == 0), so that the bands of A, B and c start on
// 16-byte boundaries
__host__ __device__ inline void band(int n, int C, int rank, int& r0, int& r1) {
  const long long nq = n >> 2;
  r0 = 4 * static_cast<int>((nq * rank) / C);
  r1 = 4 * static_cast<int>((nq * (rank + 1)) / C);
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

// acc[r] += sum_j A[row0 + r][q0 + 32 j] . xq[j] for NR consecutive rows of a shared-memory tile (row stride n
// floats); quads at or beyond q_end are skipped.  All NR x ql loads of a pass are independent.
template <int QLMAX, int NR>
__device__ __forceinline__ void rows_dot(const float* tile, int n, int row0, int q0, int q_end, int ql,
                                         const float4 (&xq)[QLMAX], float (&acc)[4]) {
  const float* base = tile + static_cast<size_t>(row0) * n + 4 * q0;
#pragma unroll
  for (int j = 0; j < QLMAX; ++j) {
    if (j < ql && q0 + 32 * j < q_end) {
#pragma unroll
      for (int r = 0; r < NR; ++r) {
        const float4 a = *reinterpret_cast<const float4*>(base + static_cast<size_t>(r) * n + 128 * j);
        acc[r] = dot4(a, xq[j], acc[r]);
      }
    }
  }
}
template <int QLMAX>
__device__ __forceinline__ void rows_dot_n(int nr, const float* tile, int n, int row0, int q0, int q_end, int ql,
                                           const float4 (&xq)[QLMAX], float (&acc)[4]) {
  switch (nr) {   // warp-uniform
    case 4: rows_dot<QLMAX, 4>(tile, n, row0, q0, q_end, ql, xq, acc); break;
    case 3: rows_dot<QLMAX, 3>(tile, n, row0, q0, q_end, ql, xq, acc); break;
    case 2: rows_dot<QLMAX, 2>(tile, n, row0, q0, q_end, ql, xq, acc); break;
    default: rows_dot<QLMAX, 1>(tile, n, row0, q0, q_end, ql, xq, acc); break;
  }
}

template <bool WIDE>
__global__ void __launch_bounds__(kRollThreads, 1) rollout_kernel(const RollParams p) {
  constexpr int QLMAX = WIDE ? 8 : 5;
  extern __shared__ __align__(128) uint8_t smem[];
  const int C = static_cast<int>(cluster_nctarank());
  const int rank = static_cast<int>(cluster_ctarank());
  const int cl = blockIdx.x / C, ncl = gridDim.x / C;   // this cluster, clusters in the grid
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n = p.n, T = p.T, m = p.m;
  int r0, r1;
  band(n, C, rank, r0, r1);
  const int rows = r1 - r0;
  const int rc = p.sp.rc, stages = p.sp.stages;
  const int nchunks = (rows + rc - 1) / rc;

  float* ring = reinterpret_cast<float*>(smem);
  float* xbuf = reinterpret_cast<float*>(smem + p.sp.off_x);   // [3][n]
  float* bvec = reinterpret_cast<float*>(smem + p.sp.off_b);   // [kBStages][rows_max]
  float* part = reinterpret_cast<float*>(smem + p.sp.off_part);  // mode B: [kGroups][2][kConsWarps][4]
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + p.sp.off_bar);
  uint64_t* full = bars;                    // [stages]  producer -> consumers (tx bytes)
  uint64_t* empty = bars + kMaxStages;      // [stages]  consumers -> producer (kConsWarps arrivals)
  uint64_t* xfull = bars + 2 * kMaxStages;  // [3]       state number g complete in xbuf[g % 3]
  uint64_t* bfull = xfull + 3;              // [kBStages] affine term number h complete in bvec[h % kBStages]
  uint64_t* bempty = bfull + kBStages;      // [kBStages] consumers are done with it (kAllCons arrivals)

  if (threadIdx.x == 0) {
    for (int s = 0; s < stages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], kConsWarps);
    }
    for (int s = 0; s < 3; ++s) mbar_init(&xfull[s], 1);
    for (int s = 0; s < kBStages; ++s) {
      mbar_init(&bfull[s], 1);
      mbar_init(&bempty[s], kAllCons);
    }
    fence_mbar_init();
  }
  __syncthreads();
  cluster_sync_all();  // every CTA's barriers are initialised before any remote st.async can target them

  // Persistent over items: cluster `cl` takes items cl, cl + ncl, ...  Steps are numbered h = j T + t over the
  // item rounds j.  x_0 is read from global memory by the consumers themselves; x_{t+1}, t + 1 < T, is
  // exchanged through xbuf[(h+1) % 3] behind xfull[(h+1) % 3] (armed by consumer thread 0 at the start of
  // step t); the affine term b_t lives in bvec[h % kBStages] behind bfull / bempty, formed up to kBStages
  // steps ahead by a warp that depends on nothing but those buffers.  The producer streams A straight
  // through item boundaries.
  if (warp == kAllCons) {
    // ------------------------------------------------------------------ producer (one thread)
    if (lane == 0 && rows > 0) {
      const uint64_t pol = l2_policy_evict_first();
      int st = 0;
      uint32_t eph = 1;   // parity of empty[st] to wait for (the first pass over the ring does not block)
      for (int item = cl; item < p.batch; item += ncl) {
        const size_t itemA = static_cast<size_t>(item) * T * n * n;
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
    }
  } else if (warp > kAllCons) {
    // ------------------------------------------------------------------ affine warp: b_t = B_t u_t + c_t
    // The bands of B_t and c_t are contiguous: all of their 128-bit loads (and u_t) are issued before the first
    // use, so a step costs one memory latency however many rows the band has; B_t is staged in shared memory
    // and reduced lane-per-row.  (Row-at-a-time loads made this warp the bottleneck at batch 1024, where B no
    // longer sits in L2.)
    float4* stB = reinterpret_cast<float4*>(smem + p.sp.off_stage);
    const bool has_bu = p.B && p.u && m > 0;
    const int nvB = has_bu ? (rows * m) >> 2 : 0, nvC = p.c ? rows >> 2 : 0;
    const bool staged = nvB <= kStageVecs;
    const int aw = warp - kAllCons - 1;
    stB += aw * kStageVecs;
    int bs = 0;
    uint32_t bph = 1;   // parity of bempty[bs] (the first pass over the buffers does not block)
    uint32_t sn = 0;    // step number over all items of this cluster
    for (int item = cl; item < p.batch; item += ncl) {
      for (int t = 0; t < T; ++t, ++sn) {
        if (static_cast<int>(sn % kAffWarps) != aw) {
          if (++bs == kBStages) { bs = 0; bph ^= 1; }
          continue;
        }
        float* bv = bvec + bs * p.sp.rows_max;
        const size_t bt = static_cast<size_t>(item) * T + t;
        const float ul = (has_bu && lane < m) ? __ldg(p.u + bt * m + lane) : 0.f;
        const float4* gB = has_bu ? reinterpret_cast<const float4*>(p.B + (bt * n + r0) * m) : nullptr;
        const float4* gC = p.c ? reinterpret_cast<const float4*>(p.c + bt * n + r0) : nullptr;
        constexpr int kVB = kStageVecs / 32, kVC = 2;
        float4 vb[kVB], vc[kVC];
        if (staged) {
#pragma unroll
          for (int j = 0; j < kVB; ++j) vb[j] = (lane + 32 * j < nvB) ? __ldg(gB + lane + 32 * j) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int j = 0; j < kVC; ++j) vc[j] = (lane + 32 * j < nvC) ? __ldg(gC + lane + 32 * j) : make_float4(0.f, 0.f, 0.f, 0.f);
        mbar_wait(&bempty[bs], bph);
        float4* bv4 = reinterpret_cast<float4*>(bv);
#pragma unroll
        for (int j = 0; j < kVC; ++j)
          if (lane + 32 * j < (rows >> 2)) bv4[lane + 32 * j] = vc[j];
        for (int v = lane + 32 * kVC; v < (rows >> 2); v += 32) bv4[v] = gC ? __ldg(gC + v) : make_float4(0.f, 0.f, 0.f, 0.f);
        if (has_bu) {
          if (staged) {
#pragma unroll
            for (int j = 0; j < kVB; ++j)
              if (lane + 32 * j < nvB) stB[lane + 32 * j] = vb[j];
          }
          __syncwarp();
          const float* sB = reinterpret_cast<const float*>(stB);
          for (int i0 = 0; i0 < rows; i0 += 32) {   // warp-uniform trip count: the shuffles need every lane
            const int i = i0 + lane;
            const bool ok = i < rows;
            float acc = ok ? bv[i] : 0.f;
            if (m <= 32) {
              for (int l = 0; l < m; ++l) {
                const float bl = !ok ? 0.f : staged ? sB[i * m + l] : __ldg(p.B + (bt * n + r0 + i) * m + l);
                acc = fmaf(bl, __shfl_sync(0xffffffffu, ul, l), acc);
              }
            } else {
              for (int l = 0; l < m; ++l) {
                const float bl = !ok ? 0.f : staged ? sB[i * m + l] : __ldg(p.B + (bt * n + r0 + i) * m + l);
                acc = fmaf(bl, __ldg(p.u + bt * m + l), acc);
              }
            }
            if (ok) bv[i] = acc;
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&bfull[bs]);
        if (++bs == kBStages) { bs = 0; bph ^= 1; }
      }
    }
  } else {
    // ------------------------------------------------------------------ consumers: shared-memory GEMV
    // Two groups take alternate chunks: a pass is a chain of latencies (shared loads, 6 shuffles, remote stores:
    // ~1500 cycles measured with clock traces) in which shared memory is busy for a quarter of the time, so
    // one group's loads run under the other group's reduction.
    const int grpid = warp / kConsWarps, gw = warp % kConsWarps;   // consumer group, warp within it
    const int n4 = n >> 2;
    const int sl = WIDE ? (n4 + kConsWarps - 1) / kConsWarps : n4;   // quads in this warp's column slice
    const int q0 = (WIDE ? gw * sl : 0) + lane;
    const int q_end = WIDE ? min(n4, (gw + 1) * sl) : n4;
    const int ql = (sl + 31) / 32;
    const int rpw = p.sp.rpw;
    const int grp = lane >> 3, sub = lane & 7;   // after reduce4_rows lane group `grp` holds row `grp` of the pass
    int st = 0;
    uint32_t fph = 0, cidx = 0;
    int bs = 0;
    uint32_t bph = 0;   // parity of bfull[bs]
    uint32_t xph = 0;   // bit s: parity of the next phase of xfull[s] (x_0 of an item never uses its slot)
    uint32_t h = 0;
    for (int item = cl; item < p.batch; item += ncl, h += T)
    for (int t = 0; t < T; ++t) {
      const uint32_t ht = h + t;
      const bool exch = t + 1 < T;   // x_T only goes to global memory
      float4 xq[QLMAX];
      if (t == 0) {
        const float4* x4 = reinterpret_cast<const float4*>(p.x0 + static_cast<size_t>(item) * n);
#pragma unroll
        for (int j = 0; j < QLMAX; ++j) {
          const int q = q0 + 32 * j;
          xq[j] = (j < ql && q < q_end) ? __ldg(x4 + q) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
      } else {
        mbar_wait_cluster(&xfull[ht % 3], (xph >> (ht % 3)) & 1u);
        xph ^= 1u << (ht % 3);
        const float4* x4 = reinterpret_cast<const float4*>(xbuf + (ht % 3) * n);
#pragma unroll
        for (int j = 0; j < QLMAX; ++j) {
          const int q = q0 + 32 * j;
          xq[j] = (j < ql && q < q_end) ? x4[q] : make_float4(0.f, 0.f, 0.f, 0.f);
        }
      }
      // every warp of every CTA has finished step t-1, so nobody reads xbuf[(ht+1) % 3] (= x_{t-2}) any more
      if (exch && threadIdx.x == 0) mbar_arrive_expect_tx(&xfull[(ht + 1) % 3], static_cast<uint32_t>(n) * 4u);
      mbar_wait(&bfull[bs], bph);
      float* xn = xbuf + ((ht + 1) % 3) * n;
      const float* bv = bvec + bs * p.sp.rows_max;
      uint64_t* xbar = &xfull[(ht + 1) % 3];
      float* xg = p.x_out + (static_cast<size_t>(item) * T + t) * n + r0;   // x_{t+1}, this CTA's rows
      for (int k = 0; k < nchunks; ++k, ++cidx) {
        if (static_cast<int>(cidx % kGroups) == grpid) {
        mbar_wait(&full[st], fph);
        const float* tile = reinterpret_cast<const float*>(reinterpret_cast<uint8_t*>(ring) +
                                                            static_cast<size_t>(st) * p.sp.stage_bytes);
        const int rk = min(rc, rows - k * rc);
        if (!WIDE) {
          // units of 4 consecutive rows are dealt round-robin to the warps of the group, one unit per pass
          const int nu = (rk + 3) >> 2;
          for (int un = gw; un < nu; un += kConsWarps) {
            const int base = 4 * un;
            const int nval = min(4, rk - base);
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
            rows_dot_n<QLMAX>(nval, tile, n, base, q0, q_end, ql, xq, acc);
            const float v = reduce4_rows(acc, lane);
            const int li0 = k * rc + base;
            if (nval == 4) {
              // all four sums into every lane: one 16-byte remote store per destination CTA, one 16-byte global store
              float4 y;
              y.x = __shfl_sync(0xffffffffu, v, 0) + bv[li0];
              y.y = __shfl_sync(0xffffffffu, v, 8) + bv[li0 + 1];
              y.z = __shfl_sync(0xffffffffu, v, 16) + bv[li0 + 2];
              y.w = __shfl_sync(0xffffffffu, v, 24) + bv[li0 + 3];
              if (exch && lane < C) st_async_remote_f32x4(xn + r0 + li0, y, xbar, lane);
              if (lane == 31) *reinterpret_cast<float4*>(xg + li0) = y;
            } else if (grp < nval) {
              const int li = li0 + grp;
              const float y = v + bv[li];
              if (exch)
                for (int cta = sub; cta < C; cta += 8) st_async_remote_f32(xn + r0 + li, y, xbar, cta);
              if (sub == 0) xg[li] = y;
            }
          }
        } else {
          // warp gw: its eighth of the columns of all (<= 4) rows of the chunk; partial sums meet in shared memory
          float acc[4] = {0.f, 0.f, 0.f, 0.f};
          rows_dot_n<QLMAX>(rk, tile, n, 0, q0, q_end, ql, xq, acc);
          const float v = reduce4_rows(acc, lane);
          float* pb = part + (grpid * 2 + ((cidx / kGroups) & 1)) * (kConsWarps * 4);
          if (sub == 0) pb[gw * 4 + grp] = v;
          named_bar_sync(1 + grpid, kConsWarps * 32);
          const int tid = gw * 32 + lane;
          if (rk == 4) {
            if (tid < C) {
              float4 y = *reinterpret_cast<const float4*>(bv + k * rc);
#pragma unroll
              for (int w = 0; w < kConsWarps; ++w) {
                const float4 pw = *reinterpret_cast<const float4*>(pb + w * 4);
                y.x += pw.x; y.y += pw.y; y.z += pw.z; y.w += pw.w;
              }
              if (exch) st_async_remote_f32x4(xn + r0 + k * rc, y, xbar, tid);
              if (tid == 0) *reinterpret_cast<float4*>(xg + k * rc) = y;
            }
          } else if (tid < rk * C) {
            const int row = tid / C, cta = tid - row * C;
            float y = bv[k * rc + row];
#pragma unroll
            for (int w = 0; w < kConsWarps; ++w) y += pb[w * 4 + row];
            if (exch) st_async_remote_f32(xn + r0 + k * rc + row, y, xbar, cta);
            if (cta == 0) xg[k * rc + row] = y;
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);
        }
        if (++st == stages) { st = 0; fph ^= 1; }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&bempty[bs]);
      if (++bs == kBStages) { bs = 0; bph ^= 1; }
    }
  }
  __syncthreads();
  cluster_sync_all();  // no CTA may exit while a peer can still write into its shared memory
}

RollSmemPlan plan_rollout(int n, int C, int occ) {
  RollSmemPlan sp{};
  sp.rows_max = 4 * (((n >> 2) + C - 1) / C) + 4;   // bands are multiples of 4 rows
  sp.wide = n > kModeAMaxN ? 1 : 0;
  const uint32_t row_bytes = static_cast<uint32_t>(n) * 4u;
  const uint32_t vec_bytes = static_cast<uint32_t>(align_up(3 * row_bytes, 128) + align_up(kBStages * sp.rows_max * 4u, 128)) +
                             512u /* part */ + kAffWarps * kStageVecs * 16u;
  // occ CTAs share the 228 KB of an SM (1 KB of each is reserved by the system)
  const uint32_t cta_bytes = occ > 1 ? (228u * 1024u) / occ - 1024u : 227u * 1024u;
  if (cta_bytes < vec_bytes + 512u) return sp;   // stages = 0: caller falls back
  const uint32_t budget = cta_bytes - vec_bytes - 256u;
  const uint32_t target = budget / 6u < 32u * 1024u ? budget / 6u : 32u * 1024u;
  int rc;
  if (sp.wide) {
    rc = static_cast<int>(target / row_bytes);
    if (rc < 1) rc = 1;
    if (rc > 4 || 4u * row_bytes <= 48u * 1024u) rc = 4;   // 4-row chunks: 16-byte state exchange
    sp.rpw = 0;
  } else {
    // a multiple of 8 rows near the 32 KB target, at most 64 (8 per warp) and no more than the band needs
    rc = static_cast<int>((target + row_bytes * 4) / (row_bytes * 8)) * 8;
    if (rc < 8) rc = 8;
    if (rc > 64) rc = 64;
    const int need = (sp.rows_max - 4 + 7) / 8 * 8;
    if (rc > need) rc = need;
    sp.rpw = rc / 8;
  }
  sp.rc = rc;
  sp.stage_bytes = static_cast<uint32_t>(align_up(static_cast<size_t>(rc) * row_bytes, 128));
  int st = static_cast<int>(budget / sp.stage_bytes);
  if (st > kMaxStages) st = kMaxStages;
  // An EVEN number of stages: the two consumer groups take alternate chunks, so with an odd ring a stage would change
  // hands every pass and a group would see only every other phase of its `full` barrier - the parity test then cannot
  // tell its own chunk from the other group's chunk of the pass before, still in flight (adjoint.cu has the story).
  st &= ~1;
  sp.stages = st;
  sp.off_x = sp.stage_bytes * st;
  sp.off_b = sp.off_x + static_cast<uint32_t>(align_up(3 * row_bytes, 128));
  sp.off_part = sp.off_b + static_cast<uint32_t>(align_up(kBStages * sp.rows_max * 4u, 128));
  sp.off_stage = sp.off_part + 512u;
  sp.off_bar = sp.off_stage + kAffWarps * kStageVecs * 16u;
  sp.total = sp.off_bar + (2 * kMaxStages + 3 + 2 * kBStages) * 8;
  return sp;
}

}  // namespace

// `cluster` CTAs per item (0 = modelled); the grid is as many clusters as can be resident at once (at most one
// per item), each looping over items
static const int* rollout_max_active(int wide) {
  static int max_active[2][17];
  static bool have[2] = {false, false};
  if (!have[wide]) {
    query_max_active_clusters(wide ? reinterpret_cast<const void*>(rollout_kernel<true>)
                                   : reinterpret_cast<const void*>(rollout_kernel<false>),
                              kRollThreads, 200 * 1024, max_active[wide]);
    have[wide] = true;
  }
  return max_active[wide];
}

int rollout_cluster_choice(const RolloutArgs& a) {
  return pick_cluster_model(a.batch, a.n, rollout_max_active(a.n > kModeAMaxN ? 1 : 0), a.sm_budget);
}

int rollout_clusters_resident(const RolloutArgs& a, int cluster) {
  return (cluster >= 1 && cluster <= 16) ? rollout_max_active(a.n > kModeAMaxN ? 1 : 0)[cluster] : 0;
}

cudaError_t launch_rollout(const RolloutArgs& a, int cluster, cudaStream_t stream, unsigned long long* launches) {
  const int wide = a.n > kModeAMaxN ? 1 : 0;
  const int* max_active = rollout_max_active(wide);
  if (cluster <= 0) cluster = pick_cluster_model(a.batch, a.n, max_active, a.sm_budget);
  RollParams p{};
  p.A = a.A; p.B = (a.m > 0) ? a.B : nullptr; p.c = a.c; p.x0 = a.x0; p.u = a.u; p.x_out = a.x_out;
  p.batch = a.batch; p.T = a.T; p.n = a.n; p.m = a.m;
  p.sp = plan_rollout(a.n, cluster, 1);
  if (p.sp.stages < 2) return cudaErrorInvalidConfiguration;

  auto kern = p.sp.wide ? rollout_kernel<true> : rollout_kernel<false>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, p.sp.total);
  if (e != cudaSuccess) return e;
  if (cluster > 8) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
  }
  cudaLaunchConfig_t cfg{};
  int ncl = max_active[cluster];
  if (ncl > a.batch) ncl = a.batch;
  if (a.sm_budget > 0 && ncl > a.sm_budget / cluster) ncl = a.sm_budget / cluster;
  if (ncl < 1) ncl = 1;
  cfg.gridDim = dim3(static_cast<unsigned>(ncl) * cluster);
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
  LTV_DBG_INSTALL();
  {
    ProfScope prof(kProfRollout, stream);
    e = cudaLaunchKernelEx(&cfg, kern, p);
  }
  if (e == cudaSuccess) ++*launches;
  return e;
}

}  // namespace ltv
