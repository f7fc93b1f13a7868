// The whole hot path of a SMALL problem in ONE launch (SURVEY section 7 hard part 6; BASELINE.json configs[0]: rope N = 8,
// n = 48, T = 16, batch 1 - the paper's own regime of tens of states and one problem):
//     rollout x_{t+1} = A_t x_t + B_t u_t + c_t                       PAPER.md:53 eq.(2), :139 eq.(12b)
//     Phi(t,s) = A_{t-1} .. A_s, r_t = sum_{s<t} |Phi(t,s)| w_s        PAPER.md:142 eq.(12c), :147 eq.(12e)
//     lam_t = A_t^T lam_{t+1} + g_t, grad_u, grad_x0                   PAPER.md:106-110 eq.(10)
// All of A (147 KB at C1) fits one SM's shared memory, so the multi-launch path (9 launches, 0.16-0.2 ms, every one of
// them launch-latency bound) is replaced by one thread-block cluster per item:
//   CTA r < C-1   owns the block COLUMNS s = r, r + (C-1), ... of Phi.  A column is a chain Phi(t,s) = A_{t-1} Phi(t-1,s),
//                 t = s+2 .. T-1, that depends on nothing outside the CTA (A_t in shared memory, the running block in
//                 shared memory): no grid- or cluster-wide synchronisation per level.  The T-1 chains have 0 .. T-2
//                 products; with one column per CTA the longest (s = 0) is the critical path, T-2 products of n^3.
//                 Each product: 4 x 4 register tiles, K split over up to 4 thread groups, fp32 FMA (the same arithmetic
//                 as the fp32-FMA combine the library uses for n < 96).  The tube term |Phi(t,s)| w_s is taken from the
//                 finished tile and kept per (column, t) in shared memory.
//   CTA C-1       runs the rollout (warps 0-7) and the adjoint (warps 8-15) side by side, A in shared memory.
//   finally       one cluster barrier; CTA q sums r_t for t = q, q + C, ... over the columns s < t in fixed order,
//                 reading the per-column terms out of the owners' shared memory (DSMEM): deterministic, no atomics.
// This is the column-sequential form of the scan (depth T-2 instead of log2 T): at n^3 = 0.2 MFLOP per product the
// log-depth schedule's extra synchronisation costs more than its shorter chain saves; the divide-and-conquer levels
// remain the path for everything that does not fit here.
#include <cooperative_groups.h>

#include "../../include/ltv_scan.h"
#include "ltv_internal.h"
#include "phi_geom.cuh"
#include "ptx.cuh"

namespace cg = cooperative_groups;

namespace ltv {

namespace {

constexpr int kFsThreads = 512;
constexpr int kFsMaxN = 64;
constexpr int kFsMaxCluster = 16;
constexpr int kFsVecGroup = 256;   // threads of the rollout group and of the adjoint group

struct FsParams {
  const float *A, *B, *c, *x0, *u, *w, *g;
  float *x, *phi, *r, *lam, *gu, *gx0;
  int batch, T, n, m;
  int tube_mode;     // 0 box, 1 row two-norm
  int ncc;           // column CTAs per cluster (cluster size - 1)
  int cps;           // column slots per column CTA = ceil((T-1) / ncc)
  int lda;           // row stride of A in shared memory (n + 4: the 4-row a-loads of a warp hit distinct banks)
  int ksplit, kchunk;
  int b_in_smem;     // vector CTA keeps B in shared memory
  uint32_t off_p, off_red, off_w, off_tube, off_rpart;                    // column CTA layout (bytes), A at 0
  uint32_t off_b, off_bs, off_gs, off_xs, off_ls, off_pa, off_us;         // vector CTA layout (bytes), A at 0
};

__device__ __forceinline__ float fs_tube_term(float d, float w, int mode) {
  const float v = d * w;
  return mode ? v * v : fabsf(v);
}

// A_t (global, row-major n x n) -> shared memory with row stride lda, 16-byte cp.async
__device__ __forceinline__ void fs_load_A(float* dst, const float* src, int n, int lda, int tid, int nthreads) {
  const int n4 = n >> 2;
  for (int e = tid; e < n * n4; e += nthreads) {
    const int i = e / n4, q = e - i * n4;
    cp_async16(dst + i * lda + 4 * q, src + static_cast<size_t>(i) * n + 4 * q);
  }
}

// ------------------------------------------------------------------------------------------------ column CTA
__device__ void fs_column_cta(const FsParams& p, uint8_t* smem, int item, int rank) {
  const int n = p.n, T = p.T, lda = p.lda, nt = n >> 2, tiles = nt * nt;
  const int tid = threadIdx.x;
  float* As = reinterpret_cast<float*>(smem);                       // [T][n][lda] (only the steps this CTA needs)
  float* Pb = reinterpret_cast<float*>(smem + p.off_p);             // [2][n][n] running block, ping-pong
  float* red = reinterpret_cast<float*>(smem + p.off_red);          // [ksplit-1][n][n] partial products
  float* wv = reinterpret_cast<float*>(smem + p.off_w);             // [n]
  float* tube = reinterpret_cast<float*>(smem + p.off_tube);        // [n][nt + 1]
  float* rpart = reinterpret_cast<float*>(smem + p.off_rpart);      // [cps][T][n]
  const float* Ag = p.A + static_cast<size_t>(item) * T * n * n;
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;

  for (int e = tid; e < p.cps * T * n; e += kFsThreads) rpart[e] = 0.f;
  // the left operands this CTA will use: A_t, t = s_min + 1 .. T-2
  const int s_min = rank;
  for (int t = s_min + 1; t <= T - 2; ++t)
    fs_load_A(As + static_cast<size_t>(t) * n * lda, Ag + static_cast<size_t>(t) * n * n, n, lda, tid, kFsThreads);
  cp_async_commit();

  // thread -> (k group, tile row, tile col)
  const int g = tid / tiles, rem = tid - g * tiles;
  const int tr = rem / nt, tc = rem - tr * nt;
  const bool active = g < p.ksplit;
  const int k0 = g * p.kchunk, k1 = min(n, k0 + p.kchunk);

  for (int slot = 0; slot < p.cps; ++slot) {
    const int s = rank + slot * p.ncc;
    if (s > T - 2) break;
    float* rp = rpart + static_cast<size_t>(slot) * T * n;
    float* phi_col = p.phi + (static_cast<size_t>(item) * P + phi_colbase(T, s)) * n * n;   // blocks t = s+1 .. T-1
    __syncthreads();   // the previous column is finished with Pb / wv
    // level 0: Phi(s+1,s) = A_s  (global -> Pb[0] and -> phi), tube term |A_s| w_s
    if (tid < n) wv[tid] = __ldg(p.w + (static_cast<size_t>(item) * T + s) * n + tid);
    {
      const float4* src = reinterpret_cast<const float4*>(Ag + static_cast<size_t>(s) * n * n);
      float4* dstg = reinterpret_cast<float4*>(phi_col);
      float4* dsts = reinterpret_cast<float4*>(Pb);
      for (int e = tid; e < n * nt; e += kFsThreads) {
        const float4 v = __ldg(src + e);
        dsts[e] = v;
        dstg[e] = v;
      }
    }
    __syncthreads();
    for (int i = tid; i < n; i += kFsThreads) {
      float acc = 0.f;
      for (int j = 0; j < n; ++j) acc += fs_tube_term(Pb[i * n + ((j + i) % n)], wv[(j + i) % n], p.tube_mode);
      rp[(s + 1) * n + i] = acc;
    }
    if (slot == 0) cp_async_wait<0>();   // the A_t of this CTA have landed (this thread's copies) ...
    __syncthreads();                  // ... and everybody's
    int cur = 0;
    for (int t = s + 2; t <= T - 1; ++t) {
      // D = A_{t-1} Pcur : thread tile rows 4 tr .. +3, cols 4 tc .. +3, k in [k0, k1)
      const float* L = As + static_cast<size_t>(t - 1) * n * lda;
      const float* R = Pb + cur * n * n;
      float acc[4][4];
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.f;
      if (active) {
        for (int k = k0; k < k1; k += 4) {
          float4 av[4], bv[4];
#pragma unroll
          for (int a = 0; a < 4; ++a) av[a] = *reinterpret_cast<const float4*>(L + (4 * tr + a) * lda + k);
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) bv[kk] = *reinterpret_cast<const float4*>(R + (k + kk) * n + 4 * tc);
#pragma unroll
          for (int a = 0; a < 4; ++a) {
            const float al[4] = {av[a].x, av[a].y, av[a].z, av[a].w};
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
              acc[a][0] = fmaf(al[kk], bv[kk].x, acc[a][0]);
              acc[a][1] = fmaf(al[kk], bv[kk].y, acc[a][1]);
              acc[a][2] = fmaf(al[kk], bv[kk].z, acc[a][2]);
              acc[a][3] = fmaf(al[kk], bv[kk].w, acc[a][3]);
            }
          }
        }
        if (g > 0) {
          float* rd = red + static_cast<size_t>(g - 1) * n * n;
#pragma unroll
          for (int a = 0; a < 4; ++a)
            *reinterpret_cast<float4*>(rd + (4 * tr + a) * n + 4 * tc) = make_float4(acc[a][0], acc[a][1], acc[a][2], acc[a][3]);
        }
      }
      __syncthreads();
      if (g == 0) {
        // fixed-order sum of the k groups, then: next running block, global Phi(t,s), tube partials
        float* Pn = Pb + (cur ^ 1) * n * n;
        float* outg = phi_col + static_cast<size_t>(t - s - 1) * n * n;
        const float4 ww = *reinterpret_cast<const float4*>(wv + 4 * tc);
#pragma unroll
        for (int a = 0; a < 4; ++a) {
          float4 v = make_float4(acc[a][0], acc[a][1], acc[a][2], acc[a][3]);
          for (int gg = 1; gg < p.ksplit; ++gg) {
            const float4 q = *reinterpret_cast<const float4*>(red + static_cast<size_t>(gg - 1) * n * n + (4 * tr + a) * n + 4 * tc);
            v.x += q.x; v.y += q.y; v.z += q.z; v.w += q.w;
          }
          *reinterpret_cast<float4*>(Pn + (4 * tr + a) * n + 4 * tc) = v;
          *reinterpret_cast<float4*>(outg + (4 * tr + a) * n + 4 * tc) = v;
          tube[(4 * tr + a) * (nt + 1) + tc] = (fs_tube_term(v.x, ww.x, p.tube_mode) + fs_tube_term(v.y, ww.y, p.tube_mode)) +
                                               (fs_tube_term(v.z, ww.z, p.tube_mode) + fs_tube_term(v.w, ww.w, p.tube_mode));
        }
      }
      __syncthreads();
      if (tid < n) {
        float acc_r = 0.f;
        for (int q = 0; q < nt; ++q) acc_r += tube[tid * (nt + 1) + q];
        rp[t * n + tid] = acc_r;
      }
      cur ^= 1;
    }
  }
}

// ------------------------------------------------------------------------------------------------ vector CTA
// warps 0-7: rollout; warps 8-15: adjoint.  All of A_0 .. A_{T-1} row-major in shared memory (row stride lda).
__device__ void fs_vector_cta(const FsParams& p, uint8_t* smem, int item) {
  const int n = p.n, T = p.T, m = p.m, lda = p.lda, n4 = n >> 2;
  const int tid = threadIdx.x, lane = tid & 31;
  float* As = reinterpret_cast<float*>(smem);
  float* Bs = reinterpret_cast<float*>(smem + p.off_b);     // [T][n][m] (if b_in_smem)
  float* bs = reinterpret_cast<float*>(smem + p.off_bs);    // [T][n] affine terms b_t = B_t u_t + c_t
  float* gs = reinterpret_cast<float*>(smem + p.off_gs);    // [T][n] g_t
  float* xs = reinterpret_cast<float*>(smem + p.off_xs);    // [2][n]
  float* ls = reinterpret_cast<float*>(smem + p.off_ls);    // [2][n]
  float* pa = reinterpret_cast<float*>(smem + p.off_pa);    // [row groups][n] partial sums of A^T lam
  float* us = reinterpret_cast<float*>(smem + p.off_us);    // [T][m]
  const size_t itT = static_cast<size_t>(item) * T;
  const float* Ag = p.A + itT * n * n;
  const bool has_bu = p.B != nullptr && p.u != nullptr && m > 0;
  const bool has_gu = p.B != nullptr && p.gu != nullptr && m > 0;

  for (int t = 0; t < T; ++t)
    fs_load_A(As + static_cast<size_t>(t) * n * lda, Ag + static_cast<size_t>(t) * n * n, n, lda, tid, kFsThreads);
  cp_async_commit();
  if (p.b_in_smem && p.B != nullptr && m > 0) {
    const float* Bg = p.B + itT * n * m;
    for (int e = tid; e < T * n * m; e += kFsThreads) Bs[e] = __ldg(Bg + e);
  }
  if (has_bu)
    for (int e = tid; e < T * m; e += kFsThreads) us[e] = __ldg(p.u + itT * m + e);
  for (int e = tid; e < T * n; e += kFsThreads) gs[e] = __ldg(p.g + itT * n + e);
  for (int e = tid; e < n; e += kFsThreads) xs[e] = __ldg(p.x0 + static_cast<size_t>(item) * n + e);
  __syncthreads();
  // affine terms of every step at once (a1: b_t = B_t u_t + c_t, never written to global memory)
  for (int e = tid; e < T * n; e += kFsThreads) {
    const int t = e / n;
    float acc = p.c ? __ldg(p.c + itT * n + e) : 0.f;
    if (has_bu) {
      const float* brow = p.b_in_smem ? Bs + static_cast<size_t>(e) * m : p.B + (itT * n + e) * m;
      for (int l = 0; l < m; ++l) acc = fmaf(p.b_in_smem ? brow[l] : __ldg(brow + l), us[t * m + l], acc);
    }
    bs[e] = acc;
  }
  cp_async_wait<0>();
  __syncthreads();

  if (tid < kFsVecGroup) {
    // ---------------------------------------------------------------- rollout: warp per row, lanes over column quads
    const int warp = tid >> 5;
    float* xg = p.x + itT * n;
    for (int t = 0; t < T; ++t) {
      const float* At = As + static_cast<size_t>(t) * n * lda;
      const float* xc = xs + (t & 1) * n;
      float* xn = xs + ((t + 1) & 1) * n;
      for (int i = warp; i < n; i += kFsVecGroup / 32) {
        float acc = 0.f;
        for (int q = lane; q < n4; q += 32) {
          const float4 a = *reinterpret_cast<const float4*>(At + i * lda + 4 * q);
          const float4 xv = *reinterpret_cast<const float4*>(xc + 4 * q);
          acc = fmaf(a.x, xv.x, fmaf(a.y, xv.y, fmaf(a.z, xv.z, fmaf(a.w, xv.w, acc))));
        }
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);   // n <= 64: quads live in lanes 0-15
        if (lane == 0) {
          const float y = acc + bs[t * n + i];
          xn[i] = y;
          xg[static_cast<size_t>(t) * n + i] = y;
        }
      }
      named_bar_sync(1, kFsVecGroup);
    }
  } else {
    // ---------------------------------------------------------------- adjoint: thread = (column j, row class)
    const int at = tid - kFsVecGroup;
    const int nrg = kFsVecGroup / n;           // row classes (n <= 64: >= 4)
    const int j = at % n, rg = at / n;
    const bool act = rg < nrg;
    float* lg = p.lam + itT * n;
    if (at < n) {
      const float v = gs[(T - 1) * n + at];    // lam_T = g_T
      ls[at] = v;
      lg[static_cast<size_t>(T - 1) * n + at] = v;
    }
    named_bar_sync(2, kFsVecGroup);
    const int nstep = (T - 1) + (p.gx0 != nullptr ? 1 : 0);
    for (int k = 0; k <= nstep; ++k) {
      // lam_{t+1} is in ls[k & 1], t = T-1-k.  grad_u[t] = B_t^T lam_{t+1} for t >= 0; then lam_t (t >= 1) / grad_x0 (t = 0)
      const int t = T - 1 - k;
      const float* lc = ls + (k & 1) * n;
      if (has_gu && t >= 0) {
        // warp w of the group takes the inputs l = w, w + 8, ..
        for (int l = (at >> 5); l < m; l += kFsVecGroup / 32) {
          float acc = 0.f;
          for (int i = lane; i < n; i += 32) {
            const float bv = p.b_in_smem ? Bs[(static_cast<size_t>(t) * n + i) * m + l] : __ldg(p.B + ((itT + t) * n + i) * m + l);
            acc = fmaf(bv, lc[i], acc);
          }
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
          if (lane == 0) p.gu[(itT + t) * m + l] = acc;
        }
      }
      if (k == nstep || t < 0) break;
      const float* At = As + static_cast<size_t>(t) * n * lda;
      if (act) {
        float acc = 0.f;
        for (int i = rg; i < n; i += nrg) acc = fmaf(At[i * lda + j], lc[i], acc);
        pa[rg * n + j] = acc;
      }
      named_bar_sync(2, kFsVecGroup);
      if (at < n) {
        float v = 0.f;
        for (int q = 0; q < nrg; ++q) v += pa[q * n + at];
        if (t >= 1) {
          v += gs[(t - 1) * n + at];                       // + g_t
          ls[((k + 1) & 1) * n + at] = v;
          lg[static_cast<size_t>(t - 1) * n + at] = v;     // lam_out[t-1] = lam_t
        } else {
          p.gx0[static_cast<size_t>(item) * n + at] = v;   // grad_x0 = A_0^T lam_1
        }
      }
      named_bar_sync(2, kFsVecGroup);
    }
  }
}

// ------------------------------------------------------------------------------------------------ kernel
__global__ void __launch_bounds__(kFsThreads, 1) fused_small_kernel(const FsParams p) {
  extern __shared__ __align__(128) uint8_t smem[];
  cg::cluster_group cluster = cg::this_cluster();
  const int C = static_cast<int>(cluster.num_blocks());
  const int rank = static_cast<int>(cluster.block_rank());
  const int item = blockIdx.x / C;
  if (rank < p.ncc) fs_column_cta(p, smem, item, rank); else fs_vector_cta(p, smem, item);
  __syncthreads();
  cluster.sync();
  // r_t = sum_{s<t} f(term(t,s)): CTA q takes t = q, q + C, ..; the terms sit in the shared memory of the column owners
  const int n = p.n, T = p.T;
  float* rpart = reinterpret_cast<float*>(smem + p.off_rpart);
  for (int t = rank; t < T; t += C) {
    for (int i = threadIdx.x; i < n; i += kFsThreads) {
      float acc = 0.f;
      for (int s = 0; s < t; ++s) {
        const float* remote = cluster.map_shared_rank(rpart, s % p.ncc);
        const float v = remote[(static_cast<size_t>(s / p.ncc) * T + t) * n + i];
        acc += p.tube_mode ? sqrtf(v) : v;
      }
      p.r[(static_cast<size_t>(item) * T + t) * n + i] = acc;
    }
  }
  cluster.sync();   // nobody exits while a peer may still read its shared memory
}

struct FsPlan {
  bool ok;
  int cluster;
  uint32_t smem;
  FsParams p;
};

FsPlan fs_plan(int batch, int T, int n, int m) {
  FsPlan pl{};
  pl.ok = false;
  if (n > kFsMaxN || n < 4 || (n & 3) || T < 2 || m < 0 || m > 64) return pl;
  FsParams& p = pl.p;
  p.batch = batch; p.T = T; p.n = n; p.m = m;
  const int ncol = T - 1;
  p.ncc = ncol < kFsMaxCluster - 1 ? ncol : kFsMaxCluster - 1;
  pl.cluster = p.ncc + 1;
  p.cps = (ncol + p.ncc - 1) / p.ncc;
  p.lda = n + 4;
  const int tiles = (n / 4) * (n / 4);
  p.ksplit = kFsThreads / tiles;
  if (p.ksplit > 4) p.ksplit = 4;
  if (p.ksplit < 1) return pl;
  p.kchunk = ((n + p.ksplit - 1) / p.ksplit + 3) & ~3;
  auto up = [](size_t v) { return static_cast<uint32_t>((v + 127) & ~static_cast<size_t>(127)); };
  const uint32_t a_bytes = up(static_cast<size_t>(T) * n * p.lda * 4);
  // column CTA
  p.off_p = a_bytes;
  p.off_red = p.off_p + up(2u * n * n * 4);
  p.off_w = p.off_red + up(static_cast<size_t>(p.ksplit > 1 ? p.ksplit - 1 : 1) * n * n * 4);
  p.off_tube = p.off_w + up(n * 4);
  p.off_rpart = p.off_tube + up(static_cast<size_t>(n) * (n / 4 + 1) * 4);
  const uint32_t col_total = p.off_rpart + up(static_cast<size_t>(p.cps) * T * n * 4);
  // vector CTA (rpart is not used there, but off_rpart must stay inside its allocation for the uniform final pass)
  p.off_bs = a_bytes;
  p.off_gs = p.off_bs + up(static_cast<size_t>(T) * n * 4);
  p.off_xs = p.off_gs + up(static_cast<size_t>(T) * n * 4);
  p.off_ls = p.off_xs + up(2u * n * 4);
  p.off_pa = p.off_ls + up(2u * n * 4);
  p.off_us = p.off_pa + up(static_cast<size_t>(kFsVecGroup / n) * n * 4);
  p.off_b = p.off_us + up(static_cast<size_t>(T) * (m > 0 ? m : 1) * 4);
  uint32_t vec_total = p.off_b;
  const uint32_t limit = 227u * 1024u;
  const uint32_t b_bytes = up(static_cast<size_t>(T) * n * (m > 0 ? m : 1) * 4);
  p.b_in_smem = (m > 0 && vec_total + b_bytes <= limit) ? 1 : 0;
  if (p.b_in_smem) vec_total += b_bytes;
  pl.smem = col_total > vec_total ? col_total : vec_total;
  if (pl.smem > limit) return pl;
  pl.ok = true;
  return pl;
}

}  // namespace

bool fused_small_supported(int batch, int T, int n, int m) { return fs_plan(batch, T, n, m).ok; }

cudaError_t launch_fused_small(const FusedSmallArgs& a, cudaStream_t stream, unsigned long long* launches) {
  FsPlan pl = fs_plan(a.batch, a.T, a.n, a.m);
  if (!pl.ok) return cudaErrorInvalidConfiguration;
  FsParams& p = pl.p;
  p.A = a.A; p.B = (a.m > 0) ? a.B : nullptr; p.c = a.c; p.x0 = a.x0; p.u = a.u; p.w = a.w; p.g = a.g;
  p.x = a.x_out; p.phi = a.phi_out; p.r = a.r_out; p.lam = a.lambda_out;
  p.gu = (a.m > 0) ? a.grad_u_out : nullptr; p.gx0 = a.grad_x0_out;
  p.tube_mode = a.tube_mode;
  cudaError_t e = cudaFuncSetAttribute(fused_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(pl.smem));
  if (e != cudaSuccess) return e;
  if (pl.cluster > 8) {
    e = cudaFuncSetAttribute(fused_small_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
  }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>(a.batch) * pl.cluster);
  cfg.blockDim = dim3(kFsThreads);
  cfg.dynamicSmemBytes = pl.smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = pl.cluster;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  {
    ProfScope prof(kProfFusedSmall, stream);
    e = cudaLaunchKernelEx(&cfg, fused_small_kernel, p);
  }
  if (e == cudaSuccess) ++*launches;
  return e;
}

}  // namespace ltv
