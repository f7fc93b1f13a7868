// Phi path, non-tensor-core kernels: level 0 (copy + tube), the fp32 FMA combine used for small n, and the
// deterministic tube finalise.  (eq.(12c), :147 eq.(12e).)
#include "ltv_internal.h"
#include "phi_geom.cuh"
#include "phi_kernels.h"
#include "ptx.cuh"

namespace ltv {

// one term of the fused tube reduction: |d| w (box tube) or (d w)^2 (row-wise two-norm tube, summed per block and
// square-rooted by the finalise kernel)
__device__ __forceinline__ float tube_term(float d, float w, int mode) {
  const float dw = d * w;
  return mode ? dw * dw : fabsf(dw);
}

// ------------------------------------------------------------------------------------------ level 0
// Phi(s+1,s) = A_s, part[b][q(s+1,s)][0][i] = sum_j |A_s[i,j]| w_s[j]; part slots 1..NT-1 are zeroed.
// HBM-bound copy.  A warp takes FOUR consecutive rows (never straddling a block: n % 4 == 0) and, per pass,
// four column quads per lane: 16 independent 128-bit loads in flight per lane, w_s read once for the four rows,
// and the four row sums finished with one transpose-reduce (6 shuffles) instead of four 5-level trees.
__device__ __forceinline__ float level0_reduce4(const float (&a)[4], int lane) {
  const bool hi16 = (lane & 16) != 0;
  const float b0 = (hi16 ? a[2] : a[0]) + __shfl_xor_sync(0xffffffffu, hi16 ? a[0] : a[2], 16);
  const float b1 = (hi16 ? a[3] : a[1]) + __shfl_xor_sync(0xffffffffu, hi16 ? a[1] : a[3], 16);
  const bool hi8 = (lane & 8) != 0;
  float v = (hi8 ? b1 : b0) + __shfl_xor_sync(0xffffffffu, hi8 ? b0 : b1, 8);
  v += __shfl_xor_sync(0xffffffffu, v, 4);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  return v;   // lanes 8g .. 8g+7 hold the sum of row g
}

__global__ void __launch_bounds__(256) phi_level0_kernel(const float* __restrict__ A, const float* __restrict__ w,
                                                         float* __restrict__ phi, float* __restrict__ part,
                                                         int batch, int T, int n, int NT, int mode) {
  const int P = T * (T - 1) / 2;
  const long long nunits = static_cast<long long>(batch) * (T - 1) * (n >> 2);
  const int lane = threadIdx.x & 31;
  const int n4 = n >> 2;
  for (long long un = static_cast<long long>(blockIdx.x) * 8 + (threadIdx.x >> 5); un < nunits;
       un += static_cast<long long>(gridDim.x) * 8) {
    const int i = 4 * static_cast<int>(un % n4);
    const long long bs = un / n4;
    const int s = static_cast<int>(bs % (T - 1));
    const int b = static_cast<int>(bs / (T - 1));
    const float4* src = reinterpret_cast<const float4*>(A + ((static_cast<size_t>(b) * T + s) * n + i) * n);
    const float4* wv = reinterpret_cast<const float4*>(w + (static_cast<size_t>(b) * T + s) * n);
    const size_t q = static_cast<size_t>(b) * P + phi_colbase(T, s);
    float* dst = phi + (q * n + i) * n;
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    for (int c0 = 0; c0 < n4; c0 += 128) {
      float4 a[4][4], ww[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int c = c0 + lane + 32 * j;
        const bool ok = c < n4;
        ww[j] = ok ? __ldg(wv + c) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int r = 0; r < 4; ++r) a[r][j] = ok ? __ldcs(src + static_cast<size_t>(r) * n4 + c) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int c = c0 + lane + 32 * j;
        if (c < n4) {
#pragma unroll
          for (int r = 0; r < 4; ++r) {
            st_global_f4_na(dst + static_cast<size_t>(r) * n + 4 * c, a[r][j]);
            acc[r] += (tube_term(a[r][j].x, ww[j].x, mode) + tube_term(a[r][j].y, ww[j].y, mode)) +
                      (tube_term(a[r][j].z, ww[j].z, mode) + tube_term(a[r][j].w, ww[j].w, mode));
          }
        }
      }
    }
    const float v = level0_reduce4(acc, lane);
    const int g = lane >> 3, sub = lane & 7;
    // lane (g, sub): row i + g, tube slots sub, sub + 8, ... (slot 0 = the sum, the others zero)
    for (int e = sub; e < NT; e += 8) part[(q * NT + e) * n + i + g] = (e == 0) ? v : 0.f;
  }
}

// ------------------------------------------------------------------------------------------ observer level 0
// Closed-loop observer propagation, eq.(14): the level-0 blocks are
//   PhiX(s+1,s) = Abar_s = A_s + Lt_s C_s   (rank-p update while A_s streams through: HBM-bound like the copy)
//   PhiY(s+1,s) = Abar_s Lt_s               (skinny product, second kernel; Abar_s is still in L2)
// written side by side in rows of nc = n + roundup4(p) floats; the tube partial is taken over PhiX.
// p > 8: the gains are first transposed (Ltt[b,t][k][j] = Lt[b,t][j][k], columns padded to pp = nc - n with zeros) so
// that the wide kernel reads them with coalesced 128-bit loads.  grid (batch T), 256 threads.
__global__ void __launch_bounds__(256) phi_obs_transpose_gains_kernel(const float* __restrict__ Lt, float* __restrict__ Ltt,
                                                                      int n, int p, int pp) {
  const size_t bt = blockIdx.x;
  const float* src = Lt + bt * n * p;
  float* dst = Ltt + bt * pp * n;
  for (int e = threadIdx.x; e < pp * n; e += 256) {
    const int k = e / n, j = e - k * n;
    dst[e] = (k < p) ? __ldg(src + static_cast<size_t>(j) * p + k) : 0.f;
  }
}

// Wide path (8 < p <= 32): a warp takes ROWS rows; per column quad it loads A (ROWS rows), the p rows of C_s and the p rows
// of Lt_s^T once, forms Abar in registers, stores it, and accumulates the tube partial and the ROWS x p products of
// PhiY(s+1,s) = Abar_s Lt_s; butterfly reductions at the end.  PG = ceil(p / 8) groups of eight columns (the padded
// columns of Ltt are zero, so they add nothing and come out as the zero padding of the row).
template <int PG, int ROWS>
__global__ void __launch_bounds__(256) phi_obs_level0_wide_kernel(const float* __restrict__ A, const float* __restrict__ Lt,
                                                                  const float* __restrict__ Ltt, const float* __restrict__ C,
                                                                  const float* __restrict__ w, float* __restrict__ phi,
                                                                  float* __restrict__ part, int batch, int T, int n, int nc,
                                                                  int p, int NT, int mode, int yshift) {
  constexpr int PP = 8 * PG;
  const int pp = nc - n;
  const int P = T * (T - 1) / 2;
  const int n4 = n >> 2;
  const int ngrp = (n + ROWS - 1) / ROWS;
  const long long nunits = static_cast<long long>(batch) * (T - 1) * ngrp;
  const int lane = threadIdx.x & 31;
  for (long long un = static_cast<long long>(blockIdx.x) * 8 + (threadIdx.x >> 5); un < nunits;
       un += static_cast<long long>(gridDim.x) * 8) {
    const int i = ROWS * static_cast<int>(un % ngrp);
    const long long bs = un / ngrp;
    const int s = static_cast<int>(bs % (T - 1));
    const int b = static_cast<int>(bs / (T - 1));
    const size_t bt = static_cast<size_t>(b) * T + s;
    const float4* wv = reinterpret_cast<const float4*>(w + bt * n);
    const float4* Cs = reinterpret_cast<const float4*>(C + bt * p * n);
    // PhiY columns: gain of step s (eq.(14) as printed) or, with yshift, of step s - 1 (the Phihat^y of (12c)/(15);
    // no such term for s = 0: the products are formed on valid memory and scaled by zero)
    const bool ynone = yshift && s == 0;
    const float4* Lts = reinterpret_cast<const float4*>(Ltt + (bt - ((yshift && s > 0) ? 1 : 0)) * pp * n);
    const size_t q = static_cast<size_t>(b) * P + phi_colbase(T, s);
    const float4* src[ROWS];
    const float* lrow[ROWS];
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
      const int ir = min(i + r, n - 1);
      src[r] = reinterpret_cast<const float4*>(A + (bt * n + ir) * n);
      lrow[r] = Lt + (bt * n + ir) * p;
    }
    float tube[ROWS], y[ROWS][PP];
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
      tube[r] = 0.f;
#pragma unroll
      for (int k = 0; k < PP; ++k) y[r][k] = 0.f;
    }
    for (int c = lane; c < n4; c += 32) {
      float4 a[ROWS];
#pragma unroll
      for (int r = 0; r < ROWS; ++r) a[r] = __ldcs(src[r] + c);
      for (int k = 0; k < p; ++k) {
        const float4 ck = __ldg(Cs + static_cast<size_t>(k) * n4 + c);
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
          const float l = __ldg(lrow[r] + k);
          a[r].x = fmaf(l, ck.x, a[r].x); a[r].y = fmaf(l, ck.y, a[r].y);
          a[r].z = fmaf(l, ck.z, a[r].z); a[r].w = fmaf(l, ck.w, a[r].w);
        }
      }
      const float4 ww = __ldg(wv + c);
#pragma unroll
      for (int r = 0; r < ROWS; ++r) {
        if (i + r < n) *reinterpret_cast<float4*>(phi + (q * n + i + r) * nc + 4 * c) = a[r];
        tube[r] += (tube_term(a[r].x, ww.x, mode) + tube_term(a[r].y, ww.y, mode)) +
                   (tube_term(a[r].z, ww.z, mode) + tube_term(a[r].w, ww.w, mode));
      }
#pragma unroll
      for (int kg = 0; kg < PP; kg += 8) {
        float4 lt[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) lt[k] = __ldg(Lts + static_cast<size_t>(min(kg + k, pp - 1)) * n4 + c);
#pragma unroll
        for (int k = 0; k < 8; ++k)
#pragma unroll
          for (int r = 0; r < ROWS; ++r)
            y[r][kg + k] = fmaf(a[r].x, lt[k].x, fmaf(a[r].y, lt[k].y, fmaf(a[r].z, lt[k].z, fmaf(a[r].w, lt[k].w, y[r][kg + k]))));
      }
    }
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) tube[r] += __shfl_xor_sync(0xffffffffu, tube[r], o);
#pragma unroll
      for (int k = 0; k < PP; ++k) {
        if (k < pp) {
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) y[r][k] += __shfl_xor_sync(0xffffffffu, y[r][k], o);
          if (lane == (k & 31) && i + r < n) phi[(q * n + i + r) * nc + n + k] = ynone ? 0.f : y[r][k];
        }
      }
      if (lane == 0 && i + r < n)
        for (int e = 0; e < NT; ++e) part[(q * NT + e) * n + i + r] = (e == 0) ? tube[r] : 0.f;
    }
  }
}

// ------------------------------------------------------------------------------------------ SIMT combine
// 64 x 64 output tile, 256 threads, 4 x 4 register micro-tile, K blocked by 16 through shared memory.
constexpr int kST = 64, kSK = 16;
__global__ void __launch_bounds__(256) phi_combine_simt_kernel(float* phi, const float* __restrict__ w,
                                                               float* __restrict__ part, PhiGeom g, int mode) {
  __shared__ float As[kSK][kST + 4];  // [k][m]
  __shared__ float Bs[kSK][kST + 4];  // [k][j]
  __shared__ float ws[kST];
  __shared__ float tube[kST][17];
  const int n = g.n, nc = g.nc;   // K extent / rows per block; columns per block = row stride
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  for (long long idx = blockIdx.x; idx < g.total; idx += gridDim.x) {
    const PhiTile t = phi_decode(g, idx);
    const size_t item = static_cast<size_t>(t.b) * g.P;
    const float* Aop = phi + (item + phi_colbase(g.T, t.mid)) * n * nc;                       // rows (t,i)
    const float* Bop = phi + (item + phi_colbase(g.T, t.s) + (t.mid - t.s - 1)) * n * nc;    // Phi(mid,s)
    float* Out = phi + (item + phi_colbase(g.T, t.s) + (t.mid - t.s)) * n * nc;             // rows (t,i), col s
    const int Mrows = t.cnt_t * n;
    const int m0 = t.m_tile * kST, j0 = t.n_tile * kST;
    if (threadIdx.x < kST) {
      const int j = j0 + threadIdx.x;
      ws[threadIdx.x] = (j < n) ? w[(static_cast<size_t>(t.b) * g.T + t.s) * n + j] : 0.f;
    }
    float acc[4][4] = {};
    for (int k0 = 0; k0 < n; k0 += kSK) {
      for (int e = threadIdx.x; e < kST * kSK; e += 256) {
        const int kk = e % kSK, mm = e / kSK;
        const int r = m0 + mm, k = k0 + kk;
        As[kk][mm] = (r < Mrows && k < n) ? Aop[static_cast<size_t>(r) * nc + k] : 0.f;
      }
      for (int e = threadIdx.x; e < kST * kSK; e += 256) {
        const int jj = e % kST, kk = e / kST;
        const int j = j0 + jj, k = k0 + kk;
        Bs[kk][jj] = (j < nc && k < n) ? Bop[static_cast<size_t>(k) * nc + j] : 0.f;
      }
      __syncthreads();
#pragma unroll
      for (int kk = 0; kk < kSK; ++kk) {
        float a[4], bb[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) a[r] = As[kk][ty * 4 + r];
#pragma unroll
        for (int c = 0; c < 4; ++c) bb[c] = Bs[kk][tx * 4 + c];
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
          for (int c = 0; c < 4; ++c) acc[r][c] = fmaf(a[r], bb[c], acc[r][c]);
      }
      __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int row = m0 + ty * 4 + r;
      float tb = 0.f;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const int j = j0 + tx * 4 + c;
        tb += tube_term(acc[r][c], ws[tx * 4 + c], mode);
        if (row < Mrows && j < nc) Out[static_cast<size_t>(row) * nc + j] = acc[r][c];
      }
      tube[ty * 4 + r][tx] = tb;
    }
    __syncthreads();
    if (threadIdx.x < kST) {
      const int row = m0 + threadIdx.x;
      if (row < Mrows) {
        float v = 0.f;
#pragma unroll
        for (int c = 0; c < 16; ++c) v += tube[threadIdx.x][c];
        const size_t q = item + phi_colbase(g.T, t.s) + (t.mid - t.s) + row / n;
        part[(q * g.NT + t.n_tile) * n + row % n] = v;
      }
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------ finalise
// r[b][t][i] = sum_{s<t} f(sum_{nt} part[b][q(t,s)][nt][i]), f = identity (box tube) or sqrt (two-norm tube: the
// partials are sums of squares over the columns of an n-tile); fixed order; r[b][0][:] = 0.
__global__ void __launch_bounds__(128) phi_tube_finalize_kernel(const float* __restrict__ part, float* __restrict__ r,
                                                                int batch, int T, int n, int NT, int mode) {
  const int P = T * (T - 1) / 2;
  const int t = blockIdx.x % T, b = blockIdx.x / T;
  for (int i = blockIdx.y * blockDim.x + threadIdx.x; i < n; i += gridDim.y * blockDim.x) {
    float acc = 0.f;
    for (int s = 0; s < t; ++s) {
      const size_t q = static_cast<size_t>(b) * P + phi_colbase(T, s) + (t - s - 1);
      float blk = 0.f;
      for (int nt = 0; nt < NT; ++nt) blk += part[(q * NT + nt) * n + i];
      acc += mode ? sqrtf(blk) : blk;
    }
    r[(static_cast<size_t>(b) * T + t) * n + i] = acc;
  }
}

// Fused fast path for p <= 8: a warp takes four rows; per column quad it loads A (4 rows), the p rows of C_s and the
// four rows j..j+3 of Lt_s (4p contiguous floats) ONCE, forms Abar in registers, stores it, and accumulates both the
// tube partial and the 4 x p products of PhiY(s+1,s) = Abar_s Lt_s; the 4 + 4p sums are finished by shuffles.
template <int PP>
__global__ void __launch_bounds__(256, 2) phi_obs_level0_fused_kernel(const float* __restrict__ A, const float* __restrict__ Lt,
                                                                   const float* __restrict__ C, const float* __restrict__ w,
                                                                   float* __restrict__ phi, float* __restrict__ part,
                                                                   int batch, int T, int n, int nc, int NT, int mode,
                                                                   int yshift) {
  constexpr int p = PP;   // exact number of measurement rows: every loop below unrolls, Lt is read as float4
  const int P = T * (T - 1) / 2;
  const int n4 = n >> 2;
  const long long nunits = static_cast<long long>(batch) * (T - 1) * n4;
  const int lane = threadIdx.x & 31;
  for (long long un = static_cast<long long>(blockIdx.x) * 8 + (threadIdx.x >> 5); un < nunits;
       un += static_cast<long long>(gridDim.x) * 8) {
    const int i = 4 * static_cast<int>(un % n4);
    const long long bs = un / n4;
    const int s = static_cast<int>(bs % (T - 1));
    const int b = static_cast<int>(bs / (T - 1));
    const size_t bt = static_cast<size_t>(b) * T + s;
    const float4* src = reinterpret_cast<const float4*>(A + (bt * n + i) * n);
    const float4* wv = reinterpret_cast<const float4*>(w + bt * n);
    const float4* Cs = reinterpret_cast<const float4*>(C + bt * p * n);
    const float* Ls = Lt + bt * n * p;
    // gain of the PhiY columns: step s (eq.(14) as printed) or, with yshift, step s - 1 (zero block for s = 0)
    const bool ynone = yshift && s == 0;
    const float* Lys = Ls - ((yshift && s > 0) ? static_cast<size_t>(n) * p : 0);
    const size_t q = static_cast<size_t>(b) * P + phi_colbase(T, s);
    float* dst = phi + (q * n + i) * nc;
    float lr[4][PP];   // Lt_s[i + r][k]: the gains of this unit's own rows
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int k = 0; k < PP; ++k) lr[r][k] = __ldg(Ls + static_cast<size_t>(i + r) * p + k);
    float tube[4] = {0.f, 0.f, 0.f, 0.f};
    float y[4][PP];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int k = 0; k < PP; ++k) y[r][k] = 0.f;
    for (int c = lane; c < n4; c += 32) {
      float4 a[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) a[r] = __ldcs(src + static_cast<size_t>(r) * n4 + c);
#pragma unroll
      for (int k = 0; k < PP; ++k) {
        const float4 ck = __ldg(Cs + static_cast<size_t>(k) * n4 + c);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          a[r].x = fmaf(lr[r][k], ck.x, a[r].x); a[r].y = fmaf(lr[r][k], ck.y, a[r].y);
          a[r].z = fmaf(lr[r][k], ck.z, a[r].z); a[r].w = fmaf(lr[r][k], ck.w, a[r].w);
        }
      }
      const float4 ww = __ldg(wv + c);
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        *reinterpret_cast<float4*>(dst + static_cast<size_t>(r) * nc + 4 * c) = a[r];
        tube[r] += (tube_term(a[r].x, ww.x, mode) + tube_term(a[r].y, ww.y, mode)) +
                   (tube_term(a[r].z, ww.z, mode) + tube_term(a[r].w, ww.w, mode));
      }
      // rows 4c .. 4c+3 of Lt_s: 4p contiguous floats
      const float4* lj4 = reinterpret_cast<const float4*>(Lys + static_cast<size_t>(4 * c) * p);
      float lt[4 * PP];   // lt[jj * p + k] = Lt_s[4c + jj][k]
#pragma unroll
      for (int v = 0; v < PP; ++v) {
        const float4 t4 = __ldg(lj4 + v);
        lt[4 * v + 0] = t4.x; lt[4 * v + 1] = t4.y; lt[4 * v + 2] = t4.z; lt[4 * v + 3] = t4.w;
      }
#pragma unroll
      for (int k = 0; k < PP; ++k)
#pragma unroll
        for (int r = 0; r < 4; ++r)
          y[r][k] = fmaf(a[r].x, lt[k], fmaf(a[r].y, lt[p + k], fmaf(a[r].z, lt[2 * p + k], fmaf(a[r].w, lt[3 * p + k], y[r][k]))));
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) tube[r] += __shfl_xor_sync(0xffffffffu, tube[r], o);
#pragma unroll
      for (int k = 0; k < PP; ++k)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) y[r][k] += __shfl_xor_sync(0xffffffffu, y[r][k], o);
    }
    if (lane < 4) {
      const int r = lane;
      float* prow = dst + static_cast<size_t>(r) * nc + n;
      float tr = tube[0];
#pragma unroll
      for (int rr = 1; rr < 4; ++rr) tr = (r == rr) ? tube[rr] : tr;
#pragma unroll
      for (int k = 0; k < PP; ++k) {
        float v = y[0][k];
#pragma unroll
        for (int rr = 1; rr < 4; ++rr) v = (r == rr) ? y[rr][k] : v;
        prow[k] = ynone ? 0.f : v;
      }
      for (int k = p; k < nc - n; ++k) prow[k] = 0.f;
      for (int e = 0; e < NT; ++e) part[(q * NT + e) * n + i + r] = (e == 0) ? tr : 0.f;
    }
  }
}

cudaError_t launch_phi_obs_level0(const PhiArgs& a, int NT, int num_sms, cudaStream_t stream) {
  const long long nrows = static_cast<long long>(a.batch) * (a.T - 1) * a.n;
  long long blocks = (nrows + 7) / 8;
  const long long cap = static_cast<long long>(num_sms) * 16;
  if (blocks > cap) blocks = cap;
  ProfScope prof(kProfPhiLevel0, stream);
  if (a.p <= 8) {
    const long long nunits = static_cast<long long>(a.batch) * (a.T - 1) * (a.n >> 2);
    long long ub = (nunits + 7) / 8;
    const long long ucap = static_cast<long long>(num_sms) * 8;
    if (ub > ucap) ub = ucap;
#define LTV_OBS_CASE(PV)                                                                                        \
  case PV:                                                                                                     \
    phi_obs_level0_fused_kernel<PV><<<static_cast<unsigned>(ub), 256, 0, stream>>>(a.A, a.Lt, a.C, a.w, a.phi, a.part, \
                                                                                   a.batch, a.T, a.n, a.nc, NT,   \
                                                                                   a.tube_mode, a.yshift);      \
    break;
    switch (a.p) {
      LTV_OBS_CASE(1) LTV_OBS_CASE(2) LTV_OBS_CASE(3) LTV_OBS_CASE(4)
      LTV_OBS_CASE(5) LTV_OBS_CASE(6) LTV_OBS_CASE(7) LTV_OBS_CASE(8)
    }
#undef LTV_OBS_CASE
    return cudaGetLastError();
  }
  // 8 < p <= 32: transpose the gains, then the wide fused kernel
  const int pp = a.nc - a.n;
  if (a.Ltt == nullptr) return cudaErrorInvalidValue;
  phi_obs_transpose_gains_kernel<<<static_cast<unsigned>(a.batch * a.T), 256, 0, stream>>>(a.Lt, a.Ltt, a.n, a.p, pp);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  constexpr int kRows = 2;
  const long long nunits = static_cast<long long>(a.batch) * (a.T - 1) * ((a.n + kRows - 1) / kRows);
  long long ub = (nunits + 7) / 8;
  const long long ucap = static_cast<long long>(num_sms) * 8;
  if (ub > ucap) ub = ucap;
#define LTV_OBSW_CASE(PGV)                                                                                         \
  case PGV:                                                                                                        \
    phi_obs_level0_wide_kernel<PGV, kRows><<<static_cast<unsigned>(ub), 256, 0, stream>>>(                          \
        a.A, a.Lt, a.Ltt, a.C, a.w, a.phi, a.part, a.batch, a.T, a.n, a.nc, a.p, NT, a.tube_mode, a.yshift);        \
    break;
  switch ((pp + 7) / 8) {
    LTV_OBSW_CASE(2) LTV_OBSW_CASE(3) LTV_OBSW_CASE(4)
    default: return cudaErrorInvalidValue;
  }
#undef LTV_OBSW_CASE
  return cudaGetLastError();
}

cudaError_t launch_phi_level0(const PhiArgs& a, int NT, int num_sms, cudaStream_t stream) {
  const long long nunits = static_cast<long long>(a.batch) * (a.T - 1) * (a.n >> 2);   // 4-row units, one per warp
  long long blocks = (nunits + 7) / 8;
  const long long cap = static_cast<long long>(num_sms) * 8;
  if (blocks > cap) blocks = cap;
  ProfScope prof(kProfPhiLevel0, stream);
  phi_level0_kernel<<<static_cast<unsigned>(blocks), 256, 0, stream>>>(a.A, a.w, a.phi, a.part, a.batch, a.T, a.n, NT,
                                                                       a.tube_mode);
  return cudaGetLastError();
}

cudaError_t launch_phi_combine_simt(const PhiArgs& a, int level, int num_sms, cudaStream_t stream) {
  const PhiGeom g = phi_geom(a.batch, a.T, a.n, a.nc, level, kST, kST);
  if (g.total == 0) return cudaSuccess;
  long long blocks = g.total;
  const long long cap = static_cast<long long>(num_sms) * 8;
  if (blocks > cap) blocks = cap;
  ProfScope prof(kProfPhiCombineSimt, stream);
  phi_combine_simt_kernel<<<static_cast<unsigned>(blocks), 256, 0, stream>>>(a.phi, a.w, a.part, g, a.tube_mode);
  return cudaGetLastError();
}

cudaError_t launch_phi_finalize(const PhiArgs& a, int NT, cudaStream_t stream) {
  dim3 grid(static_cast<unsigned>(a.batch) * a.T, static_cast<unsigned>((a.n + 127) / 128));
  if (grid.y > 64) grid.y = 64;
  ProfScope prof(kProfPhiFinalize, stream);
  phi_tube_finalize_kernel<<<grid, 128, 0, stream>>>(a.part, a.r, a.batch, a.T, a.n, NT, a.tube_mode);
  return cudaGetLastError();
}

}  // namespace ltv
