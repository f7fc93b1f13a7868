// ltv_scan_kalman_gains: the backward-Kalman recursion of eq.(13), batched over
// items and time-sequential:
//     Pi_0 = Xi Xi^T;   L_{j+1} = -(F_j F_j^T + C_j Pi_j C_j^T)^{-1} C_j Pi_j A_j^T;
//     Pi_{j+1} = E_j E_j^T + A_j Pi_j A_j^T + A_j Pi_j C_j^T L_{j+1}
// computed per step j, for all items at once, as
//     G = C_j Pi_j                     [p,n]   kalman_cpi_kernel      (rows of the symmetric Pi_j against the p rows of C_j)
//     S = F F^T + G C_j^T, K = S^{-1}G [p,n]   kalman_gain_kernel     (Cholesky of the p x p innovation covariance)
//     Lt_j = L_{j+1}^T = -A_j K^T      [n,p]   kalman_closed_loop_kernel (A_j streams through once: the same pass
//     Abar_j = A_j + Lt_j C_j          [n,n]                           writes the closed-loop matrix of eq.(14))
//     Yt = (Abar_j Pi_j)^T             [n,n]   tcgen05 3xTF32 batched GEMM, transposed store
//     Pi_{j+1} = A_j Yt + diag(e_j)^2  [n,n]   tcgen05 3xTF32 batched GEMM, E E^T added in the epilogue
// (A_j Pi_j Abar_j^T is the right-hand side of (13) with L_{j+1} substituted.)
//
// Recursion or associative scan (16)(17)?  One combination of (16) costs an n x n solve with 2n
// right-hand sides plus six n^3 products (~17 n^3 flop) against 4 n^3 for one step of (13), and a scan needs
// (T/2) log2 T of them; at T = 32 that is ~10x the flops.  The scan buys depth log T; where one step over the whole
// batch already fills all 148 SMs (C2: 384 tiles of 128 x 160) the sequential form is the faster one.  For small n and
// batch - the paper's own regime - the scan runs on the device too (riccati_scan.cu; kalman_use_scan picks), and the
// gains of all steps then come out of ONE pass of the three kernels below.  DESIGN.md section 7.
#include <cuda.h>

#include <algorithm>
#include <type_traits>

#include "ltv_internal.h"
#include "phi_kernels.h"

namespace ltv {

namespace {

constexpr int kRowWarps = 8;   // warps per CTA of the row kernels

// offset of (item b, step j) in an array, for a flattened pair index it = b * nj + j
struct Stride2 {
  long long sb, sj;
  int nj;
  __device__ __forceinline__ long long at(int it) const { return (it / nj) * sb + (it % nj) * sj; }
};
// measured on B200 (C2 p = 6, C4 p = 12; the variants differ by < 10 %): p <= 8 runs best with two CTAs per SM and the
// loop not unrolled, wider p with one CTA per SM and two passes in flight
// NP = number of accumulators per row: exactly p for p <= 8 (no padded work: the kernels are instruction-bound), else p
// rounded up to a multiple of 8 (accumulators beyond p re-read vector p - 1 and are discarded)
template <int NP> struct RowCfg {
  static constexpr int kRows = NP <= 16 ? 4 : 2;
  static constexpr int kUnroll = NP <= 8 ? 1 : 2;
  static constexpr int kMinBlocks = NP <= 8 ? 2 : 1;
};

// ROWS rows of a row-major matrix against p vectors V[q][0..n) (global memory, L1-resident: every warp reads the same
// ones): acc[r][q] = sum_k row_r[k] V[q][k], complete in every lane.  Lane = float4 column, stride 32; ROWS
// independent 128-bit loads in flight per lane and pass, the vector loads amortised over the ROWS rows.
template <int NP, int ROWS>
__device__ __forceinline__ void row_dots(const float4* const (&rows)[ROWS], const float* __restrict__ V, int n4, int p,
                                         int lane, float (&acc)[ROWS][NP]) {
  constexpr int PP = NP;
#pragma unroll
  for (int r = 0; r < ROWS; ++r)
#pragma unroll
    for (int q = 0; q < PP; ++q) acc[r][q] = 0.f;
  // no branch on q < p inside the loop: behind a branch every vector load waits for the previous one's FMAs (measured:
  // 6 serialised L2 round trips per pass).  Accumulators q >= p re-read vector p - 1 and are discarded.
  const float4* V4 = reinterpret_cast<const float4*>(V);
  size_t voff[PP];
#pragma unroll
  for (int q = 0; q < PP; ++q) voff[q] = static_cast<size_t>(min(q, p - 1)) * n4;
#pragma unroll RowCfg<NP>::kUnroll
  for (int k4 = lane; k4 < n4; k4 += 32) {
    float4 a[ROWS];
#pragma unroll
    for (int r = 0; r < ROWS; ++r) a[r] = __ldg(rows[r] + k4);
#pragma unroll
    for (int qg = 0; qg < PP; qg += 8) {   // up to eight vector loads in flight at a time
      constexpr int kGrp = PP < 8 ? PP : 8;   // PP is <= 8 or a multiple of 8
      float4 v[kGrp];
#pragma unroll
      for (int q = 0; q < kGrp; ++q) v[q] = __ldg(V4 + voff[qg + q] + k4);
#pragma unroll
      for (int q = 0; q < kGrp; ++q) {
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
          acc[r][qg + q] = fmaf(a[r].x, v[q].x, acc[r][qg + q]);
          acc[r][qg + q] = fmaf(a[r].y, v[q].y, acc[r][qg + q]);
          acc[r][qg + q] = fmaf(a[r].z, v[q].z, acc[r][qg + q]);
          acc[r][qg + q] = fmaf(a[r].w, v[q].w, acc[r][qg + q]);
        }
      }
    }
  }
#pragma unroll
  for (int q = 0; q < PP; ++q) {
    if (q < p) {
#pragma unroll
      for (int r = 0; r < ROWS; ++r)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc[r][q] += __shfl_xor_sync(0xffffffffu, acc[r][q], o);
    }
  }
}

// G[b][q][j] = sum_k Pi[b][j][k] C[b][q][k]  (= (C Pi)[q][j]: Pi is symmetric, so its ROW j serves as column j and the
// loads are contiguous).  Warp = ROWS rows of Pi; grid (ceil(n / (8 ROWS)), batch), 256 threads.
template <int NP, int ROWS>
__global__ void __launch_bounds__(32 * kRowWarps, RowCfg<NP>::kMinBlocks) kalman_cpi_kernel(const float* __restrict__ C, Stride2 c_stride,
                                                                    const float* __restrict__ Pi, Stride2 pi_stride,
                                                                    float* __restrict__ G, int n, int p) {
  const int b = blockIdx.y;   // (item, step) pair
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int j0 = (blockIdx.x * kRowWarps + warp) * ROWS;
  if (j0 >= n) return;
  const int n4 = n >> 2;
  const float4* rows[ROWS];
#pragma unroll
  for (int r = 0; r < ROWS; ++r)
    rows[r] = reinterpret_cast<const float4*>(Pi + pi_stride.at(b) + static_cast<size_t>(min(j0 + r, n - 1)) * n);
  float acc[ROWS][NP];
  row_dots<NP, ROWS>(rows, C + c_stride.at(b), n4, p, lane, acc);
  float* Gb = G + static_cast<size_t>(b) * p * n;
#pragma unroll
  for (int q = 0; q < NP; ++q) {
    if (q < p && lane == (q & 31)) {
#pragma unroll
      for (int r = 0; r < ROWS; ++r)
        if (j0 + r < n) Gb[static_cast<size_t>(q) * n + j0 + r] = acc[r][q];
    }
  }
}

// One CTA per item: S = diag(f)^2 + G C^T (lower triangle; warp per entry), Cholesky S = R R^T (warp 0, lane = row),
// K = S^{-1} G (thread per column).  256 threads; shared memory: S [32][33].
template <int PG>
__global__ void __launch_bounds__(256) kalman_gain_kernel(const float* __restrict__ C, Stride2 c_stride,
                                                          const float* __restrict__ f, Stride2 f_stride,
                                                          const float* __restrict__ G, float* __restrict__ K, int n,
                                                          int p) {
  constexpr int PP = 8 * PG;
  __shared__ float S[32][33];
  const int b = blockIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const float4* C4 = reinterpret_cast<const float4*>(C + c_stride.at(b));
  const float* Gb = G + static_cast<size_t>(b) * p * n;
  const float4* G4 = reinterpret_cast<const float4*>(Gb);
  float* Kb = K + static_cast<size_t>(b) * p * n;
  const int n4 = n >> 2;
  for (int pr = warp; pr < p * p; pr += 8) {
    const int q = pr / p, r = pr % p;
    if (r > q) continue;
    float s0 = 0.f, s1 = 0.f;
    int k4 = lane;
    for (; k4 + 32 < n4; k4 += 64) {
      const float4 g0 = __ldg(G4 + static_cast<size_t>(q) * n4 + k4), c0 = __ldg(C4 + static_cast<size_t>(r) * n4 + k4);
      const float4 g1 = __ldg(G4 + static_cast<size_t>(q) * n4 + k4 + 32), c1 = __ldg(C4 + static_cast<size_t>(r) * n4 + k4 + 32);
      s0 = fmaf(g0.x, c0.x, fmaf(g0.y, c0.y, fmaf(g0.z, c0.z, fmaf(g0.w, c0.w, s0))));
      s1 = fmaf(g1.x, c1.x, fmaf(g1.y, c1.y, fmaf(g1.z, c1.z, fmaf(g1.w, c1.w, s1))));
    }
    if (k4 < n4) {
      const float4 g0 = __ldg(G4 + static_cast<size_t>(q) * n4 + k4), c0 = __ldg(C4 + static_cast<size_t>(r) * n4 + k4);
      s0 = fmaf(g0.x, c0.x, fmaf(g0.y, c0.y, fmaf(g0.z, c0.z, fmaf(g0.w, c0.w, s0))));
    }
    float s = s0 + s1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) {
      if (q == r) {
        const float ff = __ldg(f + f_stride.at(b) + q);
        s = fmaf(ff, ff, s);
      }
      S[q][r] = s;
    }
  }
  __syncthreads();
  if (warp == 0) {
    for (int k = 0; k < p; ++k) {
      const float d = sqrtf(S[k][k]);
      __syncwarp();
      if (lane == k) S[k][k] = d;
      if (lane > k && lane < p) S[lane][k] /= d;
      __syncwarp();
      if (lane > k && lane < p)
        for (int c = k + 1; c <= lane; ++c) S[lane][c] -= S[lane][k] * S[c][k];
      __syncwarp();
    }
  }
  __syncthreads();
  for (int j = threadIdx.x; j < n; j += 256) {
    float y[PP];
#pragma unroll
    for (int q = 0; q < PP; ++q) y[q] = (q < p) ? __ldg(Gb + static_cast<size_t>(q) * n + j) : 0.f;
    // R y' = g (forward), R^T k = y' (backward)
#pragma unroll
    for (int q = 0; q < PP; ++q) {
      if (q < p) {
        float s = y[q];
#pragma unroll
        for (int r = 0; r < q; ++r) s = fmaf(-S[q][r], y[r], s);
        y[q] = s / S[q][q];
      }
    }
#pragma unroll
    for (int q = PP - 1; q >= 0; --q) {
      if (q < p) {
        float s = y[q];
#pragma unroll
        for (int r = q + 1; r < PP; ++r)
          if (r < p) s = fmaf(-S[r][q], y[r], s);
        y[q] = s / S[q][q];
      }
    }
#pragma unroll
    for (int q = 0; q < PP; ++q)
      if (q < p) Kb[static_cast<size_t>(q) * n + j] = y[q];
  }
}

// Warp = ROWS rows i of A_j: Lt[i][q] = -sum_k A[i][k] K[q][k];  Abar[i][:] = A[i][:] + sum_q Lt[i][q] C[q][:].
// grid (ceil(n / (8 ROWS)), batch), 256 threads.
template <int NP, int ROWS>
__global__ void __launch_bounds__(32 * kRowWarps, RowCfg<NP>::kMinBlocks) kalman_closed_loop_kernel(
    const float* __restrict__ A, Stride2 a_stride, const float* __restrict__ C, Stride2 c_stride,
    const float* __restrict__ K, float* __restrict__ Lt, Stride2 lt_stride, float* __restrict__ Abar, int n, int p) {
  constexpr int PP = NP;
  const int b = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i0 = (blockIdx.x * kRowWarps + warp) * ROWS;
  if (i0 >= n) return;
  const int n4 = n >> 2;
  const float4* rows[ROWS];
#pragma unroll
  for (int r = 0; r < ROWS; ++r)
    rows[r] = reinterpret_cast<const float4*>(A + a_stride.at(b) + static_cast<size_t>(min(i0 + r, n - 1)) * n);
  float acc[ROWS][PP];
  row_dots<NP, ROWS>(rows, K + static_cast<size_t>(b) * p * n, n4, p, lane, acc);
#pragma unroll
  for (int q = 0; q < PP; ++q) {
    if (q < p) {
#pragma unroll
      for (int r = 0; r < ROWS; ++r) {
        acc[r][q] = -acc[r][q];
        if (lane == (q & 31) && i0 + r < n) Lt[lt_stride.at(b) + static_cast<size_t>(i0 + r) * p + q] = acc[r][q];
      }
    }
  }
  if (Abar == nullptr) return;   // gains only (the scan path has no use for the closed-loop matrix)
  const float4* C4 = reinterpret_cast<const float4*>(C + c_stride.at(b));
#pragma unroll
  for (int q = 0; q < PP; ++q)
    if (q >= p) {
#pragma unroll
      for (int r = 0; r < ROWS; ++r) acc[r][q] = 0.f;   // discarded accumulators must not reach Abar
    }
  size_t coff[PP];
#pragma unroll
  for (int q = 0; q < PP; ++q) coff[q] = static_cast<size_t>(min(q, p - 1)) * n4;
  for (int k4 = lane; k4 < n4; k4 += 32) {
    float4 a[ROWS];
#pragma unroll
    for (int r = 0; r < ROWS; ++r) a[r] = __ldg(rows[r] + k4);
#pragma unroll
    for (int qg = 0; qg < PP; qg += 8) {
      constexpr int kGrp = PP < 8 ? PP : 8;
      float4 cc[kGrp];
#pragma unroll
      for (int q = 0; q < kGrp; ++q) cc[q] = __ldg(C4 + coff[qg + q] + k4);
#pragma unroll
      for (int q = 0; q < kGrp; ++q) {
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
          a[r].x = fmaf(acc[r][qg + q], cc[q].x, a[r].x);
          a[r].y = fmaf(acc[r][qg + q], cc[q].y, a[r].y);
          a[r].z = fmaf(acc[r][qg + q], cc[q].z, a[r].z);
          a[r].w = fmaf(acc[r][qg + q], cc[q].w, a[r].w);
        }
      }
    }
#pragma unroll
    for (int r = 0; r < ROWS; ++r)
      if (i0 + r < n) reinterpret_cast<float4*>(Abar + (static_cast<size_t>(b) * n + i0 + r) * n)[k4] = a[r];
  }
}

// Pi_out[b][0] = Pi0[b]
__global__ void kalman_copy_pi0_kernel(const float4* __restrict__ src, float4* __restrict__ dst, long long per_item4,
                                       long long dst_stride4, long long total4) {
  for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < total4;
       i += static_cast<long long>(gridDim.x) * blockDim.x) {
    const long long b = i / per_item4, r = i - b * per_item4;
    dst[b * dst_stride4 + r] = __ldg(src + i);
  }
}

// fp32-FMA batched GEMM for n < 96 (BASELINE.json configs[0]): same operands and epilogues as the tcgen05 MODE 1
// kernel.  16 x 16 output tile per CTA, one element per thread.
__global__ void __launch_bounds__(256) bgemm_simt_kernel(const BatchedGemm g) {
  __shared__ float sL[16][17], sR[16][17];
  const int b = blockIdx.z;
  const float* L = g.L + (static_cast<size_t>(g.l_row0) + static_cast<size_t>(b) * g.l_row_stride) * g.K;
  const float* R = g.R + (static_cast<size_t>(g.r_blk0) + static_cast<size_t>(b) * g.r_blk_stride) * g.K * g.N;
  float* D = g.D + (static_cast<size_t>(g.d_blk0) + static_cast<size_t>(b) * g.d_blk_stride) * (g.d_rows > 0 ? g.d_rows : g.M) * g.N +
             (static_cast<size_t>(g.d_row0) + static_cast<size_t>(b) * g.d_row_stride) * g.N;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int row = blockIdx.y * 16 + ty, col = blockIdx.x * 16 + tx;
  float acc = 0.f;
  for (int k0 = 0; k0 < g.K; k0 += 16) {
    sL[ty][tx] = (row < g.M && k0 + tx < g.K) ? L[static_cast<size_t>(row) * g.K + k0 + tx] : 0.f;
    sR[ty][tx] = (k0 + ty < g.K && col < g.N) ? R[static_cast<size_t>(k0 + ty) * g.N + col] : 0.f;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 16; ++k) acc = fmaf(sL[ty][k], sR[k][tx], acc);
    __syncthreads();
  }
  if (row < g.M && col < g.N) {
    if (g.diag != nullptr && row == col) {
      const float d = g.diag[static_cast<long long>(b) * g.diag_stride + row];
      acc += d * d;
    }
    if (g.transpose_out) D[static_cast<size_t>(col) * g.M + row] = acc; else D[static_cast<size_t>(row) * g.N + col] = acc;
  }
}

}  // namespace

cudaError_t launch_bgemm_simt(const BatchedGemm& g, cudaStream_t stream) {
  const dim3 grid((g.N + 15) / 16, (g.M + 15) / 16, g.count);
  bgemm_simt_kernel<<<grid, 256, 0, stream>>>(g);
  return cudaGetLastError();
}

namespace {

template <typename F>
cudaError_t dispatch_pg(int p, F&& fn) {
  switch ((p + 7) / 8) {
    case 1: return fn(std::integral_constant<int, 1>{});
    case 2: return fn(std::integral_constant<int, 2>{});
    case 3: return fn(std::integral_constant<int, 3>{});
    case 4: return fn(std::integral_constant<int, 4>{});
    default: return cudaErrorInvalidValue;
  }
}

// NP (accumulators of the row kernels: p itself up to 8, else p rounded up to a multiple of 8) and PG = ceil(p / 8)
template <typename F>
cudaError_t dispatch_np(int p, F&& fn) {
  using std::integral_constant;
  switch (p) {
    case 1: return fn(integral_constant<int, 1>{}, integral_constant<int, 1>{});
    case 2: return fn(integral_constant<int, 2>{}, integral_constant<int, 1>{});
    case 3: return fn(integral_constant<int, 3>{}, integral_constant<int, 1>{});
    case 4: return fn(integral_constant<int, 4>{}, integral_constant<int, 1>{});
    case 5: return fn(integral_constant<int, 5>{}, integral_constant<int, 1>{});
    case 6: return fn(integral_constant<int, 6>{}, integral_constant<int, 1>{});
    case 7: return fn(integral_constant<int, 7>{}, integral_constant<int, 1>{});
    case 8: return fn(integral_constant<int, 8>{}, integral_constant<int, 1>{});
    default: break;
  }
  switch ((p + 7) / 8) {
    case 2: return fn(integral_constant<int, 16>{}, integral_constant<int, 2>{});
    case 3: return fn(integral_constant<int, 24>{}, integral_constant<int, 3>{});
    case 4: return fn(integral_constant<int, 32>{}, integral_constant<int, 4>{});
    default: return cudaErrorInvalidValue;
  }
}

struct KalmanWs {
  float *G, *K, *Abar, *Yt;
};

size_t carve(size_t floats) { return align_up(floats * sizeof(float), 256); }

}  // namespace

// G = C Pi, K = (F F^T + G C^T)^{-1} G, Lt = -A K^T (and Abar = A + Lt C unless Abar == nullptr) for the steps
// j0 .. j0 + nj - 1 of every item at once (three launches).  The recursion calls it with nj = 1 once Pi_j exists; the
// scan path calls it once with j0 = 0, nj = T after all Pi_j are known.  G, K: [batch nj][p][n]; Abar: [batch][n][n]
// (nj = 1 only).
cudaError_t launch_kalman_gain_chain(const KalmanArgs& a, int j0, int nj, float* G, float* K, float* Abar,
                                     cudaStream_t stream) {
  const int batch = a.batch, T = a.T, n = a.n, p = a.p;
  const int pairs = batch * nj;
  const Stride2 sC{static_cast<long long>(T) * p * n, static_cast<long long>(p) * n, nj};
  const Stride2 sA{static_cast<long long>(T) * n * n, static_cast<long long>(n) * n, nj};
  const Stride2 sPi{static_cast<long long>(T + 1) * n * n, static_cast<long long>(n) * n, nj};
  const Stride2 sF{static_cast<long long>(T) * p, p, nj};
  const Stride2 sLt{static_cast<long long>(T) * n * p, static_cast<long long>(n) * p, nj};
  const float* Cj = a.C + static_cast<size_t>(j0) * p * n;
  const float* Aj = a.A + static_cast<size_t>(j0) * n * n;
  const float* Pij = a.Pi_out + static_cast<size_t>(j0) * n * n;
  return dispatch_np(p, [&](auto np_, auto pg) {
    constexpr int NP = decltype(np_)::value;
    constexpr int PG = decltype(pg)::value;
    constexpr int ROWS = RowCfg<NP>::kRows;
    const dim3 rgrid((n + kRowWarps * ROWS - 1) / (kRowWarps * ROWS), pairs);
    {
      ProfScope prof(kProfKalmanSimt, stream);
      kalman_cpi_kernel<NP, ROWS><<<rgrid, 32 * kRowWarps, 0, stream>>>(Cj, sC, Pij, sPi, G, n, p);
    }
    cudaError_t ee = cudaGetLastError();
    if (ee != cudaSuccess) return ee;
    {
      ProfScope prof(kProfKalmanSimt, stream);
      kalman_gain_kernel<PG><<<pairs, 256, 0, stream>>>(Cj, sC, a.f + static_cast<size_t>(j0) * p, sF, G, K, n, p);
    }
    if ((ee = cudaGetLastError()) != cudaSuccess) return ee;
    {
      ProfScope prof(kProfKalmanSimt, stream);
      kalman_closed_loop_kernel<NP, ROWS><<<rgrid, 32 * kRowWarps, 0, stream>>>(
          Aj, sA, Cj, sC, K, a.Lt_out + static_cast<size_t>(j0) * n * p, sLt, Abar, n, p);
    }
    return cudaGetLastError();
  });
}

size_t kalman_workspace_bytes(int batch, int T, int n, int p) {
  const size_t b = batch, nn = n, pp = p;
  const size_t rec = 2 * carve(b * pp * nn) + 2 * carve(b * nn * nn);
  if (!riccati_scan_supported(n)) return rec;
  const size_t scan = riccati_scan_workspace_bytes(batch, T, n) + 2 * carve(b * T * pp * nn);
  return rec > scan ? rec : scan;
}

// The scan (riccati_scan.cu) pays when its log2(T+1) levels of (T+1)/2 combinations per item fit the machine in about
// one wave and the recursion's T steps would each be a handful of latency-bound launches: small n, small batch.
static bool kalman_use_scan(const KalmanArgs& a, int sms) {
  if (a.mode == 2 || !riccati_scan_supported(a.n)) return false;
  if (a.mode == 1) return true;
  const int forced = env_int("KALMAN_SCAN", -1);
  if (forced >= 0) return forced != 0;
  // The scan is faster for one small problem (n = 40, batch 1: 417 vs 927 us at T = 32, 550 vs 3677 us at T = 128), but its
  // fp32 n x n solves lose digits as max(C^2 / f^2) ||Pi|| grows (measured, n = 48: Pi0 = 0.01 I, f = 1e-3: gains off by 7.5e-3;
  // Pi0 = I, f = 1e-2: 2.5e-2; NaN beyond) where the recursion stays at 1e-5 .. 5e-4.  The library cannot look at device data when
  // it picks, so the scan runs only when the caller asks for it (LTV_KALMAN_SCAN).
  (void)sms;
  return false;
}

cudaError_t launch_kalman(const KalmanArgs& a, cudaStream_t stream, unsigned long long* launches) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int batch = a.batch, T = a.T, n = a.n, p = a.p;
  const size_t b = batch, nn = n, pp = p;
  if (kalman_use_scan(a, sms)) {
    // Pi_0 .. Pi_T by the associative scan (16)(17), then the gains of all steps in one batched pass
    char* cur = static_cast<char*>(a.workspace);
    float* AD = reinterpret_cast<float*>(cur); cur += riccati_scan_workspace_bytes(batch, T, n);
    float* G = reinterpret_cast<float*>(cur); cur += carve(b * T * pp * nn);
    float* K = reinterpret_cast<float*>(cur);
    cudaError_t es = launch_riccati_scan(a, AD, stream, launches);
    if (es != cudaSuccess) return es;
    es = launch_kalman_gain_chain(a, 0, T, G, K, nullptr, stream);
    if (es == cudaSuccess) *launches += 3;
    return es;
  }
  if (kalman_small_supported(n, p)) return launch_kalman_small(a, stream, launches);   // one launch, Pi_j in shared memory
  KalmanWs w;
  char* cur = static_cast<char*>(a.workspace);
  w.G = reinterpret_cast<float*>(cur); cur += carve(b * pp * nn);
  w.K = reinterpret_cast<float*>(cur); cur += carve(b * pp * nn);
  w.Abar = reinterpret_cast<float*>(cur); cur += carve(b * nn * nn);
  w.Yt = reinterpret_cast<float*>(cur);

  cudaError_t e;
  {
    const long long per4 = static_cast<long long>(nn * nn / 4), tot4 = per4 * batch;
    const int blocks = static_cast<int>(std::min<long long>((tot4 + 255) / 256, 8ll * sms));
    ProfScope prof(kProfKalmanSimt, stream);
    kalman_copy_pi0_kernel<<<blocks, 256, 0, stream>>>(reinterpret_cast<const float4*>(a.Pi0),
                                                       reinterpret_cast<float4*>(a.Pi_out), per4,
                                                       per4 * (T + 1), tot4);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    ++*launches;
  }

  const bool tc = phi_uses_tensor_cores(n);
  const int nch = phi_pick_nch(n);
  BatchedGemm g1{}, g2{};
  // Yt[b] = (Abar[b] Pi_j[b])^T
  g1.L = w.Abar; g1.l_rows = static_cast<long long>(b * nn); g1.l_row0 = 0; g1.l_row_stride = n;
  g1.R = a.Pi_out; g1.r_blocks = batch * (T + 1); g1.r_blk_stride = T + 1;
  g1.D = w.Yt; g1.d_blocks = batch; g1.d_blk0 = 0; g1.d_blk_stride = 1;
  g1.count = batch; g1.M = n; g1.N = n; g1.K = n; g1.transpose_out = 1; g1.diag = nullptr; g1.diag_stride = 0;
  // Pi_{j+1}[b] = A_j[b] Yt[b] + diag(e_j[b])^2
  g2.L = a.A; g2.l_rows = static_cast<long long>(b * T * nn); g2.l_row_stride = T * n;
  g2.R = w.Yt; g2.r_blocks = batch; g2.r_blk0 = 0; g2.r_blk_stride = 1;
  g2.D = a.Pi_out; g2.d_blocks = batch * (T + 1); g2.d_blk_stride = T + 1;
  g2.count = batch; g2.M = n; g2.N = n; g2.K = n; g2.transpose_out = 0; g2.diag_stride = static_cast<long long>(T) * n;
  alignas(64) unsigned char maps1[1024], maps2[1024];
  if (tc) {
    if (phi_tc_maps_size() > sizeof(maps1)) return cudaErrorInvalidValue;
    if ((e = bgemm_tc_make_maps(g1, maps1)) != cudaSuccess) return e;
    if ((e = bgemm_tc_make_maps(g2, maps2)) != cudaSuccess) return e;
  }

  for (int j = 0; j < T; ++j) {
    e = launch_kalman_gain_chain(a, j, 1, w.G, w.K, w.Abar, stream);
    if (e != cudaSuccess) return e;
    *launches += 3;
    g1.r_blk0 = j;
    g2.l_row0 = j * n;
    g2.d_blk0 = j + 1;
    g2.diag = a.e + static_cast<size_t>(j) * n;
    if (tc) {
      if ((e = launch_bgemm_tc(g1, nch, maps1, sms, stream)) != cudaSuccess) return e;
      if ((e = launch_bgemm_tc(g2, nch, maps2, sms, stream)) != cudaSuccess) return e;
    } else {
      const dim3 grid((n + 15) / 16, (n + 15) / 16, batch);
      {
        ProfScope prof(kProfKalmanGemm, stream);
        bgemm_simt_kernel<<<grid, 256, 0, stream>>>(g1);
      }
      if ((e = cudaGetLastError()) != cudaSuccess) return e;
      {
        ProfScope prof(kProfKalmanGemm, stream);
        bgemm_simt_kernel<<<grid, 256, 0, stream>>>(g2);
      }
      if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    *launches += 2;
  }
  return cudaSuccess;
}

}  // namespace ltv
