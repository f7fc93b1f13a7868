// ltv_scan_kalman_gains for SMALL systems (n <= 64; the paper's own regime of tens of states, and
// BASELINE.json configs[0]): the whole backward-Kalman recursion of eq.(13) of one item in ONE CTA,
// ONE launch for the batch.  The batched path (kalman.cu) spends five dependent, latency-bound launches per step
// (29 us per step at n = 40, batch 1); here Pi_j never leaves shared memory and a step is two n^3 products in fp32 FMA
// plus the p x p Cholesky:
//     G = C_j Pi_j,  S = F_j F_j^T + G C_j^T = L L^T,  K = S^-1 G,  Lt_j = L_{j+1}^T = -A_j K^T,  Abar_j = A_j + Lt_j C_j,
//     Y = Abar_j Pi_j,  Pi_{j+1} = A_j Y^T + diag(e_j)^2
// - the same arithmetic, in the same order, as the batched path (fp32 throughout), so the two agree to rounding.  A_{j+1} and
// C_{j+1} are fetched with cp.async while step j computes.
#include "ltv_internal.h"
#include "ptx.cuh"

namespace ltv {

namespace {

constexpr int kKsThreads = 256;
constexpr int kKsMaxN = 64;
constexpr int kKsMaxP = 32;

struct KsParams {
  const float *A, *C, *e, *f, *Pi0;
  float *Lt_out, *Pi_out;
  int T, n, p;
};

// sum_k x[k sx] y[k sy], k < n (n % 4 == 0), four interleaved partial sums added pairwise: the short dot products that feed
// the p x p innovation covariance cancel heavily when the observation noise is small, and a single running sum loses a digit
// more than the warp-tree reductions of the batched path
__device__ __forceinline__ float ks_dot(const float* x, int sx, const float* y, int sy, int n) {
  float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
  for (int k = 0; k < n; k += 4) {
    a0 = fmaf(x[k * sx], y[k * sy], a0);
    a1 = fmaf(x[(k + 1) * sx], y[(k + 1) * sy], a1);
    a2 = fmaf(x[(k + 2) * sx], y[(k + 2) * sy], a2);
    a3 = fmaf(x[(k + 3) * sx], y[(k + 3) * sy], a3);
  }
  return (a0 + a1) + (a2 + a3);
}

// D[i][c] (+)= sum_k X[i][k] * Y[k][c] for a 4 x 4 tile (rows 4 tr .., cols 4 tc ..); all matrices n x n in shared memory with
// row stride ld (odd: the strided accesses below are conflict-free).  YT: use Y[c][k] instead (D = X Y^T).
template <bool YT>
__device__ __forceinline__ void ks_tile(const float* X, const float* Y, int n, int ld, int tr, int tc, float (&acc)[4][4]) {
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = 0.f;
#pragma unroll 4
  for (int k = 0; k < n; ++k) {
    float x[4], y[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) x[a] = X[(4 * tr + a) * ld + k];
#pragma unroll
    for (int b = 0; b < 4; ++b) y[b] = YT ? Y[(4 * tc + b) * ld + k] : Y[k * ld + 4 * tc + b];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int b = 0; b < 4; ++b) acc[a][b] = fmaf(x[a], y[b], acc[a][b]);
  }
}

__global__ void __launch_bounds__(kKsThreads, 1) kalman_small_kernel(const KsParams p) {
  extern __shared__ __align__(16) float ksm[];
  const int n = p.n, T = p.T, np = p.p, ld = n + 1, ldp = np + 1;
  const int tid = threadIdx.x, b = blockIdx.x;
  float* Pi = ksm;                    // [n][ld]
  float* Ab = Pi + n * ld;            // [n][ld] closed-loop matrix
  float* Y = Ab + n * ld;             // [n][ld]
  float* Abuf = Y + n * ld;           // [2][n][ld] A_j, A_{j+1}
  float* Cbuf = Abuf + 2 * n * ld;    // [2][np][ld]
  float* G = Cbuf + 2 * np * ld;      // [np][ld]
  float* K = G + np * ld;             // [np][ld]
  float* S = K + np * ld;             // [np][ldp]
  float* Lt = S + np * ldp;           // [n][np]
  float* ev = Lt + n * np;            // [n]
  float* fv = ev + n;                 // [np]
  const float* Ag = p.A + static_cast<size_t>(b) * T * n * n;
  const float* Cg = p.C + static_cast<size_t>(b) * T * np * n;
  float* Pig = p.Pi_out + static_cast<size_t>(b) * (T + 1) * n * n;
  float* Ltg = p.Lt_out + static_cast<size_t>(b) * T * n * np;

  auto fetch = [&](int j, int buf) {   // A_j, C_j -> shared memory (4-byte cp.async: the padded rows are not 16-byte aligned)
    float* As = Abuf + buf * n * ld;
    float* Cs = Cbuf + buf * np * ld;
    const float* a = Ag + static_cast<size_t>(j) * n * n;
    const float* c = Cg + static_cast<size_t>(j) * np * n;
    for (int i = tid; i < n * n; i += kKsThreads) cp_async4(As + (i / n) * ld + i % n, a + i);
    for (int i = tid; i < np * n; i += kKsThreads) cp_async4(Cs + (i / n) * ld + i % n, c + i);
    cp_async_commit();
  };
  fetch(0, 0);
  for (int i = tid; i < n * n; i += kKsThreads) {
    const float v = __ldg(p.Pi0 + static_cast<size_t>(b) * n * n + i);
    Pi[(i / n) * ld + i % n] = v;
    Pig[i] = v;   // Pi_out[b][0] = Pi0
  }
  const int nt = n >> 2, tiles = nt * nt;
  const int tr = tid / nt, tc = tid % nt;

  for (int j = 0; j < T; ++j) {
    const float* A = Abuf + (j & 1) * n * ld;
    const float* C = Cbuf + (j & 1) * np * ld;
    if (j + 1 < T) fetch(j + 1, (j + 1) & 1);   // the buffer was last read at step j-1: every thread is past it (barriers below)
    if (tid < n) ev[tid] = __ldg(p.e + (static_cast<size_t>(b) * T + j) * n + tid);
    if (tid < np) fv[tid] = __ldg(p.f + (static_cast<size_t>(b) * T + j) * np + tid);
    if (j + 1 < T) cp_async_wait<1>(); else cp_async_wait<0>();   // this thread's copies of step j have landed ...
    __syncthreads();                                               // ... and everybody's
    // G = C Pi   (Pi symmetric: row k of Pi against column k of C)
    for (int o = tid; o < np * n; o += kKsThreads) {
      const int q = o / n, c = o - q * n;
      G[q * ld + c] = ks_dot(C + q * ld, 1, Pi + c, ld, n);
    }
    __syncthreads();
    // S = F F^T + G C^T (lower triangle is enough; filled fully)
    for (int o = tid; o < np * np; o += kKsThreads) {
      const int q = o / np, r = o - q * np;
      S[q * ldp + r] = ks_dot(G + q * ld, 1, C + r * ld, 1, n) + ((q == r) ? fv[q] * fv[q] : 0.f);
    }
    __syncthreads();
    // Cholesky S = L L^T in place (one warp, lane = row)
    if (tid < 32) {
      const int lane = tid;
      for (int k = 0; k < np; ++k) {
        if (lane == k) S[k * ldp + k] = sqrtf(S[k * ldp + k]);
        __syncwarp();
        if (lane > k && lane < np) S[lane * ldp + k] /= S[k * ldp + k];
        __syncwarp();
        if (lane > k && lane < np) {
          const float lk = S[lane * ldp + k];
          for (int c2 = k + 1; c2 <= lane; ++c2) S[lane * ldp + c2] = fmaf(-lk, S[c2 * ldp + k], S[lane * ldp + c2]);
        }
        __syncwarp();
      }
    }
    __syncthreads();
    // K = S^-1 G: thread per column, forward then backward substitution
    if (tid < n) {
      const int c = tid;
      for (int q = 0; q < np; ++q) {
        float v = G[q * ld + c];
        for (int r = 0; r < q; ++r) v = fmaf(-S[q * ldp + r], K[r * ld + c], v);
        K[q * ld + c] = v / S[q * ldp + q];
      }
      for (int q = np - 1; q >= 0; --q) {
        float v = K[q * ld + c];
        for (int r = q + 1; r < np; ++r) v = fmaf(-S[r * ldp + q], K[r * ld + c], v);
        K[q * ld + c] = v / S[q * ldp + q];
      }
    }
    __syncthreads();
    // Lt = -A K^T  [n][np]  (= L_{j+1}^T), to shared and global memory
    for (int o = tid; o < n * np; o += kKsThreads) {
      const int i = o / np, q = o - i * np;
      const float acc = ks_dot(A + i * ld, 1, K + q * ld, 1, n);
      Lt[o] = -acc;
      Ltg[static_cast<size_t>(j) * n * np + o] = -acc;
    }
    __syncthreads();
    // Abar = A + Lt C
    for (int o = tid; o < n * n; o += kKsThreads) {
      const int i = o / n, c = o - i * n;
      float acc = A[i * ld + c];
      for (int q = 0; q < np; ++q) acc = fmaf(Lt[i * np + q], C[q * ld + c], acc);
      Ab[i * ld + c] = acc;
    }
    __syncthreads();
    // Y = Abar Pi
    if (tid < tiles) {
      float acc[4][4];
      ks_tile<false>(Ab, Pi, n, ld, tr, tc, acc);
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int c2 = 0; c2 < 4; ++c2) Y[(4 * tr + a) * ld + 4 * tc + c2] = acc[a][c2];
    }
    __syncthreads();
    // Pi_{j+1} = A Y^T + diag(e)^2
    if (tid < tiles) {
      float acc[4][4];
      ks_tile<true>(A, Y, n, ld, tr, tc, acc);
      float* out = Pig + static_cast<size_t>(j + 1) * n * n;
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        const int i = 4 * tr + a;
#pragma unroll
        for (int c2 = 0; c2 < 4; ++c2) {
          const int k2 = 4 * tc + c2;
          const float v = acc[a][c2] + (i == k2 ? ev[i] * ev[i] : 0.f);
          Pi[i * ld + k2] = v;
          acc[a][c2] = v;
        }
        *reinterpret_cast<float4*>(out + static_cast<size_t>(i) * n + 4 * tc) = make_float4(acc[a][0], acc[a][1], acc[a][2], acc[a][3]);
      }
    }
    __syncthreads();
  }
}

size_t ks_smem_bytes(int n, int p) {
  const size_t ld = n + 1, ldp = p + 1;
  return (5 * n * ld + 4 * p * ld + p * ldp + static_cast<size_t>(n) * p + n + p) * sizeof(float) + 64;
}

}  // namespace

bool kalman_small_supported(int n, int p) { return n <= kKsMaxN && n >= 4 && (n & 3) == 0 && p >= 1 && p <= kKsMaxP; }

cudaError_t launch_kalman_small(const KalmanArgs& a, cudaStream_t stream, unsigned long long* launches) {
  KsParams p{a.A, a.C, a.e, a.f, a.Pi0, a.Lt_out, a.Pi_out, a.T, a.n, a.p};
  const size_t smem = ks_smem_bytes(a.n, a.p);
  cudaError_t e = cudaFuncSetAttribute(kalman_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
  if (e != cudaSuccess) return e;
  {
    ProfScope prof(kProfKalmanSimt, stream);
    kalman_small_kernel<<<a.batch, kKsThreads, smem, stream>>>(p);
  }
  e = cudaGetLastError();
  if (e == cudaSuccess) ++*launches;
  return e;
}

}  // namespace ltv
