// Riccati prefix scan of PAPER.md:166-177 on the device, for the small-n / small-batch regime the paper runs it in
// (one problem, tens of states): Pi_j of eq.(13) as the P~ part of  e_{j-1} (x) ... (x) e_0 (x) e_init  with the
// elements (17)
//     e_i = (A~ = A_i^T,  D~ = C_i^T (F_i F_i^T)^{-1} C_i,  P~ = E_i E_i^T),      e_init = (0, 0, Xi Xi^T),
// and the combination rule (16) in the re-derived form of DESIGN.md q14, for x = (A1, D1, P1) newer, y = (A2, D2, P2):
//     G = I + D1 P2;   X = G^{-1} [A1 | D1]   (Gauss-Jordan with partial pivoting on [G | A1 | D1] in shared memory)
//     A = A2 X_A;      D = A2 X_D A2^T + D2;      P = A1^T P2 X_A + P1.
// Schedule: Sklansky prefix scan over the T + 1 elements x[0] = e_init, x[t] = e_{t-1}: at level l every aligned
// segment of 2^l elements combines each x[t] of its upper half with x[mid - 1], the finished aggregate of its lower
// half; ceil(log2(T + 1)) launches, one CTA per combination, in place (x[mid - 1] is not written at that level).
// Segment 0 always combines with a complete prefix (A2 = D2 = 0): only P is formed there.
// The P~ parts live in Pi_out ([batch][T+1][n][n]: element t at block t), the A~, D~ parts in the workspace.
// n <= 64 (nine n x (n+1) fp32 matrices in shared memory); everything else takes the recursion (kalman.cu), which does
// ~10x fewer flops and wins whenever one time step already fills the machine.
#include <cuda.h>

#include "ltv_internal.h"

namespace ltv {

namespace {

constexpr int kRicThreads = 256;
constexpr int kRicMaxN = 64;

struct RicParams {
  const float *A, *C, *e, *f, *Pi0;
  float* AD;   // [batch][T+1][2][n][n]  A~ and D~ of every element
  float* Pi;   // [batch][T+1][n][n]     P~ of every element (Pi_out)
  int batch, T, n, p;
};

// x[0] = (0, 0, Pi0);  x[t] = (A_{t-1}^T, C^T diag(f)^{-2} C, diag(e)^2).   grid (T + 1, batch)
__global__ void __launch_bounds__(kRicThreads) riccati_elements_kernel(const RicParams q) {
  const int t = blockIdx.x, b = blockIdx.y, n = q.n, p = q.p, T = q.T;
  float* At = q.AD + ((static_cast<size_t>(b) * (T + 1) + t) * 2) * n * n;
  float* Dt = At + static_cast<size_t>(n) * n;
  float* Pt = q.Pi + (static_cast<size_t>(b) * (T + 1) + t) * n * n;
  if (t == 0) {
    const float* P0 = q.Pi0 + static_cast<size_t>(b) * n * n;
    for (int i = threadIdx.x; i < n * n; i += kRicThreads) {
      At[i] = 0.f;
      Dt[i] = 0.f;
      Pt[i] = P0[i];
    }
    return;
  }
  const size_t bt = static_cast<size_t>(b) * T + (t - 1);
  const float* A = q.A + bt * n * n;
  const float* C = q.C + bt * p * n;
  const float* e = q.e + bt * n;
  const float* f = q.f + bt * p;
  for (int i = threadIdx.x; i < n * n; i += kRicThreads) {
    const int r = i / n, c = i % n;
    At[i] = A[static_cast<size_t>(c) * n + r];
    float d = 0.f;
    for (int k = 0; k < p; ++k) {
      const float fk = f[k];
      d = fmaf(C[k * n + r] / (fk * fk), C[k * n + c], d);
    }
    Dt[i] = d;
    const float ee = e[r];
    Pt[i] = (r == c) ? ee * ee : 0.f;
  }
}

// Out = op(X) op(Y) (+ Add): n x n, leading dimension ld, all in shared memory; 16 x 16 threads, 4 x 4 outputs each.
// Out must not alias X or Y; it may alias Add (every thread reads and writes only its own entries of it).
template <bool TX, bool TY>
__device__ __forceinline__ void smem_gemm(float* Out, int ldo, const float* X, int ldx, const float* Y, int ldy,
                                          const float* Add, int lda, int n) {
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  float acc[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int c = 0; c < 4; ++c) acc[a][c] = 0.f;
  // rows / columns beyond n are clamped to n - 1 (computed, never stored): no predicates inside the k loop
  const float* xp[4];
  const float* yp[4];
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    const int i = min(ty + 16 * a, n - 1);
    xp[a] = TX ? X + i : X + i * ldx;
  }
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const int j = min(tx + 16 * c, n - 1);
    yp[c] = TY ? Y + j * ldy : Y + j;
  }
  const int sx = TX ? ldx : 1, sy = TY ? 1 : ldy;
#pragma unroll 4
  for (int k = 0; k < n; ++k) {
    float xv[4], yv[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) xv[a] = xp[a][k * sx];
#pragma unroll
    for (int c = 0; c < 4; ++c) yv[c] = yp[c][k * sy];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int c = 0; c < 4; ++c) acc[a][c] = fmaf(xv[a], yv[c], acc[a][c]);
  }
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int i = ty + 16 * a, j = tx + 16 * c;
      if (i < n && j < n) Out[i * ldo + j] = acc[a][c] + (Add ? Add[i * lda + j] : 0.f);
    }
}

__device__ __forceinline__ void load_mat(float* dst, const float* __restrict__ src, int n, int ld) {
  for (int i = threadIdx.x; i < n * n; i += kRicThreads) dst[(i / n) * ld + (i % n)] = src[i];
}
__device__ __forceinline__ void store_mat(float* __restrict__ dst, const float* src, int n, int ld) {
  for (int i = threadIdx.x; i < n * n; i += kRicThreads) dst[i] = src[(i / n) * ld + (i % n)];
}

// One combination x[t] <- x[t] (x) x[mid - 1] per CTA (the Sklansky level is `level`); grid (T + 1, batch): CTAs whose
// element sits in the lower half of its segment exit at once.
__global__ void __launch_bounds__(kRicThreads, 1) riccati_combine_kernel(const RicParams q, int level) {
  extern __shared__ float sm[];
  __shared__ int s_piv;
  __shared__ float s_fac[kRicMaxN];
  const int n = q.n, T = q.T, t = blockIdx.x, b = blockIdx.y;
  const int S = 1 << level, H = S >> 1;
  if ((t & (S - 1)) < H) return;
  const int seg = t >> level, mid = seg * S + H;
  const bool full = seg != 0;   // segment 0: y = x[mid - 1] is a complete prefix (A2 = D2 = 0), only P is needed
  const int ld = n + 1, ldw = 3 * n + 1;
  float* W = sm;                       // [n][3n+1]: G | A1 | D1, reduced in place to  . | G^-1 A1 | G^-1 D1
  float* A1 = W + n * ldw;             // five n x (n+1) matrices and one temporary
  float* P1 = A1 + n * ld;
  float* A2 = P1 + n * ld;
  float* D2 = A2 + n * ld;
  float* P2 = D2 + n * ld;
  float* Tm = P2 + n * ld;
  const size_t nn = static_cast<size_t>(n) * n;
  float* gx = q.AD + ((static_cast<size_t>(b) * (T + 1) + t) * 2) * nn;
  const float* gy = q.AD + ((static_cast<size_t>(b) * (T + 1) + (mid - 1)) * 2) * nn;
  float* gPx = q.Pi + (static_cast<size_t>(b) * (T + 1) + t) * nn;
  const float* gPy = q.Pi + (static_cast<size_t>(b) * (T + 1) + (mid - 1)) * nn;
  const int tid = threadIdx.x;

  load_mat(A1, gx, n, ld);
  load_mat(W + n, gx, n, ldw);
  load_mat(W + 2 * n, gx + nn, n, ldw);
  load_mat(P1, gPx, n, ld);
  load_mat(P2, gPy, n, ld);
  if (full) {
    load_mat(A2, gy, n, ld);
    load_mat(D2, gy + nn, n, ld);
  }
  __syncthreads();
  smem_gemm<false, false>(W, ldw, W + 2 * n, ldw, P2, ld, nullptr, 0, n);   // D1 P2
  __syncthreads();
  for (int i = tid; i < n; i += kRicThreads) W[i * ldw + i] += 1.f;
  __syncthreads();

  // Gauss-Jordan with partial pivoting on [G | A1 | (D1)]
  const int ncols = full ? 3 * n : 2 * n;
  for (int k = 0; k < n; ++k) {
    if (tid < 32) {
      float best = -1.f;
      int bi = k;
      for (int r = k + tid; r < n; r += 32) {
        const float v = fabsf(W[r * ldw + k]);
        if (v > best) { best = v; bi = r; }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(0xffffffffu, best, o);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
      }
      if (tid == 0) s_piv = bi;
    }
    __syncthreads();
    const int piv = s_piv;
    if (piv != k) {
      for (int c = k + tid; c < ncols; c += kRicThreads) {
        const float u = W[k * ldw + c];
        W[k * ldw + c] = W[piv * ldw + c];
        W[piv * ldw + c] = u;
      }
    }
    __syncthreads();
    if (tid < n) s_fac[tid] = (tid == k) ? 0.f : W[tid * ldw + k] / W[k * ldw + k];
    __syncthreads();
    // thread = (column slot, half of the rows); eight rows per pass with all loads issued before the first store (the
    // compiler cannot prove that W and s_fac do not alias, so a plain loop serialises on every store)
    {
      const int half = tid >> 7, r0 = half ? (n >> 1) : 0, r1 = half ? n : (n >> 1);
      for (int c = k + 1 + (tid & 127); c < ncols; c += 128) {
        const float wkc = W[k * ldw + c];
        int i0 = r0;
        for (; i0 + 8 <= r1; i0 += 8) {
          float fac[8], wv[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            fac[u] = s_fac[i0 + u];
            wv[u] = W[(i0 + u) * ldw + c];
          }
#pragma unroll
          for (int u = 0; u < 8; ++u)
            if (i0 + u != k) W[(i0 + u) * ldw + c] = fmaf(-fac[u], wkc, wv[u]);   // row k is read by the other half: leave it alone
        }
        for (; i0 < r1; ++i0)
          if (i0 != k) W[i0 * ldw + c] = fmaf(-s_fac[i0], wkc, W[i0 * ldw + c]);
      }
    }
    __syncthreads();
  }
  for (int i = tid; i < n * (ncols - n); i += kRicThreads) {
    const int r = i / (ncols - n), c = n + i % (ncols - n);
    W[r * ldw + c] /= W[r * ldw + r];
  }
  __syncthreads();
  const float* XA = W + n;
  const float* XD = W + 2 * n;

  smem_gemm<false, false>(Tm, ld, P2, ld, XA, ldw, nullptr, 0, n);   // P2 X_A
  __syncthreads();
  smem_gemm<true, false>(P1, ld, A1, ld, Tm, ld, P1, ld, n);         // P = A1^T (P2 X_A) + P1
  __syncthreads();
  store_mat(gPx, P1, n, ld);
  if (!full) return;
  smem_gemm<false, false>(Tm, ld, A2, ld, XA, ldw, nullptr, 0, n);   // A = A2 X_A
  __syncthreads();
  store_mat(gx, Tm, n, ld);
  __syncthreads();
  smem_gemm<false, false>(Tm, ld, A2, ld, XD, ldw, nullptr, 0, n);   // A2 X_D
  __syncthreads();
  smem_gemm<false, true>(D2, ld, Tm, ld, A2, ld, D2, ld, n);         // D = (A2 X_D) A2^T + D2
  __syncthreads();
  store_mat(gx + nn, D2, n, ld);
}

}  // namespace

bool riccati_scan_supported(int n) { return n <= kRicMaxN; }

size_t riccati_scan_workspace_bytes(int batch, int T, int n) {
  return align_up(static_cast<size_t>(batch) * (T + 1) * 2 * n * n * sizeof(float), 256);
}

// fills Pi_out[b][0..T] (Pi_0 .. Pi_T); `AD` = workspace of riccati_scan_workspace_bytes
cudaError_t launch_riccati_scan(const KalmanArgs& a, float* AD, cudaStream_t stream, unsigned long long* launches) {
  RicParams q{a.A, a.C, a.e, a.f, a.Pi0, AD, a.Pi_out, a.batch, a.T, a.n, a.p};
  const dim3 grid(a.T + 1, a.batch);
  {
    ProfScope prof(kProfKalmanSimt, stream);
    riccati_elements_kernel<<<grid, kRicThreads, 0, stream>>>(q);
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  ++*launches;
  const int n = a.n;
  const size_t smem = (static_cast<size_t>(n) * (3 * n + 1) + 6 * static_cast<size_t>(n) * (n + 1)) * sizeof(float);
  e = cudaFuncSetAttribute(riccati_combine_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
  if (e != cudaSuccess) return e;
  for (int level = 1; (1 << (level - 1)) < a.T + 1; ++level) {
    {
      ProfScope prof(kProfKalmanGemm, stream);
      riccati_combine_kernel<<<grid, kRicThreads, smem, stream>>>(q, level);
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    ++*launches;
  }
  return cudaSuccess;
}

}  // namespace ltv
