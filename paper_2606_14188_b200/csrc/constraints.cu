// ltv_scan_constraint_tightening: the constraint-tightening margins of eq.(12d),
//     sigma_k[i] = sum_{j<k} || c_{k,i}^T Phi(k,j) E_j ||_2,   E_j = diag(w_j),   c_{k,i}^T = Hc[k,i,:],
// WITHOUT forming or re-reading Phi: Psi(k,j) = Hc_k Phi(k,j) (nc x n) obeys Psi(k,k) = Hc_k,
// Psi(k,j) = Psi(k,j+1) A_j, so one backward sweep over j carries the stack of all rows with k > j,
//     X_j = [Psi(T-1,j); Psi(T-2,j); ...; Psi(j+1,j)] = [X_{j+1}; Hc_{j+1}] A_j        ((T-1-j) nc rows),
// as one batched GEMM per step (the MODE 1 tcgen05 3xTF32 kernel of phi_tc.cu; fp32 FMA for n < 96) that reads A_j
// once, followed by a row-norm kernel that adds ||row E_j||_2 to sigma.  It is the adjoint recursion of eq.(10) run
// for every constraint row of every step at once: 2 n^2 nc (T-1-j) flop per step instead of the n^3 of Phi.
// Two ping-pong stacks; Hc_k is placed beforehand at its slot in the stack that is the left operand of step k-1
// (no later GEMM writes that slot before it is read, because ragged tiles are stored row-masked).
#include <cuda.h>

#include "ltv_internal.h"
#include "phi_kernels.h"

namespace ltv {

namespace {

// X[(k-1)&1][b][(T-1-k) nc + i][:] = Hc[b][k][i][:], k = 1..T-1;  sigma[b][:][:] = 0.   grid (T, batch)
__global__ void __launch_bounds__(256) constraint_prefill_kernel(const float* __restrict__ Hc, float* __restrict__ X0,
                                                                 float* __restrict__ X1, float* __restrict__ sigma,
                                                                 int T, int n, int nc, int rmax) {
  const int k = blockIdx.x, b = blockIdx.y;
  for (int i = threadIdx.x; i < nc; i += 256) sigma[(static_cast<size_t>(b) * T + k) * nc + i] = 0.f;
  if (k == 0) return;
  float* X = ((k - 1) & 1) ? X1 : X0;
  const float4* src = reinterpret_cast<const float4*>(Hc + (static_cast<size_t>(b) * T + k) * nc * n);
  float4* dst = reinterpret_cast<float4*>(X + (static_cast<size_t>(b) * rmax + static_cast<size_t>(T - 1 - k) * nc) * n);
  for (int i = threadIdx.x; i < nc * n / 4; i += 256) dst[i] = __ldg(src + i);
}

// sigma[b][k][i] += || X[b][row][:] * w_j ||_2 for the R_j rows of the stack; warp per row.  grid (ceil(R_j/8), batch)
__global__ void __launch_bounds__(256) constraint_rownorm_kernel(const float* __restrict__ X,
                                                                 const float* __restrict__ w, long long w_stride,
                                                                 float* __restrict__ sigma, int T, int n, int nc,
                                                                 int rmax, int rows) {
  const int b = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row = blockIdx.x * 8 + warp;
  if (row >= rows) return;
  const float4* x4 = reinterpret_cast<const float4*>(X + (static_cast<size_t>(b) * rmax + row) * n);
  const float4* w4 = reinterpret_cast<const float4*>(w + b * w_stride);
  float s0 = 0.f, s1 = 0.f;
  for (int k4 = lane; k4 < (n >> 2); k4 += 32) {
    const float4 x = x4[k4];
    const float4 ww = __ldg(w4 + k4);
    const float a = x.x * ww.x, c = x.y * ww.y, d = x.z * ww.z, e = x.w * ww.w;
    s0 = fmaf(a, a, fmaf(c, c, s0));
    s1 = fmaf(d, d, fmaf(e, e, s1));
  }
  float s = s0 + s1;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) {
    const int k = T - 1 - row / nc, i = row % nc;
    float* out = sigma + (static_cast<size_t>(b) * T + k) * nc + i;
    *out += sqrtf(s);   // one warp owns this entry in this launch; launches are stream-ordered: deterministic
  }
}

size_t carve(size_t floats) { return align_up(floats * sizeof(float), 256); }

}  // namespace

size_t constraint_workspace_bytes(int batch, int T, int n, int nc) {
  const size_t rmax = static_cast<size_t>(T > 1 ? T - 1 : 1) * nc;
  return 2 * carve(static_cast<size_t>(batch) * rmax * n);
}

cudaError_t launch_constraint_tightening(const ConstraintArgs& a, cudaStream_t stream, unsigned long long* launches) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int batch = a.batch, T = a.T, n = a.n, nc = a.nc;
  const int rmax = (T > 1 ? T - 1 : 1) * nc;
  float* X[2];
  X[0] = static_cast<float*>(a.workspace);
  X[1] = reinterpret_cast<float*>(static_cast<char*>(a.workspace) + carve(static_cast<size_t>(batch) * rmax * n));
  cudaError_t e;
  {
    ProfScope prof(kProfKalmanSimt, stream);
    constraint_prefill_kernel<<<dim3(T, batch), 256, 0, stream>>>(a.Hc, X[0], X[1], a.sigma_out, T, n, nc, rmax);
  }
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  ++*launches;
  if (T < 2) return cudaSuccess;

  const bool tc = phi_uses_tensor_cores(n);
  const int nch = phi_pick_nch(n);
  BatchedGemm g[2];
  alignas(64) unsigned char maps[2][1024];
  for (int q = 0; q < 2; ++q) {   // q = parity of the step: left operand X[q], output X[q ^ 1]
    g[q] = BatchedGemm{};
    g[q].L = X[q]; g[q].l_rows = static_cast<long long>(batch) * rmax; g[q].l_row0 = 0; g[q].l_row_stride = rmax;
    g[q].R = a.A; g[q].r_blocks = batch * T; g[q].r_blk_stride = T;
    g[q].D = X[q ^ 1]; g[q].d_blocks = batch; g[q].d_blk0 = 0; g[q].d_blk_stride = 1;
    g[q].count = batch; g[q].M = rmax; g[q].N = n; g[q].K = n; g[q].d_rows = rmax;
    g[q].transpose_out = 0; g[q].diag = nullptr; g[q].diag_stride = 0;
    if (tc) {
      if (phi_tc_maps_size() > sizeof(maps[q])) return cudaErrorInvalidValue;
      if ((e = bgemm_tc_make_maps(g[q], maps[q])) != cudaSuccess) return e;
    }
  }
  for (int j = T - 2; j >= 0; --j) {
    const int q = j & 1;
    const int rows = (T - 1 - j) * nc;
    g[q].M = rows;
    g[q].r_blk0 = j;
    if (tc) {
      e = launch_bgemm_tc(g[q], nch, maps[q], sms, stream);
    } else {
      ProfScope prof(kProfKalmanGemm, stream);
      e = launch_bgemm_simt(g[q], stream);
    }
    if (e != cudaSuccess) return e;
    {
      ProfScope prof(kProfKalmanSimt, stream);
      constraint_rownorm_kernel<<<dim3((rows + 7) / 8, batch), 256, 0, stream>>>(
          X[q ^ 1], a.w + static_cast<size_t>(j) * n, static_cast<long long>(T) * n, a.sigma_out, T, n, nc, rmax, rows);
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    *launches += 2;
  }
  return cudaSuccess;
}

}  // namespace ltv
