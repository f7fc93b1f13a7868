// ltv_scan_system_response_tube_rows: the block ROWS k_lo <= k < k_hi of the system response Phi(k,j) = A_{k-1} .. A_j
// (eq.(12c)) and their tube rows r_k (eq.(12e)) - the piece of ONE item's response that one GPU
// computes when a single large item is split over several GPUs (optional).  The split is by ROWS, not by columns:
// a block row depends on nothing outside itself,
//     Phi(k,j) = Phi(k,j+1) A_j,    Phi(k,k) = I,    j = k-1 .. 0,
// so a shard needs A (replicated) and no other shard's blocks, and r_k = sum_j |Phi(k,j)| w_j is COMPLETE on the GPU that owns
// row k: no reduction across GPUs (a column split - SURVEY's sketch - needs an all-reduce of r and the left operands of other
// columns).  Same flop count as the time-parallel scan (one n^3 product per block), k_hi - 2 sequential steps: at step j all
// blocks (k, j+1) of the shard are one contiguous tall matrix in the shard's column-packed order, multiplied by A_j in ONE batched
// GEMM (tcgen05 3xTF32, MODE 1 of phi_tc.cu; fp32 FMA for n < 96) into column j; a row kernel then sets block (j+1, j) = A_j
// (if the shard owns row j+1) and adds the tube terms of column j (one owner per (k, i) and step, stream-ordered: deterministic).
#include <cuda.h>

#include <algorithm>

#include "ltv_internal.h"
#include "phi_kernels.h"

namespace ltv {

namespace {

struct RowShard {
  int T, k_lo, k_hi;
  __host__ __device__ int kmin(int j) const { return k_lo > j + 1 ? k_lo : j + 1; }
  __host__ __device__ int cnt(int j) const { const int c = k_hi - kmin(j); return c > 0 ? c : 0; }
  __host__ __device__ long long colbase(int j) const {   // blocks of the shard in columns < j
    // columns j' < k_lo - 1 hold k_hi - k_lo blocks each; columns j' >= k_lo - 1 hold k_hi - (j' + 1)
    const long long full = j < k_lo - 1 ? j : k_lo - 1;
    long long v = full * (k_hi - k_lo);
    for (int jj = k_lo - 1 > 0 ? k_lo - 1 : 0; jj < j; ++jj) v += cnt(jj);
    return v;
  }
};

// warp per row of column j of the shard: (k, i), k = kmin(j) .. k_hi-1.  k = j+1: row := A_j[i] (written); then
// r_k[i] += sum_c |row[c]| w_j[c]   (mode 1: sqrt(sum_c (row[c] w_j[c])^2)).  grid (ceil(rows / 8), batch).
__global__ void __launch_bounds__(256) phi_rows_step_kernel(const float* __restrict__ A, const float* __restrict__ w,
                                                            float* phi, float* r, RowShard sh, long long cb_j, long long Ps,
                                                            int n, int j, int mode) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row = blockIdx.x * 8 + warp;
  const int rows = sh.cnt(j) * n;
  if (row >= rows) return;
  const int b = blockIdx.y;
  const int kk = row / n, i = row - kk * n;
  const int k = sh.kmin(j) + kk;
  const int n4 = n >> 2;
  float4* prow = reinterpret_cast<float4*>(phi + ((static_cast<size_t>(b) * Ps + cb_j + kk) * n + i) * n);
  const float4* arow = (k == j + 1) ? reinterpret_cast<const float4*>(A + ((static_cast<size_t>(b) * sh.T + j) * n + i) * n) : nullptr;
  const float4* wj = reinterpret_cast<const float4*>(w + (static_cast<size_t>(b) * sh.T + j) * n);
  float* rp = r + (static_cast<size_t>(b) * sh.T + k) * n + i;
  const float r_old = lane == 0 ? *rp : 0.f;
  float acc = 0.f;
  for (int c = lane; c < n4; c += 32) {
    float4 x;
    if (arow != nullptr) {
      x = __ldg(arow + c);
      prow[c] = x;
    } else {
      x = prow[c];
    }
    const float4 ww = __ldg(wj + c);
    const float e0 = x.x * ww.x, e1 = x.y * ww.y, e2 = x.z * ww.z, e3 = x.w * ww.w;
    acc += mode ? (e0 * e0 + e1 * e1) + (e2 * e2 + e3 * e3) : (fabsf(e0) + fabsf(e1)) + (fabsf(e2) + fabsf(e3));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) *rp = r_old + (mode ? sqrtf(acc) : acc);
}

// r[b, k, :] = 0 for the rows of the shard (and row 0 if the shard starts at k = 1)
__global__ void phi_rows_zero_kernel(float* r, int T, int n, int k0, int k1) {
  const int b = blockIdx.y;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < (k1 - k0) * n; e += gridDim.x * blockDim.x)
    r[(static_cast<size_t>(b) * T + k0) * n + e] = 0.f;
}

}  // namespace

long long phi_row_shard_blocks(int T, int k_lo, int k_hi) {
  (void)T;
  long long s = 0;
  for (int k = k_lo; k < k_hi; ++k) s += k;
  return s;
}

long long phi_row_shard_index(int T, int k_lo, int k_hi, int k, int j) {
  if (T < 1 || k_lo < 1 || k_hi > T || k < k_lo || k >= k_hi || j < 0 || j >= k) return -1;
  RowShard sh{T, k_lo, k_hi};
  return sh.colbase(j) + (k - sh.kmin(j));
}

cudaError_t launch_phi_rows(const PhiRowsArgs& a, cudaStream_t stream, unsigned long long* launches) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int batch = a.batch, T = a.T, n = a.n;
  RowShard sh{T, a.k_lo, a.k_hi};
  const long long Ps = phi_row_shard_blocks(T, a.k_lo, a.k_hi);
  cudaError_t e;
  {
    const int k0 = a.k_lo == 1 ? 0 : a.k_lo;
    ProfScope prof(kProfPhiFinalize, stream);
    phi_rows_zero_kernel<<<dim3(std::max(1, std::min(64, ((a.k_hi - k0) * n + 255) / 256)), batch), 256, 0, stream>>>(a.r, T, n, k0, a.k_hi);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    ++*launches;
  }
  if (Ps == 0) return cudaSuccess;
  const bool tc = phi_uses_tensor_cores(n);
  const int nch = phi_pick_nch(n);
  BatchedGemm g{};
  alignas(64) unsigned char maps[1024];
  g.L = a.phi; g.l_rows = static_cast<long long>(batch) * Ps * n; g.l_row_stride = static_cast<int>(Ps * n);
  g.R = a.A; g.r_blocks = batch * T; g.r_blk_stride = T;
  g.D = a.phi; g.d_blocks = 1; g.d_blk0 = 0; g.d_blk_stride = 0;
  g.d_rows = static_cast<int>(static_cast<long long>(batch) * Ps * n); g.d_row_stride = static_cast<int>(Ps * n);
  g.count = batch; g.N = n; g.K = n; g.M = n;
  if (tc) {
    if (phi_tc_maps_size() > sizeof(maps)) return cudaErrorInvalidValue;
    if ((e = bgemm_tc_make_maps(g, maps)) != cudaSuccess) return e;
  }
  for (int j = a.k_hi - 2; j >= 0; --j) {
    const long long cb_j = sh.colbase(j), cb_n = sh.colbase(j + 1);
    const int cn = sh.cnt(j + 1);              // blocks of column j+1 = rows k >= max(k_lo, j+2) of the shard
    if (cn > 0) {
      g.M = cn * n;
      g.l_row0 = static_cast<int>(cb_n * n);
      g.d_row0 = static_cast<int>((cb_j + (sh.kmin(j) == j + 1 ? 1 : 0)) * n);   // behind block (j+1, j) if the shard owns it
      g.r_blk0 = j;
      if (tc) {
        e = launch_bgemm_tc(g, nch, maps, sms, stream);
      } else {
        ProfScope prof(kProfKalmanGemm, stream);
        e = launch_bgemm_simt(g, stream);
      }
      if (e != cudaSuccess) return e;
      ++*launches;
    }
    const int rows = sh.cnt(j) * n;
    if (rows > 0) {
      ProfScope prof(kProfPhiLevel0, stream);
      phi_rows_step_kernel<<<dim3((rows + 7) / 8, batch), 256, 0, stream>>>(a.A, a.w, a.phi, a.r, sh, cb_j, Ps, n, j, a.tube_mode);
      if ((e = cudaGetLastError()) != cudaSuccess) return e;
      ++*launches;
    }
  }
  return cudaSuccess;
}

}  // namespace ltv
