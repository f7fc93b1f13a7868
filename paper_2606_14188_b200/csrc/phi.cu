// ltv_scan_system_response_tube orchestration: level 0, ceil(log2(T-1)) combine levels, tube finalise.
// All launches go to one stream in level order; no host synchronisation.
#include <cuda.h>

#include "../../include/ltv_scan.h"
#include "ltv_internal.h"
#include "phi_geom.cuh"
#include "phi_kernels.h"

namespace ltv {

bool phi_uses_tensor_cores(int n) { return n >= 96 && env_int("PHI_SIMT", 0) == 0; }

// n-tile width: the multiple of 32 in [64, 160] with the least padding, ties to the wider tile
// (2 * NT accumulator columns + 192 columns of L-operand ring must fit the 512 TMEM columns)
static int pick_nch(int n) {
  int forced = env_int("PHI_NCH", 0);
  if (forced >= 2 && forced <= 5) return forced;
  int best = 2;
  long long best_pad = -1;
  for (int nch = 2; nch <= 5; ++nch) {
    const int nt = 32 * nch;
    const long long padded = static_cast<long long>((n + nt - 1) / nt) * nt;
    if (best_pad < 0 || padded <= best_pad) {
      best_pad = padded;
      best = nch;
    }
  }
  return best;
}

int phi_pick_nch(int n) { return pick_nch(n); }

int phi_tile_n(int n, int nc) { return phi_uses_tensor_cores(n) ? 32 * pick_nch(nc) : 64; }

// bytes of the tube partials `part` (the first region of the Phi workspace)
size_t phi_part_bytes(int batch, int T, int n, int nc) {
  const int tn = phi_tile_n(n, nc);
  const size_t NT = (nc + tn - 1) / tn;
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
  size_t bytes = static_cast<size_t>(batch) * P * NT * n * sizeof(float);
  if (bytes == 0) bytes = 16;
  return align_up(bytes, 256);
}

// observer with p > 8 (nc - n > 8): a second region holds the gains transposed, Lt^T [batch,T,nc-n,n]
size_t phi_workspace_bytes(int batch, int T, int n, int nc) {
  size_t bytes = phi_part_bytes(batch, T, n, nc);
  if (nc - n > 8) bytes += align_up(static_cast<size_t>(batch) * T * (nc - n) * n * sizeof(float), 256);
  return bytes;
}

// ------------------------------------------------------------------------------------------ block re-ordering
// COLUMN_PACKED -> ROW_PACKED (block (t,s) at t(t-1)/2 + s) or SQUARE_GRID (block (t,s) at t T + s of a T x T grid; blocks
// with s >= t are not touched).  Blocks are contiguous n x n matrices in every layout, so this is a streaming copy of
// whole blocks: unit = (block, 32 KB chunk), 128-bit loads / stores, read-once / write-once cache hints.
namespace {
constexpr int kRelayoutVecs = 2048;   // float4 per unit
__global__ void __launch_bounds__(256) phi_relayout_kernel(const float4* __restrict__ src, float4* __restrict__ dst,
                                                           int batch, int T, long long vecs_per_block, int layout) {
  const int P = T * (T - 1) / 2;
  const long long cpb = (vecs_per_block + kRelayoutVecs - 1) / kRelayoutVecs;   // chunks per block
  const long long nunits = static_cast<long long>(batch) * P * cpb;
  for (long long un = blockIdx.x; un < nunits; un += gridDim.x) {
    const long long blk = un / cpb;
    const long long ch = un - blk * cpb;
    const int b = static_cast<int>(blk / P);
    const int q = static_cast<int>(blk - static_cast<long long>(b) * P);
    // invert q = colbase(s) + (t - s - 1): s is the largest column with colbase(s) <= q
    int s = 0;
    while (s + 1 < T - 1 && phi_colbase(T, s + 1) <= q) ++s;
    const int t = s + 1 + (q - static_cast<int>(phi_colbase(T, s)));
    const long long dblk = (layout == LTV_PHI_ROW_PACKED)
                               ? static_cast<long long>(b) * P + static_cast<long long>(t) * (t - 1) / 2 + s
                               : (static_cast<long long>(b) * T + t) * T + s;
    const float4* sp = src + blk * vecs_per_block + ch * kRelayoutVecs;
    float4* dp = dst + dblk * vecs_per_block + ch * kRelayoutVecs;
    const long long lim = vecs_per_block - ch * kRelayoutVecs;
    const int cnt = lim < kRelayoutVecs ? static_cast<int>(lim) : kRelayoutVecs;
    float4 v[kRelayoutVecs / 256];
#pragma unroll
    for (int j = 0; j < kRelayoutVecs / 256; ++j)
      if (threadIdx.x + 256 * j < cnt) v[j] = __ldcs(sp + threadIdx.x + 256 * j);
#pragma unroll
    for (int j = 0; j < kRelayoutVecs / 256; ++j)
      if (threadIdx.x + 256 * j < cnt) __stcs(dp + threadIdx.x + 256 * j, v[j]);
  }
}
}  // namespace

size_t phi_colpacked_bytes(int batch, int T, int n, int nc) {
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
  return align_up(static_cast<size_t>(batch) * P * n * nc * sizeof(float) + 16, 256);
}

cudaError_t launch_phi_relayout(const float* src, float* dst, int batch, int T, int n, int nc, int layout, int num_sms,
                                cudaStream_t stream) {
  if (T < 2) return cudaSuccess;
  const long long vecs = static_cast<long long>(n) * nc / 4;
  const long long nunits = static_cast<long long>(batch) * (T * (T - 1) / 2) * ((vecs + kRelayoutVecs - 1) / kRelayoutVecs);
  long long blocks = nunits < static_cast<long long>(num_sms) * 8 ? nunits : static_cast<long long>(num_sms) * 8;
  ProfScope prof(kProfPhiRelayout, stream);
  phi_relayout_kernel<<<static_cast<unsigned>(blocks), 256, 0, stream>>>(reinterpret_cast<const float4*>(src),
                                                                        reinterpret_cast<float4*>(dst), batch, T, vecs, layout);
  return cudaGetLastError();
}

cudaError_t launch_phi_tube(const PhiArgs& a, cudaStream_t stream, unsigned long long* launches) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int tn = phi_tile_n(a.n, a.nc);
  const int NT = (a.nc + tn - 1) / tn;
  cudaError_t e;
  const int NS = a.T - 1;
  if (NS >= 1) {
    e = a.Lt ? launch_phi_obs_level0(a, NT, sms, stream) : launch_phi_level0(a, NT, sms, stream);
    if (e != cudaSuccess) return e;
    *launches += (a.Lt && a.p > 8) ? 2 : 1;   // the observer's level 0 is two kernels beyond the fused p <= 8 path
    const bool tc = phi_uses_tensor_cores(a.n);
    alignas(64) unsigned char maps[1024];
    if (tc && NS >= 2) {
      if (phi_tc_maps_size() > sizeof(maps)) return cudaErrorInvalidValue;
      e = phi_tc_make_maps(a, tn / 32, maps);
      if (e != cudaSuccess) return e;
    }
    for (int level = 1; (1 << (level - 1)) < NS; ++level) {
      e = tc ? launch_phi_combine_tc(a, level, tn / 32, maps, sms, stream)
             : launch_phi_combine_simt(a, level, sms, stream);
      if (e != cudaSuccess) return e;
      ++*launches;
    }
  }
  e = launch_phi_finalize(a, NT, stream);
  if (e == cudaSuccess) ++*launches;
  return e;
}

}  // namespace ltv
