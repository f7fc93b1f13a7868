// ltv_scan_operator_constraint_margins: the constraint-tightening margins of eq.(12d), BOTH terms, constraint
// rows on the stacked pair [z_k; v_k], evaluated on ASSEMBLED output-feedback operators Phi^xw, Phi^uw, Phi^xe, Phi^ue - whatever
// produced them (ltv_scan_output_feedback_assemble for a general Phibar, or the gain-defined calls):
//     sigma_0 = 0;  sigma_k[i] = sum_{j<k} || (Hx_k[i] Phi^xw(k,j) + Hu_k[i] Phi^uw(k,j)) diag(w_j) ||_2
//                             + sum_{1<=j<k} || (Hx_k[i] Phi^xe(k,j) + Hu_k[i] Phi^ue(k,j)) diag(f_{j-1}) ||_2
// One CTA per (item b, step k) walks j = 0 .. k-1 in order and keeps the nc sums of its step: deterministic, no partial
// buffers, every operator block read exactly once (HBM-bound: 4 n^2 bytes per block, 2 nc n^2 flop).  Per block the warps
// split the rows r of Phi^xw(k,j) (and of Phi^uw), a lane owns the column quads lane, lane + 32, ..: each loaded quad meets the
// nc constraint coefficients Hx_k[i][r] out of shared memory; the eight warps' partial rows are added in fixed order.
#include "ltv_internal.h"
#include "phi_geom.cuh"

namespace ltv {

namespace {

constexpr int kMgThreads = 256;
constexpr int kMgMaxNc = 8;     // constraint rows per pass (more rows: further passes over the operators)
constexpr int kMgMaxQ = 4;      // column quads per lane: n <= 512

struct MgParams {
  const float *xw, *uw, *xe, *ue, *Hx, *Hu, *w, *f;
  float* sigma;
  int T, n, m, p, nc;
};

// A WARP owns whole blocks: warp w of the CTA of (b, k) takes j = w, w + 8, .. < k, reduces all n (+ m) rows of the block into
// its own nc x n accumulators (lane = column quads lane, lane + 32, ..), takes the nc norms with shuffles and leaves one term
// per (j, i) in shared memory; a last pass adds the terms of each constraint in the order of j (deterministic).  No barrier
// and no partial buffer per block.
template <int QN>
__global__ void __launch_bounds__(kMgThreads) margins_kernel(const MgParams s, int i0 /* first constraint row of this pass */) {
  extern __shared__ float mg_sm[];
  const int T = s.T, n = s.n, m = s.m, p = s.p;
  const int nci = min(kMgMaxNc, s.nc - i0);
  const int k = T - 1 - static_cast<int>(blockIdx.x);   // long steps first
  const int b = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n4 = n >> 2;
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
  const size_t bT = static_cast<size_t>(b) * T;
  float* hx = mg_sm;                              // [kMgMaxNc][n]
  float* hu = hx + kMgMaxNc * n;                  // [kMgMaxNc][m]
  float* term = hu + kMgMaxNc * (m > 0 ? m : 1);  // [T][kMgMaxNc]
  if (k == 0) {
    if (threadIdx.x < nci) s.sigma[bT * s.nc + i0 + threadIdx.x] = 0.f;
    return;
  }
  for (int e = threadIdx.x; e < kMgMaxNc * n; e += kMgThreads) {
    const int i = e / n, c = e - i * n;
    hx[e] = i < nci ? __ldg(s.Hx + ((bT + k) * s.nc + i0 + i) * n + c) : 0.f;
  }
  for (int e = threadIdx.x; e < kMgMaxNc * m; e += kMgThreads) {
    const int i = e / m, c = e - i * m;
    hu[e] = (i < nci && s.Hu != nullptr) ? __ldg(s.Hu + ((bT + k) * s.nc + i0 + i) * m + c) : 0.f;
  }
  __syncthreads();
  const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int j = warp; j < k; j += 8) {
    const size_t blk = static_cast<size_t>(b) * P + phi_colbase(T, j) + (k - j - 1);
    // ---- w term
    float4 acc[kMgMaxNc][QN];
#pragma unroll
    for (int i = 0; i < kMgMaxNc; ++i)
#pragma unroll
      for (int q = 0; q < QN; ++q) acc[i][q] = z4;
    constexpr int RU = QN <= 2 ? 4 : 2;   // rows per pass: RU QN independent 128-bit loads in flight per lane
    for (int side = 0; side < 2; ++side) {
      const int rows = side == 0 ? n : ((s.uw != nullptr) ? m : 0);
      const float4* base = side == 0 ? reinterpret_cast<const float4*>(s.xw + blk * n * n)
                                     : reinterpret_cast<const float4*>(s.uw + blk * m * n);
      const float* h = side == 0 ? hx : hu;
      const int hstr = side == 0 ? n : m;
      for (int r0 = 0; r0 < rows; r0 += RU) {
        float4 v[RU][QN];
#pragma unroll
        for (int u = 0; u < RU; ++u)
#pragma unroll
          for (int q = 0; q < QN; ++q)
            v[u][q] = (r0 + u < rows && lane + 32 * q < n4) ? __ldcs(base + static_cast<size_t>(r0 + u) * n4 + lane + 32 * q) : z4;
#pragma unroll
        for (int u = 0; u < RU; ++u) {
          const int r = min(r0 + u, rows - 1);   // beyond the block v is zero: any coefficient will do
#pragma unroll
          for (int i = 0; i < kMgMaxNc; ++i) {
            const float hc = h[i * hstr + r];
#pragma unroll
            for (int q = 0; q < QN; ++q) {
              acc[i][q].x = fmaf(hc, v[u][q].x, acc[i][q].x); acc[i][q].y = fmaf(hc, v[u][q].y, acc[i][q].y);
              acc[i][q].z = fmaf(hc, v[u][q].z, acc[i][q].z); acc[i][q].w = fmaf(hc, v[u][q].w, acc[i][q].w);
            }
          }
        }
      }
    }
    float ss[kMgMaxNc];
    {
      const float4* wj = reinterpret_cast<const float4*>(s.w + (bT + j) * n);
      float4 wq[QN];
#pragma unroll
      for (int q = 0; q < QN; ++q) wq[q] = (lane + 32 * q < n4) ? __ldg(wj + lane + 32 * q) : z4;
#pragma unroll
      for (int i = 0; i < kMgMaxNc; ++i) {
        float t = 0.f;
#pragma unroll
        for (int q = 0; q < QN; ++q) {
          const float e0 = acc[i][q].x * wq[q].x, e1 = acc[i][q].y * wq[q].y, e2 = acc[i][q].z * wq[q].z, e3 = acc[i][q].w * wq[q].w;
          t = fmaf(e0, e0, fmaf(e1, e1, fmaf(e2, e2, fmaf(e3, e3, t))));
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        ss[i] = sqrtf(t);
      }
    }
    // ---- e term (j >= 1): (Hx Phi^xe + Hu Phi^ue)(k,j), nc x p; lanes split the rows, one measurement column at a time
    if (j >= 1 && s.xe != nullptr) {
      float se[kMgMaxNc];
#pragma unroll
      for (int i = 0; i < kMgMaxNc; ++i) se[i] = 0.f;
      const float* xe = s.xe + blk * n * p;
      const float* ue = s.ue != nullptr ? s.ue + blk * m * p : nullptr;
      for (int q = 0; q < p; ++q) {
        float a[kMgMaxNc];
#pragma unroll
        for (int i = 0; i < kMgMaxNc; ++i) a[i] = 0.f;
        for (int r = lane; r < n; r += 32) {
          const float x = __ldg(xe + static_cast<size_t>(r) * p + q);
#pragma unroll
          for (int i = 0; i < kMgMaxNc; ++i) a[i] = fmaf(hx[i * n + r], x, a[i]);
        }
        if (ue != nullptr) {
          for (int r = lane; r < m; r += 32) {
            const float x = __ldg(ue + static_cast<size_t>(r) * p + q);
#pragma unroll
            for (int i = 0; i < kMgMaxNc; ++i) a[i] = fmaf(hu[i * m + r], x, a[i]);
          }
        }
        const float fq = __ldg(s.f + (bT + j - 1) * p + q);
#pragma unroll
        for (int i = 0; i < kMgMaxNc; ++i) {
          float t = a[i];
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
          t *= fq;
          se[i] = fmaf(t, t, se[i]);
        }
      }
#pragma unroll
      for (int i = 0; i < kMgMaxNc; ++i) ss[i] += sqrtf(se[i]);
    }
#pragma unroll
    for (int i = 0; i < kMgMaxNc; ++i)
      if (lane == i) term[j * kMgMaxNc + i] = ss[i];
  }
  __syncthreads();
  if (threadIdx.x < nci) {
    float acc = 0.f;
    for (int j = 0; j < k; ++j) acc += term[j * kMgMaxNc + threadIdx.x];
    s.sigma[(bT + k) * s.nc + i0 + threadIdx.x] = acc;
  }
}

size_t mg_smem(int n, int m, int T) {
  return (static_cast<size_t>(kMgMaxNc) * n + kMgMaxNc * (m > 0 ? m : 1) + static_cast<size_t>(T) * kMgMaxNc) * sizeof(float);
}

template <int QN>
cudaError_t launch_mg(const MgParams& s, int batch, size_t smem, cudaStream_t stream) {
  cudaError_t e = cudaFuncSetAttribute(margins_kernel<QN>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
  if (e != cudaSuccess) return e;
  for (int i0 = 0; i0 < s.nc; i0 += kMgMaxNc) {
    ProfScope prof(kProfOfbSupport, stream);
    margins_kernel<QN><<<dim3(s.T, batch), kMgThreads, smem, stream>>>(s, i0);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace

bool margins_supported(int n, int m, int T) { return n <= 32 * 4 * kMgMaxQ && mg_smem(n, m, T) <= 200u * 1024u; }

cudaError_t launch_operator_margins(const MarginArgs& a, cudaStream_t stream, unsigned long long* launches) {
  MgParams s{a.phi_xw, a.phi_uw, a.phi_xe, a.phi_ue, a.Hx, a.Hu, a.w, a.f, a.sigma, a.T, a.n, a.m, a.p, a.nc};
  const size_t smem = mg_smem(a.n, a.m, a.T);
  const int qn = (a.n / 4 + 31) / 32;
  cudaError_t e;
  switch (qn) {
    case 1: e = launch_mg<1>(s, a.batch, smem, stream); break;
    case 2: e = launch_mg<2>(s, a.batch, smem, stream); break;
    case 3: e = launch_mg<3>(s, a.batch, smem, stream); break;
    default: e = launch_mg<4>(s, a.batch, smem, stream); break;
  }
  if (e == cudaSuccess) *launches += (a.nc + kMgMaxNc - 1) / kMgMaxNc;
  return e;
}

}  // namespace ltv
