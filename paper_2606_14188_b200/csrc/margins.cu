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
#include "ptx.cuh"

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
// The rows of a block reach the warp through its own two-stage cp.async ring in shared memory (rb rows per stage): with the
// rows loaded straight into registers a warp had 6 quads in flight and the SM 16 warps at most (96 accumulator registers) -
// 34 % of the HBM copy peak; the ring keeps 2 rb rows per warp in flight whatever the register count.  NCT = accumulator rows
// (2, 4, 6 or 8 >= the constraint rows of the pass).
template <int QN, int NCT>
__global__ void __launch_bounds__(kMgThreads) margins_kernel(const MgParams s, int i0 /* first constraint row of this pass */, int rb) {
  extern __shared__ __align__(16) float mg_sm[];
  const int T = s.T, n = s.n, m = s.m, p = s.p;
  const int nci = min(NCT, s.nc - i0);
  const int k = T - 1 - static_cast<int>(blockIdx.x);   // long steps first
  const int b = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n4 = n >> 2;
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
  const size_t bT = static_cast<size_t>(b) * T;
  float* hx = mg_sm;                              // [kMgMaxNc][n]
  float* hu = hx + kMgMaxNc * n;                  // [kMgMaxNc][m]
  float* term = hu + kMgMaxNc * (m > 0 ? ((m + 3) & ~3) : 4);  // [T][kMgMaxNc]
  float4* ring = reinterpret_cast<float4*>(term + static_cast<size_t>(T) * kMgMaxNc) + static_cast<size_t>(warp) * 2 * rb * n4;
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
    float4 acc[NCT][QN];
#pragma unroll
    for (int i = 0; i < NCT; ++i)
#pragma unroll
      for (int q = 0; q < QN; ++q) acc[i][q] = z4;
    const float4* xwb = reinterpret_cast<const float4*>(s.xw + blk * n * n);
    const float4* uwb = s.uw != nullptr ? reinterpret_cast<const float4*>(s.uw + blk * m * n) : nullptr;
    const int nch0 = (n + rb - 1) / rb, nch = nch0 + (uwb != nullptr ? (m + rb - 1) / rb : 0);
    // chunk ch = rb consecutive rows (contiguous in memory) of Phi^xw(k,j), then of Phi^uw(k,j)
    auto prefetch = [&](int ch, int stage) {
      if (ch < nch) {
        const bool u_side = ch >= nch0;
        const int r0 = (u_side ? ch - nch0 : ch) * rb;
        const int cnt = min(rb, (u_side ? m : n) - r0) * n4;
        const float4* src = (u_side ? uwb : xwb) + static_cast<size_t>(r0) * n4;
        float4* dst = ring + static_cast<size_t>(stage) * rb * n4;
        for (int c = lane; c < cnt; c += 32) cp_async16(dst + c, src + c);
      }
      cp_async_commit();
    };
    prefetch(0, 0);
    for (int ch = 0; ch < nch; ++ch) {
      prefetch(ch + 1, (ch + 1) & 1);
      cp_async_wait<1>();
      __syncwarp();
      const bool u_side = ch >= nch0;
      const int r0 = (u_side ? ch - nch0 : ch) * rb;
      const int rows = min(rb, (u_side ? m : n) - r0);
      const float* h = u_side ? hu : hx;
      const int hstr = u_side ? m : n;
      const float4* st = ring + static_cast<size_t>(ch & 1) * rb * n4;
      for (int u = 0; u < rows; ++u) {
        float4 v[QN];
#pragma unroll
        for (int q = 0; q < QN; ++q) v[q] = (lane + 32 * q < n4) ? st[u * n4 + lane + 32 * q] : z4;
#pragma unroll
        for (int i = 0; i < NCT; ++i) {
          const float hc = h[i * hstr + r0 + u];
#pragma unroll
          for (int q = 0; q < QN; ++q) {
            acc[i][q].x = fmaf(hc, v[q].x, acc[i][q].x); acc[i][q].y = fmaf(hc, v[q].y, acc[i][q].y);
            acc[i][q].z = fmaf(hc, v[q].z, acc[i][q].z); acc[i][q].w = fmaf(hc, v[q].w, acc[i][q].w);
          }
        }
      }
      __syncwarp();   // every lane is done with this stage before the prefetch of the next iteration refills it
    }
    float ss[NCT];
    {
      const float4* wj = reinterpret_cast<const float4*>(s.w + (bT + j) * n);
      float4 wq[QN];
#pragma unroll
      for (int q = 0; q < QN; ++q) wq[q] = (lane + 32 * q < n4) ? __ldg(wj + lane + 32 * q) : z4;
#pragma unroll
      for (int i = 0; i < NCT; ++i) {
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
      float se[NCT];
#pragma unroll
      for (int i = 0; i < NCT; ++i) se[i] = 0.f;
      const float* xe = s.xe + blk * n * p;
      const float* ue = s.ue != nullptr ? s.ue + blk * m * p : nullptr;
      for (int q = 0; q < p; ++q) {
        float a[NCT];
#pragma unroll
        for (int i = 0; i < NCT; ++i) a[i] = 0.f;
        for (int r = lane; r < n; r += 32) {
          const float x = __ldg(xe + static_cast<size_t>(r) * p + q);
#pragma unroll
          for (int i = 0; i < NCT; ++i) a[i] = fmaf(hx[i * n + r], x, a[i]);
        }
        if (ue != nullptr) {
          for (int r = lane; r < m; r += 32) {
            const float x = __ldg(ue + static_cast<size_t>(r) * p + q);
#pragma unroll
            for (int i = 0; i < NCT; ++i) a[i] = fmaf(hu[i * m + r], x, a[i]);
          }
        }
        const float fq = __ldg(s.f + (bT + j - 1) * p + q);
#pragma unroll
        for (int i = 0; i < NCT; ++i) {
          float t = a[i];
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
          t *= fq;
          se[i] = fmaf(t, t, se[i]);
        }
      }
#pragma unroll
      for (int i = 0; i < NCT; ++i) ss[i] += sqrtf(se[i]);
    }
#pragma unroll
    for (int i = 0; i < NCT; ++i)
      if (lane == i) term[j * kMgMaxNc + i] = ss[i];
  }
  __syncthreads();
  if (threadIdx.x < nci) {
    float acc = 0.f;
    for (int j = 0; j < k; ++j) acc += term[j * kMgMaxNc + threadIdx.x];
    s.sigma[(bT + k) * s.nc + i0 + threadIdx.x] = acc;
  }
}

size_t mg_smem(int n, int m, int T, int rb) {
  return (static_cast<size_t>(kMgMaxNc) * n + kMgMaxNc * (m > 0 ? ((m + 3) & ~3) : 4) + static_cast<size_t>(T) * kMgMaxNc +
          static_cast<size_t>(kMgThreads / 32) * 2 * rb * n) * sizeof(float);
}

// rows per ring stage: 4 while two CTAs still share an SM, else 2
int mg_rows_per_stage(int n, int m, int T) { return mg_smem(n, m, T, 4) <= 100u * 1024u ? 4 : 2; }

template <int QN, int NCT>
cudaError_t launch_mg(const MgParams& s, int batch, size_t smem, int rb, cudaStream_t stream) {
  cudaError_t e = cudaFuncSetAttribute(margins_kernel<QN, NCT>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
  if (e != cudaSuccess) return e;
  for (int i0 = 0; i0 < s.nc; i0 += NCT) {
    ProfScope prof(kProfOfbSupport, stream);
    margins_kernel<QN, NCT><<<dim3(s.T, batch), kMgThreads, smem, stream>>>(s, i0, rb);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  return cudaSuccess;
}

template <int QN>
cudaError_t launch_mg_nc(const MgParams& s, int batch, size_t smem, int rb, cudaStream_t stream, int* passes) {
  // accumulator rows: the smallest of 2, 4, 6, 8 that holds the constraint rows (more than 8: passes of 8)
  const int nct = s.nc >= 7 ? 8 : s.nc >= 5 ? 6 : s.nc >= 3 ? 4 : 2;
  *passes = (s.nc + nct - 1) / nct;
  switch (nct) {
    case 2: return launch_mg<QN, 2>(s, batch, smem, rb, stream);
    case 4: return launch_mg<QN, 4>(s, batch, smem, rb, stream);
    case 6: return launch_mg<QN, 6>(s, batch, smem, rb, stream);
    default: return launch_mg<QN, 8>(s, batch, smem, rb, stream);
  }
}

}  // namespace

bool margins_supported(int n, int m, int T) { return n <= 32 * 4 * kMgMaxQ && mg_smem(n, m, T, 2) <= 200u * 1024u; }

cudaError_t launch_operator_margins(const MarginArgs& a, cudaStream_t stream, unsigned long long* launches) {
  MgParams s{a.phi_xw, a.phi_uw, a.phi_xe, a.phi_ue, a.Hx, a.Hu, a.w, a.f, a.sigma, a.T, a.n, a.m, a.p, a.nc};
  const int rb = mg_rows_per_stage(a.n, a.m, a.T);
  const size_t smem = mg_smem(a.n, a.m, a.T, rb);
  const int qn = (a.n / 4 + 31) / 32;
  int passes = 0;
  cudaError_t e;
  switch (qn) {
    case 1: e = launch_mg_nc<1>(s, a.batch, smem, rb, stream, &passes); break;
    case 2: e = launch_mg_nc<2>(s, a.batch, smem, rb, stream, &passes); break;
    case 3: e = launch_mg_nc<3>(s, a.batch, smem, rb, stream, &passes); break;
    default: e = launch_mg_nc<4>(s, a.batch, smem, rb, stream, &passes); break;
  }
  if (e == cudaSuccess) *launches += passes;
  return e;
}

}  // namespace ltv
