// ltv_scan_output_feedback_assemble: eq.(15) for a GENERAL state-feedback response Phibar = (Phibar^x,
// Phibar^u) - any block-lower-triangular operators with Phibar^x(k,k) = I, e.g. the solution of the SLS program's first stage -
// and the observer response Phihat of the gains of (13)/(14):
//     Phi^xw = Phibar^x + Phihat^x - Phibar^x M Phihat^x,   Phi^uw = Phibar^u (I - M Phihat^x),   M = I - Z A,
//     Phi^xe = Phihat^y - Phibar^x M Phihat^y,              Phi^ue = -Phibar^u M Phihat^y,
// with Phihat^x(k,j) = Abar_{k-1} .. Abar_j, Abar_j = A_j + Lt_j C_j, Phihat^y(k,j) = Phihat^x(k,j) Lt_{j-1} (DESIGN.md q20, q21).
//
// No block-triangular operator product is formed (that would be T^3/6 products of n^3).  M is block bidiagonal and Phihat^x
// obeys Phihat^x(i,j) = Phihat^x(i,j+1) Abar_j, so the assembled operators satisfy a backward recursion over the column index
// (pinned against the oracle's dense evaluation of (15): tests/test_oracle_pins_assembly.py):
//     Phi^xw(k,j) = Phi^xw(k,j+1) Abar_j - [Phibar^x(k,j+1) Lt_j] C_j,    Phi^xw(k,k) = I,
//     Phi^uw(k,j) = Phi^uw(k,j+1) Abar_j - [Phibar^u(k,j+1) Lt_j] C_j,    Phi^uw(k,k) = 0,
//     Phi^xe(k,j) = (Phi^xw - Phibar^x)(k,j) Lt_{j-1},   Phi^ue(k,j) = (Phi^uw - Phibar^u)(k,j) Lt_{j-1}    (j >= 1)
// i.e. ONE n^3 product per block - as many as the Phi scan itself - plus rank-p corrections.  In COLUMN_PACKED order all
// blocks (k, j+1), k >= j+2, are one contiguous tall matrix: step j is one batched GEMM [stack of column j+1] x Abar_j into
// column j (tcgen05 3xTF32, MODE 1 of phi_tc.cu; fp32 FMA for n < 96), then one fused row kernel that applies the rank-p
// correction, writes Phi^xe / Phi^ue and adds the two row norms of the tube (12e) - one owner per (k, i) and step,
// stream-ordered: deterministic.  T-1 steps, sequential in j, parallel over k and the batch.
#include <cuda.h>

#include "ltv_internal.h"
#include "phi_geom.cuh"
#include "phi_kernels.h"

namespace ltv {

namespace {

// Abar = A + Lt C and the gains transposed, Ltt[b,t,q,:] = Lt[b,t,:,q].  Warp per row; grid (batch T, ceil(n / 32)).
__global__ void __launch_bounds__(256) asm_prep_kernel(const float* __restrict__ A, const float* __restrict__ Lt,
                                                       const float* __restrict__ C, float* __restrict__ Abar,
                                                       float* __restrict__ Ltt, int n, int p) {
  const size_t bt = blockIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n4 = n >> 2;
  for (int i = blockIdx.y * 32 + warp; i < min(n, static_cast<int>(blockIdx.y) * 32 + 32); i += 8) {
    const float4* Ar = reinterpret_cast<const float4*>(A + (bt * n + i) * n);
    const float* Li = Lt + (bt * n + i) * p;
    if (lane < p) Ltt[(bt * p + lane) * n + i] = __ldg(Li + lane);
    const float4* C4 = reinterpret_cast<const float4*>(C + bt * p * n);
    float4* o = reinterpret_cast<float4*>(Abar + (bt * n + i) * n);
    for (int c = lane; c < n4; c += 32) {
      float4 a = __ldg(Ar + c);
      for (int q = 0; q < p; ++q) {
        const float s = __ldg(Li + q);
        const float4 c4 = __ldg(C4 + static_cast<size_t>(q) * n4 + c);
        a.x = fmaf(s, c4.x, a.x); a.y = fmaf(s, c4.y, a.y); a.z = fmaf(s, c4.z, a.z); a.w = fmaf(s, c4.w, a.w);
      }
      o[c] = a;
    }
  }
}

struct AsmStep {
  float* out;            // [batch, P, R, n] COLUMN_PACKED strictly-lower blocks of Phi^xw (R = n) or Phi^uw (R = m)
  float* oute;           // [batch, P, R, p] Phi^xe / Phi^ue, or null
  const float* pbar;     // Phibar: x: [batch, P, n, n] strictly-lower blocks (diagonal = I implied);
                         //         u: [batch, P + T, m, n] blocks 0 <= j <= k, column j has T - j blocks starting with the diagonal
  const float* A;        // [batch, T, n, n] (x side: block (j+1, j) = A_j)
  const float *Ltt, *C, *w, *f;
  float* tau;            // [batch, T, n], x side only, or null
  int T, n, p, R, is_u, j;
};

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Step j of the backward recursion for the rows of column j: warp per row (b, k, i), k = j+1 .. T-1, i < R.
//   k = j+1:  x: row = A_j[i]                                   u: row = -(Phibar^u(j+1,j+1)[i] Lt_j) C_j
//   k > j+1:  row = (GEMM result already in out) - (Phibar(k,j+1)[i] Lt_j) C_j
// then e = (row - Phibar(k,j)[i]) Lt_{j-1} (j >= 1) and, x side, tau_k[i] += ||row o w_j|| + ||e o f_{j-1}||.
// grid (ceil(rows / 8), batch), rows = (T-1-j) R.
__global__ void __launch_bounds__(256) asm_step_kernel(const AsmStep s) {
  const int T = s.T, n = s.n, p = s.p, R = s.R, j = s.j;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row = blockIdx.x * 8 + warp;
  if (row >= (T - 1 - j) * R) return;
  const int b = blockIdx.y;
  const int kk = row / R, i = row - kk * R;
  const int k = j + 1 + kk;
  const int n4 = n >> 2;
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
  const size_t bT = static_cast<size_t>(b) * T;
  // Phibar blocks (k, j+1) and (k, j)
  const float4 *pb_next = nullptr, *pb_cur;
  if (s.is_u) {
    const size_t item = static_cast<size_t>(b) * (P + T);
    auto qd = [&](int kq, int jq) { return static_cast<size_t>(jq) * T - static_cast<size_t>(jq) * (jq - 1) / 2 + (kq - jq); };
    pb_next = reinterpret_cast<const float4*>(s.pbar + ((item + qd(k, j + 1)) * R + i) * n);
    pb_cur = reinterpret_cast<const float4*>(s.pbar + ((item + qd(k, j)) * R + i) * n);
  } else {
    const size_t item = static_cast<size_t>(b) * P;
    if (kk > 0) pb_next = reinterpret_cast<const float4*>(s.pbar + ((item + phi_colbase(T, j + 1) + (k - j - 2)) * R + i) * n);
    pb_cur = reinterpret_cast<const float4*>(s.pbar + ((item + phi_colbase(T, j) + (k - j - 1)) * R + i) * n);
  }
  const size_t oblk = static_cast<size_t>(b) * P + phi_colbase(T, j) + (k - j - 1);
  float4* orow = reinterpret_cast<float4*>(s.out + (oblk * R + i) * n);
  const float4* Lj = reinterpret_cast<const float4*>(s.Ltt + (bT + j) * p * n);
  const float4* Cj = reinterpret_cast<const float4*>(s.C + (bT + j) * p * n);
  const float4* Ljm = (j >= 1) ? reinterpret_cast<const float4*>(s.Ltt + (bT + j - 1) * p * n) : nullptr;
  const float4* wj = reinterpret_cast<const float4*>(s.w + (bT + j) * n);

  // u[q] = Phibar(k,j+1)[i] . Lt_j[:,q]
  float u[32];
  if (pb_next != nullptr) {
    for (int q0 = 0; q0 < p; q0 += 8) {
      float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      for (int c = lane; c < n4; c += 32) {
        const float4 a = __ldg(pb_next + c);
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          if (q0 + q < p) {
            const float4 l = __ldg(Lj + static_cast<size_t>(q0 + q) * n4 + c);
            acc[q] = fmaf(a.x, l.x, fmaf(a.y, l.y, fmaf(a.z, l.z, fmaf(a.w, l.w, acc[q]))));
          }
        }
      }
#pragma unroll
      for (int q = 0; q < 8; ++q) u[(q0 + q) & 31] = warp_sum(acc[q]);
    }
  }
  // the row, its tube term and e = (row - Phibar(k,j)[i]) Lt_{j-1}
  float s1 = 0.f;
  float e[32];
#pragma unroll
  for (int q = 0; q < 32; ++q) e[q] = 0.f;
  for (int c = lane; c < n4; c += 32) {
    float4 x;
    if (kk == 0) {
      x = s.is_u ? make_float4(0.f, 0.f, 0.f, 0.f) : __ldg(reinterpret_cast<const float4*>(s.A + ((bT + j) * n + i) * n) + c);
    } else {
      x = orow[c];
    }
    if (pb_next != nullptr) {
      for (int q = 0; q < p; ++q) {
        const float4 cq = __ldg(Cj + static_cast<size_t>(q) * n4 + c);
        const float uq = u[q];
        x.x = fmaf(-uq, cq.x, x.x); x.y = fmaf(-uq, cq.y, x.y); x.z = fmaf(-uq, cq.z, x.z); x.w = fmaf(-uq, cq.w, x.w);
      }
    }
    orow[c] = x;
    if (!s.is_u) {
      const float4 ww = __ldg(wj + c);
      const float e0 = x.x * ww.x, e1 = x.y * ww.y, e2 = x.z * ww.z, e3 = x.w * ww.w;
      s1 = fmaf(e0, e0, fmaf(e1, e1, fmaf(e2, e2, fmaf(e3, e3, s1))));
    }
    if (Ljm != nullptr) {
      const float4 pc = __ldg(pb_cur + c);
      const float4 v = make_float4(x.x - pc.x, x.y - pc.y, x.z - pc.z, x.w - pc.w);
      for (int q = 0; q < p; ++q) {
        const float4 l = __ldg(Ljm + static_cast<size_t>(q) * n4 + c);
        e[q] = fmaf(v.x, l.x, fmaf(v.y, l.y, fmaf(v.z, l.z, fmaf(v.w, l.w, e[q]))));
      }
    }
  }
  float s2 = 0.f;
  if (Ljm != nullptr) {
    const float* fj = s.f + (bT + j - 1) * p;
    for (int q = 0; q < p; ++q) {
      const float eq = warp_sum(e[q]);
      const float t = eq * __ldg(fj + q);
      s2 = fmaf(t, t, s2);
      if (s.oute != nullptr && lane == (q & 31)) s.oute[(oblk * R + i) * p + q] = eq;
    }
  } else if (s.oute != nullptr && lane < p) {
    s.oute[(oblk * R + i) * p + lane] = 0.f;   // j = 0: no measurement noise has entered yet
  }
  if (!s.is_u && s.tau != nullptr) {
    s1 = warp_sum(s1);
    if (lane == 0) s.tau[(bT + k) * n + i] += sqrtf(s1) + sqrtf(s2);
  }
}

size_t carve(size_t floats) { return align_up(floats * sizeof(float), 256); }

}  // namespace

size_t asm_workspace_bytes(int batch, int T, int n, int p) {
  const size_t b = batch, t = T;
  return carve(b * t * n * n) + carve(b * t * p * n);
}

cudaError_t launch_ofb_assemble(const AsmArgs& a, cudaStream_t stream, unsigned long long* launches) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int batch = a.batch, T = a.T, n = a.n, m = a.m, p = a.p;
  const size_t b = batch, t = T;
  const int P = T * (T - 1) / 2;
  char* cur = static_cast<char*>(a.workspace);
  float* Abar = reinterpret_cast<float*>(cur); cur += carve(b * t * n * n);
  float* Ltt = reinterpret_cast<float*>(cur);
  cudaError_t e;
  if (a.tau != nullptr && (e = cudaMemsetAsync(a.tau, 0, b * t * n * sizeof(float), stream)) != cudaSuccess) return e;
  {
    ProfScope prof(kProfOfbSupport, stream);
    asm_prep_kernel<<<dim3(batch * T, (n + 31) / 32), 256, 0, stream>>>(a.A, a.Lt, a.C, Abar, Ltt, n, p);
  }
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  ++*launches;
  if (T < 2) return cudaSuccess;
  const bool want_u = a.phi_uw != nullptr;
  const bool tc = phi_uses_tensor_cores(n);
  const int nch = phi_pick_nch(n);
  // side 0: Phi^xw (R = n rows per block), side 1: Phi^uw (R = m).  Both GEMMs: [stack of column j+1] x Abar_j -> column j,
  // the array viewed as ONE matrix of batch P R rows; problem b starts at row b P R + (block offset) R.
  BatchedGemm g[2];
  alignas(64) unsigned char maps[2][1024];
  for (int sd = 0; sd < (want_u ? 2 : 1); ++sd) {
    const int R = sd ? m : n;
    float* arr = sd ? a.phi_uw : a.phi_xw;
    g[sd] = BatchedGemm{};
    g[sd].L = arr; g[sd].l_rows = static_cast<long long>(b) * P * R; g[sd].l_row_stride = P * R;
    g[sd].R = Abar; g[sd].r_blocks = batch * T; g[sd].r_blk_stride = T;
    g[sd].D = arr; g[sd].d_blocks = 1; g[sd].d_blk0 = 0; g[sd].d_blk_stride = 0;
    g[sd].d_rows = static_cast<int>(b * P * R); g[sd].d_row_stride = P * R;
    g[sd].count = batch; g[sd].N = n; g[sd].K = n; g[sd].M = R;
    if (tc) {
      if (phi_tc_maps_size() > sizeof(maps[sd])) return cudaErrorInvalidValue;
      if ((e = bgemm_tc_make_maps(g[sd], maps[sd])) != cudaSuccess) return e;
    }
  }
  for (int j = T - 2; j >= 0; --j) {
    for (int sd = 0; sd < (want_u ? 2 : 1); ++sd) {
      const int R = sd ? m : n;
      const int mrows = (T - 2 - j) * R;   // blocks k = j+2 .. T-1
      if (mrows > 0) {
        g[sd].M = mrows;
        g[sd].l_row0 = static_cast<int>(phi_colbase(T, j + 1)) * R;      // block (j+2, j+1)
        g[sd].d_row0 = (static_cast<int>(phi_colbase(T, j)) + 1) * R;    // block (j+2, j)
        g[sd].r_blk0 = j;
        if (tc) {
          e = launch_bgemm_tc(g[sd], nch, maps[sd], sms, stream);
        } else {
          ProfScope prof(kProfKalmanGemm, stream);
          e = launch_bgemm_simt(g[sd], stream);
        }
        if (e != cudaSuccess) return e;
        ++*launches;
      }
      AsmStep s{};
      s.out = sd ? a.phi_uw : a.phi_xw; s.oute = sd ? a.phi_ue : a.phi_xe; s.pbar = sd ? a.phibar_u : a.phibar_x;
      s.A = a.A; s.Ltt = Ltt; s.C = a.C; s.w = a.w; s.f = a.f; s.tau = sd ? nullptr : a.tau;
      s.T = T; s.n = n; s.p = p; s.R = R; s.is_u = sd; s.j = j;
      const int rows = (T - 1 - j) * R;
      {
        ProfScope prof(kProfOfbSupport, stream);
        asm_step_kernel<<<dim3((rows + 7) / 8, batch), 256, 0, stream>>>(s);
      }
      if ((e = cudaGetLastError()) != cudaSuccess) return e;
      ++*launches;
    }
  }
  return cudaSuccess;
}

}  // namespace ltv
