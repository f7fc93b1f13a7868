// ltv_scan_output_feedback_response: the assembled output-feedback responses of eq.(15) and the
// reachable tube of eq.(12e) (:147) with both terms, for controllers given by gains (first form).
// With the predictor-form observer xhat+ = A xhat + B u - Lt (y - C xhat) and u = K xhat, the closed loop is the LTV
// system in xi = (x, x - xhat)
//     xi_{k+1} = [[A_k + B_k K_k, -B_k K_k], [0, A_k + Lt_k C_k]] xi_k + [I; I] w~_{k+1} + [0; Lt_k] e~_{k+1},
// so with G = Phi_aug(k,j) = A_aug,k-1 ... A_aug,j (the system response of the augmented Jacobians):
//     Phi^xw(k,j) = G11 + G12,        Phi^xe(k,j) = G12 Lt_{j-1}  (j >= 1),
// which equals (15) evaluated on Phibar = (I - Z(A + BK))^-1, Phihat = (I - Z(A + LtC))^-1 (pinned in the oracle tests).
// Three steps, all on the device: (1) form the 2n x 2n augmented Jacobians; (2) the time-parallel Phi scan of phi.cu on
// them (tcgen05 3xTF32 for 2n >= 96); (3) one pass over Phi_aug that writes Phi^xw, Phi^xe and accumulates
//     tau_k[i] = sum_{j<k} ||row_i(Phi^xw(k,j) diag(w_j))||_2 + ||row_i(Phi^xe(k,j) diag(f_{j-1}))||_2
// with one warp per (k, i) walking j in order (deterministic, no partial buffers).
// The augmented matrix is block upper triangular, and so is every Phi_aug(k,j): G11 = Phibar^x, G22 = Phihat^x and the
// cross block obeys G12(t,s) = G11(t,mid) G12(mid,s) + G12(t,mid) G22(mid,s).  For n >= 96 the call therefore runs two
// n-state scans and one cross scan (MODE 2 of the tcgen05 kernel: one K loop over both operand pairs) - 4 instead of 8
// n^3 products per block and 3 instead of 4 n x n blocks of storage; below that the plain 2n-state scan is used.
// The low-rank form for a general Phibar is the next step (NEXT-4).
#include <cuda.h>

#include <algorithm>

#include "../../include/ltv_scan.h"
#include "ltv_internal.h"
#include "phi_geom.cuh"
#include "phi_kernels.h"

namespace ltv {

namespace {

// warp per row i of (b, t): top row i = [A + B K | -B K], bottom row n + i = [0 | A + Lt C].  grid (batch T, ceil(n/32)); four rows per warp, one after the other
__global__ void __launch_bounds__(256) ofb_build_aug_kernel(const float* __restrict__ A, const float* __restrict__ B,
                                                            const float* __restrict__ Kfb, const float* __restrict__ Lt,
                                                            const float* __restrict__ C, float* __restrict__ Aaug,
                                                            float* __restrict__ Ltt, int n, int m, int p) {
  const size_t bt = blockIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n4 = n >> 2, n2 = 2 * n;
  for (int i = blockIdx.y * 32 + warp; i < min(n, static_cast<int>(blockIdx.y) * 32 + 32); i += 8) {
  const float4* Ar = reinterpret_cast<const float4*>(A + (bt * n + i) * n);
  const float* Bi = B + (bt * n + i) * m;
  const float* Li = Lt + (bt * n + i) * p;
  if (lane < p) Ltt[(bt * p + lane) * n + i] = __ldg(Li + lane);   // gains with n contiguous, for the extraction pass
  const float4* K4 = reinterpret_cast<const float4*>(Kfb + bt * m * n);
  const float4* C4 = reinterpret_cast<const float4*>(C + bt * p * n);
  float4* top = reinterpret_cast<float4*>(Aaug + (bt * n2 + i) * n2);
  float4* bot = reinterpret_cast<float4*>(Aaug + (bt * n2 + n + i) * n2);
  for (int c = lane; c < n4; c += 32) {
    const float4 a = __ldg(Ar + c);
    float4 bk = make_float4(0.f, 0.f, 0.f, 0.f), lc = bk;
    for (int q = 0; q < m; ++q) {
      const float s = __ldg(Bi + q);
      const float4 k4 = __ldg(K4 + static_cast<size_t>(q) * n4 + c);
      bk.x = fmaf(s, k4.x, bk.x); bk.y = fmaf(s, k4.y, bk.y); bk.z = fmaf(s, k4.z, bk.z); bk.w = fmaf(s, k4.w, bk.w);
    }
    for (int q = 0; q < p; ++q) {
      const float s = __ldg(Li + q);
      const float4 c4 = __ldg(C4 + static_cast<size_t>(q) * n4 + c);
      lc.x = fmaf(s, c4.x, lc.x); lc.y = fmaf(s, c4.y, lc.y); lc.z = fmaf(s, c4.z, lc.z); lc.w = fmaf(s, c4.w, lc.w);
    }
    top[c] = make_float4(a.x + bk.x, a.y + bk.y, a.z + bk.z, a.w + bk.w);
    top[n4 + c] = make_float4(-bk.x, -bk.y, -bk.z, -bk.w);
    bot[c] = make_float4(0.f, 0.f, 0.f, 0.f);
    bot[n4 + c] = make_float4(a.x + lc.x, a.y + lc.y, a.z + lc.z, a.w + lc.w);
  }
  }
}

// structured path: warp per row i of (b, t): Atil = A + B K, Abar = A + Lt C (n x n each), and the level-0 cross block
// G12(t+1,t) = -B_t K_t into block (t+1, t) of the column-packed G (t <= T-2).  grid (batch T, ceil(n/32)); four rows per warp, one after the other
__global__ void __launch_bounds__(256) ofb_build_split_kernel(const float* __restrict__ A, const float* __restrict__ B,
                                                              const float* __restrict__ Kfb, const float* __restrict__ Lt,
                                                              const float* __restrict__ C, float* __restrict__ Atil,
                                                              float* __restrict__ Abar, float* __restrict__ G,
                                                              float* __restrict__ Ltt, int T, int n, int m, int p) {
  const size_t bt = blockIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n4 = n >> 2;
  const int t = static_cast<int>(bt % T);
  const size_t b = bt / T;
  for (int i = blockIdx.y * 32 + warp; i < min(n, static_cast<int>(blockIdx.y) * 32 + 32); i += 8) {
  const float4* Ar = reinterpret_cast<const float4*>(A + (bt * n + i) * n);
  const float* Bi = B + (bt * n + i) * m;
  const float* Li = Lt + (bt * n + i) * p;
  if (lane < p) Ltt[(bt * p + lane) * n + i] = __ldg(Li + lane);   // gains with n contiguous, for the extraction pass
  const float4* K4 = reinterpret_cast<const float4*>(Kfb + bt * m * n);
  const float4* C4 = reinterpret_cast<const float4*>(C + bt * p * n);
  float4* o1 = reinterpret_cast<float4*>(Atil + (bt * n + i) * n);
  float4* o2 = reinterpret_cast<float4*>(Abar + (bt * n + i) * n);
  float4* o3 = nullptr;
  if (t <= T - 2) {
    const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
    o3 = reinterpret_cast<float4*>(G + ((b * P + phi_colbase(T, t)) * n + i) * n);
  }
  for (int c = lane; c < n4; c += 32) {
    const float4 a = __ldg(Ar + c);
    float4 bk = make_float4(0.f, 0.f, 0.f, 0.f), lc = bk;
    for (int q = 0; q < m; ++q) {
      const float s = __ldg(Bi + q);
      const float4 k4 = __ldg(K4 + static_cast<size_t>(q) * n4 + c);
      bk.x = fmaf(s, k4.x, bk.x); bk.y = fmaf(s, k4.y, bk.y); bk.z = fmaf(s, k4.z, bk.z); bk.w = fmaf(s, k4.w, bk.w);
    }
    for (int q = 0; q < p; ++q) {
      const float s = __ldg(Li + q);
      const float4 c4 = __ldg(C4 + static_cast<size_t>(q) * n4 + c);
      lc.x = fmaf(s, c4.x, lc.x); lc.y = fmaf(s, c4.y, lc.y); lc.z = fmaf(s, c4.z, lc.z); lc.w = fmaf(s, c4.w, lc.w);
    }
    o1[c] = make_float4(a.x + bk.x, a.y + bk.y, a.z + bk.z, a.w + bk.w);
    o2[c] = make_float4(a.x + lc.x, a.y + lc.y, a.z + lc.z, a.w + lc.w);
    if (o3 != nullptr) o3[c] = make_float4(-bk.x, -bk.y, -bk.z, -bk.w);
  }
  }
}

// warp per (b, k, i): for j = 0 .. k-1 reads row i of Phi_aug(k,j) (2n floats), writes row i of Phi^xw(k,j) and of
// Phi^xe(k,j), adds the two row norms of (12e) to tau_k[i].  Lane = column quad: it keeps 8 PG partial sums of
// Phi^xe[i][q] = sum_c G12[i][c] Lt_{j-1}[c][q] over its own columns (accumulators q >= p re-read column p - 1 and are
// discarded), finished by butterfly shuffles.  grid (ceil(n/8), T, batch); k = blockIdx.y (k = 0: tau_0 = 0).
template <int PG>
__global__ void __launch_bounds__(256) ofb_extract_kernel(const float* P1, const float* __restrict__ P2, int ld, int brows,
                                                          const float* __restrict__ Lt /* transposed: [b,T,p,n] */,
                                                          const float* __restrict__ w, const float* __restrict__ f,
                                                          float* phi_xw, float* __restrict__ phi_xe,
                                                          float* __restrict__ tau, int T, int n, int p) {
  constexpr int PP = 8 * PG;
  const int b = blockIdx.z, k = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = blockIdx.x * 8 + warp;
  if (i >= n) return;
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
  const int n4 = n >> 2;
  int qoff[PP];
#pragma unroll
  for (int q = 0; q < PP; ++q) qoff[q] = min(q, p - 1);
  float acc = 0.f;
  for (int j = 0; j < k; ++j) {
    const size_t blk = static_cast<size_t>(b) * P + phi_colbase(T, j) + (k - j - 1);
    // G11 row from P1, G12 row from P2 (augmented scan: the two halves of one 2n-float row; structured: two arrays; P1 may
    // be phi_xw itself - each element is read, then written, by the same thread)
    const float4* g1 = reinterpret_cast<const float4*>(P1 + (blk * brows + i) * ld);
    const float4* g2 = reinterpret_cast<const float4*>(P2 + (blk * brows + i) * ld);
    const float4* w4 = reinterpret_cast<const float4*>(w + (static_cast<size_t>(b) * T + j) * n);
    float4* out = reinterpret_cast<float4*>(phi_xw + (blk * n + i) * n);
    const float4* Lj = (j >= 1) ? reinterpret_cast<const float4*>(Lt + (static_cast<size_t>(b) * T + (j - 1)) * n * p) : nullptr;
    float s1 = 0.f;
    float xe[PP];
#pragma unroll
    for (int q = 0; q < PP; ++q) xe[q] = 0.f;
    for (int c = lane; c < n4; c += 32) {
      const float4 a = g1[c];
      const float4 h = __ldcs(g2 + c);
      const float4 ww = __ldg(w4 + c);
      const float4 x = make_float4(a.x + h.x, a.y + h.y, a.z + h.z, a.w + h.w);
      out[c] = x;
      const float e0 = x.x * ww.x, e1 = x.y * ww.y, e2 = x.z * ww.z, e3 = x.w * ww.w;
      s1 = fmaf(e0, e0, fmaf(e1, e1, fmaf(e2, e2, fmaf(e3, e3, s1))));
      if (Lj != nullptr) {
#pragma unroll
        for (int q = 0; q < PP; ++q) {
          const float4 l = __ldg(Lj + static_cast<size_t>(qoff[q]) * n4 + c);   // row q of Lt_{j-1}^T, coalesced
          xe[q] = fmaf(h.x, l.x, fmaf(h.y, l.y, fmaf(h.z, l.z, fmaf(h.w, l.w, xe[q]))));
        }
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    float s2 = 0.f;
    if (Lj != nullptr) {
      const float* fj = f + (static_cast<size_t>(b) * T + (j - 1)) * p;
#pragma unroll
      for (int q = 0; q < PP; ++q) {
        if (q < p) {
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) xe[q] += __shfl_xor_sync(0xffffffffu, xe[q], o);
          const float v = xe[q] * __ldg(fj + q);
          s2 = fmaf(v, v, s2);
          if (phi_xe != nullptr && lane == (q & 31)) phi_xe[(blk * n + i) * p + q] = xe[q];
        }
      }
    } else if (phi_xe != nullptr && lane < p) {
      phi_xe[(blk * n + i) * p + lane] = 0.f;
    }
    acc += sqrtf(s1) + sqrtf(s2);
  }
  if (lane == 0) tau[(static_cast<size_t>(b) * T + k) * n + i] = acc;
}

size_t carve(size_t floats) { return align_up(floats * sizeof(float), 256); }

// ------------------------------------------------------------------------------------------------------------------
// Closed-loop backward sweep (ltv_scan_output_feedback_constraints): input-side responses of eq.(15) and both terms of
// the margins (12d).  A row s^T acting on xi_k = (x_k, x_k - xhat_k) propagates as psi(k,j) = psi(k,j+1) A_aug,j with
// psi(k,k) = s^T.  For a constraint row c = [hx, hu] on [z_k; v_k] (u = K xhat = K [I -I] xi): s = [hx + hu K_k | -hu K_k];
// for row a of the input response: s = [K_k[a] | -K_k[a]].  With psi = [psi1 | psi2] (n floats each):
//     c^T Phi^w(k,j) = psi1 + psi2  (= psi(k,j) [I; I]),       c^T Phi^e(k,j) = psi2 Lt_{j-1}  (j >= 1),
// and the same two expressions are rows of Phi^uw(k,j), Phi^ue(k,j) for the K rows.

// start rows: X[(k-1)&1][b][(T-1-k) nr + i][0 .. 2n), k = 1 .. T-1, i < nr = nc + mu (mu = m if the input responses are
// wanted, else 0); sigma[b][k][:] = 0.  grid (T, batch), 256 threads.
__global__ void __launch_bounds__(256) cls_prefill_kernel(const float* __restrict__ Hx, const float* __restrict__ Hu,
                                                          const float* __restrict__ Kfb, float* __restrict__ X0,
                                                          float* __restrict__ X1, float* __restrict__ sigma, int T, int n,
                                                          int m, int nc, int mu, int rmax) {
  const int k = blockIdx.x, b = blockIdx.y;
  const int nr = nc + mu, n2 = 2 * n;
  if (sigma != nullptr)
    for (int i = threadIdx.x; i < nc; i += 256) sigma[(static_cast<size_t>(b) * T + k) * nc + i] = 0.f;
  if (k == 0) return;
  float* X = ((k - 1) & 1) ? X1 : X0;
  float* dst = X + (static_cast<size_t>(b) * rmax + static_cast<size_t>(T - 1 - k) * nr) * n2;
  const size_t bk = static_cast<size_t>(b) * T + k;
  const float* Kk = Kfb + bk * m * n;
  for (int e = threadIdx.x; e < nr * n; e += 256) {
    const int i = e / n, c = e - i * n;
    float s1, s2;
    if (i < nc) {
      const float* hu = Hu + (bk * nc + i) * m;
      float hk = 0.f;
      for (int a = 0; a < m; ++a) hk = fmaf(__ldg(hu + a), __ldg(Kk + static_cast<size_t>(a) * n + c), hk);
      s1 = __ldg(Hx + (bk * nc + i) * n + c) + hk;
      s2 = -hk;
    } else {
      s1 = __ldg(Kk + static_cast<size_t>(i - nc) * n + c);
      s2 = -s1;
    }
    dst[static_cast<size_t>(i) * n2 + c] = s1;
    dst[static_cast<size_t>(i) * n2 + n + c] = s2;
  }
}

// after the GEMM of step j: warp per stacked row (k, i) of X = [psi(T-1,j); ..; psi(j+1,j)].  Constraint rows add the two
// norms of (12d) to sigma[b][k][i] (one owner per entry and launch, launches stream-ordered: deterministic); K rows are
// written out as rows of Phi^uw(k,j) (n floats) and Phi^ue(k,j) (p floats).  grid (ceil(rows/8), batch).
__global__ void __launch_bounds__(256) cls_post_kernel(const float* __restrict__ X, const float* __restrict__ Ltt,
                                                       const float* __restrict__ w, const float* __restrict__ f,
                                                       float* __restrict__ sigma, float* __restrict__ phi_uw,
                                                       float* __restrict__ phi_ue, int T, int n, int m, int p, int nc,
                                                       int mu, int rmax, int rows, int j) {
  const int b = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row = blockIdx.x * 8 + warp;
  if (row >= rows) return;
  const int nr = nc + mu, n4 = n >> 2;
  const int k = T - 1 - row / nr, i = row % nr;
  const float4* p1 = reinterpret_cast<const float4*>(X + (static_cast<size_t>(b) * rmax + row) * 2 * n);
  const float4* p2 = p1 + n4;
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
  const size_t blk = static_cast<size_t>(b) * P + phi_colbase(T, j) + (k - j - 1);
  const bool krow = i >= nc;
  const float4* w4 = reinterpret_cast<const float4*>(w + (static_cast<size_t>(b) * T + j) * n);
  float4* uw = (krow && phi_uw != nullptr) ? reinterpret_cast<float4*>(phi_uw + (blk * m + (i - nc)) * n) : nullptr;
  float s1 = 0.f;
  for (int c = lane; c < n4; c += 32) {
    const float4 a = p1[c], h = p2[c];
    const float4 x = make_float4(a.x + h.x, a.y + h.y, a.z + h.z, a.w + h.w);
    if (uw != nullptr) uw[c] = x;
    if (!krow) {
      const float4 ww = __ldg(w4 + c);
      const float e0 = x.x * ww.x, e1 = x.y * ww.y, e2 = x.z * ww.z, e3 = x.w * ww.w;
      s1 = fmaf(e0, e0, fmaf(e1, e1, fmaf(e2, e2, fmaf(e3, e3, s1))));
    }
  }
  float s2 = 0.f;
  if (j >= 1) {
    const float4* L4 = reinterpret_cast<const float4*>(Ltt + (static_cast<size_t>(b) * T + (j - 1)) * p * n);
    const float* fj = f + (static_cast<size_t>(b) * T + (j - 1)) * p;
    for (int q = 0; q < p; ++q) {
      float y = 0.f;
      for (int c = lane; c < n4; c += 32) {
        const float4 h = p2[c];
        const float4 l = __ldg(L4 + static_cast<size_t>(q) * n4 + c);
        y = fmaf(h.x, l.x, fmaf(h.y, l.y, fmaf(h.z, l.z, fmaf(h.w, l.w, y))));
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) y += __shfl_xor_sync(0xffffffffu, y, o);
      if (krow) {
        if (phi_ue != nullptr && lane == 0) phi_ue[(blk * m + (i - nc)) * p + q] = y;
      } else {
        const float v = y * __ldg(fj + q);
        s2 = fmaf(v, v, s2);
      }
    }
  } else if (krow && phi_ue != nullptr && lane < p) {
    phi_ue[(blk * m + (i - nc)) * p + lane] = 0.f;
  }
  if (!krow) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    if (lane == 0) sigma[(static_cast<size_t>(b) * T + k) * nc + i] += sqrtf(s1) + sqrtf(s2);
  }
}

}  // namespace

static bool ofb_structured(int n) { return phi_uses_tensor_cores(n) && env_int("OFB_AUGMENTED", 0) == 0; }

// Route of the structured path (n >= 96), LTV_OPT_OUTPUT_FEEDBACK_ROUTE: 1 = CROSS SCAN (two n-state scans + the cross scan with
// the two-source K loop: 4 n^3 products per block, log depth), 2 = COLUMN RECURSION (assemble.cu: one scan for Phibar^x, then
// the backward recursion over the columns on D = Phi^xw - Phibar^x: 2 n^3 products per block, half the passes over the
// blocks, but a chain of 2 (T - 1) launches; needs m, p <= 8), 0 = by size: the column recursion wins once the GEMM of a
// middle step is worth about four waves of tiles (C2 batch 64: 1.33x, one n = 1200 or 2400 item: 1.75x; C2 batch 4: 0.95x).
static int ofb_route(int batch, int T, int n, int m, int p) {
  if (!ofb_columns_supported(n, m, p)) return 1;
  const int forced = option(LTV_OPT_OUTPUT_FEEDBACK_ROUTE);
  if (forced == 1 || forced == 2) return forced;
  const long long rows = static_cast<long long>(batch) * (T / 2) * n;   // column T/2 holds T/2 blocks per item
  const long long tiles = (rows / 128) * ((n + 159) / 160);
  return tiles >= 4 * 148 ? 2 : 1;
}

// m = p = 0: the gains' sizes are not known to the caller of ltv_scan_workspace_bytes - room for either route
size_t ofb_workspace_bytes(int batch, int T, int n, int m, int p) {
  const size_t b = batch, t = T, nn = n, n2 = 2 * nn, P = t * (t - 1) / 2;
  if (ofb_structured(n)) {
    // Atil, Abar; Phihat, G (Phibar lives in phi_xw_out); zero w, scratch r; tube partials of a scan
    const size_t cross = carve(b * t * 32 * nn) + 2 * carve(b * t * nn * nn) + 2 * carve(b * P * nn * nn + 4) + 2 * carve(b * t * nn) + phi_workspace_bytes(batch, T, n, n);
    if (m < 1 || p < 1) return std::max(cross, ofb_columns_workspace_bytes(batch, T, n));
    return ofb_route(batch, T, n, m, p) == 2 ? ofb_columns_workspace_bytes(batch, T, n) : cross;
  }
  return carve(b * t * 32 * nn) + carve(b * t * n2 * n2) + carve(b * P * n2 * n2 + 4) + 2 * carve(b * t * n2) + phi_workspace_bytes(batch, T, 2 * n, 2 * n);
}

template <typename... Args>
static cudaError_t launch_extract(int p, dim3 grid, cudaStream_t stream, Args... args) {
  ProfScope prof(kProfKalmanSimt, stream);
  switch ((p + 7) / 8) {
    case 1: ofb_extract_kernel<1><<<grid, 256, 0, stream>>>(args...); break;
    case 2: ofb_extract_kernel<2><<<grid, 256, 0, stream>>>(args...); break;
    case 3: ofb_extract_kernel<3><<<grid, 256, 0, stream>>>(args...); break;
    default: ofb_extract_kernel<4><<<grid, 256, 0, stream>>>(args...); break;
  }
  return cudaGetLastError();
}

cudaError_t launch_output_feedback(const OfbArgs& a, cudaStream_t stream, unsigned long long* launches) {
  const int batch = a.batch, T = a.T, n = a.n;
  const size_t b = batch, t = T, nn = n, n2 = 2 * nn, P = t * (t - 1) / 2;
  char* cur = static_cast<char*>(a.workspace);
  const dim3 xgrid((n + 7) / 8, T, batch);
  cudaError_t e;
  if (ofb_structured(n) && ofb_route(batch, T, n, a.m, a.p) == 2) return launch_ofb_response_columns(a, stream, launches);
  float* Ltt = reinterpret_cast<float*>(cur); cur += carve(b * t * 32 * nn);   // [b,T,p,n] (sized for p = 32)
  if (ofb_structured(n)) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    float* Atil = reinterpret_cast<float*>(cur); cur += carve(b * t * nn * nn);
    float* Abar = reinterpret_cast<float*>(cur); cur += carve(b * t * nn * nn);
    float* phat = reinterpret_cast<float*>(cur); cur += carve(b * P * nn * nn + 4);
    float* G = reinterpret_cast<float*>(cur); cur += carve(b * P * nn * nn + 4);
    float* wz = reinterpret_cast<float*>(cur); cur += carve(b * t * nn);
    float* rz = reinterpret_cast<float*>(cur); cur += carve(b * t * nn);
    float* part = reinterpret_cast<float*>(cur);
    float* pbar = a.phi_xw;   // Phibar^x is scanned straight into the output and completed in place by the last pass
    if ((e = cudaMemsetAsync(wz, 0, b * t * nn * sizeof(float), stream)) != cudaSuccess) return e;
    {
      ProfScope prof(kProfKalmanSimt, stream);
      ofb_build_split_kernel<<<dim3(batch * T, (n + 31) / 32), 256, 0, stream>>>(a.A, a.B, a.Kfb, a.Lt, a.C, Atil, Abar, G, Ltt,
                                                                               T, n, a.m, a.p);
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    ++*launches;
    PhiArgs pb{Atil, wz, pbar, rz, part, batch, T, n, n, 0};
    if ((e = launch_phi_tube(pb, stream, launches)) != cudaSuccess) return e;
    PhiArgs ph{Abar, wz, phat, rz, part, batch, T, n, n, 0};
    if ((e = launch_phi_tube(ph, stream, launches)) != cudaSuccess) return e;
    if (T - 1 >= 2) {
      PhiArgs pg{nullptr, nullptr, G, nullptr, nullptr, batch, T, n, n, 0};
      const int nch = phi_pick_nch(n);
      alignas(64) unsigned char maps[1024];
      if (phi_tc_maps_size() > sizeof(maps)) return cudaErrorInvalidValue;
      if ((e = phi_tc_make_cross_maps(pg, pbar, phat, nch, maps)) != cudaSuccess) return e;
      for (int level = 1; (1 << (level - 1)) < T - 1; ++level) {
        if ((e = launch_phi_cross_tc(pg, level, nch, maps, sms, stream)) != cudaSuccess) return e;
        ++*launches;
      }
    }
    if ((e = launch_extract(a.p, xgrid, stream, static_cast<const float*>(pbar), static_cast<const float*>(G), n, n,
                            static_cast<const float*>(Ltt), a.w, a.f, a.phi_xw, a.phi_xe, a.tau, T, n, a.p)) != cudaSuccess)
      return e;
    ++*launches;
    return cudaSuccess;
  }
  float* Aaug = reinterpret_cast<float*>(cur); cur += carve(b * t * n2 * n2);
  float* phi_aug = reinterpret_cast<float*>(cur); cur += carve(b * P * n2 * n2 + 4);
  float* wz = reinterpret_cast<float*>(cur); cur += carve(b * t * n2);
  float* rz = reinterpret_cast<float*>(cur); cur += carve(b * t * n2);
  float* part = reinterpret_cast<float*>(cur);
  if ((e = cudaMemsetAsync(wz, 0, b * t * n2 * sizeof(float), stream)) != cudaSuccess) return e;   // the scan's own tube is not used
  {
    ProfScope prof(kProfKalmanSimt, stream);
    ofb_build_aug_kernel<<<dim3(batch * T, (n + 31) / 32), 256, 0, stream>>>(a.A, a.B, a.Kfb, a.Lt, a.C, Aaug, Ltt, n, a.m, a.p);
  }
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  ++*launches;
  PhiArgs ph{Aaug, wz, phi_aug, rz, part, batch, T, 2 * n, 2 * n, 0};
  if ((e = launch_phi_tube(ph, stream, launches)) != cudaSuccess) return e;
  if ((e = launch_extract(a.p, xgrid, stream, static_cast<const float*>(phi_aug), static_cast<const float*>(phi_aug + n), 2 * n,
                          2 * n, static_cast<const float*>(Ltt), a.w, a.f, a.phi_xw, a.phi_xe, a.tau, T, n, a.p)) != cudaSuccess)
    return e;
  ++*launches;
  return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------------------------
// ltv_scan_output_feedback_constraints: Phi^uw, Phi^ue of eq.(15) and the closed-loop margins of eq.(12d), both terms.
// One backward sweep over j on the 2n-state augmented closed loop carries the stack of all start rows with k > j,
//     X_j = [X_{j+1}; S_{j+1}] A_aug,j        ((T-1-j) nr rows of 2n floats, nr = nc + m),
// as one batched GEMM per step (MODE 1 of the tcgen05 3xTF32 kernel for 2n >= 96, fp32 FMA below), followed by
// cls_post_kernel.  Phi_aug is never formed: 2 (2n)^2 nr (T-1-j) flop per step.
size_t ofb_constraints_workspace_bytes(int batch, int T, int n, int nc, int m) {
  const size_t b = batch, t = T, nn = n, n2 = 2 * nn;
  const size_t rmax = static_cast<size_t>(T > 1 ? T - 1 : 1) * (nc + m);
  return carve(b * t * 32 * nn) + carve(b * t * n2 * n2) + 2 * carve(b * rmax * n2);
}

cudaError_t launch_ofb_constraints(const OfbConArgs& a, cudaStream_t stream, unsigned long long* launches) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int batch = a.batch, T = a.T, n = a.n, n2 = 2 * a.n, nc = a.nc;
  const int mu = (a.phi_uw != nullptr || a.phi_ue != nullptr) ? a.m : 0;
  const int nr = nc + mu;
  const int rmax = (T > 1 ? T - 1 : 1) * (nc + a.m);   // sized as the workspace query (which does not know mu)
  const size_t b = batch, t = T, nn = n;
  char* cur = static_cast<char*>(a.workspace);
  float* Ltt = reinterpret_cast<float*>(cur); cur += carve(b * t * 32 * nn);
  float* Aaug = reinterpret_cast<float*>(cur); cur += carve(b * t * n2 * static_cast<size_t>(n2));
  float* X[2];
  X[0] = reinterpret_cast<float*>(cur); cur += carve(b * rmax * n2);
  X[1] = reinterpret_cast<float*>(cur);
  cudaError_t e;
  {
    ProfScope prof(kProfOfbSupport, stream);
    ofb_build_aug_kernel<<<dim3(batch * T, (n + 31) / 32), 256, 0, stream>>>(a.A, a.B, a.Kfb, a.Lt, a.C, Aaug, Ltt, n, a.m, a.p);
  }
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  {
    ProfScope prof(kProfOfbSupport, stream);
    cls_prefill_kernel<<<dim3(T, batch), 256, 0, stream>>>(a.Hx, a.Hu, a.Kfb, X[0], X[1], a.sigma, T, n, a.m, nc, mu, rmax);
  }
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  *launches += 2;
  if (T < 2 || nr == 0) return cudaSuccess;

  const bool tc = phi_uses_tensor_cores(n2);
  const int nch = phi_pick_nch(n2);
  BatchedGemm g[2];
  alignas(64) unsigned char maps[2][1024];
  for (int q = 0; q < 2; ++q) {   // q = parity of the step: left operand X[q], output X[q ^ 1]
    g[q] = BatchedGemm{};
    g[q].L = X[q]; g[q].l_rows = static_cast<long long>(batch) * rmax; g[q].l_row0 = 0; g[q].l_row_stride = rmax;
    g[q].R = Aaug; g[q].r_blocks = batch * T; g[q].r_blk_stride = T;
    g[q].D = X[q ^ 1]; g[q].d_blocks = batch; g[q].d_blk0 = 0; g[q].d_blk_stride = 1;
    g[q].count = batch; g[q].M = rmax; g[q].N = n2; g[q].K = n2; g[q].d_rows = rmax;
    g[q].transpose_out = 0; g[q].diag = nullptr; g[q].diag_stride = 0;
    if (tc) {
      if (phi_tc_maps_size() > sizeof(maps[q])) return cudaErrorInvalidValue;
      if ((e = bgemm_tc_make_maps(g[q], maps[q])) != cudaSuccess) return e;
    }
  }
  for (int j = T - 2; j >= 0; --j) {
    const int q = j & 1;
    const int rows = (T - 1 - j) * nr;
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
      ProfScope prof(kProfOfbSupport, stream);
      cls_post_kernel<<<dim3((rows + 7) / 8, batch), 256, 0, stream>>>(X[q ^ 1], Ltt, a.w, a.f, a.sigma, a.phi_uw, a.phi_ue, T, n,
                                                                     a.m, a.p, nc, mu, rmax, rows, j);
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    *launches += 2;
  }
  return cudaSuccess;
}

}  // namespace ltv
