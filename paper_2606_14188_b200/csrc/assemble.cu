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

#include <algorithm>

#include "ltv_internal.h"
#include "phi_geom.cuh"
#include "phi_kernels.h"
#include "ptx.cuh"

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
  // DIFFERENCE mode (gain-defined controllers, x side only; see launch_ofb_response_columns): the recursion carries
  // D = Phi^xw - Phibar^x.  Ltt / C above are replaced by Gt = B^T [batch,T,pc,n] and Cm = Kfb [batch,T,pc,n] for the rank-pc
  // correction, Lte = Lt^T [batch,T,p,n] gives e = D Lt_{j-1}; dcol = the D blocks (k, j), k = j+1 .. T-1, of this column
  // ([batch, T-1, n, n], block k-j-1), read (GEMM result) and written in place; out receives Phi^xw = D + Phibar^x.
  const float *Gt, *Cm, *Lte;
  float* dcol;
  int pc;
};

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Step j of the backward recursion for the rows of column j: a warp takes kAsmRows consecutive rows i of one block (b, k),
// k = j+1 .. T-1 (the p gain / measurement vectors are then loaded once per kAsmRows rows, and kAsmRows independent row loads
// are in flight per lane).
//   k = j+1:  x: row = A_j[i]                                   u: row = -(Phibar^u(j+1,j+1)[i] Lt_j) C_j
//   k > j+1:  row = (GEMM result already in out) - (Phibar(k,j+1)[i] Lt_j) C_j
// then e = (row - Phibar(k,j)[i]) Lt_{j-1} (j >= 1) and, x side, tau_k[i] += ||row o w_j|| + ||e o f_{j-1}||.
// NP = p exactly for p <= 8 (every loop over the measurements unrolls, the sums stay in registers); NP = 0: any p <= 32
// (32 guarded accumulators, one row per warp).  grid (ceil(groups / 8), batch), groups = (T-1-j) ceil(R / ROWS).
template <int NP, int ROWS, bool DIFF = false>
__global__ void __launch_bounds__(256) asm_step_kernel(const AsmStep s) {
  constexpr int PMAX = NP > 0 ? NP : 32;
  const int T = s.T, n = s.n, R = s.R, j = s.j;
  const int p = (NP > 0 && !DIFF) ? NP : s.p;   // rank of the noise term (DIFF: p <= NP, the rest of the accumulators idle)
  const int pcr = DIFF ? s.pc : p;             // rank of the correction
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int gpb = (R + ROWS - 1) / ROWS;   // row groups per block
  const int grp = blockIdx.x * 8 + warp;
  if (grp >= (T - 1 - j) * gpb) return;
  const int b = blockIdx.y;
  const int kk = grp / gpb, i0 = (grp - kk * gpb) * ROWS;
  const int nr = min(ROWS, R - i0);        // rows of this group that exist
  const int k = j + 1 + kk;
  const int n4 = n >> 2;
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
  const size_t bT = static_cast<size_t>(b) * T;
  // Phibar blocks (k, j+1) and (k, j), row i0
  const float4 *pb_next = nullptr, *pb_cur;
  if (s.is_u) {
    const size_t item = static_cast<size_t>(b) * (P + T);
    auto qd = [&](int kq, int jq) { return static_cast<size_t>(jq) * T - static_cast<size_t>(jq) * (jq - 1) / 2 + (kq - jq); };
    pb_next = reinterpret_cast<const float4*>(s.pbar + ((item + qd(k, j + 1)) * R + i0) * n);
    pb_cur = reinterpret_cast<const float4*>(s.pbar + ((item + qd(k, j)) * R + i0) * n);
  } else {
    const size_t item = static_cast<size_t>(b) * P;
    if (kk > 0) pb_next = reinterpret_cast<const float4*>(s.pbar + ((item + phi_colbase(T, j + 1) + (k - j - 2)) * R + i0) * n);
    pb_cur = reinterpret_cast<const float4*>(s.pbar + ((item + phi_colbase(T, j) + (k - j - 1)) * R + i0) * n);
  }
  const size_t oblk = static_cast<size_t>(b) * P + phi_colbase(T, j) + (k - j - 1);
  float4* orow = DIFF ? reinterpret_cast<float4*>(s.dcol + ((static_cast<size_t>(b) * (T - 1) + kk) * n + i0) * n)
                      : reinterpret_cast<float4*>(s.out + (oblk * R + i0) * n);
  float4* xrow = DIFF ? reinterpret_cast<float4*>(s.out + (oblk * R + i0) * n) : nullptr;   // Phi^xw = D + Phibar^x
  const float4* Lj = reinterpret_cast<const float4*>((DIFF ? s.Gt : s.Ltt) + (bT + j) * pcr * n);
  const float4* Cj = reinterpret_cast<const float4*>((DIFF ? s.Cm : s.C) + (bT + j) * pcr * n);
  const float4* Ljm = (j >= 1) ? reinterpret_cast<const float4*>((DIFF ? s.Lte : s.Ltt) + (bT + j - 1) * p * n) : nullptr;
  const float4* wj = reinterpret_cast<const float4*>(s.w + (bT + j) * n);
  const float4* arow = (!DIFF && !s.is_u && kk == 0) ? reinterpret_cast<const float4*>(s.A + ((bT + j) * n + i0) * n) : nullptr;
  const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
  const bool corr = pb_next != nullptr || (DIFF && kk == 0);   // DIFF, k = j+1: Phibar^x(j+1,j+1) = I, the gain row is B_j[i]

  // u[r][q] = Phibar(k,j+1)[i0 + r] . Lt_j[:,q]
  float u[ROWS][PMAX];
#pragma unroll
  for (int r = 0; r < ROWS; ++r)
#pragma unroll
    for (int q = 0; q < PMAX; ++q) u[r][q] = 0.f;
  if (pb_next != nullptr) {
    for (int c = lane; c < n4; c += 32) {
      float4 a[ROWS];
#pragma unroll
      for (int r = 0; r < ROWS; ++r) a[r] = (r < nr) ? __ldg(pb_next + static_cast<size_t>(r) * n4 + c) : z4;
#pragma unroll
      for (int q = 0; q < PMAX; ++q) {
        if ((NP > 0 && !DIFF) || q < pcr) {
          const float4 l = __ldg(Lj + static_cast<size_t>(q) * n4 + c);
#pragma unroll
          for (int r = 0; r < ROWS; ++r)
            u[r][q] = fmaf(a[r].x, l.x, fmaf(a[r].y, l.y, fmaf(a[r].z, l.z, fmaf(a[r].w, l.w, u[r][q]))));
        }
      }
    }
#pragma unroll
    for (int r = 0; r < ROWS; ++r)
#pragma unroll
      for (int q = 0; q < PMAX; ++q)
        if ((NP > 0 && !DIFF) || q < pcr) u[r][q] = warp_sum(u[r][q]);
  } else if (DIFF && kk == 0) {
    const float* Bt = s.Gt + (bT + j) * pcr * n;
#pragma unroll
    for (int r = 0; r < ROWS; ++r)
#pragma unroll
      for (int q = 0; q < PMAX; ++q)
        if (q < pcr && r < nr) u[r][q] = __ldg(Bt + static_cast<size_t>(q) * n + i0 + r);
  }
  // the rows, their tube terms and e = (row - Phibar(k,j)[i]) Lt_{j-1}
  float s1[ROWS];
  float e[ROWS][PMAX];
#pragma unroll
  for (int r = 0; r < ROWS; ++r) {
    s1[r] = 0.f;
#pragma unroll
    for (int q = 0; q < PMAX; ++q) e[r][q] = 0.f;
  }
  for (int c = lane; c < n4; c += 32) {
    float4 x[ROWS], pc[ROWS];
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
      if (r < nr) {
        if (kk == 0) x[r] = (s.is_u || DIFF) ? z4 : __ldg(arow + static_cast<size_t>(r) * n4 + c); else x[r] = orow[static_cast<size_t>(r) * n4 + c];
        pc[r] = (DIFF || Ljm != nullptr) ? __ldg(pb_cur + static_cast<size_t>(r) * n4 + c) : z4;
      } else {
        x[r] = z4; pc[r] = z4;
      }
    }
    if (corr) {
#pragma unroll
      for (int q = 0; q < PMAX; ++q) {
        if ((NP > 0 && !DIFF) || q < pcr) {
          const float4 cq = __ldg(Cj + static_cast<size_t>(q) * n4 + c);
#pragma unroll
          for (int r = 0; r < ROWS; ++r) {
            x[r].x = fmaf(-u[r][q], cq.x, x[r].x); x[r].y = fmaf(-u[r][q], cq.y, x[r].y);
            x[r].z = fmaf(-u[r][q], cq.z, x[r].z); x[r].w = fmaf(-u[r][q], cq.w, x[r].w);
          }
        }
      }
    }
#pragma unroll
    for (int r = 0; r < ROWS; ++r)
      if (r < nr && (!DIFF || j > 0)) orow[static_cast<size_t>(r) * n4 + c] = x[r];   // DIFF: column 0 feeds no further product
    if (DIFF) {
      // x = row of D: the response row is D + Phibar^x, and e = D Lt_{j-1} runs over D itself (no subtraction)
#pragma unroll
      for (int r = 0; r < ROWS; ++r) {
        const float4 d = x[r];
        x[r].x += pc[r].x; x[r].y += pc[r].y; x[r].z += pc[r].z; x[r].w += pc[r].w;
        if (r < nr) xrow[static_cast<size_t>(r) * n4 + c] = x[r];
        pc[r] = d;
      }
    }
    if (!s.is_u) {
      const float4 ww = __ldg(wj + c);
#pragma unroll
      for (int r = 0; r < ROWS; ++r) {
        const float e0 = x[r].x * ww.x, e1 = x[r].y * ww.y, e2 = x[r].z * ww.z, e3 = x[r].w * ww.w;
        s1[r] = fmaf(e0, e0, fmaf(e1, e1, fmaf(e2, e2, fmaf(e3, e3, s1[r]))));
      }
    }
    if (Ljm != nullptr) {
      if (!DIFF) {
#pragma unroll
        for (int r = 0; r < ROWS; ++r) {
          pc[r].x = x[r].x - pc[r].x; pc[r].y = x[r].y - pc[r].y; pc[r].z = x[r].z - pc[r].z; pc[r].w = x[r].w - pc[r].w;
        }
      }
#pragma unroll
      for (int q = 0; q < PMAX; ++q) {
        if ((NP > 0 && !DIFF) || q < p) {
          const float4 l = __ldg(Ljm + static_cast<size_t>(q) * n4 + c);
#pragma unroll
          for (int r = 0; r < ROWS; ++r)
            e[r][q] = fmaf(pc[r].x, l.x, fmaf(pc[r].y, l.y, fmaf(pc[r].z, l.z, fmaf(pc[r].w, l.w, e[r][q]))));
        }
      }
    }
  }
  const float* fj = (Ljm != nullptr) ? s.f + (bT + j - 1) * p : nullptr;
#pragma unroll
  for (int r = 0; r < ROWS; ++r) {
    if (r >= nr) continue;   // warp-uniform
    float s2 = 0.f;
    float* er = s.oute ? s.oute + (oblk * R + i0 + r) * p : nullptr;
    if (Ljm != nullptr) {
#pragma unroll
      for (int q = 0; q < PMAX; ++q) {
        if ((NP > 0 && !DIFF) || q < p) {
          const float eq = warp_sum(e[r][q]);
          const float t = eq * __ldg(fj + q);
          s2 = fmaf(t, t, s2);
          if (er != nullptr && lane == q) er[q] = eq;
        }
      }
    } else if (er != nullptr && lane < p) {
      er[lane] = 0.f;   // j = 0: no measurement noise has entered yet
    }
    if (!s.is_u && s.tau != nullptr) {
      const float t1 = warp_sum(s1[r]);
      if (lane == 0) s.tau[(bT + k) * n + i0 + r] += sqrtf(t1) + sqrtf(s2);
    }
  }
}

// The same step as a small persistent pipeline (p <= 8 and the buffers below fit shared memory; C2: 80 KB, C3: 160 KB).
// ncu on the register version: 24 % dram throughput, long-scoreboard stalls 7 per issue - a warp lived for one row, waited
// out a DRAM latency per pass, and every CTA re-fetched the 3 p gain / measurement vectors of its (b, j) through L1.  Here a
// CTA stays on one item, stages Lt_j^T, C_j, Lt_{j-1}^T and w_j in shared memory ONCE, and each warp walks its rows with a
// two-stage cp.async ring: the (up to) three rows of row r+1 - Phibar(k,j+1)[i], the GEMM result, Phibar(k,j)[i] - are in
// flight while row r is reduced out of shared memory.
// DIFF (difference mode, see AsmStep): NP = max(pc, p); the vectors beyond a rank are staged as zeros.
template <int NP, bool DIFF = false>
__global__ void __launch_bounds__(256) asm_step_pipe_kernel(const AsmStep s) {
  extern __shared__ float4 asm_sm[];
  const int T = s.T, n = s.n, R = s.R, j = s.j;
  constexpr int p = NP;
  const int pe = DIFF ? s.p : NP;     // rank of the noise term = row length of oute and f
  const int pcr = DIFF ? s.pc : NP;   // rank of the correction
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int b = blockIdx.y;
  const int n4 = n >> 2;
  const int rtot = (T - 1 - j) * R;
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
  const size_t bT = static_cast<size_t>(b) * T;
  float4* vL = asm_sm;                 // [p][n4] Lt_j^T
  float4* vC = vL + p * n4;            // [p][n4] C_j
  float4* vLm = vC + p * n4;           // [p][n4] Lt_{j-1}^T (j >= 1)
  float4* vw = vLm + p * n4;           // [n4]    w_j
  float4* ring = vw + n4 + static_cast<size_t>(warp) * 6 * n4;   // [2 stages][3 rows][n4] of this warp
  {
    const float4* Lj = reinterpret_cast<const float4*>((DIFF ? s.Gt : s.Ltt) + (bT + j) * pcr * n);
    const float4* Cj = reinterpret_cast<const float4*>((DIFF ? s.Cm : s.C) + (bT + j) * pcr * n);
    const float4* wj = reinterpret_cast<const float4*>(s.w + (bT + j) * n);
    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int e = threadIdx.x; e < p * n4; e += 256) {
      const bool in_c = !DIFF || e < pcr * n4, in_e = !DIFF || e < pe * n4;
      vL[e] = in_c ? __ldg(Lj + e) : z4;
      vC[e] = in_c ? __ldg(Cj + e) : z4;
      if (j >= 1) vLm[e] = in_e ? __ldg(reinterpret_cast<const float4*>((DIFF ? s.Lte : s.Ltt) + (bT + j - 1) * pe * n) + e) : z4;
    }
    for (int e = threadIdx.x; e < n4; e += 256) vw[e] = __ldg(wj + e);
  }
  __syncthreads();
  const bool has_e = j >= 1;
  const size_t item_x = static_cast<size_t>(b) * P, item_u = static_cast<size_t>(b) * (P + T);
  auto qd = [&](int kq, int jq) { return static_cast<size_t>(jq) * T - static_cast<size_t>(jq) * (jq - 1) / 2 + (kq - jq); };
  // global rows of row index `row` of this step: Phibar(k,j+1)[i] (or null), base row (or null = zero), Phibar(k,j)[i], out row
  auto rows_of = [&](int row, const float4*& nx, const float4*& bs, const float4*& cu, float4*& orow, size_t& oidx, int& k) {
    const int kk = row / R, i = row - kk * R;
    k = j + 1 + kk;
    oidx = (item_x + phi_colbase(T, j) + (k - j - 1)) * R + i;
    orow = reinterpret_cast<float4*>(s.out + oidx * n);
    if (DIFF) {
      orow = reinterpret_cast<float4*>(s.dcol + ((static_cast<size_t>(b) * (T - 1) + kk) * n + i) * n);   // row of D(k,j)
      nx = kk > 0 ? reinterpret_cast<const float4*>(s.pbar + ((item_x + phi_colbase(T, j + 1) + (k - j - 2)) * R + i) * n) : nullptr;
      cu = reinterpret_cast<const float4*>(s.pbar + ((item_x + phi_colbase(T, j) + (k - j - 1)) * R + i) * n);
      bs = kk == 0 ? nullptr : orow;
    } else if (s.is_u) {
      nx = reinterpret_cast<const float4*>(s.pbar + ((item_u + qd(k, j + 1)) * R + i) * n);
      cu = reinterpret_cast<const float4*>(s.pbar + ((item_u + qd(k, j)) * R + i) * n);
      bs = kk == 0 ? nullptr : orow;
    } else {
      nx = kk > 0 ? reinterpret_cast<const float4*>(s.pbar + ((item_x + phi_colbase(T, j + 1) + (k - j - 2)) * R + i) * n) : nullptr;
      cu = reinterpret_cast<const float4*>(s.pbar + ((item_x + phi_colbase(T, j) + (k - j - 1)) * R + i) * n);
      bs = kk == 0 ? reinterpret_cast<const float4*>(s.A + ((bT + j) * n + i) * n) : orow;
    }
  };
  auto prefetch = [&](int row, int stage) {
    if (row < rtot) {
      const float4 *nx, *bs, *cu; float4* orow; size_t oidx; int k;
      rows_of(row, nx, bs, cu, orow, oidx, k);
      float4* dst = ring + static_cast<size_t>(stage) * 3 * n4;
      for (int c = lane; c < n4; c += 32) {
        if (nx != nullptr) cp_async16(dst + c, nx + c);
        if (bs != nullptr) cp_async16(dst + n4 + c, bs + c);
        if (has_e || DIFF) cp_async16(dst + 2 * n4 + c, cu + c);
      }
    }
    cp_async_commit();
  };
  float fq[NP];   // f_{j-1}: the scaling of the measurement noise that enters through Lt_{j-1}
#pragma unroll
  for (int q = 0; q < NP; ++q) fq[q] = (has_e && q < pe) ? __ldg(s.f + (bT + j - 1) * pe + q) : 0.f;
  const int stride = gridDim.x * 8;
  int row = blockIdx.x * 8 + warp;
  prefetch(row, 0);
  for (int it = 0; row < rtot; row += stride, ++it) {
    const int stage = it & 1;
    prefetch(row + stride, stage ^ 1);
    cp_async_wait<1>();
    __syncwarp();
    const float4 *nx, *bs, *cu; float4* orow; size_t oidx; int k;
    rows_of(row, nx, bs, cu, orow, oidx, k);
    // tau_k[i] so far: loaded now, needed only at the end of the row (one owner per entry and step: no race)
    float* tau_p = (!s.is_u && s.tau != nullptr) ? s.tau + (bT + k) * n + row % R : nullptr;
    const float tau_old = (tau_p != nullptr && lane == 0) ? *tau_p : 0.f;
    const float4* s_next = ring + static_cast<size_t>(stage) * 3 * n4;
    const float4* s_base = s_next + n4;
    const float4* s_cur = s_base + n4;
    float u[NP];
#pragma unroll
    for (int q = 0; q < NP; ++q) u[q] = 0.f;
    if (nx != nullptr) {
      for (int c = lane; c < n4; c += 32) {
        const float4 a = s_next[c];
#pragma unroll
        for (int q = 0; q < NP; ++q) {
          const float4 l = vL[q * n4 + c];
          u[q] = fmaf(a.x, l.x, fmaf(a.y, l.y, fmaf(a.z, l.z, fmaf(a.w, l.w, u[q]))));
        }
      }
#pragma unroll
      for (int q = 0; q < NP; ++q) u[q] = warp_sum(u[q]);
    } else if (DIFF) {
      // k = j+1: Phibar^x(j+1,j+1) = I, so the gain row is row i of B_j = column i of the staged B_j^T (zeros beyond pc)
      const float* vLf = reinterpret_cast<const float*>(vL);
#pragma unroll
      for (int q = 0; q < NP; ++q) u[q] = vLf[static_cast<size_t>(q) * n + row % R];
    }
    const bool corr = nx != nullptr || DIFF;
    float4* xrow = DIFF ? reinterpret_cast<float4*>(s.out + oidx * n) : nullptr;   // Phi^xw = D + Phibar^x
    float s1 = 0.f;
    float e[NP];
#pragma unroll
    for (int q = 0; q < NP; ++q) e[q] = 0.f;
    for (int c = lane; c < n4; c += 32) {
      float4 x = (bs != nullptr) ? s_base[c] : make_float4(0.f, 0.f, 0.f, 0.f);
      if (corr) {
#pragma unroll
        for (int q = 0; q < NP; ++q) {
          const float4 cq = vC[q * n4 + c];
          x.x = fmaf(-u[q], cq.x, x.x); x.y = fmaf(-u[q], cq.y, x.y); x.z = fmaf(-u[q], cq.z, x.z); x.w = fmaf(-u[q], cq.w, x.w);
        }
      }
      if (!DIFF || j > 0) orow[c] = x;   // DIFF: column 0 of D feeds no further product
      const float4 d = x;
      if (DIFF) {
        const float4 pc = s_cur[c];
        x.x += pc.x; x.y += pc.y; x.z += pc.z; x.w += pc.w;
        xrow[c] = x;
      }
      if (!s.is_u) {
        const float4 ww = vw[c];
        const float e0 = x.x * ww.x, e1 = x.y * ww.y, e2 = x.z * ww.z, e3 = x.w * ww.w;
        s1 = fmaf(e0, e0, fmaf(e1, e1, fmaf(e2, e2, fmaf(e3, e3, s1))));
      }
      if (has_e) {
        float4 v = d;   // DIFF: e = D Lt_{j-1}
        if (!DIFF) {
          const float4 pc = s_cur[c];
          v = make_float4(x.x - pc.x, x.y - pc.y, x.z - pc.z, x.w - pc.w);
        }
#pragma unroll
        for (int q = 0; q < NP; ++q) {
          const float4 l = vLm[q * n4 + c];
          e[q] = fmaf(v.x, l.x, fmaf(v.y, l.y, fmaf(v.z, l.z, fmaf(v.w, l.w, e[q]))));
        }
      }
    }
    float s2 = 0.f;
    if (has_e) {
#pragma unroll
      for (int q = 0; q < NP; ++q) {
        const float eq = warp_sum(e[q]);
        const float t = eq * fq[q];
        s2 = fmaf(t, t, s2);
        if (s.oute != nullptr && lane == q && q < pe) s.oute[oidx * pe + q] = eq;
      }
    } else if (s.oute != nullptr && lane < pe) {
      s.oute[oidx * pe + lane] = 0.f;   // j = 0: no measurement noise has entered yet
    }
    if (tau_p != nullptr) {
      s1 = warp_sum(s1);
      if (lane == 0) *tau_p = tau_old + (sqrtf(s1) + sqrtf(s2));
    }
    __syncwarp();   // every lane is done with this stage before the next iteration's prefetch overwrites the other one's successor
  }
  cp_async_wait<0>();
}

size_t asm_pipe_smem_bytes(int n, int p) { return (static_cast<size_t>(3) * p * n + n + static_cast<size_t>(8) * 6 * n) * sizeof(float); }

constexpr int kAsmWaves = 8;

template <int NP, bool DIFF = false>
cudaError_t launch_asm_step_pipe(const AsmStep& s, int batch, int sms, cudaStream_t stream) {
  const size_t smem = asm_pipe_smem_bytes(s.n, NP);
  if (smem > 48 * 1024) {   // every launch: the attribute belongs to the current device's copy of the function
    cudaError_t e = cudaFuncSetAttribute(asm_step_pipe_kernel<NP, DIFF>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    if (e != cudaSuccess) return e;
  }
  const int rtot = (s.T - 1 - s.j) * s.R;
  const int per_sm = static_cast<int>(std::max<size_t>(1, std::min<size_t>(4, (200u * 1024u) / smem)));
  // CTAs per item: about kAsmWaves waves of resident CTAs (a single wave wants batch to divide the slots - 64 items on 296
  // slots left 14 % of them empty -, two or three waves end in a long tail; with eight the tail is <= 1/8 of a wave and the
  // staging of the vectors is still amortised over >= 30 rows per warp on the long steps)
  int cx = (env_int("ASM_WAVES", kAsmWaves) * per_sm * sms + batch - 1) / batch;
  cx = std::max(1, std::min(cx, (rtot + 7) / 8));
  asm_step_pipe_kernel<NP, DIFF><<<dim3(cx, batch), 256, smem, stream>>>(s);
  return cudaGetLastError();
}

constexpr int kAsmRows = 2;

cudaError_t launch_asm_step(const AsmStep& s, int batch, int sms, cudaStream_t stream) {
  if (s.p <= 8 && asm_pipe_smem_bytes(s.n, s.p) <= 200u * 1024u) {
    switch (s.p) {
      case 1: return launch_asm_step_pipe<1>(s, batch, sms, stream);
      case 2: return launch_asm_step_pipe<2>(s, batch, sms, stream);
      case 3: return launch_asm_step_pipe<3>(s, batch, sms, stream);
      case 4: return launch_asm_step_pipe<4>(s, batch, sms, stream);
      case 5: return launch_asm_step_pipe<5>(s, batch, sms, stream);
      case 6: return launch_asm_step_pipe<6>(s, batch, sms, stream);
      case 7: return launch_asm_step_pipe<7>(s, batch, sms, stream);
      default: return launch_asm_step_pipe<8>(s, batch, sms, stream);
    }
  }
  const int rows = s.p <= 8 ? kAsmRows : 1;
  const int groups = (s.T - 1 - s.j) * ((s.R + rows - 1) / rows);
  const dim3 grid((groups + 7) / 8, batch);
  switch (s.p <= 8 ? s.p : 0) {
    case 1: asm_step_kernel<1, kAsmRows><<<grid, 256, 0, stream>>>(s); break;
    case 2: asm_step_kernel<2, kAsmRows><<<grid, 256, 0, stream>>>(s); break;
    case 3: asm_step_kernel<3, kAsmRows><<<grid, 256, 0, stream>>>(s); break;
    case 4: asm_step_kernel<4, kAsmRows><<<grid, 256, 0, stream>>>(s); break;
    case 5: asm_step_kernel<5, kAsmRows><<<grid, 256, 0, stream>>>(s); break;
    case 6: asm_step_kernel<6, kAsmRows><<<grid, 256, 0, stream>>>(s); break;
    case 7: asm_step_kernel<7, kAsmRows><<<grid, 256, 0, stream>>>(s); break;
    case 8: asm_step_kernel<8, kAsmRows><<<grid, 256, 0, stream>>>(s); break;
    default: asm_step_kernel<0, 1><<<grid, 256, 0, stream>>>(s); break;
  }
  return cudaGetLastError();
}

// Difference mode, second form: TWO rows per warp and the gain products stashed one step ahead.
// ncu on the one-row pipeline: 38 % of the HBM copy peak at 56 % issue-slot use - ~1060 warp instructions per 1.2 KB row, most of
// them the 3 NP shared-memory vector loads per column quad and the 5-step butterflies of 2 NP + 1 sums.  Here
//   * a warp reduces rows i, i+1 of a block together: every staged vector is loaded once for both rows, and the butterflies
//     start with an exchange between the two rows (lanes 0-15 end with row i's sums, lanes 16-31 with row i+1's): half the shuffles;
//   * the skinny product S(k,j+1)[i] = Phibar^x(k,j+1)[i] B_j that the correction of step j needs is formed at step j+1, when the
//     row of Phibar^x(k,j+1) is in shared memory anyway (for Phi^xw = D + Phibar^x), and stashed in sbuf[b,k,i,0..7]: the row of
//     Phibar^x(k,j+1) is not read a second time (4 instead of 5 row passes per step, two rows instead of three in the ring).
// Shared memory: K_j, B_{j-1}^T, Lt_{j-1}^T, w_j + per warp 2 stages x (2 rows of D + 2 rows of Phibar^x + 16 floats of S).
// GEN = true: the same pipeline for the x side of the GENERAL assembly (Phibar given as operators): the recursion runs on
// Phi^xw itself (rows of column j in `out`: GEMM result, or A_j for k = j+1), correction vectors C_j, gain rows
// S(k,j+1) = Phibar^x(k,j+1) Lt_j stashed the same way (Lt_{j-1}^T serves both e = (row - Phibar^x(k,j)) Lt_{j-1} and the stash),
// three row passes per step (read GEMM result, read Phibar^x(k,j), write Phi^xw(k,j)).
template <int NP, bool GEN>
__global__ void __launch_bounds__(256) asm_diff2_kernel(const AsmStep s, float* __restrict__ sbuf) {
  extern __shared__ float4 asm_sm[];
  const int T = s.T, n = s.n, j = s.j;
  const int pe = s.p, pcr = s.pc;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int half = lane >> 4;   // which row of the pair this lane ends up owning
  const int b = blockIdx.y;
  const int n4 = n >> 2;
  const int ptot = (T - 1 - j) * (n >> 1);   // row pairs of this column (n is even)
  const size_t P = static_cast<size_t>(T) * (T - 1) / 2;
  const size_t bT = static_cast<size_t>(b) * T;
  const bool has_e = j >= 1;
  float4* vK = asm_sm;                  // [NP][n4] Kfb_j          (zeros beyond pc)
  float4* vB = vK + NP * n4;            // [NP][n4] B_{j-1}^T      (zeros beyond pc; j >= 1)
  float4* vLm = vB + NP * n4;           // [NP][n4] Lt_{j-1}^T     (zeros beyond p;  j >= 1)
  float4* vw = vLm + NP * n4;           // [n4]     w_j
  const int stage_f4 = 4 * n4 + 4;      // 2 rows of D, 2 rows of Phibar^x, 2 x 8 floats of S
  float4* ring = vw + n4 + static_cast<size_t>(warp) * 2 * stage_f4;
  {
    const float4* Kj = reinterpret_cast<const float4*>(s.Cm + (bT + j) * pcr * n);
    const float4* wj = reinterpret_cast<const float4*>(s.w + (bT + j) * n);
    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int e = threadIdx.x; e < NP * n4; e += 256) {
      vK[e] = e < pcr * n4 ? __ldg(Kj + e) : z4;
      if (has_e) {
        if (!GEN) vB[e] = e < pcr * n4 ? __ldg(reinterpret_cast<const float4*>(s.Gt + (bT + j - 1) * pcr * n) + e) : z4;
        vLm[e] = e < pe * n4 ? __ldg(reinterpret_cast<const float4*>(s.Lte + (bT + j - 1) * pe * n) + e) : z4;
      }
    }
    for (int e = threadIdx.x; e < n4; e += 256) vw[e] = __ldg(wj + e);
  }
  __syncthreads();
  const size_t item_x = static_cast<size_t>(b) * P;
  const float* Btj = s.Gt + (bT + j) * pcr * n;   // B_j^T: the gain rows of the blocks (j+1, j)
  auto prefetch = [&](int pr, int stage) {
    if (pr < ptot) {
      const int row = pr * 2, kk = row / n, i = row - kk * n, k = j + 1 + kk;
      float4* dst = ring + static_cast<size_t>(stage) * stage_f4;
      const size_t orow = ((item_x + phi_colbase(T, j) + kk) * n + i) * n;   // row i of block (k, j), COLUMN_PACKED
      const float4* bs = GEN ? reinterpret_cast<const float4*>(kk > 0 ? s.out + orow : s.A + ((bT + j) * n + i) * n)
                             : reinterpret_cast<const float4*>(s.dcol + ((static_cast<size_t>(b) * (T - 1) + kk) * n + i) * n);
      const float4* cu = reinterpret_cast<const float4*>(s.pbar + orow);
      for (int c = lane; c < 2 * n4; c += 32) {   // rows i and i+1 are contiguous in every array
        if (GEN || kk > 0) cp_async16(dst + c, bs + c);
        if (!GEN || has_e) cp_async16(dst + 2 * n4 + c, cu + c);
      }
      float* su = reinterpret_cast<float*>(dst + 4 * n4);   // [2][8]
      if (kk > 0) {
        if (lane < 4) cp_async16(dst + 4 * n4 + lane, reinterpret_cast<const float4*>(sbuf + ((bT + k) * n + i) * 8) + lane);
      } else if (lane < 16) {
        const int r = lane >> 3, q = lane & 7;
        if (!GEN && q < pcr) cp_async4(su + lane, Btj + static_cast<size_t>(q) * n + i + r); else su[lane] = 0.f;
      }
    }
    cp_async_commit();
  };
  float fq[NP];
#pragma unroll
  for (int q = 0; q < NP; ++q) fq[q] = (has_e && q < pe) ? __ldg(s.f + (bT + j - 1) * pe + q) : 0.f;
  const int stride = gridDim.x * 8;
  int pr = blockIdx.x * 8 + warp;
  prefetch(pr, 0);
  for (int it = 0; pr < ptot; pr += stride, ++it) {
    const int stage = it & 1;
    prefetch(pr + stride, stage ^ 1);
    cp_async_wait<1>();
    __syncwarp();
    const int row = pr * 2, kk = row / n, i = row - kk * n, k = j + 1 + kk;
    const size_t oidx = (item_x + phi_colbase(T, j) + kk) * n + i;   // row i of block (k, j) in COLUMN_PACKED order
    float* tau_p = s.tau != nullptr ? s.tau + (bT + k) * n + i + half : nullptr;
    const float tau_old = (tau_p != nullptr && (lane & 15) == 0) ? *tau_p : 0.f;
    const float4* sD = ring + static_cast<size_t>(stage) * stage_f4;
    const float4* sP = sD + 2 * n4;
    const float* su = reinterpret_cast<const float*>(sD + 4 * n4);
    float4* drow = reinterpret_cast<float4*>(s.dcol + ((static_cast<size_t>(b) * (T - 1) + kk) * n + i) * n);
    float4* xrow = reinterpret_cast<float4*>(s.out + oidx * n);
    float u0[NP], u1[NP], e0[NP], e1[NP], g0[NP], g1[NP];
#pragma unroll
    for (int q = 0; q < NP; ++q) { u0[q] = su[q]; u1[q] = su[8 + q]; e0[q] = e1[q] = g0[q] = g1[q] = 0.f; }
    float t0 = 0.f, t1 = 0.f;
    for (int c = lane; c < n4; c += 32) {
      float4 x0 = make_float4(0.f, 0.f, 0.f, 0.f), x1 = x0;
      if (GEN || kk > 0) { x0 = sD[c]; x1 = sD[n4 + c]; }
      if (!GEN || kk > 0) {   // GEN, k = j+1: the row is A_j[i] as it stands
#pragma unroll
        for (int q = 0; q < NP; ++q) {
          const float4 kq = vK[q * n4 + c];
          x0.x = fmaf(-u0[q], kq.x, x0.x); x0.y = fmaf(-u0[q], kq.y, x0.y); x0.z = fmaf(-u0[q], kq.z, x0.z); x0.w = fmaf(-u0[q], kq.w, x0.w);
          x1.x = fmaf(-u1[q], kq.x, x1.x); x1.y = fmaf(-u1[q], kq.y, x1.y); x1.z = fmaf(-u1[q], kq.z, x1.z); x1.w = fmaf(-u1[q], kq.w, x1.w);
        }
      }
      if (GEN) {
        if (has_e) {
          const float4 p0 = sP[c], p1 = sP[n4 + c];
          const float4 v0 = make_float4(x0.x - p0.x, x0.y - p0.y, x0.z - p0.z, x0.w - p0.w);
          const float4 v1 = make_float4(x1.x - p1.x, x1.y - p1.y, x1.z - p1.z, x1.w - p1.w);
#pragma unroll
          for (int q = 0; q < NP; ++q) {
            const float4 l = vLm[q * n4 + c];
            e0[q] = fmaf(v0.x, l.x, fmaf(v0.y, l.y, fmaf(v0.z, l.z, fmaf(v0.w, l.w, e0[q]))));
            e1[q] = fmaf(v1.x, l.x, fmaf(v1.y, l.y, fmaf(v1.z, l.z, fmaf(v1.w, l.w, e1[q]))));
            g0[q] = fmaf(p0.x, l.x, fmaf(p0.y, l.y, fmaf(p0.z, l.z, fmaf(p0.w, l.w, g0[q]))));
            g1[q] = fmaf(p1.x, l.x, fmaf(p1.y, l.y, fmaf(p1.z, l.z, fmaf(p1.w, l.w, g1[q]))));
          }
        }
      } else {
        const float4 p0 = sP[c], p1 = sP[n4 + c];
        if (has_e) {   // column 0 of D feeds no further product
          drow[c] = x0; drow[n4 + c] = x1;
#pragma unroll
          for (int q = 0; q < NP; ++q) {
            const float4 l = vLm[q * n4 + c];
            e0[q] = fmaf(x0.x, l.x, fmaf(x0.y, l.y, fmaf(x0.z, l.z, fmaf(x0.w, l.w, e0[q]))));
            e1[q] = fmaf(x1.x, l.x, fmaf(x1.y, l.y, fmaf(x1.z, l.z, fmaf(x1.w, l.w, e1[q]))));
            const float4 bq = vB[q * n4 + c];
            g0[q] = fmaf(p0.x, bq.x, fmaf(p0.y, bq.y, fmaf(p0.z, bq.z, fmaf(p0.w, bq.w, g0[q]))));
            g1[q] = fmaf(p1.x, bq.x, fmaf(p1.y, bq.y, fmaf(p1.z, bq.z, fmaf(p1.w, bq.w, g1[q]))));
          }
        }
        x0.x += p0.x; x0.y += p0.y; x0.z += p0.z; x0.w += p0.w;
        x1.x += p1.x; x1.y += p1.y; x1.z += p1.z; x1.w += p1.w;
      }
      xrow[c] = x0; xrow[n4 + c] = x1;
      const float4 ww = vw[c];
      {
        const float a0 = x0.x * ww.x, a1 = x0.y * ww.y, a2 = x0.z * ww.z, a3 = x0.w * ww.w;
        t0 = fmaf(a0, a0, fmaf(a1, a1, fmaf(a2, a2, fmaf(a3, a3, t0))));
        const float b0 = x1.x * ww.x, b1 = x1.y * ww.y, b2 = x1.z * ww.z, b3 = x1.w * ww.w;
        t1 = fmaf(b0, b0, fmaf(b1, b1, fmaf(b2, b2, fmaf(b3, b3, t1))));
      }
    }
    // pair reduction: lanes 0-15 keep row i's partial and take the partner's, lanes 16-31 the same for row i+1; then four
    // butterfly steps inside each half
    auto pair_sum = [&](float a0, float a1) {
      float v = (half ? a1 : a0) + __shfl_xor_sync(0xffffffffu, half ? a0 : a1, 16);
#pragma unroll
      for (int o = 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      return v;
    };
    const float s1 = pair_sum(t0, t1);
    float s2 = 0.f;
    if (has_e) {
      float* er = s.oute != nullptr ? s.oute + (oidx + half) * pe : nullptr;
      float* sn = sbuf + ((bT + k) * n + i + half) * 8;
#pragma unroll
      for (int q = 0; q < NP; ++q) {
        const float eq = pair_sum(e0[q], e1[q]);
        const float gq = pair_sum(g0[q], g1[q]);
        const float t = eq * fq[q];
        s2 = fmaf(t, t, s2);
        if ((lane & 15) == q) {
          if (er != nullptr && q < pe) er[q] = eq;
          sn[q] = gq;   // S(k,j)[i] = Phibar^x(k,j)[i] B_{j-1}: the gain row of step j-1
        }
      }
    } else if (s.oute != nullptr && (lane & 15) < pe) {
      s.oute[(oidx + half) * pe + (lane & 15)] = 0.f;   // j = 0: no measurement noise has entered yet
    }
    if (tau_p != nullptr && (lane & 15) == 0) *tau_p = tau_old + (sqrtf(s1) + sqrtf(s2));
    __syncwarp();
  }
  cp_async_wait<0>();
}

size_t asm_diff2_smem_bytes(int n, int np) { return (static_cast<size_t>(3) * np * n + n + static_cast<size_t>(8) * 2 * (4 * n + 16)) * sizeof(float); }

template <int NP, bool GEN = false>
cudaError_t launch_asm_diff2(const AsmStep& s, float* sbuf, int batch, int sms, cudaStream_t stream) {
  const size_t smem = asm_diff2_smem_bytes(s.n, NP);
  if (smem > 48 * 1024) {   // every launch: the attribute belongs to the current device's copy of the function
    cudaError_t e = cudaFuncSetAttribute(asm_diff2_kernel<NP, GEN>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    if (e != cudaSuccess) return e;
  }
  const int ptot = (s.T - 1 - s.j) * (s.n / 2);
  const int per_sm = static_cast<int>(std::max<size_t>(1, std::min<size_t>(4, (200u * 1024u) / smem)));
  int cx = (env_int("ASM_WAVES", kAsmWaves) * per_sm * sms + batch - 1) / batch;
  cx = std::max(1, std::min(cx, (ptot + 7) / 8));
  asm_diff2_kernel<NP, GEN><<<dim3(cx, batch), 256, smem, stream>>>(s, sbuf);
  return cudaGetLastError();
}

// difference mode: NP = max(pc, p) <= 8
cudaError_t launch_asm_step_diff(const AsmStep& s, float* sbuf, bool two_rows, int batch, int sms, cudaStream_t stream) {
  const int np = std::max(s.pc, s.p);
  if (two_rows) {
    switch (np) {
      case 1: return launch_asm_diff2<1>(s, sbuf, batch, sms, stream);
      case 2: return launch_asm_diff2<2>(s, sbuf, batch, sms, stream);
      case 3: return launch_asm_diff2<3>(s, sbuf, batch, sms, stream);
      case 4: return launch_asm_diff2<4>(s, sbuf, batch, sms, stream);
      case 5: return launch_asm_diff2<5>(s, sbuf, batch, sms, stream);
      case 6: return launch_asm_diff2<6>(s, sbuf, batch, sms, stream);
      case 7: return launch_asm_diff2<7>(s, sbuf, batch, sms, stream);
      default: return launch_asm_diff2<8>(s, sbuf, batch, sms, stream);
    }
  }
  if (asm_pipe_smem_bytes(s.n, np) <= 200u * 1024u) {
    switch (np) {
      case 1: return launch_asm_step_pipe<1, true>(s, batch, sms, stream);
      case 2: return launch_asm_step_pipe<2, true>(s, batch, sms, stream);
      case 3: return launch_asm_step_pipe<3, true>(s, batch, sms, stream);
      case 4: return launch_asm_step_pipe<4, true>(s, batch, sms, stream);
      case 5: return launch_asm_step_pipe<5, true>(s, batch, sms, stream);
      case 6: return launch_asm_step_pipe<6, true>(s, batch, sms, stream);
      case 7: return launch_asm_step_pipe<7, true>(s, batch, sms, stream);
      default: return launch_asm_step_pipe<8, true>(s, batch, sms, stream);
    }
  }
  const int groups = (s.T - 1 - s.j) * ((s.R + kAsmRows - 1) / kAsmRows);
  const dim3 grid((groups + 7) / 8, batch);
  switch (np) {
    case 1: asm_step_kernel<1, kAsmRows, true><<<grid, 256, 0, stream>>>(s); break;
    case 2: asm_step_kernel<2, kAsmRows, true><<<grid, 256, 0, stream>>>(s); break;
    case 3: asm_step_kernel<3, kAsmRows, true><<<grid, 256, 0, stream>>>(s); break;
    case 4: asm_step_kernel<4, kAsmRows, true><<<grid, 256, 0, stream>>>(s); break;
    case 5: asm_step_kernel<5, kAsmRows, true><<<grid, 256, 0, stream>>>(s); break;
    case 6: asm_step_kernel<6, kAsmRows, true><<<grid, 256, 0, stream>>>(s); break;
    case 7: asm_step_kernel<7, kAsmRows, true><<<grid, 256, 0, stream>>>(s); break;
    default: asm_step_kernel<8, kAsmRows, true><<<grid, 256, 0, stream>>>(s); break;
  }
  return cudaGetLastError();
}

// Gain-defined controllers: Atil = A + B K, Abar = A + Lt C and both gains transposed, Btt[b,t,q,:] = B[b,t,:,q],
// Ltt[b,t,q,:] = Lt[b,t,:,q], in one pass over A.  Warp per row; grid (batch T, ceil(n / 32)).
__global__ void __launch_bounds__(256) asm_prep_gains_kernel(const float* __restrict__ A, const float* __restrict__ B,
                                                             const float* __restrict__ Kfb, const float* __restrict__ Lt,
                                                             const float* __restrict__ C, float* __restrict__ Atil,
                                                             float* __restrict__ Abar, float* __restrict__ Btt,
                                                             float* __restrict__ Ltt, int n, int m, int p) {
  const size_t bt = blockIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n4 = n >> 2;
  const float4* K4 = reinterpret_cast<const float4*>(Kfb + bt * m * n);
  const float4* C4 = reinterpret_cast<const float4*>(C + bt * p * n);
  for (int i = blockIdx.y * 32 + warp; i < min(n, static_cast<int>(blockIdx.y) * 32 + 32); i += 8) {
    const float4* Ar = reinterpret_cast<const float4*>(A + (bt * n + i) * n);
    const float* Bi = B + (bt * n + i) * m;
    const float* Li = Lt + (bt * n + i) * p;
    if (lane < m) Btt[(bt * m + lane) * n + i] = __ldg(Bi + lane);
    if (lane < p) Ltt[(bt * p + lane) * n + i] = __ldg(Li + lane);
    float4* o1 = reinterpret_cast<float4*>(Atil + (bt * n + i) * n);
    float4* o2 = reinterpret_cast<float4*>(Abar + (bt * n + i) * n);
    for (int c = lane; c < n4; c += 32) {
      const float4 a = __ldg(Ar + c);
      float4 bk = a, lc = a;
      for (int q = 0; q < m; ++q) {
        const float sc = __ldg(Bi + q);
        const float4 k4 = __ldg(K4 + static_cast<size_t>(q) * n4 + c);
        bk.x = fmaf(sc, k4.x, bk.x); bk.y = fmaf(sc, k4.y, bk.y); bk.z = fmaf(sc, k4.z, bk.z); bk.w = fmaf(sc, k4.w, bk.w);
      }
      for (int q = 0; q < p; ++q) {
        const float sc = __ldg(Li + q);
        const float4 c4 = __ldg(C4 + static_cast<size_t>(q) * n4 + c);
        lc.x = fmaf(sc, c4.x, lc.x); lc.y = fmaf(sc, c4.y, lc.y); lc.z = fmaf(sc, c4.z, lc.z); lc.w = fmaf(sc, c4.w, lc.w);
      }
      o1[c] = bk;
      o2[c] = lc;
    }
  }
}

size_t carve(size_t floats) { return align_up(floats * sizeof(float), 256); }

}  // namespace

// ------------------------------------------------------------------------------------------------------------------
// ltv_scan_output_feedback_response, COLUMN route (gain-defined controller u = Kfb xhat; n >= 96, m, p <= 8): eq.(15) by the
// backward column recursion above, carried on the DIFFERENCE D = Phi^xw - Phibar^x.  With Atil = A + B Kfb (Phibar^x(k,j) =
// Phibar^x(k,j+1) Atil_j) the recursion of Phi^xw turns into
//     D(k,j) = D(k,j+1) Abar_j - [Phibar^x(k,j+1) B_j] Kfb_j,    D(k,k) = 0,    Phibar^x(j+1,j+1) = I,
//     Phi^xw(k,j) = Phibar^x(k,j) + D(k,j),    Phi^xe(k,j) = D(k,j) Lt_{j-1}
// (D = the cross block G12 of the augmented closed loop): no subtraction of nearly equal operators - for small gains
// D << Phi^xw and (Phi^xw - Phibar^x) Lt computed in fp32 loses the digits the cross-scan route keeps (measured 7e-4 at C2-size
// items) - and D only ever needs TWO column buffers (the column being read and the one being written: 2 (T-1) n^2 floats per
// item instead of a third T(T-1)/2 n^2 array).  Work: one scan (Phibar^x, into the workspace) + one n^3 product per block.
size_t ofb_columns_workspace_bytes(int batch, int T, int n) {
  const size_t b = batch, t = T, nn = n, P = t * (t - 1) / 2;
  return 2 * carve(b * t * nn * nn) + 2 * carve(b * t * 8 * nn) + carve(b * P * nn * nn + 4) + 2 * carve(b * t * nn) +
         align_up(phi_workspace_bytes(batch, T, n, n), 256) + 2 * carve(b * (t - 1) * nn * nn + 4) + carve(b * t * nn * 8);
}

bool ofb_columns_supported(int n, int m, int p) { return phi_uses_tensor_cores(n) && m >= 1 && m <= 8 && p >= 1 && p <= 8; }

cudaError_t launch_ofb_response_columns(const OfbArgs& a, cudaStream_t stream, unsigned long long* launches) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int batch = a.batch, T = a.T, n = a.n, m = a.m, p = a.p;
  const size_t b = batch, t = T, nn = n, P = t * (t - 1) / 2;
  char* cur = static_cast<char*>(a.workspace);
  float* Atil = reinterpret_cast<float*>(cur); cur += carve(b * t * nn * nn);
  float* Abar = reinterpret_cast<float*>(cur); cur += carve(b * t * nn * nn);
  float* Btt = reinterpret_cast<float*>(cur); cur += carve(b * t * 8 * nn);
  float* Ltt = reinterpret_cast<float*>(cur); cur += carve(b * t * 8 * nn);
  float* pbar = reinterpret_cast<float*>(cur); cur += carve(b * P * nn * nn + 4);
  float* wz = reinterpret_cast<float*>(cur); cur += carve(b * t * nn);
  float* rz = reinterpret_cast<float*>(cur); cur += carve(b * t * nn);
  float* part = reinterpret_cast<float*>(cur); cur += align_up(phi_workspace_bytes(batch, T, n, n), 256);
  float* dbuf[2];
  dbuf[0] = reinterpret_cast<float*>(cur); cur += carve(b * (t - 1) * nn * nn + 4);
  dbuf[1] = reinterpret_cast<float*>(cur); cur += carve(b * (t - 1) * nn * nn + 4);
  float* sbuf = reinterpret_cast<float*>(cur);   // [b, T, n, 8] stashed gain rows S(k, .)[i] of the two-row kernel
  // the two-row kernel while its buffers fit shared memory (every step of a call takes the same kernel: the stash links the steps)
  const bool two_rows = env_int("ASM_DIFF2", 1) != 0 && asm_diff2_smem_bytes(n, std::max(m, p)) <= 200u * 1024u;
  cudaError_t e;
  if ((e = cudaMemsetAsync(wz, 0, b * t * nn * sizeof(float), stream)) != cudaSuccess) return e;   // the scan's own tube is not used
  if ((e = cudaMemsetAsync(a.tau, 0, b * t * nn * sizeof(float), stream)) != cudaSuccess) return e;
  {
    ProfScope prof(kProfOfbSupport, stream);
    asm_prep_gains_kernel<<<dim3(batch * T, (n + 31) / 32), 256, 0, stream>>>(a.A, a.B, a.Kfb, a.Lt, a.C, Atil, Abar, Btt, Ltt, n, m, p);
  }
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  ++*launches;
  if (T < 2) return cudaSuccess;
  PhiArgs pb{Atil, wz, pbar, rz, part, batch, T, n, n, 0};
  if ((e = launch_phi_tube(pb, stream, launches)) != cudaSuccess) return e;
  // step j: [D blocks (k, j+1), k = j+2 .. T-1: the first T-2-j blocks of the buffer of column j+1] x Abar_j -> blocks 1 .. of
  // the buffer of column j; buffers alternate with the parity of the column
  const int nch = phi_pick_nch(n);
  const int rows_item = (T - 1) * n;
  BatchedGemm g[2];
  alignas(64) unsigned char maps[2][1024];
  for (int q = 0; q < 2; ++q) {   // q = parity of the column being WRITTEN
    g[q] = BatchedGemm{};
    g[q].L = dbuf[q ^ 1]; g[q].l_rows = static_cast<long long>(b) * rows_item; g[q].l_row_stride = rows_item; g[q].l_row0 = 0;
    g[q].R = Abar; g[q].r_blocks = batch * T; g[q].r_blk_stride = T;
    g[q].D = dbuf[q]; g[q].d_blocks = 1; g[q].d_blk0 = 0; g[q].d_blk_stride = 0;
    g[q].d_rows = static_cast<int>(b * rows_item); g[q].d_row_stride = rows_item; g[q].d_row0 = n;
    g[q].count = batch; g[q].N = n; g[q].K = n; g[q].M = n;
    if (phi_tc_maps_size() > sizeof(maps[q])) return cudaErrorInvalidValue;
    if ((e = bgemm_tc_make_maps(g[q], maps[q])) != cudaSuccess) return e;
  }
  for (int j = T - 2; j >= 0; --j) {
    const int q = j & 1;
    const int mrows = (T - 2 - j) * n;
    if (mrows > 0) {
      g[q].M = mrows;
      g[q].r_blk0 = j;
      if ((e = launch_bgemm_tc(g[q], nch, maps[q], sms, stream)) != cudaSuccess) return e;
      ++*launches;
    }
    AsmStep s{};
    s.out = a.phi_xw; s.oute = a.phi_xe; s.pbar = pbar; s.A = a.A; s.w = a.w; s.f = a.f; s.tau = a.tau;
    s.Gt = Btt; s.Cm = a.Kfb; s.Lte = Ltt; s.dcol = dbuf[q]; s.pc = m;
    s.T = T; s.n = n; s.p = p; s.R = n; s.is_u = 0; s.j = j;
    {
      ProfScope prof(kProfOfbSupport, stream);
      e = launch_asm_step_diff(s, sbuf, two_rows, batch, sms, stream);
    }
    if (e != cudaSuccess) return e;
    ++*launches;
  }
  return cudaSuccess;
}

size_t asm_workspace_bytes(int batch, int T, int n, int p) {
  const size_t b = batch, t = T;
  return carve(b * t * n * n) + carve(b * t * p * n) + carve(b * t * n * 8);   // Abar, Lt^T, stashed gain rows of the two-row kernel
}

// x side of the general assembly through the two-row kernel (p <= 8, buffers fit shared memory)
static cudaError_t launch_asm_gen2(const AsmStep& s, float* sbuf, int batch, int sms, cudaStream_t stream) {
  switch (s.p) {
    case 1: return launch_asm_diff2<1, true>(s, sbuf, batch, sms, stream);
    case 2: return launch_asm_diff2<2, true>(s, sbuf, batch, sms, stream);
    case 3: return launch_asm_diff2<3, true>(s, sbuf, batch, sms, stream);
    case 4: return launch_asm_diff2<4, true>(s, sbuf, batch, sms, stream);
    case 5: return launch_asm_diff2<5, true>(s, sbuf, batch, sms, stream);
    case 6: return launch_asm_diff2<6, true>(s, sbuf, batch, sms, stream);
    case 7: return launch_asm_diff2<7, true>(s, sbuf, batch, sms, stream);
    default: return launch_asm_diff2<8, true>(s, sbuf, batch, sms, stream);
  }
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
  float* Ltt = reinterpret_cast<float*>(cur); cur += carve(b * t * p * n);
  float* sbuf = reinterpret_cast<float*>(cur);
  const bool two_rows = p <= 8 && env_int("ASM_GEN2", 1) != 0 && asm_diff2_smem_bytes(n, p) <= 200u * 1024u;
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
      s.Cm = a.C; s.Lte = Ltt; s.pc = p;
      {
        ProfScope prof(kProfOfbSupport, stream);
        e = (sd == 0 && two_rows) ? launch_asm_gen2(s, sbuf, batch, sms, stream) : launch_asm_step(s, batch, sms, stream);
      }
      if (e != cudaSuccess) return e;
      ++*launches;
    }
  }
  return cudaSuccess;
}

}  // namespace ltv
