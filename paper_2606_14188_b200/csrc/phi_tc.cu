// Phi path, levels >= 1, n >= 96: the divide-and-conquer combine Phi(t,s) = Phi(t,mid) Phi(mid,s) as a
// persistent, warp-specialised tcgen05 GEMM with 3xTF32 operand splitting and the tube reduction
// r_t += |Phi(t,s)| w_s fused into the TMEM epilogue (eq.(12c), :147 eq.(12e), :166, :177).
//
//   D[(t,i), j] = sum_k  L[(t,i), k] * R[k, j],   L = stacked Phi(t,mid) (K-major), R = Phi(mid,s) (N-major)
//
// Per CTA tile: 128 rows x NT = 32*NCH columns (NCH <= 5), K = n in blocks of 32.
//   warp 0       TMA producer: fp32 tiles of L (one 128x32 box, SWIZZLE_128B) and R (NCH boxes of 32x32,
//                SWIZZLE_128B_ATOM_32B: the only MN-major layout kind::tf32 accepts) into a ring of R stages
//   warps 8-15   split (lo = rna_tf32(a - trunc_tf32(a))): the L tile goes from shared memory into TMEM as two
//                128-lane x 32-column operands (raw bits = hi, since kind::tf32 reads only the top 19 bits, and
//                lo); the lo plane of R is written to shared memory at the same byte offsets as the raw tile
//                (position-preserving, so no knowledge of the swizzle is needed).  Ring of 3.
//   warp 1       one thread issues, per 8-deep k-step: D += Llo*Rhi, D += Lhi*Rlo, D += Lhi*Rhi (small first),
//                L from TMEM, R from shared memory
//   warps 4-7    epilogue: TMEM -> registers -> global (row per thread) + per-row |D| w partial sum
// Why L goes through TMEM: with both operands in shared memory a k-block moves 216 KB through the 128 B/clk
// shared-memory port against 960 cycles of MMA issue (measured 47 % tensor-pipe activity, profiles/r1_v1_*);
// L in TMEM removes 48 KB of MMA operand reads and 16 KB of split writes per k-block.
// The accumulator is double-buffered in TMEM (2 * NT columns) so the epilogue of tile i overlaps the MMAs of
// tile i+1; TMEM columns: [0, 2NT) accumulators, [2NT, 2NT + 192) L-operand ring.
#include <cuda.h>

#include "ltv_internal.h"
#include "phi_geom.cuh"
#include "phi_kernels.h"
#include "ptx.cuh"

namespace ltv {

namespace {

constexpr int kTcThreads = 512;
constexpr int kConvWarps = 8;
constexpr int kConvStages = 3;  // ring of split operands: L (hi, lo) in TMEM, R lo plane in shared memory
constexpr int kTM = 128;
constexpr int kKB = 32;  // k-block = one 128-byte swizzle row of fp32
constexpr uint32_t kABytes = kTM * kKB * 4;  // 16 KB
constexpr int kTcMaxStages = 6;

struct TcParams {
  float* phi;
  const float* w;
  float* part;
  PhiGeom g;
  int stages;
  int dbg;  // experiment knock-outs (LTV_SCAN_TC_DBG): 1 = no stores, 2 = no R split, 4 = no L split, 8 = no TMA store
};

struct TcMaps {
  CUtensorMap L;  // 2-D [batch*P*n rows][n]           box 32 x 128
  CUtensorMap R;  // 3-D [batch*P blocks][n][n]        box 32 x 32 x 1
  CUtensorMap O;  // 2-D [batch*P*n rows][n]           box 32 x 32 (epilogue stores)
};

__device__ __forceinline__ float tf32_lo(float a, float& hi) {
  hi = __uint_as_float(__float_as_uint(a) & 0xffffe000u);
  const float d = a - hi;
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(d));
  return __uint_as_float(r);
}

template <int NCH>
__global__ void __launch_bounds__(kTcThreads, 1)
phi_combine_tc_kernel(const TcParams p, const __grid_constant__ CUtensorMap mapL,
                      const __grid_constant__ CUtensorMap mapR, const __grid_constant__ CUtensorMap mapO) {
  constexpr int NT = 32 * NCH;
  constexpr uint32_t kBBytes = NCH * 4096u;
  constexpr uint32_t kRawBytes = kABytes + kBBytes;       // one TMA stage: L tile + R tile, fp32
  constexpr uint32_t kTmemA = 2 * NT;                      // first TMEM column of the L-operand ring
  static_assert(2 * NT + kConvStages * 64 <= 512, "TMEM budget");
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const PhiGeom& g = p.g;
  const int n = g.n;
  const int R = p.stages;
  const int nkb = (n + kKB - 1) / kKB;
  const int ks_last = ((n - (nkb - 1) * kKB) + 7) / 8;  // k-steps of the last k-block that hold data

  uint8_t* lo_ring = smem + static_cast<size_t>(R) * kRawBytes;               // [kConvStages][kBBytes]
  uint8_t* stage_out = lo_ring + kConvStages * kBBytes;                        // [4 warps][32 rows x 128 B]
  uint8_t* misc = stage_out + 4 * 4096;
  float* wbuf = reinterpret_cast<float*>(misc);  // [2][NT]
  uint64_t* bars = reinterpret_cast<uint64_t*>(misc + 2 * NT * 4);
  uint64_t* full = bars;                            // [R] TMA bytes landed
  uint64_t* rempty = bars + kTcMaxStages;           // [R] MMAs reading the raw stage have completed
  uint64_t* conv = bars + 2 * kTcMaxStages;         // [kConvStages] split operands ready (8 warp arrivals)
  uint64_t* cempty = conv + kConvStages;            // [kConvStages] MMAs reading them have completed
  uint64_t* tfull = cempty + kConvStages;           // [2] accumulator ready
  uint64_t* tempty = tfull + 2;                     // [2] accumulator drained (4 warp arrivals)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);

  if (threadIdx.x == 0) {
    for (int s = 0; s < R; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&rempty[s], 1);
    }
    for (int s = 0; s < kConvStages; ++s) {
      mbar_init(&conv[s], kConvWarps);
      mbar_init(&cempty[s], 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(&tfull[a], 1);
      mbar_init(&tempty[a], 4);
    }
    fence_mbar_init();
    tma_prefetch_desc(&mapL);
    tma_prefetch_desc(&mapR);
    tma_prefetch_desc(&mapO);
  }
  if (warp == 2) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  // NOTE on the two single-thread roles: the whole warp runs the loops and the mbarrier waits (warp-uniform
  // control flow) and one lane is picked with elect.sync only around the TMA / MMA instructions.  Those
  // instructions live on the uniform datapath; issued from a divergent `lane == 0` branch the compiler wraps
  // every one of them in an election loop, which made the MMA warp issue-bound (measured: ~110 instead of 80
  // cycles per MMA).
  if (warp == 0) {
    // ---------------------------------------------------------------------------------- TMA producer
    const uint64_t pol = l2_policy_evict_last();  // operands are re-read by many tiles: keep them in L2
    uint32_t it = 0;
    for (long long idx = blockIdx.x; idx < g.total; idx += gridDim.x) {
      const PhiTile t = phi_decode(g, idx);
      const long long item = static_cast<long long>(t.b) * g.P;
      const int rowL = static_cast<int>((item + phi_colbase(g.T, t.mid)) * n) + t.m_tile * kTM;
      const int blkR = static_cast<int>(item + phi_colbase(g.T, t.s) + (t.mid - t.s - 1));
      const int j0 = t.n_tile * NT;
      for (int kb = 0; kb < nkb; ++kb, ++it) {
        const int rs = it % R;
        const uint32_t use = it / R;
        if (use > 0) mbar_wait(&rempty[rs], (use - 1) & 1);
        uint8_t* sp = smem + static_cast<size_t>(rs) * kRawBytes;
        if (elect_one()) {
          mbar_arrive_expect_tx(&full[rs], ((p.dbg & 32) ? 0u : kABytes) + ((p.dbg & 64) ? 0u : kBBytes));
          if (!(p.dbg & 32)) tma_load_2d(sp, &mapL, kb * kKB, rowL, &full[rs], pol);
          if (!(p.dbg & 64)) {
#pragma unroll
            for (int c = 0; c < NCH; ++c)
              tma_load_3d(sp + kABytes + c * 4096, &mapR, j0 + 32 * c, kb * kKB, blkR, &full[rs], pol);
          }
        }
        __syncwarp();
      }
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------------------------- MMA issuer
    constexpr uint32_t idesc = umma_idesc_tf32(kTM, NT, 0, 1);
    uint32_t it = 0, lt = 0;
    for (long long idx = blockIdx.x; idx < g.total; idx += gridDim.x, ++lt) {
      const uint32_t acc = lt & 1;
      if (lt >= 2) mbar_wait(&tempty[acc], ((lt >> 1) - 1) & 1);
      tc_fence_after();
      const uint32_t d_tmem = tmem_base + acc * NT;
      for (int kb = 0; kb < nkb; ++kb, ++it) {
        const int rs = it % R, cs = it % kConvStages;
        if (!(p.dbg & 256)) mbar_wait(&conv[cs], (it / kConvStages) & 1);
        tc_fence_after();
        const uint32_t sb_hi = smem_u32(smem + static_cast<size_t>(rs) * kRawBytes + kABytes);
        const uint32_t sb_lo = smem_u32(lo_ring + static_cast<size_t>(cs) * kBBytes);
        const uint32_t a_hi = tmem_base + kTmemA + cs * 64;   // raw fp32 bits: the MMA keeps the top 19
        const uint32_t a_lo = a_hi + 32;
        const int nks = (kb == nkb - 1) ? ks_last : 4;
        if (elect_one()) {
#pragma unroll
          for (int ks = 0; ks < 4; ++ks) {
            if (ks < nks) {
              const uint64_t b_hi = umma_smem_desc(sb_hi + ks * 1024, 4096, 512, kUmmaSw128Base32);
              const uint64_t b_lo = umma_smem_desc(sb_lo + ks * 1024, 4096, 512, kUmmaSw128Base32);
              if (!(p.dbg & 16)) {
                umma_tf32_ts(d_tmem, a_lo + ks * 8, b_hi, idesc, (kb | ks) != 0);
                umma_tf32_ts(d_tmem, a_hi + ks * 8, b_lo, idesc, 1);
              }
              umma_tf32_ts(d_tmem, a_hi + ks * 8, b_hi, idesc, (p.dbg & 16) ? ((kb | ks) != 0) : 1);
            }
          }
          umma_commit(&rempty[rs]);
          umma_commit(&cempty[cs]);
          if (kb == nkb - 1) umma_commit(&tfull[acc]);
        }
        __syncwarp();
      }
    }
  } else if (warp >= 8) {
    // ---------------------------------------------------------------------------------- operand split
    // L: warp (q, h) moves rows 32q..32q+31, k-columns 16h..16h+15 of the swizzled landing tile into TMEM
    // (raw bits = hi, and lo); R: lo plane written to shared memory at the same byte offsets as the raw tile.
    const int ctid = threadIdx.x - 256;
    const int q = warp & 3, h = (warp - 8) >> 2;
    const int row = q * 32 + lane;
    uint32_t it = 0;
    for (long long idx = blockIdx.x; idx < g.total; idx += gridDim.x) {
      for (int kb = 0; kb < nkb; ++kb, ++it) {
        const int rs = it % R, cs = it % kConvStages;
        const uint32_t cuse = it / kConvStages;
        mbar_wait(&full[rs], (it / R) & 1);
        if (cuse > 0) {
          mbar_wait(&cempty[cs], (cuse - 1) & 1);
          tc_fence_after();
        }
        const uint8_t* sp = smem + static_cast<size_t>(rs) * kRawBytes;
        uint32_t vh[16], vl[16];
        if (!(p.dbg & 4))
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const float4 f = *reinterpret_cast<const float4*>(sp + row * 128 + (((4 * h + c) ^ (row & 7)) << 4));
          float hh;
          vh[4 * c + 0] = __float_as_uint(f.x); vl[4 * c + 0] = __float_as_uint(tf32_lo(f.x, hh));
          vh[4 * c + 1] = __float_as_uint(f.y); vl[4 * c + 1] = __float_as_uint(tf32_lo(f.y, hh));
          vh[4 * c + 2] = __float_as_uint(f.z); vl[4 * c + 2] = __float_as_uint(tf32_lo(f.z, hh));
          vh[4 * c + 3] = __float_as_uint(f.w); vl[4 * c + 3] = __float_as_uint(tf32_lo(f.w, hh));
        }
        const uint32_t ta = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + kTmemA + cs * 64 + h * 16;
        if (!(p.dbg & 128)) {
          tmem_st_32x16(ta, vh);
          tmem_st_32x16(ta + 32, vl);
        }
        const float4* br = reinterpret_cast<const float4*>(sp + kABytes);
        float4* bl = reinterpret_cast<float4*>(lo_ring + static_cast<size_t>(cs) * kBBytes);
        if (!(p.dbg & 2))
#pragma unroll
        for (int i = ctid; i < static_cast<int>(kBBytes / 16); i += 32 * kConvWarps) {
          const float4 a = br[i];
          float4 l;
          float hh;
          l.x = tf32_lo(a.x, hh); l.y = tf32_lo(a.y, hh); l.z = tf32_lo(a.z, hh); l.w = tf32_lo(a.w, hh);
          bl[i] = l;
        }
        if (!(p.dbg & 128)) {
          tmem_st_wait();
          fence_proxy_async_smem();
          tc_fence_before();
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&conv[cs]);
      }
    }
  } else if (warp >= 4) {
    // ---------------------------------------------------------------------------------- epilogue
    const int wq = warp - 4;            // == warp % 4: the TMEM lane quarter this warp may read
    const int etid = threadIdx.x - 128;
    uint32_t lt = 0;
    for (long long idx = blockIdx.x; idx < g.total; idx += gridDim.x, ++lt) {
      const PhiTile t = phi_decode(g, idx);
      const uint32_t acc = lt & 1;
      const int j0 = t.n_tile * NT;
      float* wb = wbuf + acc * NT;
      for (int j = etid; j < NT; j += 128)
        wb[j] = (j0 + j < n) ? __ldg(p.w + (static_cast<size_t>(t.b) * g.T + t.s) * n + j0 + j) : 0.f;
      named_bar_sync(1, 128);
      const size_t item = static_cast<size_t>(t.b) * g.P;
      const size_t qcol = item + phi_colbase(g.T, t.s) + (t.mid - t.s);  // block (mid+1, s)
      const int rho = t.m_tile * kTM + wq * 32 + lane;
      const bool valid = rho < t.cnt_t * n;
      float* out = p.phi + (qcol * n + rho) * n + j0;
      mbar_wait(&tfull[acc], (lt >> 1) & 1);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(wq * 32) << 16) + acc * NT;
      // all 32 rows of this warp inside the interval: swizzled shared-memory box + TMA store (coalesced, off the
      // LSU); otherwise (ragged last m-tile) masked row-per-thread stores
      const bool box_ok = (t.m_tile * kTM + wq * 32 + 31) < t.cnt_t * n && !(p.dbg & 8);
      const int row0 = static_cast<int>(qcol * n) + t.m_tile * kTM + wq * 32;
      uint8_t* sbox = stage_out + wq * 4096;
      float tube = 0.f;
#pragma unroll
      for (int cc = 0; cc < NCH; ++cc) {
        uint32_t v[32];
        tmem_ld_32x32(taddr + cc * 32, v);
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 32; ++e) tube = fmaf(fabsf(__uint_as_float(v[e])), wb[cc * 32 + e], tube);
        if (p.dbg & 1) continue;
        if (box_ok) {
          if (j0 + cc * 32 < n) {
            if (lane == 0) tma_store_wait_read<0>();   // the previous box of this warp has been read out
            __syncwarp();
#pragma unroll
            for (int e = 0; e < 8; ++e)
              *reinterpret_cast<uint4*>(sbox + lane * 128 + ((e ^ (lane & 7)) << 4)) =
                  make_uint4(v[4 * e], v[4 * e + 1], v[4 * e + 2], v[4 * e + 3]);
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) {
              tma_store_2d(&mapO, j0 + cc * 32, row0, sbox);
              tma_store_commit();
            }
          }
        } else if (valid) {
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            if (j0 + cc * 32 + 4 * e < n)
              st_global_f4_na(out + cc * 32 + 4 * e,
                              make_float4(__uint_as_float(v[4 * e]), __uint_as_float(v[4 * e + 1]),
                                          __uint_as_float(v[4 * e + 2]), __uint_as_float(v[4 * e + 3])));
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&tempty[acc]);
      if (valid) p.part[((qcol + rho / n) * g.NT + t.n_tile) * n + rho % n] = tube;
    }
    if (lane == 0) tma_store_wait_all<0>();   // shared memory must outlive the last bulk store
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc<512>(tmem_base);
  }
}

template <int NCH>
cudaError_t launch_tc(const TcParams& p, const TcMaps& maps, int num_sms, cudaStream_t stream) {
  constexpr uint32_t kBBytes = NCH * 4096u;
  constexpr uint32_t kRawBytes = kABytes + kBBytes;
  const uint32_t misc = 4 * 4096 + 2 * 32 * NCH * 4 + (2 * kTcMaxStages + 2 * kConvStages + 4) * 8 + 16;
  TcParams q = p;
  int st = static_cast<int>((227u * 1024u - 1024u - misc - kConvStages * kBBytes) / kRawBytes);
  if (st > kTcMaxStages) st = kTcMaxStages;
  if (st < 2) return cudaErrorInvalidConfiguration;
  q.stages = st;
  const uint32_t smem = 1024u + st * kRawBytes + kConvStages * kBBytes + misc;
  cudaError_t e = cudaFuncSetAttribute(phi_combine_tc_kernel<NCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e != cudaSuccess) return e;
  long long blocks = q.g.total < num_sms ? q.g.total : num_sms;
  ProfScope prof(kProfPhiCombineTc, stream);
  phi_combine_tc_kernel<NCH><<<static_cast<unsigned>(blocks), kTcThreads, smem, stream>>>(q, maps.L, maps.R, maps.O);
  return cudaGetLastError();
}

// =====================================================================================================
// cta_group::2 variant: a CTA pair (cluster of 2, the two SMs of one TPC) computes one 256 x NT tile.
// CTA `rank` owns rows [128 rank, 128 rank + 128) of the tile (its own L tile, TMEM accumulators and epilogue)
// and supplies columns [rank NT/2, (rank+1) NT/2) of the right operand, so per CTA the right-operand share of
// everything that goes through the 128 B/clk shared-memory port (TMA writes, split traffic, MMA operand
// reads) is halved - the port, not the tensor pipe, bounds the single-CTA kernel.
// Rank 0 issues every MMA (tcgen05.mma.cta_group::2); its `conv` / `tempty` barriers count the warps of BOTH
// CTAs (the peer arrives remotely), and its commits are multicast to the barriers of both CTAs.
template <int NCH>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kTcThreads, 1)
phi_combine_tc2_kernel(const TcParams p, const __grid_constant__ CUtensorMap mapL,
                       const __grid_constant__ CUtensorMap mapR, const __grid_constant__ CUtensorMap mapO) {
  constexpr int NT = 32 * NCH;
  constexpr int NH = NT / 2;                               // right-operand columns held by this CTA
  constexpr int NBOX = (NH + 31) / 32;                     // 32-column TMA boxes covering them
  constexpr uint32_t kBBytes = NBOX * 4096u;
  constexpr uint32_t kRawBytes = kABytes + kBBytes;
  constexpr uint32_t kTmemA = 2 * NT;
  static_assert(2 * NT + kConvStages * 64 <= 512, "TMEM budget");
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const PhiGeom& g = p.g;                                  // decoded with tm = 256
  const int n = g.n;
  const int R = p.stages;
  const int nkb = (n + kKB - 1) / kKB;
  const int ks_last = ((n - (nkb - 1) * kKB) + 7) / 8;
  const long long pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;

  uint8_t* lo_ring = smem + static_cast<size_t>(R) * kRawBytes;
  uint8_t* stage_out = lo_ring + kConvStages * kBBytes;
  uint8_t* misc = stage_out + 4 * 4096;
  float* wbuf = reinterpret_cast<float*>(misc);  // [2][NT]
  uint64_t* bars = reinterpret_cast<uint64_t*>(misc + 2 * NT * 4);
  uint64_t* full = bars;                            // [R] local TMA bytes landed
  uint64_t* rempty = bars + kTcMaxStages;           // [R] multicast commit
  uint64_t* conv = bars + 2 * kTcMaxStages;         // [kConvStages] rank 0 only: 16 warp arrivals (both CTAs)
  uint64_t* cempty = conv + kConvStages;            // [kConvStages] multicast commit
  uint64_t* tfull = cempty + kConvStages;           // [2] multicast commit
  uint64_t* tempty = tfull + 2;                     // [2] rank 0 only: 8 warp arrivals (both CTAs)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);

  if (threadIdx.x == 0) {
    for (int s = 0; s < R; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&rempty[s], 1);
    }
    for (int s = 0; s < kConvStages; ++s) {
      mbar_init(&conv[s], 2 * kConvWarps);
      mbar_init(&cempty[s], 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(&tfull[a], 1);
      mbar_init(&tempty[a], 8);
    }
    fence_mbar_init();
    tma_prefetch_desc(&mapL);
    tma_prefetch_desc(&mapR);
    tma_prefetch_desc(&mapO);
  }
  if (warp == 2) tmem_alloc_2cta<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();   // both CTAs' barriers and TMEM allocations exist before anything crosses the pair
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ---------------------------------------------------------------------------------- TMA producer (both CTAs)
    const uint64_t pol = l2_policy_evict_last();
    uint32_t it = 0;
    for (long long idx = pair; idx < g.total; idx += npairs) {
      const PhiTile t = phi_decode(g, idx);
      const long long item = static_cast<long long>(t.b) * g.P;
      const int rowL = static_cast<int>((item + phi_colbase(g.T, t.mid)) * n) + t.m_tile * 256 + rank * kTM;
      const int blkR = static_cast<int>(item + phi_colbase(g.T, t.s) + (t.mid - t.s - 1));
      const int j0 = t.n_tile * NT + rank * NH;
      for (int kb = 0; kb < nkb; ++kb, ++it) {
        const int rs = it % R;
        const uint32_t use = it / R;
        if (use > 0) mbar_wait(&rempty[rs], (use - 1) & 1);
        uint8_t* sp = smem + static_cast<size_t>(rs) * kRawBytes;
        if (elect_one()) {
          mbar_arrive_expect_tx(&full[rs], kRawBytes);
          tma_load_2d(sp, &mapL, kb * kKB, rowL, &full[rs], pol);
#pragma unroll
          for (int c = 0; c < NBOX; ++c)
            tma_load_3d(sp + kABytes + c * 4096, &mapR, j0 + 32 * c, kb * kKB, blkR, &full[rs], pol);
        }
        __syncwarp();
      }
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------------------------- MMA issuer (rank 0 only)
    if (rank == 0) {
      constexpr uint32_t idesc = umma_idesc_tf32(256, NT, 0, 1);
      uint32_t it = 0, lt = 0;
      for (long long idx = pair; idx < g.total; idx += npairs, ++lt) {
        const uint32_t acc = lt & 1;
        if (lt >= 2) mbar_wait(&tempty[acc], ((lt >> 1) - 1) & 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * NT;
        for (int kb = 0; kb < nkb; ++kb, ++it) {
          const int rs = it % R, cs = it % kConvStages;
          mbar_wait(&conv[cs], (it / kConvStages) & 1);
          tc_fence_after();
          const uint32_t sb_hi = smem_u32(smem + static_cast<size_t>(rs) * kRawBytes + kABytes);
          const uint32_t sb_lo = smem_u32(lo_ring + static_cast<size_t>(cs) * kBBytes);
          const uint32_t a_hi = tmem_base + kTmemA + cs * 64;
          const uint32_t a_lo = a_hi + 32;
          const int nks = (kb == nkb - 1) ? ks_last : 4;
          if (elect_one()) {
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
              if (ks < nks) {
                const uint64_t b_hi = umma_smem_desc(sb_hi + ks * 1024, 4096, 512, kUmmaSw128Base32);
                const uint64_t b_lo = umma_smem_desc(sb_lo + ks * 1024, 4096, 512, kUmmaSw128Base32);
                umma_tf32_ts_2cta(d_tmem, a_lo + ks * 8, b_hi, idesc, (kb | ks) != 0);
                umma_tf32_ts_2cta(d_tmem, a_hi + ks * 8, b_lo, idesc, 1);
                umma_tf32_ts_2cta(d_tmem, a_hi + ks * 8, b_hi, idesc, 1);
              }
            }
            umma_commit_2cta(&rempty[rs], 3);
            umma_commit_2cta(&cempty[cs], 3);
            if (kb == nkb - 1) umma_commit_2cta(&tfull[acc], 3);
          }
          __syncwarp();
        }
      }
    }
  } else if (warp >= 8) {
    // ---------------------------------------------------------------------------------- operand split (both CTAs)
    const int ctid = threadIdx.x - 256;
    const int q = warp & 3, h = (warp - 8) >> 2;
    const int row = q * 32 + lane;
    uint32_t it = 0;
    for (long long idx = pair; idx < g.total; idx += npairs) {
      for (int kb = 0; kb < nkb; ++kb, ++it) {
        const int rs = it % R, cs = it % kConvStages;
        const uint32_t cuse = it / kConvStages;
        mbar_wait(&full[rs], (it / R) & 1);
        if (cuse > 0) {
          mbar_wait(&cempty[cs], (cuse - 1) & 1);
          tc_fence_after();
        }
        const uint8_t* sp = smem + static_cast<size_t>(rs) * kRawBytes;
        uint32_t vh[16], vl[16];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const float4 f = *reinterpret_cast<const float4*>(sp + row * 128 + (((4 * h + c) ^ (row & 7)) << 4));
          float hh;
          vh[4 * c + 0] = __float_as_uint(f.x); vl[4 * c + 0] = __float_as_uint(tf32_lo(f.x, hh));
          vh[4 * c + 1] = __float_as_uint(f.y); vl[4 * c + 1] = __float_as_uint(tf32_lo(f.y, hh));
          vh[4 * c + 2] = __float_as_uint(f.z); vl[4 * c + 2] = __float_as_uint(tf32_lo(f.z, hh));
          vh[4 * c + 3] = __float_as_uint(f.w); vl[4 * c + 3] = __float_as_uint(tf32_lo(f.w, hh));
        }
        const uint32_t ta = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + kTmemA + cs * 64 + h * 16;
        tmem_st_32x16(ta, vh);
        tmem_st_32x16(ta + 32, vl);
        const float4* br = reinterpret_cast<const float4*>(sp + kABytes);
        float4* bl = reinterpret_cast<float4*>(lo_ring + static_cast<size_t>(cs) * kBBytes);
#pragma unroll
        for (int i = ctid; i < static_cast<int>(kBBytes / 16); i += 32 * kConvWarps) {
          const float4 a = br[i];
          float4 l;
          float hh;
          l.x = tf32_lo(a.x, hh); l.y = tf32_lo(a.y, hh); l.z = tf32_lo(a.z, hh); l.w = tf32_lo(a.w, hh);
          bl[i] = l;
        }
        tmem_st_wait();
        fence_proxy_async_smem();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_remote_relaxed(&conv[cs], 0);
      }
    }
  } else if (warp >= 4) {
    // ---------------------------------------------------------------------------------- epilogue (both CTAs)
    const int wq = warp - 4;
    const int etid = threadIdx.x - 128;
    uint32_t lt = 0;
    for (long long idx = pair; idx < g.total; idx += npairs, ++lt) {
      const PhiTile t = phi_decode(g, idx);
      const uint32_t acc = lt & 1;
      const int j0 = t.n_tile * NT;
      float* wb = wbuf + acc * NT;
      for (int j = etid; j < NT; j += 128)
        wb[j] = (j0 + j < n) ? __ldg(p.w + (static_cast<size_t>(t.b) * g.T + t.s) * n + j0 + j) : 0.f;
      named_bar_sync(1, 128);
      const size_t item = static_cast<size_t>(t.b) * g.P;
      const size_t qcol = item + phi_colbase(g.T, t.s) + (t.mid - t.s);
      const int rbase = t.m_tile * 256 + static_cast<int>(rank) * kTM + wq * 32;
      const int rho = rbase + lane;
      const bool valid = rho < t.cnt_t * n;
      float* out = p.phi + (qcol * n + rho) * n + j0;
      mbar_wait(&tfull[acc], (lt >> 1) & 1);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(wq * 32) << 16) + acc * NT;
      const bool box_ok = (rbase + 31) < t.cnt_t * n;
      const int row0 = static_cast<int>(qcol * n) + rbase;
      uint8_t* sbox = stage_out + wq * 4096;
      float tube = 0.f;
#pragma unroll
      for (int cc = 0; cc < NCH; ++cc) {
        uint32_t v[32];
        tmem_ld_32x32(taddr + cc * 32, v);
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 32; ++e) tube = fmaf(fabsf(__uint_as_float(v[e])), wb[cc * 32 + e], tube);
        if (box_ok) {
          if (j0 + cc * 32 < n) {
            if (lane == 0) tma_store_wait_read<0>();
            __syncwarp();
#pragma unroll
            for (int e = 0; e < 8; ++e)
              *reinterpret_cast<uint4*>(sbox + lane * 128 + ((e ^ (lane & 7)) << 4)) =
                  make_uint4(v[4 * e], v[4 * e + 1], v[4 * e + 2], v[4 * e + 3]);
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) {
              tma_store_2d(&mapO, j0 + cc * 32, row0, sbox);
              tma_store_commit();
            }
          }
        } else if (valid) {
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            if (j0 + cc * 32 + 4 * e < n)
              st_global_f4_na(out + cc * 32 + 4 * e,
                              make_float4(__uint_as_float(v[4 * e]), __uint_as_float(v[4 * e + 1]),
                                          __uint_as_float(v[4 * e + 2]), __uint_as_float(v[4 * e + 3])));
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_remote_relaxed(&tempty[acc], 0);
      if (valid) p.part[((qcol + rho / n) * g.NT + t.n_tile) * n + rho % n] = tube;
    }
    if (lane == 0) tma_store_wait_all<0>();
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();   // the peer may still be reading this CTA's TMEM / shared memory through the pair MMA
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc_2cta<512>(tmem_base);
  }
}

template <int NCH>
cudaError_t launch_tc2(const TcParams& p, const TcMaps& maps, int num_sms, cudaStream_t stream) {
  constexpr uint32_t kBBytes = ((32 * NCH / 2 + 31) / 32) * 4096u;
  constexpr uint32_t kRawBytes = kABytes + kBBytes;
  const uint32_t misc = 4 * 4096 + 2 * 32 * NCH * 4 + (2 * kTcMaxStages + 2 * kConvStages + 4) * 8 + 16;
  TcParams q = p;
  int st = static_cast<int>((227u * 1024u - 1024u - misc - kConvStages * kBBytes) / kRawBytes);
  if (st > kTcMaxStages) st = kTcMaxStages;
  if (st < 2) return cudaErrorInvalidConfiguration;
  q.stages = st;
  const uint32_t smem = 1024u + st * kRawBytes + kConvStages * kBBytes + misc;
  cudaError_t e =
      cudaFuncSetAttribute(phi_combine_tc2_kernel<NCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e != cudaSuccess) return e;
  const long long max_pairs = num_sms / 2;
  const long long pairs = q.g.total < max_pairs ? q.g.total : max_pairs;
  ProfScope prof(kProfPhiCombineTc, stream);
  phi_combine_tc2_kernel<NCH><<<static_cast<unsigned>(2 * pairs), kTcThreads, smem, stream>>>(q, maps.L, maps.R,
                                                                                               maps.O);
  return cudaGetLastError();
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

size_t phi_tc_maps_size() { return sizeof(TcMaps); }

cudaError_t phi_tc_make_maps(const PhiArgs& a, int nch, void* maps_out) {
  (void)nch;
  EncodeTiledFn enc = reinterpret_cast<EncodeTiledFn>(get_encode_tiled());
  if (!enc) return cudaErrorNotSupported;
  TcMaps* m = static_cast<TcMaps*>(maps_out);
  const cuuint64_t P = static_cast<cuuint64_t>(a.T) * (a.T - 1) / 2;
  const cuuint64_t n = a.n;
  const cuuint32_t estr[3] = {1, 1, 1};
  {
    const cuuint64_t dims[2] = {n, static_cast<cuuint64_t>(a.batch) * P * n};
    const cuuint64_t strides[1] = {n * 4};
    const cuuint32_t box[2] = {kKB, kTM};
    if (enc(&m->L, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, a.phi, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  {
    const cuuint64_t dims[3] = {n, n, static_cast<cuuint64_t>(a.batch) * P};
    const cuuint64_t strides[2] = {n * 4, n * n * 4};
    const cuuint32_t box[3] = {32, kKB, 1};
    if (enc(&m->R, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, a.phi, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  {
    const cuuint64_t dims[2] = {n, static_cast<cuuint64_t>(a.batch) * P * n};
    const cuuint64_t strides[1] = {n * 4};
    const cuuint32_t box[2] = {32, 32};
    if (enc(&m->O, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, a.phi, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  return cudaSuccess;
}

cudaError_t launch_phi_combine_tc(const PhiArgs& a, int level, int nch, const void* maps, int num_sms,
                                  cudaStream_t stream) {
  TcParams p{};
  p.phi = a.phi; p.w = a.w; p.part = a.part;
  p.dbg = env_int("TC_DBG", 0);
  const TcMaps& m = *static_cast<const TcMaps*>(maps);
  // CTA pairs (256-row tiles) when the level's stacked left operand is tall enough to fill them; the
  // single-CTA kernel (128-row tiles) on the low levels where 256-row tiles would be mostly padding
  const PhiGeom g1 = phi_geom(a.batch, a.T, a.n, level, kTM, 32 * nch);
  const PhiGeom g2 = phi_geom(a.batch, a.T, a.n, level, 2 * kTM, 32 * nch);
  if (g1.total == 0) return cudaSuccess;
  const int mode = env_int("TC_PAIR", -1);   // -1 auto, 0 never, 1 always
  const bool pair = (mode == 1) || (mode == -1 && (nch % 2 == 1 || nch >= 2) && 2 * g2.total * 100 <= g1.total * 108);
  if (pair) {
    p.g = g2;
    switch (nch) {
      case 2: return launch_tc2<2>(p, m, num_sms, stream);
      case 3: return launch_tc2<3>(p, m, num_sms, stream);
      case 4: return launch_tc2<4>(p, m, num_sms, stream);
      case 5: return launch_tc2<5>(p, m, num_sms, stream);
      default: return cudaErrorInvalidValue;
    }
  }
  p.g = g1;
  switch (nch) {
    case 2: return launch_tc<2>(p, m, num_sms, stream);
    case 3: return launch_tc<3>(p, m, num_sms, stream);
    case 4: return launch_tc<4>(p, m, num_sms, stream);
    case 5: return launch_tc<5>(p, m, num_sms, stream);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace ltv
