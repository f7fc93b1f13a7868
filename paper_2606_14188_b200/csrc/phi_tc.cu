// Phi path, levels >= 1, n >= 96: the divide-and-conquer combine Phi(t,s) = Phi(t,mid) Phi(mid,s) as a
// persistent, warp-specialised tcgen05 GEMM with 3xTF32 operand splitting and the tube reduction
// r_t += |Phi(t,s)| w_s fused into the TMEM epilogue (eq.(12c), :147 eq.(12e), :166, :177).
//
//   D[(t,i), j] = sum_k  L[(t,i), k] * R[k, j],   L = stacked Phi(t,mid) (K-major), R = Phi(mid,s) (N-major)
//
// One kernel template, two shapes:
//   PAIR = false  one CTA per 128 x NT tile (tcgen05 cta_group::1); used on the low levels whose stacked
//                 left operand is too short to fill 256 rows
//   PAIR = true   a CTA pair (cluster of 2, the two SMs of a TPC) per 256 x NT tile (cta_group::2): CTA
//                 `rank` owns rows [128 rank, 128 rank + 128) (its own L tile, accumulators, epilogue) and
//                 supplies columns [rank NT/2, (rank+1) NT/2) of the right operand, which halves the
//                 right-operand share of everything that crosses the 128 B/clk shared-memory port.  Rank 0
//                 issues every MMA; its `conv` / `tempty` barriers count the warps of both CTAs (the peer
//                 arrives remotely) and its commits are multicast to the barriers of both CTAs.
// NT = 32 NCH columns (NCH <= 5), K = n in blocks of 32.  Roles (512 threads):
//   warp 0       TMA producer: fp32 tiles of L (one 128x32 box, SWIZZLE_128B) and R (32x32 boxes,
//                SWIZZLE_128B_ATOM_32B: the only MN-major layout kind::tf32 accepts) into a ring of R stages
//   warps 8-15   operand split, lo = rna_tf32(a - trunc_tf32(a)).  Two groups of four warps take ALTERNATE
//                k-blocks: the split of one k-block is a serial chain of latencies (barrier waits, shared
//                loads, TMEM stores, proxy fence; measured ~1100 cycles with in-kernel clock traces) against
//                960 cycles of MMA issue per k-block, so two k-blocks must be in flight.  The L tile goes
//                from shared memory into TMEM as two 128-lane x 32-column operands (raw bits = hi, since
//                kind::tf32 reads only the top 19 bits, and lo); the lo plane of R is written to shared
//                memory at the same byte offsets as the raw tile (position-preserving, so no knowledge of
//                the swizzle is needed).  Ring of 3.
//   warp 1       one thread issues, per 8-deep k-step: D += Llo*Rhi, D += Lhi*Rlo, D += Lhi*Rhi (small first),
//                L from TMEM, R from shared memory
//   warps 4-7    epilogue: TMEM -> registers (next chunk's tcgen05.ld in flight) -> per-row |D| w partial sum
//                -> swizzled 32x32 shared-memory box -> bulk tensor store (masked row-per-thread stores on the
//                ragged last m-tile of a column)
// Why L goes through TMEM: with both operands in shared memory a k-block moves 216 KB through the shared-
// memory port against 960 cycles of MMA issue (measured 47 % tensor-pipe activity with the first version of round 1).
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
constexpr int kConvStages = 3;  // ring of split operands: L (hi, lo) in TMEM, R lo plane in shared memory
constexpr int kTM = 128;        // rows per CTA
constexpr int kKB = 32;         // k-block = one 128-byte swizzle row of fp32
constexpr uint32_t kABytes = kTM * kKB * 4;  // 16 KB
constexpr int kTcMaxStages = 6;

// MODE 1 of the kernel: `count` independent products D[b] = L[b] R[b] (batched GEMM of the Kalman recursion,
// eq.(13)); problem b reads rows [l_row0 + b l_row_stride, +M) of the L map, block r_blk0 + b r_blk_stride of the R
// map and writes block d_blk0 + b d_blk_stride of the (3-D) O map
struct TcGemm {
  int count, M, Mt;
  int d_rows;              // rows of one D block in memory (>= M; rows [M, d_rows) are never written)
  int l_row0, l_row_stride, r_blk0, r_blk_stride, d_blk0, d_blk_stride;
  int transpose_out;       // store D^T (the O map then describes [blocks][N][M])
  const float* diag;       // adds diag[b diag_stride + i]^2 to D[b][i][i] (E E^T with E = diag(e)); may be null
  long long diag_stride;
  int d_row0, d_row_stride;   // row offset of problem b inside its D block: d_row0 + b d_row_stride (plain stores only)
};

struct TcParams {
  TcGemm gm;
  float* phi;
  const float* w;
  float* part;
  PhiGeom g;
  int stages;
  int tube_mode;              // 0: |d| w, 1: (d w)^2 (row-wise two-norm tube; the finalise kernel takes the root)
};

struct TcMaps {
  CUtensorMap L;  // 2-D [batch*P*n rows][n]           box 32 x 128
  CUtensorMap R;  // 3-D [batch*P blocks][n][n]        box 32 x 32 x 1
  CUtensorMap O;  // 2-D [batch*P*n rows][n]           box 32 x 32 (epilogue stores)
  CUtensorMap L2, R2;   // MODE 2: second operand pair of the K loop (same geometry, other arrays)
};

__device__ __forceinline__ float tf32_lo(float a) {
  const float hi = __uint_as_float(__float_as_uint(a) & 0xffffe000u);
  const float d = a - hi;
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(d));
  return __uint_as_float(r);
}

struct GemmTile { int b, m_tile, n_tile; };
// m_tile fastest: CTAs running at the same time share the right-operand tile out of L2
__device__ __forceinline__ GemmTile gemm_decode(const TcGemm& gm, int NTiles, long long idx) {
  GemmTile t;
  int rem = static_cast<int>(idx);
  t.m_tile = rem % gm.Mt;
  rem /= gm.Mt;
  t.n_tile = rem % NTiles;
  t.b = rem / NTiles;
  return t;
}

template <int NCH, bool PAIR>
struct TcShape {
  static constexpr int NT = 32 * NCH;
  static constexpr int NCTA = PAIR ? 2 : 1;
  static constexpr int NH = NT / NCTA;                      // right-operand columns held by one CTA
  static constexpr int NBOX = (NH + 31) / 32;               // 32-column TMA boxes covering them
  static constexpr uint32_t kBBytes = NBOX * 4096u;
  static constexpr uint32_t kRawBytes = kABytes + kBBytes;  // one TMA stage: L tile + R tile, fp32
  static constexpr uint32_t kTmemA = 2 * NT;                // first TMEM column of the L-operand ring
  static constexpr uint32_t kMisc = 4 * 4096 + 2 * NT * 4 + (2 * kTcMaxStages + 2 * kConvStages + 4) * 8 + 16;
  static_assert(2 * NT + kConvStages * 64 <= 512, "TMEM budget");
  static_assert(NT % (16 * NCTA) == 0, "UMMA N granularity");
};

template <int NCH, bool PAIR, int MODE>
__global__ void __launch_bounds__(kTcThreads, 1)
phi_combine_tc_kernel(const TcParams p, const __grid_constant__ CUtensorMap mapL,
                      const __grid_constant__ CUtensorMap mapR, const __grid_constant__ CUtensorMap mapO,
                      const __grid_constant__ CUtensorMap mapL2, const __grid_constant__ CUtensorMap mapR2) {
  using S = TcShape<NCH, PAIR>;
  constexpr int NT = S::NT, NH = S::NH, NBOX = S::NBOX, NCTA = S::NCTA;
  constexpr uint32_t kBBytes = S::kBBytes, kRawBytes = S::kRawBytes, kTmemA = S::kTmemA;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = PAIR ? cluster_ctarank() : 0u;
  const PhiGeom& g = p.g;   // decoded with tm = 128 NCTA
  const int n = g.n;     // K extent and rows per block
  const int nc = g.nc;   // columns per block = row stride of Phi (n, or n + padded p: the observer's PhiY columns)
  const int R = p.stages;
  const int nkb = (n + kKB - 1) / kKB;
  const int ks_last = ((n - (nkb - 1) * kKB) + 7) / 8;  // k-steps of the last k-block that hold data
  // MODE 2 (cross block of a block-triangular system): D = L1 R1 + L2 R2, the K loop runs over both operand pairs
  const int nkb_tot = (MODE == 2) ? 2 * nkb : nkb;
  const long long unit = PAIR ? (blockIdx.x >> 1) : blockIdx.x;
  const long long nunits = PAIR ? (gridDim.x >> 1) : gridDim.x;

  uint8_t* lo_ring = smem + static_cast<size_t>(R) * kRawBytes;               // [kConvStages][kBBytes]
  uint8_t* stage_out = lo_ring + kConvStages * kBBytes;                        // [4 warps][32 rows x 128 B]
  uint8_t* misc = stage_out + 4 * 4096;
  float* wbuf = reinterpret_cast<float*>(misc);  // [2][NT]
  uint64_t* bars = reinterpret_cast<uint64_t*>(misc + 2 * NT * 4);
  uint64_t* full = bars;                            // [R] local TMA bytes landed
  uint64_t* rempty = bars + kTcMaxStages;           // [R] MMAs reading the raw stage have completed
  uint64_t* conv = bars + 2 * kTcMaxStages;         // [kConvStages] leader: split operands ready (4 NCTA warps)
  uint64_t* cempty = conv + kConvStages;            // [kConvStages] MMAs reading them have completed
  uint64_t* tfull = cempty + kConvStages;           // [2] accumulator ready
  uint64_t* tempty = tfull + 2;                     // [2] leader: accumulator drained (4 NCTA warps)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);

  if (threadIdx.x == 0) {
    for (int s = 0; s < R; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&rempty[s], 1);
    }
    for (int s = 0; s < kConvStages; ++s) {
      mbar_init(&conv[s], 4 * NCTA);
      mbar_init(&cempty[s], 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(&tfull[a], 1);
      mbar_init(&tempty[a], 4 * NCTA);
    }
    fence_mbar_init();
    tma_prefetch_desc(&mapL);
    tma_prefetch_desc(&mapR);
    tma_prefetch_desc(&mapO);
    if (MODE == 2) {
      tma_prefetch_desc(&mapL2);
      tma_prefetch_desc(&mapR2);
    }
  }
  if (warp == 2) {
    if (PAIR) tmem_alloc_2cta<512>(tmem_slot); else tmem_alloc<512>(tmem_slot);
  }
  tc_fence_before();
  __syncthreads();
  if (PAIR) cluster_sync_all();   // both CTAs' barriers and TMEM allocations exist before anything crosses the pair
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  auto arrive_leader = [&](uint64_t* bar) {
    if (PAIR) mbar_arrive_remote_relaxed(bar, 0); else mbar_arrive(bar);
  };

  // NOTE on the two single-thread roles: the whole warp runs the loops and the mbarrier waits (warp-uniform
  // control flow) and one lane is picked with elect.sync only around the TMA / MMA instructions.  Those
  // instructions live on the uniform datapath; issued from a divergent `lane == 0` branch the compiler wraps
  // every one of them in an election loop, which made the MMA warp issue-bound.
  if (warp == 0) {
    // ---------------------------------------------------------------------------------- TMA producer
    const uint64_t pol = l2_policy_evict_last();  // operands are re-read by many tiles: keep them in L2
    uint32_t it = 0;
    int rs = 0;
    uint32_t eph = 1;   // parity of rempty[rs] to wait for (the first pass over the ring does not block)
    for (long long idx = unit; idx < g.total; idx += nunits) {
      int rowL, blkR, j0;
      if (MODE != 1) {
        const PhiTile t = phi_decode(g, idx);
        const long long item = static_cast<long long>(t.b) * g.P;
        rowL = static_cast<int>((item + phi_colbase(g.T, t.mid)) * n) + t.m_tile * (kTM * NCTA) +
               static_cast<int>(rank) * kTM;
        blkR = static_cast<int>(item + phi_colbase(g.T, t.s) + (t.mid - t.s - 1));
        j0 = t.n_tile * NT + static_cast<int>(rank) * NH;
      } else {
        const GemmTile t = gemm_decode(p.gm, g.NT, idx);
        rowL = p.gm.l_row0 + t.b * p.gm.l_row_stride + t.m_tile * (kTM * NCTA) + static_cast<int>(rank) * kTM;
        blkR = p.gm.r_blk0 + t.b * p.gm.r_blk_stride;
        j0 = t.n_tile * NT + static_cast<int>(rank) * NH;
      }
      for (int kb = 0; kb < nkb_tot; ++kb, ++it) {
        mbar_wait(&rempty[rs], eph);
        uint8_t* sp = smem + static_cast<size_t>(rs) * kRawBytes;
        const bool second = (MODE == 2) && kb >= nkb;
        const int kc = (second ? kb - nkb : kb) * kKB;
        const CUtensorMap* mL = second ? &mapL2 : &mapL;
        const CUtensorMap* mR = second ? &mapR2 : &mapR;
        if (elect_one()) {
          mbar_arrive_expect_tx(&full[rs], kRawBytes);
          tma_load_2d(sp, mL, kc, rowL, &full[rs], pol);
#pragma unroll
          for (int c = 0; c < NBOX; ++c)
            tma_load_3d(sp + kABytes + c * 4096, mR, j0 + 32 * c, kc, blkR, &full[rs], pol);
        }
        __syncwarp();
        if (++rs == R) { rs = 0; eph ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------------------------- MMA issuer (leader CTA)
    if (rank == 0) {
      constexpr uint32_t idesc = umma_idesc_tf32(kTM * NCTA, NT, 0, 1);
      uint32_t it = 0, lt = 0;
      int rs = 0, cs = 0;
      uint32_t cph = 0;
      for (long long idx = unit; idx < g.total; idx += nunits, ++lt) {
        const uint32_t acc = lt & 1;
        if (lt >= 2) mbar_wait(&tempty[acc], ((lt >> 1) - 1) & 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * NT;
        for (int kb = 0; kb < nkb_tot; ++kb, ++it) {
          mbar_wait(&conv[cs], cph);
          tc_fence_after();
          const uint32_t sb_hi = smem_u32(smem + static_cast<size_t>(rs) * kRawBytes + kABytes);
          const uint32_t sb_lo = smem_u32(lo_ring + static_cast<size_t>(cs) * kBBytes);
          const uint32_t a_hi = tmem_base + kTmemA + cs * 64;   // raw fp32 bits: the MMA keeps the top 19
          const uint32_t a_lo = a_hi + 32;
          const int nks = (kb == nkb - 1 || kb == nkb_tot - 1) ? ks_last : 4;
          if (elect_one()) {
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
              if (ks < nks) {
                const uint64_t b_hi = umma_smem_desc(sb_hi + ks * 1024, 4096, 512, kUmmaSw128Base32);
                const uint64_t b_lo = umma_smem_desc(sb_lo + ks * 1024, 4096, 512, kUmmaSw128Base32);
                umma_tf32_ts<PAIR>(d_tmem, a_lo + ks * 8, b_hi, idesc, (kb | ks) != 0);
                umma_tf32_ts<PAIR>(d_tmem, a_hi + ks * 8, b_lo, idesc, 1);
                umma_tf32_ts<PAIR>(d_tmem, a_hi + ks * 8, b_hi, idesc, 1);
              }
            }
            umma_commit_all<PAIR>(&rempty[rs]);
            umma_commit_all<PAIR>(&cempty[cs]);
            if (kb == nkb_tot - 1) umma_commit_all<PAIR>(&tfull[acc]);
          }
          __syncwarp();
          if (++rs == R) rs = 0;
          if (++cs == kConvStages) { cs = 0; cph ^= 1; }
        }
      }
    }
  } else if (warp >= 8) {
    // ---------------------------------------------------------------------------------- operand split
    // group warp q: rows 32q..32q+31 of the L tile (all 32 k-columns) -> TMEM; a quarter of the R tile's lo plane
    const int grp = (warp - 8) >> 2;
    const int q = warp & 3;
    const int gtid = q * 32 + lane;
    const int row = q * 32 + lane;
    constexpr int kRVec = static_cast<int>(kBBytes / 16) / 128;   // float4 per thread of the R tile
    static_assert(kRVec * 128 * 16 == kBBytes, "R tile must split evenly over the 128 threads of a group");
    uint32_t it = 0;
    int rs = 0, cs = 0;
    uint32_t rph = 0, cph = 1;   // parity of full[rs]; parity of cempty[cs] (the first use does not block)
    for (long long idx = unit; idx < g.total; idx += nunits) {
      for (int kb = 0; kb < nkb_tot; ++kb, ++it) {
        if (static_cast<int>(it & 1) == grp) {
          mbar_wait(&full[rs], rph);
          const uint8_t* sp = smem + static_cast<size_t>(rs) * kRawBytes;
          // the raw tile is only read: load the L rows before waiting for the split ring slot
          uint32_t v[32];
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            const uint4 f = *reinterpret_cast<const uint4*>(sp + row * 128 + ((c ^ (row & 7)) << 4));
            v[4 * c + 0] = f.x; v[4 * c + 1] = f.y; v[4 * c + 2] = f.z; v[4 * c + 3] = f.w;
          }
          mbar_wait(&cempty[cs], cph);
          tc_fence_after();
          const uint32_t ta = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + kTmemA + cs * 64;
          tmem_st_32x32(ta, v);
#pragma unroll
          for (int e = 0; e < 32; ++e) v[e] = __float_as_uint(tf32_lo(__uint_as_float(v[e])));
          tmem_st_32x32(ta + 32, v);
          {
            const float4* br = reinterpret_cast<const float4*>(sp + kABytes);
            float4* bl = reinterpret_cast<float4*>(lo_ring + static_cast<size_t>(cs) * kBBytes);
#pragma unroll
            for (int i = 0; i < kRVec; ++i) {
              const float4 a = br[gtid + 128 * i];
              bl[gtid + 128 * i] = make_float4(tf32_lo(a.x), tf32_lo(a.y), tf32_lo(a.z), tf32_lo(a.w));
            }
          }
          tmem_st_wait();
          fence_proxy_async_smem();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) arrive_leader(&conv[cs]);
        }
        if (++rs == R) { rs = 0; rph ^= 1; }
        if (++cs == kConvStages) { cs = 0; cph ^= 1; }
      }
    }
  } else if (warp >= 4) {
    // ---------------------------------------------------------------------------------- epilogue
    const int wq = warp - 4;            // == warp % 4: the TMEM lane quarter this warp may read
    const int etid = threadIdx.x - 128;
    uint8_t* sbox = stage_out + wq * 4096;
    const bool two_norm = p.tube_mode != 0;
    uint32_t lt = 0;
    for (long long idx = unit; idx < g.total; idx += nunits, ++lt) {
      const uint32_t acc = lt & 1;
      if (MODE == 1) {
        // ------------------------------------------------------------ batched GEMM epilogue (Kalman recursion)
        const GemmTile t = gemm_decode(p.gm, g.NT, idx);
        const int j0 = t.n_tile * NT;
        const int rbase = t.m_tile * (kTM * NCTA) + static_cast<int>(rank) * kTM + wq * 32;
        const int rr = rbase + lane;                 // row of D[b] held by this thread
        const int rows_valid = p.gm.M - rbase;
        const int oblk = p.gm.d_blk0 + t.b * p.gm.d_blk_stride;
        const int roff = p.gm.d_row0 + t.b * p.gm.d_row_stride;
        const bool tr = p.gm.transpose_out != 0;
        float dd = 0.f;
        if (p.gm.diag != nullptr && rr < p.gm.M) {
          const float d = __ldg(p.gm.diag + static_cast<long long>(t.b) * p.gm.diag_stride + rr);
          dd = d * d;
        }
        mbar_wait(&tfull[acc], (lt >> 1) & 1);
        tc_fence_after();
        const uint32_t taddr = tmem_base + (static_cast<uint32_t>(wq * 32) << 16) + acc * NT;
        uint32_t v[2][32];
        tmem_ld_32x32(taddr, v[0]);
#pragma unroll
        for (int cc = 0; cc < NCH; ++cc) {
          uint32_t (&vc)[32] = v[cc & 1];
          tmem_ld_wait();
          if (cc + 1 < NCH) tmem_ld_32x32(taddr + (cc + 1) * 32, v[(cc + 1) & 1]);
          const int jc = j0 + cc * 32;
          if (jc >= nc || rows_valid <= 0) continue;
          if (rr >= jc && rr < jc + 32) {
#pragma unroll
            for (int e = 0; e < 32; ++e)
              if (jc + e == rr) vc[e] = __float_as_uint(__uint_as_float(vc[e]) + dd);
          }
          if (!tr && rows_valid < 32) {
            // ragged last m-tile, plain store: rows [M, d_rows) of the block belong to the caller (masked stores)
            if (lane < rows_valid) {
              float* out = p.phi + (static_cast<size_t>(oblk) * p.gm.d_rows + rr + roff) * nc + jc;
#pragma unroll
              for (int e = 0; e < 8; ++e) {
                if (jc + 4 * e < nc)
                  st_global_f4_na(out + 4 * e, make_float4(__uint_as_float(vc[4 * e]), __uint_as_float(vc[4 * e + 1]),
                                                           __uint_as_float(vc[4 * e + 2]), __uint_as_float(vc[4 * e + 3])));
              }
            }
            continue;
          }
          if (lane == 0) tma_store_wait_read<0>();
          __syncwarp();
          if (!tr) {
#pragma unroll
            for (int e = 0; e < 8; ++e)
              *reinterpret_cast<uint4*>(sbox + lane * 128 + ((e ^ (lane & 7)) << 4)) =
                  make_uint4(vc[4 * e], vc[4 * e + 1], vc[4 * e + 2], vc[4 * e + 3]);
          } else {
            // box row e = column jc + e of D, position `lane` = row rbase + lane of D: the transposed tile
#pragma unroll
            for (int e = 0; e < 32; ++e)
              *reinterpret_cast<uint32_t*>(sbox + e * 128 + ((((lane >> 2) ^ (e & 7)) << 4) | ((lane & 3) << 2))) = vc[e];
          }
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            // rows / columns beyond the block are clipped by the 3-D tensor map
            if (!tr) tma_store_3d(&mapO, jc, rbase + roff, oblk, sbox); else tma_store_3d(&mapO, rbase, jc, oblk, sbox);
            tma_store_commit();
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) arrive_leader(&tempty[acc]);
        continue;
      }
      const PhiTile t = phi_decode(g, idx);
      const int j0 = t.n_tile * NT;
      float* wb = wbuf + acc * NT;
      for (int j = etid; j < NT; j += 128)
        wb[j] = (MODE == 0 && j0 + j < n) ? __ldg(p.w + (static_cast<size_t>(t.b) * g.T + t.s) * n + j0 + j) : 0.f;
      named_bar_sync(1, 128);
      const size_t item = static_cast<size_t>(t.b) * g.P;
      const size_t qcol = item + phi_colbase(g.T, t.s) + (t.mid - t.s);  // block (mid+1, s)
      const int rbase = t.m_tile * (kTM * NCTA) + static_cast<int>(rank) * kTM + wq * 32;
      const int rho = rbase + lane;
      const int rows_valid = t.cnt_t * n - rbase;   // rows of this warp's 32 that exist (may be <= 0 or >= 32)
      float* out = p.phi + (qcol * n + rbase) * nc + j0;
      const int row0 = static_cast<int>(qcol * n) + rbase;
      mbar_wait(&tfull[acc], (lt >> 1) & 1);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(wq * 32) << 16) + acc * NT;
      float tube4[4] = {0.f, 0.f, 0.f, 0.f};
      uint32_t v[2][32];
      tmem_ld_32x32(taddr, v[0]);
#pragma unroll
      for (int cc = 0; cc < NCH; ++cc) {
        uint32_t (&vc)[32] = v[cc & 1];
        tmem_ld_wait();
        if (cc + 1 < NCH) tmem_ld_32x32(taddr + (cc + 1) * 32, v[(cc + 1) & 1]);
        if (MODE == 0) {
          const float4* w4 = reinterpret_cast<const float4*>(wb + cc * 32);
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            const float4 ww = w4[e];
            const float d0 = __uint_as_float(vc[4 * e + 0]) * ww.x, d1 = __uint_as_float(vc[4 * e + 1]) * ww.y;
            const float d2 = __uint_as_float(vc[4 * e + 2]) * ww.z, d3 = __uint_as_float(vc[4 * e + 3]) * ww.w;
            tube4[0] += two_norm ? d0 * d0 : fabsf(d0);
            tube4[1] += two_norm ? d1 * d1 : fabsf(d1);
            tube4[2] += two_norm ? d2 * d2 : fabsf(d2);
            tube4[3] += two_norm ? d3 * d3 : fabsf(d3);
          }
        }
        const int jc = j0 + cc * 32;
        if (jc >= nc || rows_valid <= 0) continue;
        if (rows_valid >= 32) {
          // all 32 rows exist: swizzled shared-memory box + bulk tensor store (coalesced, off the LSU; columns
          // beyond n are clipped by the tensor map)
          if (lane == 0) tma_store_wait_read<0>();   // the previous box of this warp has been read out
          __syncwarp();
#pragma unroll
          for (int e = 0; e < 8; ++e)
            *reinterpret_cast<uint4*>(sbox + lane * 128 + ((e ^ (lane & 7)) << 4)) =
                make_uint4(vc[4 * e], vc[4 * e + 1], vc[4 * e + 2], vc[4 * e + 3]);
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            tma_store_2d(&mapO, jc, row0, sbox);
            tma_store_commit();
          }
        } else if (lane < rows_valid) {
          // ragged last m-tile of a stacked column: masked row-per-thread stores
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            if (jc + 4 * e < nc)
              st_global_f4_na(out + static_cast<size_t>(lane) * nc + cc * 32 + 4 * e,
                              make_float4(__uint_as_float(vc[4 * e]), __uint_as_float(vc[4 * e + 1]),
                                          __uint_as_float(vc[4 * e + 2]), __uint_as_float(vc[4 * e + 3])));
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) arrive_leader(&tempty[acc]);
      if (MODE == 0 && lane < rows_valid)
        p.part[((qcol + rho / n) * g.NT + t.n_tile) * n + rho % n] = (tube4[0] + tube4[1]) + (tube4[2] + tube4[3]);
    }
    if (lane == 0) tma_store_wait_all<0>();   // shared memory must outlive the last bulk store
  }
  tc_fence_before();
  __syncthreads();
  if (PAIR) cluster_sync_all();   // the peer may still be reading this CTA's TMEM / shared memory through the pair MMA
  if (warp == 2) {
    tc_fence_after();
    if (PAIR) tmem_dealloc_2cta<512>(tmem_base); else tmem_dealloc<512>(tmem_base);
  }
}

template <int NCH, bool PAIR, int MODE>
cudaError_t launch_tc(const TcParams& p, const TcMaps& maps, int num_sms, cudaStream_t stream) {
  using S = TcShape<NCH, PAIR>;
  TcParams q = p;
  int st = static_cast<int>((227u * 1024u - 1024u - S::kMisc - kConvStages * S::kBBytes) / S::kRawBytes);
  if (st > kTcMaxStages) st = kTcMaxStages;
  if (st < 2) return cudaErrorInvalidConfiguration;
  q.stages = st;
  const uint32_t smem = 1024u + st * S::kRawBytes + kConvStages * S::kBBytes + S::kMisc;
  auto kern = phi_combine_tc_kernel<NCH, PAIR, MODE>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e != cudaSuccess) return e;
  const long long max_units = num_sms / S::NCTA;
  const long long units = q.g.total < max_units ? q.g.total : max_units;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>(units * S::NCTA));
  cfg.blockDim = dim3(kTcThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = S::NCTA;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  ProfScope prof(MODE == 1 ? kProfKalmanGemm : kProfPhiCombineTc, stream);
  return cudaLaunchKernelEx(&cfg, kern, q, maps.L, maps.R, maps.O, MODE == 2 ? maps.L2 : maps.L, MODE == 2 ? maps.R2 : maps.R);
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
  const cuuint64_t n = a.n, nc = a.nc;   // rows (= K) and columns (= row stride) of a block
  const cuuint32_t estr[3] = {1, 1, 1};
  {
    const cuuint64_t dims[2] = {n, static_cast<cuuint64_t>(a.batch) * P * n};
    const cuuint64_t strides[1] = {nc * 4};
    const cuuint32_t box[2] = {kKB, kTM};
    if (enc(&m->L, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, a.phi, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  {
    const cuuint64_t dims[3] = {nc, n, static_cast<cuuint64_t>(a.batch) * P};
    const cuuint64_t strides[2] = {nc * 4, n * nc * 4};
    const cuuint32_t box[3] = {32, kKB, 1};
    if (enc(&m->R, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, a.phi, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  {
    const cuuint64_t dims[2] = {nc, static_cast<cuuint64_t>(a.batch) * P * n};
    const cuuint64_t strides[1] = {nc * 4};
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
  p.phi = a.phi; p.w = a.w; p.part = a.part; p.tube_mode = a.tube_mode;
  const TcMaps& m = *static_cast<const TcMaps*>(maps);
  // CTA pairs (256-row tiles) when the level's stacked left operand is tall enough to fill them; the
  // single-CTA kernel (128-row tiles) on the low levels where 256-row tiles would be mostly padding
  const PhiGeom g1 = phi_geom(a.batch, a.T, a.n, a.nc, level, kTM, 32 * nch);
  const PhiGeom g2 = phi_geom(a.batch, a.T, a.n, a.nc, level, 2 * kTM, 32 * nch);
  if (g1.total == 0) return cudaSuccess;
  const int mode = env_int("TC_PAIR", -1);   // -1 auto, 0 never, 1 always
  const bool pair = (mode == 1) || (mode == -1 && 2 * g2.total * 100 <= g1.total * 108);
  p.g = pair ? g2 : g1;
#define LTV_NCH_CASE(N) \
  case N: return pair ? launch_tc<N, true, 0>(p, m, num_sms, stream) : launch_tc<N, false, 0>(p, m, num_sms, stream);
  switch (nch) {
    LTV_NCH_CASE(2) LTV_NCH_CASE(3) LTV_NCH_CASE(4) LTV_NCH_CASE(5)
    default: return cudaErrorInvalidValue;
  }
#undef LTV_NCH_CASE
}

// ---------------------------------------------------------------------------------------- cross block (MODE 2)
// G(t,s) = Pbar(t,mid) G(mid,s) + G(t,mid) Phat(mid,s) on the geometry of the Phi scan (a.phi = G; no tube).
cudaError_t phi_tc_make_cross_maps(const PhiArgs& a, const float* pbar, const float* phat, int nch, void* maps_out) {
  TcMaps mg, mb, mh;
  PhiArgs t = a;
  cudaError_t e = phi_tc_make_maps(t, nch, &mg);
  if (e != cudaSuccess) return e;
  t.phi = const_cast<float*>(pbar);
  if ((e = phi_tc_make_maps(t, nch, &mb)) != cudaSuccess) return e;
  t.phi = const_cast<float*>(phat);
  if ((e = phi_tc_make_maps(t, nch, &mh)) != cudaSuccess) return e;
  TcMaps* m = static_cast<TcMaps*>(maps_out);
  m->L = mb.L;    // Pbar(t,mid) stack
  m->R = mg.R;    // G(mid,s)
  m->L2 = mg.L;   // G(t,mid) stack
  m->R2 = mh.R;   // Phat(mid,s)
  m->O = mg.O;
  return cudaSuccess;
}

cudaError_t launch_phi_cross_tc(const PhiArgs& a, int level, int nch, const void* maps, int num_sms, cudaStream_t stream) {
  TcParams p{};
  p.phi = a.phi; p.w = nullptr; p.part = nullptr; p.tube_mode = 0;
  const TcMaps& m = *static_cast<const TcMaps*>(maps);
  const PhiGeom g1 = phi_geom(a.batch, a.T, a.n, a.nc, level, kTM, 32 * nch);
  const PhiGeom g2 = phi_geom(a.batch, a.T, a.n, a.nc, level, 2 * kTM, 32 * nch);
  if (g1.total == 0) return cudaSuccess;
  const bool pair = 2 * g2.total * 100 <= g1.total * 108;
  p.g = pair ? g2 : g1;
#define LTV_NCH_CASE(N_)                                                              \
  case N_: return pair ? launch_tc<N_, true, 2>(p, m, num_sms, stream)         \
                       : launch_tc<N_, false, 2>(p, m, num_sms, stream);
  switch (nch) {
    LTV_NCH_CASE(2) LTV_NCH_CASE(3) LTV_NCH_CASE(4) LTV_NCH_CASE(5)
    default: return cudaErrorInvalidValue;
  }
#undef LTV_NCH_CASE
}

// ---------------------------------------------------------------------------------------- batched GEMM (MODE 1)
cudaError_t bgemm_tc_make_maps(const BatchedGemm& a, void* maps_out) {
  EncodeTiledFn enc = reinterpret_cast<EncodeTiledFn>(get_encode_tiled());
  if (!enc) return cudaErrorNotSupported;
  TcMaps* m = static_cast<TcMaps*>(maps_out);
  const cuuint64_t M = a.M, N = a.N, K = a.K;
  const cuuint32_t estr[3] = {1, 1, 1};
  {
    const cuuint64_t dims[2] = {K, static_cast<cuuint64_t>(a.l_rows)};
    const cuuint64_t strides[1] = {K * 4};
    const cuuint32_t box[2] = {kKB, kTM};
    if (enc(&m->L, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(a.L), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  {
    const cuuint64_t dims[3] = {N, K, static_cast<cuuint64_t>(a.r_blocks)};
    const cuuint64_t strides[2] = {N * 4, K * N * 4};
    const cuuint32_t box[3] = {32, kKB, 1};
    if (enc(&m->R, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(a.R), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  {
    // D[b] is M x N, stored as it is or transposed (N x M); either way one block per problem, clipped per block
    const cuuint64_t cols = a.transpose_out ? M : N;
    const cuuint64_t rows = a.transpose_out ? N : (a.d_rows > 0 ? static_cast<cuuint64_t>(a.d_rows) : M);
    const cuuint64_t dims[3] = {cols, rows, static_cast<cuuint64_t>(a.d_blocks)};
    const cuuint64_t strides[2] = {cols * 4, rows * cols * 4};
    const cuuint32_t box[3] = {32, 32, 1};
    if (enc(&m->O, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, a.D, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  return cudaSuccess;
}

cudaError_t launch_bgemm_tc(const BatchedGemm& a, int nch, const void* maps, int num_sms, cudaStream_t stream) {
  if (a.count <= 0) return cudaSuccess;
  TcParams p{};
  const TcMaps& m = *static_cast<const TcMaps*>(maps);
  const int Mt1 = (a.M + kTM - 1) / kTM, Mt2 = (a.M + 2 * kTM - 1) / (2 * kTM);
  const int mode = env_int("TC_PAIR", -1);
  const int nt = 32 * nch;
  // Shape by a wave model: rounds of tiles over the CTAs (or CTA pairs) x relative time per tile.  A pair tile keeps the
  // tensor pipe ~92 % busy against ~65 % for the single-CTA shape (profiles/r2_kernels_full.md) but pays a
  // cluster launch and two cluster barriers (15 %, fitted: C2 384 single tiles 33.3 us vs 256 pair tiles 35.6 us;
  // C3 320 vs 192: 49.4 vs 45.3 us).
  const long long ntile = (a.N + nt - 1) / nt;
  const long long r1 = (static_cast<long long>(a.count) * Mt1 * ntile + num_sms - 1) / num_sms;
  const long long r2 = (static_cast<long long>(a.count) * Mt2 * ntile + num_sms / 2 - 1) / (num_sms / 2);
  const bool pair = (mode == 1) || (mode == -1 && r2 * 125 < r1 * 154);
  p.g = PhiGeom{};
  p.g.n = a.K;
  p.g.nc = a.N;
  p.g.tm = pair ? 2 * kTM : kTM;
  p.g.tn = nt;
  p.g.NT = (a.N + nt - 1) / nt;
  p.phi = a.D;
  p.gm.count = a.count; p.gm.M = a.M; p.gm.Mt = pair ? Mt2 : Mt1;
  p.gm.d_rows = a.d_rows > 0 ? a.d_rows : a.M;
  p.gm.l_row0 = a.l_row0; p.gm.l_row_stride = a.l_row_stride;
  p.gm.r_blk0 = a.r_blk0; p.gm.r_blk_stride = a.r_blk_stride;
  p.gm.d_blk0 = a.d_blk0; p.gm.d_blk_stride = a.d_blk_stride;
  p.gm.transpose_out = a.transpose_out;
  p.gm.diag = a.diag; p.gm.diag_stride = a.diag_stride;
  p.gm.d_row0 = a.d_row0; p.gm.d_row_stride = a.d_row_stride;
  if (a.transpose_out && (a.d_row0 != 0 || a.d_row_stride != 0)) return cudaErrorInvalidValue;
  p.g.total = static_cast<long long>(p.gm.Mt) * p.g.NT * a.count;
#define LTV_NCH_CASE(N_)                                                              \
  case N_: return pair ? launch_tc<N_, true, 1>(p, m, num_sms, stream)         \
                       : launch_tc<N_, false, 1>(p, m, num_sms, stream);
  switch (nch) {
    LTV_NCH_CASE(2) LTV_NCH_CASE(3) LTV_NCH_CASE(4) LTV_NCH_CASE(5)
    default: return cudaErrorInvalidValue;
  }
#undef LTV_NCH_CASE
}

}  // namespace ltv
