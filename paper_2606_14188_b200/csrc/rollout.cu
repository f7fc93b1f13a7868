// ltv_scan_rollout: x_{t+1} = A_t x_t + B_t u_t + c_t   (eq.(2), :139 eq.(12b))
//
// HBM-bound GEMV chain.  One thread-block cluster per batch item; CTA `rank` of the cluster owns a
// contiguous band of rows of every A_t.  A dedicated producer thread streams that band through a
// shared-memory ring with 1-D bulk TMA copies (the band of one step is contiguous in memory), running
// ahead of the consumers across step boundaries, so the only thing on the sequential critical path is the
// shared-memory GEMV and the exchange of the new state: every consumer warp writes its rows of x_{t+1}
// straight into the x buffer of EVERY CTA of the cluster (st.async through DSMEM) and the byte count of an
// mbarrier in each CTA tells that CTA when x_{t+1} is complete.  The affine term b_t = B_t u_t + c_t is
// formed one step ahead by a helper warp and never touches global memory.
#include "ltv_internal.h"
#include "ptx.cuh"

namespace ltv {

namespace {

constexpr int kConsWarps = 8;
constexpr int kRollThreads = (kConsWarps + 2) * 32;  // + producer warp + affine warp
constexpr int kMaxStages = 8;

struct RollSmemPlan {
  int rc;              // rows per ring chunk
  int stages;
  uint32_t stage_bytes;
  uint32_t off_x, off_b, off_bar, total;
  int rows_max;        // max rows owned by one CTA
};

__host__ __device__ inline void band(int n, int C, int rank, int& r0, int& r1) {
  r0 = static_cast<int>((static_cast<long long>(n) * rank) / C);
  r1 = static_cast<int>((static_cast<long long>(n) * (rank + 1)) / C);
}

struct RollParams {
  const float *A, *B, *c, *x0, *u;
  float* x_out;
  int batch, T, n, m;
  RollSmemPlan sp;
};

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void __launch_bounds__(kRollThreads, 1) rollout_kernel(const RollParams p) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int C = static_cast<int>(cluster_nctarank());
  const int rank = static_cast<int>(cluster_ctarank());
  const int item = blockIdx.x / C;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n = p.n, T = p.T, m = p.m;
  int r0, r1;
  band(n, C, rank, r0, r1);
  const int rows = r1 - r0;
  const int rc = p.sp.rc, stages = p.sp.stages;
  const int nchunks = (rows + rc - 1) / rc;

  float* ring = reinterpret_cast<float*>(smem);
  float* xbuf = reinterpret_cast<float*>(smem + p.sp.off_x);   // [2][n]
  float* bvec = reinterpret_cast<float*>(smem + p.sp.off_b);   // [2][rows_max]
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + p.sp.off_bar);
  uint64_t* full = bars;                    // [stages]  producer -> consumers (tx bytes)
  uint64_t* empty = bars + kMaxStages;      // [stages]  consumers -> producer (kConsWarps arrivals)
  uint64_t* xfull = bars + 2 * kMaxStages;  // [2]       x_{t} complete in xbuf[t&1] (n*4 tx bytes + 1 arrival)
  uint64_t* bfull = xfull + 2;              // [2]       b_t complete in bvec[t&1]

  if (threadIdx.x == 0) {
    for (int s = 0; s < stages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], kConsWarps);
    }
    mbar_init(&xfull[0], 1);
    mbar_init(&xfull[1], 1);
    mbar_init(&bfull[0], 1);
    mbar_init(&bfull[1], 1);
    fence_mbar_init();
  }
  for (int j = threadIdx.x; j < n; j += kRollThreads) xbuf[j] = p.x0[static_cast<size_t>(item) * n + j];
  __syncthreads();
  cluster_sync_all();  // every CTA's barriers are initialised before any remote st.async can target them

  const size_t itemA = static_cast<size_t>(item) * T * n * n;

  if (warp == kConsWarps) {
    // ------------------------------------------------------------------ producer (one thread)
    if (lane == 0 && rows > 0) {
      const uint64_t pol = l2_policy_evict_first();
      uint32_t it = 0;
      for (int t = 0; t < T; ++t) {
        const float* At = p.A + itemA + (static_cast<size_t>(t) * n + r0) * n;
        for (int k = 0; k < nchunks; ++k, ++it) {
          const int st = it % stages;
          const uint32_t use = it / stages;
          if (use > 0) mbar_wait(&empty[st], (use - 1) & 1);
          const int rk = min(rc, rows - k * rc);
          const uint32_t bytes = static_cast<uint32_t>(rk) * n * 4u;
          mbar_arrive_expect_tx(&full[st], bytes);
          bulk_g2s(reinterpret_cast<uint8_t*>(ring) + static_cast<size_t>(st) * p.sp.stage_bytes,
                   At + static_cast<size_t>(k) * rc * n, bytes, &full[st], pol);
        }
      }
    }
  } else if (warp == kConsWarps + 1) {
    // ------------------------------------------------------------------ affine / output warp
    // step t: wait x_t, arm the barrier of x_{t+1}, write x_t to global, form b_{t+1}
    auto form_b = [&](int t) {
      float* bv = bvec + (t & 1) * p.sp.rows_max;
      const size_t bt = static_cast<size_t>(item) * T + t;
      for (int i = lane; i < rows; i += 32) {
        float acc = p.c ? p.c[bt * n + r0 + i] : 0.f;
        if (p.B && p.u) {
          const float* Brow = p.B + (bt * n + r0 + i) * m;
          const float* ut = p.u + bt * m;
          for (int l = 0; l < m; ++l) acc = fmaf(__ldg(Brow + l), __ldg(ut + l), acc);
        }
        bv[i] = acc;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&bfull[t & 1]);
    };
    form_b(0);
    for (int t = 0; t <= T; ++t) {
      if (t >= 1) {
        mbar_wait_cluster(&xfull[t & 1], (((t + 1) >> 1) - 1) & 1);
        const float* xt = xbuf + (t & 1) * n;
        float* dst = p.x_out + (static_cast<size_t>(item) * T + (t - 1)) * n;
        for (int i = r0 + lane; i < r1; i += 32) dst[i] = xt[i];
      }
      if (t < T) {
        if (lane == 0) mbar_arrive_expect_tx(&xfull[(t + 1) & 1], static_cast<uint32_t>(n) * 4u);
        if (t + 1 < T) form_b(t + 1);
      }
    }
  } else {
    // ------------------------------------------------------------------ consumers: shared-memory GEMV
    const int n4 = n >> 2;
    uint32_t it = 0;
    for (int t = 0; t < T; ++t) {
      if (t >= 1) mbar_wait_cluster(&xfull[t & 1], (((t + 1) >> 1) - 1) & 1);
      mbar_wait(&bfull[t & 1], (t >> 1) & 1);
      const float4* x4 = reinterpret_cast<const float4*>(xbuf + (t & 1) * n);
      float* xn = xbuf + ((t + 1) & 1) * n;
      const float* bv = bvec + (t & 1) * p.sp.rows_max;
      uint64_t* xbar = &xfull[(t + 1) & 1];
      for (int k = 0; k < nchunks; ++k, ++it) {
        const int st = it % stages;
        mbar_wait(&full[st], (it / stages) & 1);
        const float* tile = reinterpret_cast<const float*>(reinterpret_cast<uint8_t*>(ring) +
                                                            static_cast<size_t>(st) * p.sp.stage_bytes);
        const int rk = min(rc, rows - k * rc);
        // rows of the band are dealt round-robin to the warps; two rows per pass share the x loads
        int i = (warp - (k * rc) % kConsWarps + kConsWarps) % kConsWarps;
        for (; i < rk; i += 2 * kConsWarps) {
          const bool two = (i + kConsWarps) < rk;
          const float4* a0 = reinterpret_cast<const float4*>(tile + static_cast<size_t>(i) * n);
          const float4* a1 = reinterpret_cast<const float4*>(tile + static_cast<size_t>(two ? i + kConsWarps : i) * n);
          float s0 = 0.f, s1 = 0.f;
#pragma unroll 2
          for (int q = lane; q < n4; q += 32) {
            const float4 xv = x4[q];
            const float4 v0 = a0[q];
            const float4 v1 = a1[q];
            s0 = fmaf(v0.x, xv.x, fmaf(v0.y, xv.y, fmaf(v0.z, xv.z, fmaf(v0.w, xv.w, s0))));
            s1 = fmaf(v1.x, xv.x, fmaf(v1.y, xv.y, fmaf(v1.z, xv.z, fmaf(v1.w, xv.w, s1))));
          }
          s0 = warp_sum(s0);
          s1 = warp_sum(s1);
          const int l0 = k * rc + i, l1 = l0 + kConsWarps;
          s0 += bv[l0];
          if (two) s1 += bv[l1];
          if (lane < C) {
            st_async_remote_f32(xn + r0 + l0, s0, xbar, lane);
            if (two) st_async_remote_f32(xn + r0 + l1, s1, xbar, lane);
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);
      }
    }
  }
  __syncthreads();
  cluster_sync_all();  // no CTA may exit while a peer can still write into its shared memory
}

RollSmemPlan plan_rollout(int n, int C) {
  RollSmemPlan sp{};
  sp.rows_max = (n + C - 1) / C + 1;
  const uint32_t row_bytes = static_cast<uint32_t>(n) * 4u;
  const uint32_t vec_bytes = static_cast<uint32_t>(align_up(2 * row_bytes, 128) + align_up(2u * sp.rows_max * 4u, 128));
  const uint32_t budget = 227u * 1024u - vec_bytes - 256u;
  const uint32_t target = 32u * 1024u;
  int rc = static_cast<int>(target / row_bytes);
  if (rc < 1) rc = 1;
  if (rc > sp.rows_max) rc = sp.rows_max;
  sp.rc = rc;
  sp.stage_bytes = static_cast<uint32_t>(align_up(static_cast<size_t>(rc) * row_bytes, 128));
  int st = static_cast<int>(budget / sp.stage_bytes);
  if (st > kMaxStages) st = kMaxStages;
  sp.stages = st;
  sp.off_x = sp.stage_bytes * st;
  sp.off_b = sp.off_x + static_cast<uint32_t>(align_up(2 * row_bytes, 128));
  sp.off_bar = sp.off_b + static_cast<uint32_t>(align_up(2u * sp.rows_max * 4u, 128));
  sp.total = sp.off_bar + (2 * kMaxStages + 4) * 8;
  return sp;
}

}  // namespace

cudaError_t launch_rollout(const RolloutArgs& a, int cluster, cudaStream_t stream, unsigned long long* launches) {
  RollParams p{};
  p.A = a.A; p.B = (a.m > 0) ? a.B : nullptr; p.c = a.c; p.x0 = a.x0; p.u = a.u; p.x_out = a.x_out;
  p.batch = a.batch; p.T = a.T; p.n = a.n; p.m = a.m;
  p.sp = plan_rollout(a.n, cluster);
  if (p.sp.stages < 2) return cudaErrorInvalidConfiguration;

  cudaError_t e = cudaFuncSetAttribute(rollout_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, p.sp.total);
  if (e != cudaSuccess) return e;
  if (cluster > 8) {
    e = cudaFuncSetAttribute(rollout_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
  }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(static_cast<unsigned>(a.batch) * cluster);
  cfg.blockDim = dim3(kRollThreads);
  cfg.dynamicSmemBytes = p.sp.total;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = cluster;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  {
    ProfScope prof(kProfRollout, stream);
    e = cudaLaunchKernelEx(&cfg, rollout_kernel, p);
  }
  if (e == cudaSuccess) ++*launches;
  return e;
}

}  // namespace ltv
