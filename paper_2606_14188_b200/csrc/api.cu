// extern "C" boundary of libltvscan.so (include/ltv_scan.h): argument validation, workspace sizing,
// device check, dispatch to the launchers.  No torch types, no exceptions across the ABI.
#include <algorithm>
#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/ltv_scan.h"
#include "ltv_internal.h"
#include "phi_geom.cuh"

namespace ltv {

static thread_local int g_last_cuda_error = 0;
static std::atomic<unsigned long long> g_launches{0};

// Developer overrides LTV_SCAN_<name> exist only in builds made with -DLTV_TUNING (kernel experiments: tile shape, forced
// code paths).  The product build ignores the environment: its only knobs are the documented ltv_set_option values.
int env_int(const char* name, int dflt) {
#ifdef LTV_TUNING
  char key[64] = "LTV_SCAN_";
  std::strncat(key, name, sizeof(key) - std::strlen(key) - 1);
  const char* v = std::getenv(key);
  return (v && *v) ? std::atoi(v) : dflt;
#else
  (void)name;
  return dflt;
#endif
}

#ifdef LTV_TUNING
static unsigned int* g_dbg_host = nullptr;
unsigned int* dbg_buffer_device() {
  static unsigned int* dptr = nullptr;
  if (!dptr) {
    if (cudaHostAlloc(reinterpret_cast<void**>(&g_dbg_host), 65536, cudaHostAllocMapped) != cudaSuccess) return nullptr;
    std::memset(g_dbg_host, 0, 65536);
    if (cudaHostGetDevicePointer(reinterpret_cast<void**>(&dptr), g_dbg_host, 0) != cudaSuccess) return nullptr;
  }
  return dptr;
}
extern "C" LTV_API unsigned int* ltv_debug_buffer(void) { return g_dbg_host; }
#endif

static std::atomic<int> g_options[LTV_OPT_COUNT] = {{0}, {16}, {0}};
int option(int which) { return g_options[which].load(std::memory_order_relaxed); }

int pick_cluster_model(int batch, int n, const int* max_active, int sm_budget) {
  const int forced = option(LTV_OPT_VECTOR_CLUSTER);
  if (forced >= 1 && forced <= 16 && max_active[forced] > 0) return forced;
  const double sm_gbs = 70.0, dev_gbs = 6500.0;
  int best = 1;
  double best_t = 1e300;
  for (int c = 1; c <= 16; ++c) {
    if (max_active[c] <= 0) continue;
    if (c > 1 && (n / c < 32 || (n >> 2) < c)) continue;   // keep at least ~32 rows / columns per CTA
    int cap = max_active[c];
    if (sm_budget > 0 && cap > sm_budget / c) cap = sm_budget / c > 0 ? sm_budget / c : 1;
    double t = 0.0;
    for (int rem = batch; rem > 0;) {
      const int w = rem < cap ? rem : cap;
      const double rate = (w * c * sm_gbs < dev_gbs) ? w * c * sm_gbs : dev_gbs;
      t += w / rate;
      rem -= w;
    }
    t *= 1.0 + 0.01 * c;   // ties go to the smaller cluster (less exchange per step)
    if (t < best_t) {
      best_t = t;
      best = c;
    }
  }
  return best;
}

void query_max_active_clusters(const void* kernel, int threads, size_t smem, int* max_active) {
  cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
  cudaFuncSetAttribute(kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  max_active[0] = 0;
  for (int c = 1; c <= 16; ++c) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(c * 64);
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = c;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    int nact = 0;
    if (cudaOccupancyMaxActiveClusters(&nact, kernel, &cfg) != cudaSuccess) {
      cudaGetLastError();
      nact = 0;
    }
    max_active[c] = nact;
  }
}

// ---- optional kernel timing --------------------------------------------------------------------------
namespace {
struct ProfState {
  std::mutex mu;
  std::atomic<bool> on{false};
  std::vector<cudaEvent_t> beg, end;
  std::vector<int> cls;
  size_t used = 0;
};
ProfState& prof() {
  static ProfState p;
  return p;
}
}  // namespace

ProfScope::ProfScope(int cls_, cudaStream_t s) : slot(-1), stream(s), end_event(nullptr) {
  ProfState& p = prof();
  if (!p.on.load(std::memory_order_acquire)) return;
  std::lock_guard<std::mutex> lk(p.mu);
  if (!p.on.load(std::memory_order_relaxed)) return;
  if (p.used == p.beg.size()) {
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
    p.beg.push_back(a);
    p.end.push_back(b);
    p.cls.push_back(0);
  }
  slot = static_cast<int>(p.used++);
  p.cls[slot] = cls_;
  end_event = p.end[slot];   // the handle is captured under the lock: the vectors may be reallocated by other threads
  cudaEventRecord(p.beg[slot], stream);
}
ProfScope::~ProfScope() {
  if (slot >= 0) cudaEventRecord(static_cast<cudaEvent_t>(end_event), stream);
}

static int fail_cuda(cudaError_t e) {
  g_last_cuda_error = static_cast<int>(e);
  cudaGetLastError();  // clear the sticky-free error state of the runtime
  return LTV_ERR_CUDA;
}

void count_launches(unsigned long long n) { g_launches += n; }
int report_cuda_error(cudaError_t e) { return fail_cuda(e); }

// several kernels of the NEXT calls map the batch (or batch x steps) onto gridDim.y / gridDim.z (<= 65535)
static bool grid_yz_overflow(long long v) { return v > 65535; }

static bool misaligned(const void* p) { return p && (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

static int check_dims(int batch, int T, int n, int m) {
  if (batch < 1 || T < 1 || n < 1 || m < 0) return LTV_ERR_BAD_DIM;
  if (n % 4 != 0 || n > 8192) return LTV_ERR_UNSUPPORTED_SHAPE;
  // TMA row coordinates and block indices are 32-bit
  if (static_cast<long long>(batch) * T * n >= (1ll << 31)) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (static_cast<long long>(batch) * T * (T - 1) / 2 * n >= (1ll << 31)) return LTV_ERR_UNSUPPORTED_SHAPE;
  return LTV_OK;
}

// current device must be sm_100-class; returns the SM count through *sms
static int check_device(int* sms) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_cuda(e);
  int major = 0;
  e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e != cudaSuccess) return fail_cuda(e);
  if (major != 10) return LTV_ERR_ARCH;
  e = cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return fail_cuda(e);
  return LTV_OK;
}

}  // namespace ltv

using namespace ltv;

extern "C" {

long long ltv_phi_block_index(int T, int t, int s) {
  if (T < 1 || s < 0 || t <= s || t > T - 1) return -1;
  return phi_colbase(T, s) + (t - s - 1);
}

long long ltv_phi_block_index_layout(int T, int t, int s, int phi_layout) {
  if (T < 1 || s < 0 || t <= s || t > T - 1) return -1;
  switch (phi_layout) {
    case LTV_PHI_ROW_PACKED: return static_cast<long long>(t) * (t - 1) / 2 + s;
    case LTV_PHI_SQUARE_GRID: return static_cast<long long>(t) * T + s;
    case LTV_PHI_COLUMN_PACKED: return phi_colbase(T, s) + (t - s - 1);
    default: return -1;
  }
}

size_t ltv_scan_workspace_bytes(int op, int batch, int T, int n, int m) {
  if (check_dims(batch, T, n, m) != LTV_OK) return 0;
  switch (op) {
    case LTV_OP_ROLLOUT:
    case LTV_OP_ADJOINT:
      return 0;
    case LTV_OP_SYSTEM_RESPONSE_TUBE:
      return phi_workspace_bytes(batch, T, n, n);
    case LTV_OP_SYSTEM_RESPONSE_TUBE_RELAYOUT:
      return phi_workspace_bytes(batch, T, n, n) + phi_colpacked_bytes(batch, T, n, n);
    case LTV_OP_OBSERVER_RESPONSE:
      if (m < 1 || m > 32) return 0;
      return phi_workspace_bytes(batch, T, n, n + ((m + 3) & ~3));
    case LTV_OP_KALMAN_GAINS:
      if (m < 1 || m > 32) return 0;
      return kalman_workspace_bytes(batch, T, n, m);
    case LTV_OP_CONSTRAINT_TIGHTENING:
      if (m < 1 || static_cast<long long>(batch) * T * m >= (1ll << 31) / n) return 0;
      return constraint_workspace_bytes(batch, T, n, m);
    case LTV_OP_OUTPUT_FEEDBACK:
      if (check_dims(batch, T, 2 * n, 0) != LTV_OK) return 0;
      return ofb_workspace_bytes(batch, T, n, m, m);   // m = max(m, p) of the call, or 0 = unknown
    case LTV_OP_PIPELINE_HOST:
    case LTV_OP_PIPELINE_HOST_NO_PHI: {
      const bool with_phi = op == LTV_OP_PIPELINE_HOST;
      const size_t b = batch, t = T, nn = n, mm = m;
      const size_t P = t * (t - 1) / 2;
      size_t tot = 0;
      auto add = [&](size_t floats) { tot += align_up(floats * 4 + 16, 256); };
      add(b * t * nn * nn);  // A
      add(b * t * nn * mm);  // B
      add(b * t * nn);       // c
      add(b * nn);           // x0
      add(b * t * mm);       // u
      add(b * t * nn);       // w
      add(b * t * nn);       // g
      add(b * t * nn);       // x
      add(with_phi ? b * P * nn * nn : 0);  // phi
      add(b * t * nn);       // r
      add(b * t * nn);       // lambda
      add(b * t * mm);       // grad_u
      add(b * nn);           // grad_x0
      if (with_phi) tot += phi_workspace_bytes(batch, T, n, n);
      return tot;
    }
    default:
      return 0;
  }
}

int ltv_scan_rollout(const float* A, const float* B, const float* c, const float* x0, const float* u, float* x_out,
                     int batch, int T, int n, int m, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  (void)workspace; (void)workspace_bytes;
  if (!A || !x0 || !x_out) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, m);
  if (st != LTV_OK) return st;
  if (misaligned(A) || misaligned(B) || misaligned(c) || misaligned(x0) || misaligned(u) || misaligned(x_out))
    return LTV_ERR_ALIGNMENT;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  RolloutArgs a{A, B, c, x0, u, x_out, batch, T, n, m};
  unsigned long long l = 0;
  cudaError_t e = cudaErrorUnknown;
  e = launch_rollout(a, 0, static_cast<cudaStream_t>(cuda_stream), &l);
  if (e != cudaSuccess) {   // the modelled cluster could not be placed: one CTA per item always can
    cudaGetLastError();
    e = launch_rollout(a, 1, static_cast<cudaStream_t>(cuda_stream), &l);
  }
  g_launches += l;
  return e == cudaSuccess ? LTV_OK : fail_cuda(e);
}

int ltv_scan_adjoint(const float* A, const float* B, const float* g, float* lambda_out, float* grad_u_out,
                     float* grad_x0_out, int batch, int T, int n, int m, void* workspace, size_t workspace_bytes,
                     void* cuda_stream) {
  (void)workspace; (void)workspace_bytes;
  if (!A || !g || !lambda_out) return LTV_ERR_NULL_PTR;
  if (grad_u_out && m > 0 && !B) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, m);
  if (st != LTV_OK) return st;
  if (misaligned(A) || misaligned(B) || misaligned(g) || misaligned(lambda_out) || misaligned(grad_u_out) ||
      misaligned(grad_x0_out))
    return LTV_ERR_ALIGNMENT;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  AdjointArgs a{A, B, g, lambda_out, grad_u_out, grad_x0_out, batch, T, n, m};
  unsigned long long l = 0;
  cudaError_t e = cudaErrorUnknown;
  e = launch_adjoint(a, 0, static_cast<cudaStream_t>(cuda_stream), &l);
  if (e != cudaSuccess) {
    cudaGetLastError();
    e = launch_adjoint(a, 1, static_cast<cudaStream_t>(cuda_stream), &l);
  }
  g_launches += l;
  return e == cudaSuccess ? LTV_OK : fail_cuda(e);
}

namespace {
// side stream + fork / join events of ltv_scan_rollout_adjoint: created once per host thread and device (the only
// state the library keeps besides cached function attributes); never destroyed (a handful of handles per thread)
struct PairCtx {
  int dev = -1;
  cudaStream_t side = nullptr;
  cudaEvent_t fork = nullptr, join = nullptr;
};
cudaError_t pair_ctx(PairCtx** out) {
  static thread_local PairCtx ctx[16];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  PairCtx& c = ctx[dev & 15];
  if (c.dev != dev) {
    if ((e = cudaStreamCreateWithFlags(&c.side, cudaStreamNonBlocking)) != cudaSuccess) return e;
    if ((e = cudaEventCreateWithFlags(&c.fork, cudaEventDisableTiming)) != cudaSuccess) return e;
    if ((e = cudaEventCreateWithFlags(&c.join, cudaEventDisableTiming)) != cudaSuccess) return e;
    c.dev = dev;
  }
  *out = &c;
  return cudaSuccess;
}
}  // namespace

int ltv_scan_rollout_adjoint(const float* A, const float* B, const float* c, const float* x0, const float* u,
                             const float* g, float* x_out, float* lambda_out, float* grad_u_out, float* grad_x0_out,
                             int batch, int T, int n, int m, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  (void)workspace; (void)workspace_bytes;
  if (!A || !x0 || !x_out || !g || !lambda_out) return LTV_ERR_NULL_PTR;
  if (grad_u_out && m > 0 && !B) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, m);
  if (st != LTV_OK) return st;
  if (misaligned(A) || misaligned(B) || misaligned(c) || misaligned(x0) || misaligned(u) || misaligned(x_out) ||
      misaligned(g) || misaligned(lambda_out) || misaligned(grad_u_out) || misaligned(grad_x0_out))
    return LTV_ERR_ALIGNMENT;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  PairCtx* pc = nullptr;
  cudaError_t e = pair_ctx(&pc);
  if (e != cudaSuccess) return fail_cuda(e);
  // The two scans are independent (g is an input).  Measured on B200: running them side by side pays
  // only when each one, in the configuration it would choose alone, leaves at least half of the SMs idle (one small
  // problem, or few items whose clusters cannot be wider than 16 CTAs); once either saturates HBM on its own the two only
  // get in each other's way (C2: 0.55 ms side by side on 64 + 64 SMs against 0.25 ms back to back).  So: on half the machine
  // each when both fit there, else each in its own configuration on two streams (the second fills the SMs the first leaves idle).
  RolloutArgs ra{A, B, c, x0, u, x_out, batch, T, n, m};
  AdjointArgs aa{A, B, g, lambda_out, grad_u_out, grad_x0_out, batch, T, n, m};
  const int cfr = rollout_cluster_choice(ra), cfa = adjoint_cluster_choice(aa);
  // Side by side or back to back?  Measured on B200 ("the pair"):
  //  - a scan that ALONE runs on >= 80 % of the SMs with >= 128 rows (columns) per CTA streams at 0.8-1.0 of the HBM peak
  //    (n = 300 x 64 items): splitting the SMs would only get the two in each other's way -> each keeps its configuration;
  //  - otherwise each scan alone is short of CTAs (few items: 4 x 16-CTA clusters = 64 SMs) or of work per step (n = 180: two
  //    CTAs per item exchange the state every 1.3 us), and both at once on half the machine each move more, PROVIDED every
  //    cluster of both kernels is resident at the same time - else the last cluster waits for a slot and the pair is slower
  //    than back to back (n = 2400 x 4 items: 4 + 4 clusters of 16 on 7 slots 0.665 ms, back to back 0.631, 4 + 4 clusters of
  //    10 side by side 0.536).  So: the widest cluster size c with batch c <= SMs / 2 and 2 batch clusters resident.
  auto slots = [&](int c) { return std::min(rollout_clusters_resident(ra, c), adjoint_clusters_resident(aa, c)); };
  const bool alone_good = std::min(batch * cfr, batch * cfa) * 10 >= sms * 8 && n / std::max(cfr, cfa) >= 128;
  int cl_r = 0, cl_a = 0;   // CTAs per item of the two scans; 0 = each kernel's own model
  bool side_by_side = false;
  if (!alone_good && option(LTV_OPT_VECTOR_CLUSTER) == 0) {
    int c = 0;
    for (int cc = 1; cc <= 16; ++cc) {
      if (static_cast<long long>(batch) * cc > sms / 2 || 2 * batch > slots(cc)) continue;
      if (cc > 1 && (n / cc < 32 || (n >> 2) < cc)) continue;
      c = cc;
    }
    if (c > 0) {
      side_by_side = true;
      cl_r = cl_a = c;
    }
  }
  // back to back, but on two streams: the second scan's clusters take the SMs the first leaves idle (64 items x 2 CTAs = 128
  // of 148) and fill in as its clusters finish - clusters are independent, so any interleaving is correct
  if (!side_by_side && alone_good && option(LTV_OPT_VECTOR_CLUSTER) == 0 && env_int("PAIR_OVERLAP", 1) != 0) side_by_side = true;
  unsigned long long l = 0;
  {
    ProfScope prof(kProfVectorPair, s);
    cudaStream_t sa = s;
    if (side_by_side) {
      if ((e = cudaEventRecord(pc->fork, s)) != cudaSuccess) return fail_cuda(e);
      if ((e = cudaStreamWaitEvent(pc->side, pc->fork, 0)) != cudaSuccess) return fail_cuda(e);
      sa = pc->side;
    }
    e = launch_adjoint(aa, cl_a, sa, &l);
    if (e != cudaSuccess) {
      cudaGetLastError();
      e = launch_adjoint(aa, 1, sa, &l);
    }
    cudaError_t e2 = launch_rollout(ra, cl_r, s, &l);
    if (e2 != cudaSuccess) {
      cudaGetLastError();
      e2 = launch_rollout(ra, 1, s, &l);
    }
    cudaError_t e3 = cudaSuccess;
    if (side_by_side) {
      // always join, so that the caller's stream is ordered after whatever did get enqueued on the side stream
      e3 = cudaEventRecord(pc->join, pc->side);
      if (e3 == cudaSuccess) e3 = cudaStreamWaitEvent(s, pc->join, 0);
    }
    if (e == cudaSuccess) e = e2;
    if (e == cudaSuccess) e = e3;
  }
  g_launches += l;
  return e == cudaSuccess ? LTV_OK : fail_cuda(e);
}

int ltv_scan_system_response_tube(const float* A, const float* w, float* phi_out, float* r_out, int batch, int T,
                                  int n, int phi_layout, unsigned flags, void* workspace, size_t workspace_bytes,
                                  void* cuda_stream) {
  if (!A || !w || !r_out) return LTV_ERR_NULL_PTR;
  if (T > 1 && !phi_out) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, 0);
  if (st != LTV_OK) return st;
  const bool native = phi_layout == LTV_PHI_COLUMN_PACKED;
  if ((!native && phi_layout != LTV_PHI_ROW_PACKED && phi_layout != LTV_PHI_SQUARE_GRID) ||
      (flags & ~static_cast<unsigned>(LTV_TUBE_ROW_2NORM)) != 0)
    return LTV_ERR_BAD_DIM;
  if (misaligned(A) || misaligned(w) || misaligned(phi_out) || misaligned(r_out) || misaligned(workspace))
    return LTV_ERR_ALIGNMENT;
  const size_t need = phi_workspace_bytes(batch, T, n, n) + (native ? 0 : phi_colpacked_bytes(batch, T, n, n));
  if (!workspace) return LTV_ERR_NULL_PTR;
  if (workspace_bytes < need) return LTV_ERR_WORKSPACE_TOO_SMALL;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  // the scan computes column-packed: straight into phi_out, or into the workspace followed by one block re-ordering copy
  float* phi_cp = native ? phi_out
                         : reinterpret_cast<float*>(static_cast<char*>(workspace) + phi_workspace_bytes(batch, T, n, n));
  PhiArgs a{A, w, phi_cp, r_out, static_cast<float*>(workspace), batch, T, n, n, (flags & LTV_TUBE_ROW_2NORM) ? 1 : 0};
  unsigned long long l = 0;
  cudaError_t e = launch_phi_tube(a, static_cast<cudaStream_t>(cuda_stream), &l);
  if (e == cudaSuccess && !native && T > 1) {
    e = launch_phi_relayout(phi_cp, phi_out, batch, T, n, n, phi_layout, sms, static_cast<cudaStream_t>(cuda_stream));
    if (e == cudaSuccess) ++l;
  }
  g_launches += l;
  return e == cudaSuccess ? LTV_OK : fail_cuda(e);
}

int ltv_scan_all_is_fused(int batch, int T, int n, int m, int phi_layout) {
  return (check_dims(batch, T, n, m) == LTV_OK && phi_layout == LTV_PHI_COLUMN_PACKED && fused_small_supported(batch, T, n, m)) ? 1 : 0;
}

int ltv_scan_all(const float* A, const float* B, const float* c, const float* x0, const float* u, const float* w,
                 const float* g, float* x_out, float* phi_out, float* r_out, float* lambda_out, float* grad_u_out,
                 float* grad_x0_out, int batch, int T, int n, int m, int phi_layout, unsigned flags, void* workspace,
                 size_t workspace_bytes, void* cuda_stream) {
  if (!A || !x0 || !w || !g || !x_out || !r_out || !lambda_out) return LTV_ERR_NULL_PTR;
  if (T > 1 && !phi_out) return LTV_ERR_NULL_PTR;
  if (grad_u_out && m > 0 && !B) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, m);
  if (st != LTV_OK) return st;
  if ((flags & ~static_cast<unsigned>(LTV_TUBE_ROW_2NORM)) != 0) return LTV_ERR_BAD_DIM;
  if (!ltv_scan_all_is_fused(batch, T, n, m, phi_layout)) {
    st = ltv_scan_rollout_adjoint(A, B, c, x0, u, g, x_out, lambda_out, grad_u_out, grad_x0_out, batch, T, n, m, nullptr, 0,
                                  cuda_stream);
    if (st != LTV_OK) return st;
    return ltv_scan_system_response_tube(A, w, phi_out, r_out, batch, T, n, phi_layout, flags, workspace, workspace_bytes,
                                         cuda_stream);
  }
  if (misaligned(A) || misaligned(B) || misaligned(c) || misaligned(x0) || misaligned(u) || misaligned(w) || misaligned(g) ||
      misaligned(x_out) || misaligned(phi_out) || misaligned(r_out) || misaligned(lambda_out) || misaligned(grad_u_out) ||
      misaligned(grad_x0_out))
    return LTV_ERR_ALIGNMENT;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  FusedSmallArgs a{A, B, c, x0, u, w, g, x_out, phi_out, r_out, lambda_out, grad_u_out, grad_x0_out, batch, T, n, m,
                   (flags & LTV_TUBE_ROW_2NORM) ? 1 : 0};
  unsigned long long l = 0;
  cudaError_t e = launch_fused_small(a, static_cast<cudaStream_t>(cuda_stream), &l);
  g_launches += l;
  return e == cudaSuccess ? LTV_OK : fail_cuda(e);
}

int ltv_observer_row_floats(int n, int p) { return (n < 1 || p < 1) ? 0 : n + ((p + 3) & ~3); }

int ltv_scan_observer_response(const float* A, const float* Lt, const float* C, const float* w, float* phi_out,
                               float* r_out, int batch, int T, int n, int p, int phi_layout, unsigned flags,
                               void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!A || !Lt || !C || !w || !r_out) return LTV_ERR_NULL_PTR;
  if (T > 1 && !phi_out) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, 0);
  if (st != LTV_OK) return st;
  if (p < 1) return LTV_ERR_BAD_DIM;
  if (p > 32) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (phi_layout != LTV_PHI_COLUMN_PACKED || (flags & ~static_cast<unsigned>(LTV_TUBE_ROW_2NORM | LTV_OBSERVER_SHIFTED_GAIN)) != 0)
    return LTV_ERR_BAD_DIM;
  const int nc = n + ((p + 3) & ~3);
  if (static_cast<long long>(batch) * T * (T - 1) / 2 * n * nc >= (1ll << 40)) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (misaligned(A) || misaligned(Lt) || misaligned(C) || misaligned(w) || misaligned(phi_out) || misaligned(r_out) ||
      misaligned(workspace))
    return LTV_ERR_ALIGNMENT;
  const size_t need = phi_workspace_bytes(batch, T, n, nc);
  if (!workspace) return LTV_ERR_NULL_PTR;
  if (workspace_bytes < need) return LTV_ERR_WORKSPACE_TOO_SMALL;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  PhiArgs a{A, w, phi_out, r_out, static_cast<float*>(workspace), batch, T, n, nc, (flags & LTV_TUBE_ROW_2NORM) ? 1 : 0};
  a.Lt = Lt;
  a.C = C;
  a.p = p;
  a.yshift = (flags & LTV_OBSERVER_SHIFTED_GAIN) ? 1 : 0;
  if (p > 8) a.Ltt = reinterpret_cast<float*>(static_cast<char*>(workspace) + phi_part_bytes(batch, T, n, nc));
  unsigned long long l = 0;
  cudaError_t e = launch_phi_tube(a, static_cast<cudaStream_t>(cuda_stream), &l);
  g_launches += l;
  return e == cudaSuccess ? LTV_OK : fail_cuda(e);
}

int ltv_scan_kalman_gains(const float* A, const float* C, const float* e, const float* f, const float* Pi0,
                          float* Lt_out, float* Pi_out, int batch, int T, int n, int p, unsigned flags,
                          void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!A || !C || !e || !f || !Pi0 || !Lt_out || !Pi_out || !workspace) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, 0);
  if (st != LTV_OK) return st;
  if (p < 1 || (flags & ~3u) != 0 || flags == 3u) return LTV_ERR_BAD_DIM;
  if (p > 32) return LTV_ERR_UNSUPPORTED_SHAPE;
  if ((flags & LTV_KALMAN_SCAN) && !riccati_scan_supported(n)) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (grid_yz_overflow(batch) || ((flags & LTV_KALMAN_SCAN) && grid_yz_overflow(static_cast<long long>(batch) * (T + 1))))
    return LTV_ERR_UNSUPPORTED_SHAPE;
  if (static_cast<long long>(batch) * (T + 1) * n >= (1ll << 31)) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (misaligned(A) || misaligned(C) || misaligned(e) || misaligned(f) || misaligned(Pi0) || misaligned(Lt_out) ||
      misaligned(Pi_out) || misaligned(workspace))
    return LTV_ERR_ALIGNMENT;
  if (workspace_bytes < kalman_workspace_bytes(batch, T, n, p)) return LTV_ERR_WORKSPACE_TOO_SMALL;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  KalmanArgs a{A, C, e, f, Pi0, Lt_out, Pi_out, batch, T, n, p, workspace};
  a.mode = (flags & LTV_KALMAN_SCAN) ? 1 : ((flags & LTV_KALMAN_RECURSION) ? 2 : 0);
  unsigned long long l = 0;
  cudaError_t err = launch_kalman(a, static_cast<cudaStream_t>(cuda_stream), &l);
  g_launches += l;
  return err == cudaSuccess ? LTV_OK : fail_cuda(err);
}

int ltv_scan_constraint_tightening(const float* A, const float* w, const float* Hc, float* sigma_out, int batch, int T,
                                   int n, int nc, unsigned flags, void* workspace, size_t workspace_bytes,
                                   void* cuda_stream) {
  if (!A || !w || !Hc || !sigma_out || !workspace) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, 0);
  if (st != LTV_OK) return st;
  if (nc < 1 || flags != 0) return LTV_ERR_BAD_DIM;
  if (static_cast<long long>(batch) * T * nc >= (1ll << 31) / n || grid_yz_overflow(batch)) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (misaligned(A) || misaligned(w) || misaligned(Hc) || misaligned(sigma_out) || misaligned(workspace))
    return LTV_ERR_ALIGNMENT;
  if (workspace_bytes < constraint_workspace_bytes(batch, T, n, nc)) return LTV_ERR_WORKSPACE_TOO_SMALL;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  ConstraintArgs a{A, w, Hc, sigma_out, batch, T, n, nc, workspace};
  unsigned long long l = 0;
  cudaError_t err = launch_constraint_tightening(a, static_cast<cudaStream_t>(cuda_stream), &l);
  g_launches += l;
  return err == cudaSuccess ? LTV_OK : fail_cuda(err);
}

int ltv_scan_output_feedback_response(const float* A, const float* B, const float* Kfb, const float* Lt, const float* C,
                                      const float* w, const float* f, float* phi_xw_out, float* phi_xe_out,
                                      float* tau_out, int batch, int T, int n, int m, int p, unsigned flags,
                                      void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!A || !B || !Kfb || !Lt || !C || !w || !f || !tau_out || !workspace) return LTV_ERR_NULL_PTR;
  if (T > 1 && !phi_xw_out) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, m);
  if (st != LTV_OK) return st;
  if (m < 1 || p < 1 || flags != 0) return LTV_ERR_BAD_DIM;
  if (p > 32 || grid_yz_overflow(batch)) return LTV_ERR_UNSUPPORTED_SHAPE;
  st = check_dims(batch, T, 2 * n, 0);   // the scan runs on 2n states
  if (st != LTV_OK) return st;
  if (misaligned(A) || misaligned(B) || misaligned(Kfb) || misaligned(Lt) || misaligned(C) || misaligned(w) ||
      misaligned(f) || misaligned(phi_xw_out) || misaligned(phi_xe_out) || misaligned(tau_out) || misaligned(workspace))
    return LTV_ERR_ALIGNMENT;
  if (workspace_bytes < ofb_workspace_bytes(batch, T, n, m, p)) return LTV_ERR_WORKSPACE_TOO_SMALL;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  OfbArgs a{A, B, Kfb, Lt, C, w, f, phi_xw_out, phi_xe_out, tau_out, batch, T, n, m, p, workspace};
  unsigned long long l = 0;
  cudaError_t err = launch_output_feedback(a, static_cast<cudaStream_t>(cuda_stream), &l);
  g_launches += l;
  return err == cudaSuccess ? LTV_OK : fail_cuda(err);
}

size_t ltv_scan_output_feedback_constraints_workspace_bytes(int batch, int T, int n, int m, int nc) {
  if (check_dims(batch, T, n, m) != LTV_OK || check_dims(batch, T, 2 * n, 0) != LTV_OK || m < 1 || nc < 0) return 0;
  if (static_cast<long long>(batch) * T * (nc + m) >= (1ll << 31) / (2 * n)) return 0;
  return ofb_constraints_workspace_bytes(batch, T, n, nc, m);
}

int ltv_scan_output_feedback_constraints(const float* A, const float* B, const float* Kfb, const float* Lt, const float* C,
                                         const float* w, const float* f, const float* Hx, const float* Hu,
                                         float* phi_uw_out, float* phi_ue_out, float* sigma_out, int batch, int T, int n,
                                         int m, int p, int nc, unsigned flags, void* workspace, size_t workspace_bytes,
                                         void* cuda_stream) {
  if (!A || !B || !Kfb || !Lt || !C || !w || !f || !workspace) return LTV_ERR_NULL_PTR;
  if (nc > 0 && (!Hx || !Hu || !sigma_out)) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, m);
  if (st != LTV_OK) return st;
  if (m < 1 || p < 1 || nc < 0 || flags != 0) return LTV_ERR_BAD_DIM;
  if (p > 32 || grid_yz_overflow(batch)) return LTV_ERR_UNSUPPORTED_SHAPE;
  st = check_dims(batch, T, 2 * n, 0);   // the sweep runs on 2n states
  if (st != LTV_OK) return st;
  if (static_cast<long long>(batch) * T * (nc + m) >= (1ll << 31) / (2 * n)) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (misaligned(A) || misaligned(B) || misaligned(Kfb) || misaligned(Lt) || misaligned(C) || misaligned(w) ||
      misaligned(f) || misaligned(Hx) || misaligned(Hu) || misaligned(phi_uw_out) || misaligned(phi_ue_out) ||
      misaligned(sigma_out) || misaligned(workspace))
    return LTV_ERR_ALIGNMENT;
  if (workspace_bytes < ofb_constraints_workspace_bytes(batch, T, n, nc, m)) return LTV_ERR_WORKSPACE_TOO_SMALL;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  OfbConArgs a{A, B, Kfb, Lt, C, w, f, Hx, Hu, phi_uw_out, phi_ue_out, nc > 0 ? sigma_out : nullptr, batch, T, n, m, p, nc, workspace};
  unsigned long long l = 0;
  cudaError_t err = launch_ofb_constraints(a, static_cast<cudaStream_t>(cuda_stream), &l);
  g_launches += l;
  return err == cudaSuccess ? LTV_OK : fail_cuda(err);
}

size_t ltv_scan_output_feedback_assemble_workspace_bytes(int batch, int T, int n, int m, int p) {
  if (check_dims(batch, T, n, m) != LTV_OK || p < 1 || p > 32) return 0;
  return asm_workspace_bytes(batch, T, n, p);
}

int ltv_scan_output_feedback_assemble(const float* A, const float* Lt, const float* C, const float* w, const float* f,
                                      const float* phibar_x, const float* phibar_u, float* phi_xw_out, float* phi_xe_out,
                                      float* phi_uw_out, float* phi_ue_out, float* tau_out, int batch, int T, int n, int m,
                                      int p, unsigned flags, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!A || !Lt || !C || !w || !f || !workspace) return LTV_ERR_NULL_PTR;
  if (T > 1 && (!phibar_x || !phi_xw_out)) return LTV_ERR_NULL_PTR;
  if ((phi_uw_out || phi_ue_out) && !phibar_u) return LTV_ERR_NULL_PTR;
  if (phi_ue_out && !phi_uw_out) return LTV_ERR_NULL_PTR;   // Phi^ue is derived from Phi^uw
  int st = check_dims(batch, T, n, m);
  if (st != LTV_OK) return st;
  if (p < 1 || flags != 0 || (phi_uw_out && m < 1)) return LTV_ERR_BAD_DIM;
  if (p > 32 || grid_yz_overflow(batch)) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (misaligned(A) || misaligned(Lt) || misaligned(C) || misaligned(w) || misaligned(f) || misaligned(phibar_x) ||
      misaligned(phibar_u) || misaligned(phi_xw_out) || misaligned(phi_xe_out) || misaligned(phi_uw_out) ||
      misaligned(phi_ue_out) || misaligned(tau_out) || misaligned(workspace))
    return LTV_ERR_ALIGNMENT;
  if (workspace_bytes < asm_workspace_bytes(batch, T, n, p)) return LTV_ERR_WORKSPACE_TOO_SMALL;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  AsmArgs a{A, Lt, C, w, f, phibar_x, phi_uw_out ? phibar_u : nullptr, phi_xw_out, phi_xe_out, phi_uw_out, phi_ue_out,
            tau_out, batch, T, n, m, p, workspace};
  unsigned long long l = 0;
  cudaError_t err = launch_ofb_assemble(a, static_cast<cudaStream_t>(cuda_stream), &l);
  g_launches += l;
  return err == cudaSuccess ? LTV_OK : fail_cuda(err);
}

int ltv_scan_operator_constraint_margins(const float* phi_xw, const float* phi_uw, const float* phi_xe, const float* phi_ue,
                                         const float* Hx, const float* Hu, const float* w, const float* f, float* sigma_out,
                                         int batch, int T, int n, int m, int p, int nc, unsigned flags, void* cuda_stream) {
  if (!Hx || !w || !sigma_out) return LTV_ERR_NULL_PTR;
  if (T > 1 && !phi_xw) return LTV_ERR_NULL_PTR;
  if ((phi_uw != nullptr) != (Hu != nullptr)) return LTV_ERR_NULL_PTR;   // input part of the rows and of the operators go together
  if (phi_ue && !phi_uw) return LTV_ERR_NULL_PTR;
  if (phi_xe && !f) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, m);
  if (st != LTV_OK) return st;
  if (nc < 1 || flags != 0 || (phi_uw && m < 1) || (phi_xe && p < 1)) return LTV_ERR_BAD_DIM;
  if (p > 32 || grid_yz_overflow(batch) || !margins_supported(n, phi_uw ? m : 0, T)) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (misaligned(phi_xw) || misaligned(phi_uw) || misaligned(phi_xe) || misaligned(phi_ue) || misaligned(Hx) || misaligned(Hu) ||
      misaligned(w) || misaligned(f) || misaligned(sigma_out))
    return LTV_ERR_ALIGNMENT;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  MarginArgs a{phi_xw, phi_uw, phi_xe, phi_xe ? phi_ue : nullptr, Hx, Hu, w, f, sigma_out, batch, T, n, phi_uw ? m : 0,
               phi_xe ? p : 0, nc};
  unsigned long long l = 0;
  cudaError_t err = launch_operator_margins(a, static_cast<cudaStream_t>(cuda_stream), &l);
  g_launches += l;
  return err == cudaSuccess ? LTV_OK : fail_cuda(err);
}

long long ltv_phi_row_shard_blocks(int T, int k_lo, int k_hi) {
  if (T < 1 || k_lo < 1 || k_hi > T || k_lo >= k_hi) return -1;
  return phi_row_shard_blocks(T, k_lo, k_hi);
}

long long ltv_phi_row_shard_block_index(int T, int k_lo, int k_hi, int k, int j) { return phi_row_shard_index(T, k_lo, k_hi, k, j); }

int ltv_scan_system_response_tube_rows(const float* A, const float* w, float* phi_rows_out, float* r_out, int batch, int T,
                                       int n, int k_lo, int k_hi, unsigned flags, void* cuda_stream) {
  if (!A || !w || !phi_rows_out || !r_out) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, 0);
  if (st != LTV_OK) return st;
  if (k_lo < 1 || k_hi > T || k_lo >= k_hi || (flags & ~static_cast<unsigned>(LTV_TUBE_ROW_2NORM)) != 0) return LTV_ERR_BAD_DIM;
  if (grid_yz_overflow(batch)) return LTV_ERR_UNSUPPORTED_SHAPE;
  if (misaligned(A) || misaligned(w) || misaligned(phi_rows_out) || misaligned(r_out)) return LTV_ERR_ALIGNMENT;
  int sms = 0;
  st = check_device(&sms);
  if (st != LTV_OK) return st;
  PhiRowsArgs a{A, w, phi_rows_out, r_out, batch, T, n, k_lo, k_hi, (flags & LTV_TUBE_ROW_2NORM) ? 1 : 0};
  unsigned long long l = 0;
  cudaError_t err = launch_phi_rows(a, static_cast<cudaStream_t>(cuda_stream), &l);
  g_launches += l;
  return err == cudaSuccess ? LTV_OK : fail_cuda(err);
}

int ltv_scan_pipeline_host(const float* A_host, const float* B_host, const float* c_host, const float* x0_host,
                           const float* u_host, const float* w_host, const float* g_host, float* x_host,
                           float* phi_host, float* r_host, float* lambda_host, float* grad_u_host,
                           float* grad_x0_host, int batch, int T, int n, int m, void* workspace,
                           size_t workspace_bytes, void* cuda_stream, float** phi_device_out) {
  const bool with_phi = w_host != nullptr;
  if (!A_host || !x0_host || !g_host || !x_host || !lambda_host || !workspace) return LTV_ERR_NULL_PTR;
  if (with_phi && !r_host) return LTV_ERR_NULL_PTR;
  if (grad_u_host && m > 0 && !B_host) return LTV_ERR_NULL_PTR;
  int st = check_dims(batch, T, n, m);
  if (st != LTV_OK) return st;
  if (misaligned(workspace)) return LTV_ERR_ALIGNMENT;
  if (workspace_bytes < ltv_scan_workspace_bytes(with_phi ? LTV_OP_PIPELINE_HOST : LTV_OP_PIPELINE_HOST_NO_PHI, batch, T, n, m))
    return LTV_ERR_WORKSPACE_TOO_SMALL;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const size_t b = batch, t = T, nn = n, mm = m, P = t * (t - 1) / 2;
  char* cur = static_cast<char*>(workspace);
  auto carve = [&](size_t floats) {
    float* p = reinterpret_cast<float*>(cur);
    cur += align_up(floats * 4 + 16, 256);
    return p;
  };
  float* dA = carve(b * t * nn * nn);
  float* dB = carve(b * t * nn * mm);
  float* dc = carve(b * t * nn);
  float* dx0 = carve(b * nn);
  float* du = carve(b * t * mm);
  float* dw = carve(b * t * nn);
  float* dg = carve(b * t * nn);
  float* dx = carve(b * t * nn);
  float* dphi = carve(with_phi ? b * P * nn * nn : 0);
  float* dr = carve(b * t * nn);
  float* dl = carve(b * t * nn);
  float* dgu = carve(b * t * mm);
  float* dgx = carve(b * nn);
  void* phi_ws = cur;
  const size_t phi_ws_bytes = with_phi ? phi_workspace_bytes(batch, T, n, n) : 0;
  if (phi_device_out) *phi_device_out = with_phi ? dphi : nullptr;

  cudaError_t e;
#define LTV_D2H(dst, src, floats)                                                                   \
  if ((dst) && (floats) > 0) {                                                                      \
    e = cudaMemcpyAsync((dst), (src), (floats) * sizeof(float), cudaMemcpyDeviceToHost, s);         \
    if (e != cudaSuccess) {                                                                         \
      cudaStreamSynchronize(cs);                                                                    \
      cleanup();                                                                                    \
      return fail_cuda(e);                                                                          \
    }                                                                                               \
  }
  // Chunks of the batch are pipelined: an internal copy stream uploads chunk i+1 while chunk i is computed on
  // the caller's stream (items are independent; the upload, 97 % of it A, is the longer leg at PCIe rates).
  // Chunks are multiples of 4 items so that every slice stays 16-byte aligned.
  int cb = batch;
  if (batch >= 8 && option(LTV_OPT_PIPELINE_CHUNKS) > 1) {
    const int want = option(LTV_OPT_PIPELINE_CHUNKS);
    cb = ((batch + want - 1) / want + 3) & ~3;
  }
  const int nchunk = (batch + cb - 1) / cb;
  cudaStream_t cs = nullptr;
  cudaEvent_t ev_start = nullptr, ev_up[16] = {};
  if (nchunk > 16) return LTV_ERR_BAD_DIM;
  auto cleanup = [&]() {
    for (int i = 0; i < 16; ++i)
      if (ev_up[i]) cudaEventDestroy(ev_up[i]);
    if (ev_start) cudaEventDestroy(ev_start);
    if (cs) cudaStreamDestroy(cs);
  };
#define LTV_TRY(call)                     \
  if ((e = (call)) != cudaSuccess) {      \
    cleanup();                            \
    return fail_cuda(e);                  \
  }
  LTV_TRY(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
  LTV_TRY(cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming));
  LTV_TRY(cudaEventRecord(ev_start, s));        // earlier work on the caller's stream may still use the workspace
  LTV_TRY(cudaStreamWaitEvent(cs, ev_start, 0));
  auto up = [&](float* dst, const float* src, size_t per_item, int c0, int cn) -> cudaError_t {
    if (!src || per_item == 0) return cudaSuccess;
    return cudaMemcpyAsync(dst + per_item * c0, src + per_item * c0, per_item * cn * sizeof(float),
                           cudaMemcpyHostToDevice, cs);
  };
  for (int ci = 0; ci < nchunk; ++ci) {
    const int c0 = ci * cb, cn = (c0 + cb <= batch) ? cb : batch - c0;
    LTV_TRY(up(dA, A_host, t * nn * nn, c0, cn));
    LTV_TRY(up(dB, B_host, t * nn * mm, c0, cn));
    LTV_TRY(up(dc, c_host, t * nn, c0, cn));
    LTV_TRY(up(dx0, x0_host, nn, c0, cn));
    LTV_TRY(up(du, u_host, t * mm, c0, cn));
    LTV_TRY(up(dw, w_host, t * nn, c0, cn));
    LTV_TRY(up(dg, g_host, t * nn, c0, cn));
    LTV_TRY(cudaEventCreateWithFlags(&ev_up[ci], cudaEventDisableTiming));
    LTV_TRY(cudaEventRecord(ev_up[ci], cs));
  }
  for (int ci = 0; ci < nchunk; ++ci) {
    const size_t c0 = static_cast<size_t>(ci) * cb;
    const int cn = (c0 + cb <= b) ? cb : static_cast<int>(b - c0);
    LTV_TRY(cudaStreamWaitEvent(s, ev_up[ci], 0));
    st = ltv_scan_rollout_adjoint(dA + c0 * t * nn * nn, B_host ? dB + c0 * t * nn * mm : nullptr,
                                  c_host ? dc + c0 * t * nn : nullptr, dx0 + c0 * nn, u_host ? du + c0 * t * mm : nullptr,
                                  dg + c0 * t * nn, dx + c0 * t * nn, dl + c0 * t * nn,
                                  (grad_u_host && B_host) ? dgu + c0 * t * mm : nullptr,
                                  grad_x0_host ? dgx + c0 * nn : nullptr, cn, T, n, m, nullptr, 0, cuda_stream);
    if (st == LTV_OK && with_phi)
      st = ltv_scan_system_response_tube(dA + c0 * t * nn * nn, dw + c0 * t * nn, dphi + c0 * P * nn * nn,
                                         dr + c0 * t * nn, cn, T, n, LTV_PHI_COLUMN_PACKED, 0, phi_ws, phi_ws_bytes,
                                         cuda_stream);
    if (st != LTV_OK) {
      cudaStreamSynchronize(cs);
      cleanup();
      return st;
    }
  }
  LTV_D2H(x_host, dx, b * t * nn);
  if (with_phi) LTV_D2H(r_host, dr, b * t * nn);
  LTV_D2H(lambda_host, dl, b * t * nn);
  if (B_host) LTV_D2H(grad_u_host, dgu, b * t * mm);
  LTV_D2H(grad_x0_host, dgx, b * nn);
  if (with_phi) LTV_D2H(phi_host, dphi, b * P * nn * nn);
  e = cudaStreamSynchronize(s);
  cudaStreamSynchronize(cs);
  cleanup();
  if (e != cudaSuccess) return fail_cuda(e);
  return LTV_OK;
#undef LTV_TRY
#undef LTV_D2H
}

const char* ltv_status_string(int status) {
  switch (status) {
    case LTV_OK: return "LTV_OK";
    case LTV_ERR_NULL_PTR: return "LTV_ERR_NULL_PTR";
    case LTV_ERR_BAD_DIM: return "LTV_ERR_BAD_DIM";
    case LTV_ERR_UNSUPPORTED_SHAPE: return "LTV_ERR_UNSUPPORTED_SHAPE";
    case LTV_ERR_ALIGNMENT: return "LTV_ERR_ALIGNMENT";
    case LTV_ERR_WORKSPACE_TOO_SMALL: return "LTV_ERR_WORKSPACE_TOO_SMALL";
    case LTV_ERR_ARCH: return "LTV_ERR_ARCH";
    case LTV_ERR_CUDA: return "LTV_ERR_CUDA";
    case LTV_ERR_STATIC_SCRATCH_LIMIT: return "LTV_ERR_STATIC_SCRATCH_LIMIT";
    default: return "LTV_ERR_UNKNOWN";
  }
}

int ltv_profile_enable(int on) {
  ProfState& p = prof();
  std::lock_guard<std::mutex> lk(p.mu);
  p.on.store(on != 0, std::memory_order_release);
  p.used = 0;   // scopes still open on other threads keep their (already captured) events; their record is dropped
  return LTV_OK;
}

const char* ltv_profile_class_name(int cls) {
  static const char* const names[LTV_PROFILE_CLASSES] = {
      "rollout", "adjoint", "phi_level0", "phi_combine_tc", "phi_combine_simt", "phi_finalize", "kalman_gemm",
      "kalman_simt", "phi_relayout", "vector_pair", "ofb_support", "fused_small"};
  return (cls >= 0 && cls < LTV_PROFILE_CLASSES) ? names[cls] : nullptr;
}

int ltv_profile_collect(double* ms_by_class, unsigned long long* launches_by_class) {
  if (!ms_by_class || !launches_by_class) return LTV_ERR_NULL_PTR;
  ProfState& p = prof();
  std::lock_guard<std::mutex> lk(p.mu);
  for (int c = 0; c < LTV_PROFILE_CLASSES; ++c) {
    ms_by_class[c] = 0.0;
    launches_by_class[c] = 0;
  }
  for (size_t i = 0; i < p.used; ++i) {
    cudaError_t e = cudaEventSynchronize(p.end[i]);
    if (e != cudaSuccess) return fail_cuda(e);
    float ms = 0.f;
    e = cudaEventElapsedTime(&ms, p.beg[i], p.end[i]);
    if (e != cudaSuccess) return fail_cuda(e);
    ms_by_class[p.cls[i]] += ms;
    launches_by_class[p.cls[i]] += 1;
  }
  p.used = 0;
  return LTV_OK;
}

int ltv_set_option(int opt, int value) {
  switch (opt) {
    case LTV_OPT_VECTOR_CLUSTER:
      if (value < 0 || value > 16) return LTV_ERR_BAD_DIM;
      break;
    case LTV_OPT_PIPELINE_CHUNKS:
      if (value < 1 || value > 16) return LTV_ERR_BAD_DIM;
      break;
    case LTV_OPT_OUTPUT_FEEDBACK_ROUTE:
      if (value < 0 || value > 2) return LTV_ERR_BAD_DIM;
      break;
    default:
      return LTV_ERR_BAD_DIM;
  }
  g_options[opt].store(value, std::memory_order_relaxed);
  return LTV_OK;
}

int ltv_get_option(int opt) { return (opt >= 0 && opt < LTV_OPT_COUNT) ? option(opt) : -1; }

int ltv_last_cuda_error(void) { return g_last_cuda_error; }
int ltv_version(void) { return 100; }
unsigned long long ltv_launch_count(void) { return g_launches.load(); }

}  // extern "C"
