// Internal host-side declarations shared by the translation units of libltvscan.so.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

namespace ltv {

// Every launcher enqueues on `stream`, never synchronises, and returns the cudaError_t of the launch.
// `launches` is incremented by the number of kernels enqueued.

struct RolloutArgs {
  const float *A, *B, *c, *x0, *u;
  float* x_out;
  int batch, T, n, m;
  int sm_budget = 0;   // > 0: use at most this many SMs (the rollout / adjoint pair shares the machine); 0 = all
};
// cluster = 0: chosen by pick_cluster_model
cudaError_t launch_rollout(const RolloutArgs& a, int cluster, cudaStream_t stream, unsigned long long* launches);
int rollout_cluster_choice(const RolloutArgs& a);   // the cluster size `cluster = 0` would pick
int rollout_clusters_resident(const RolloutArgs& a, int cluster);   // clusters of that size that can be resident at once

struct AdjointArgs {
  const float *A, *B, *g;
  float *lambda_out, *grad_u_out, *grad_x0_out;
  int batch, T, n, m;
  int sm_budget = 0;   // as RolloutArgs (cluster choice only: the adjoint grid is one cluster per item)
};
cudaError_t launch_adjoint(const AdjointArgs& a, int cluster, cudaStream_t stream, unsigned long long* launches);
int adjoint_cluster_choice(const AdjointArgs& a);
int adjoint_clusters_resident(const AdjointArgs& a, int cluster);

struct PhiArgs {
  const float *A, *w;
  float *phi, *r;
  float* part;  // workspace: [batch, P, NT, n] per-(block, n-tile) tube partial sums
  int batch, T, n;
  int nc;         // columns per Phi block = its row stride: n, or n + roundup4(p) when the observer's PhiY rides along
  int tube_mode;  // 0: sum_j |Phi_ij| w_j (box tube); 1: sqrt(sum_j (Phi_ij w_j)^2) per block (row-wise two-norm, eq.(12e))
  // closed-loop observer propagation (eq.(14)): level 0 forms Abar_s = A_s + Lt_s C_s and PhiY(s+1,s) = Abar_s Lt_s
  const float* Lt = nullptr;  // [batch,T,n,p] = L_j^T, or nullptr: plain system response
  const float* C = nullptr;   // [batch,T,p,n]
  int p = 0;
  float* Ltt = nullptr;       // workspace [batch,T,nc-n,n]: the gains transposed (p > 8 only)
  int yshift = 0;             // 1: PhiY(t,s) = PhiX(t,s) Lt_{s-1} (zero for s = 0): the Phihat^y of (12c)/(15)
};
// n-tile width the Phi path uses for this n (decides the size of `part`) and whether it is the tcgen05 path
int phi_tile_n(int n, int nc);
bool phi_uses_tensor_cores(int n);
size_t phi_workspace_bytes(int batch, int T, int n, int nc);
size_t phi_part_bytes(int batch, int T, int n, int nc);
cudaError_t launch_phi_tube(const PhiArgs& a, cudaStream_t stream, unsigned long long* launches);
// bytes of a COLUMN_PACKED Phi staging buffer (the scan's native order) and the block re-ordering copy into
// LTV_PHI_ROW_PACKED / LTV_PHI_SQUARE_GRID
size_t phi_colpacked_bytes(int batch, int T, int n, int nc);
cudaError_t launch_phi_relayout(const float* src, float* dst, int batch, int T, int n, int nc, int layout, int num_sms,
                                cudaStream_t stream);

// Kalman recursion of eq.(13) (kalman.cu)
struct KalmanArgs {
  const float *A, *C, *e, *f, *Pi0;
  float *Lt_out, *Pi_out;
  int batch, T, n, p;
  void* workspace;
  int mode = 0;   // 0: pick (kalman_use_scan), 1: associative scan (16)(17) (n <= 64), 2: recursion (13)
};
// riccati_scan.cu
bool riccati_scan_supported(int n);
size_t riccati_scan_workspace_bytes(int batch, int T, int n);
cudaError_t launch_riccati_scan(const KalmanArgs& a, float* AD, cudaStream_t stream, unsigned long long* launches);
size_t kalman_workspace_bytes(int batch, int T, int n, int p);
// kalman_small.cu: the whole recursion of an item in one CTA (n <= 64)
bool kalman_small_supported(int n, int p);
cudaError_t launch_kalman_small(const KalmanArgs& a, cudaStream_t stream, unsigned long long* launches);
cudaError_t launch_kalman(const KalmanArgs& a, cudaStream_t stream, unsigned long long* launches);

// Constraint-tightening margins of eq.(12d) (constraints.cu)
struct ConstraintArgs {
  const float *A, *w, *Hc;
  float* sigma_out;
  int batch, T, n, nc;
  void* workspace;
};
size_t constraint_workspace_bytes(int batch, int T, int n, int nc);
cudaError_t launch_constraint_tightening(const ConstraintArgs& a, cudaStream_t stream, unsigned long long* launches);

// Output-feedback responses of eq.(15) + tube (12e) for gain-defined controllers (output_feedback.cu)
struct OfbArgs {
  const float *A, *B, *Kfb, *Lt, *C, *w, *f;
  float *phi_xw, *phi_xe, *tau;
  int batch, T, n, m, p;
  void* workspace;
};
size_t ofb_workspace_bytes(int batch, int T, int n, int m, int p);   // m = p = 0: sizes of the gains unknown
cudaError_t launch_output_feedback(const OfbArgs& a, cudaStream_t stream, unsigned long long* launches);
// column route of the same call (assemble.cu): one scan + the backward column recursion on D = Phi^xw - Phibar^x
size_t ofb_columns_workspace_bytes(int batch, int T, int n);
bool ofb_columns_supported(int n, int m, int p);
cudaError_t launch_ofb_response_columns(const OfbArgs& a, cudaStream_t stream, unsigned long long* launches);

// Input-side responses of eq.(15) and closed-loop margins of eq.(12d) (output_feedback.cu)
struct OfbConArgs {
  const float *A, *B, *Kfb, *Lt, *C, *w, *f, *Hx, *Hu;   // Hx, Hu null iff nc == 0
  float *phi_uw, *phi_ue, *sigma;                        // each may be null
  int batch, T, n, m, p, nc;
  void* workspace;
};
size_t ofb_constraints_workspace_bytes(int batch, int T, int n, int nc, int m);
cudaError_t launch_ofb_constraints(const OfbConArgs& a, cudaStream_t stream, unsigned long long* launches);

// Eq.(15) for a general Phibar (assemble.cu)
struct AsmArgs {
  const float *A, *Lt, *C, *w, *f;
  const float *phibar_x, *phibar_u;            // phibar_u null iff phi_uw null
  float *phi_xw, *phi_xe, *phi_uw, *phi_ue, *tau;   // phi_xe, phi_uw, phi_ue, tau may be null
  int batch, T, n, m, p;
  void* workspace;
};
size_t asm_workspace_bytes(int batch, int T, int n, int p);
cudaError_t launch_ofb_assemble(const AsmArgs& a, cudaStream_t stream, unsigned long long* launches);

// Block rows of the system response of one shard (phi_rows.cu)
struct PhiRowsArgs {
  const float *A, *w;
  float *phi, *r;      // phi [batch, Ps, n, n] (the shard's column-packed order), r [batch, T, n] (rows k_lo .. k_hi-1 written)
  int batch, T, n, k_lo, k_hi, tube_mode;
};
long long phi_row_shard_blocks(int T, int k_lo, int k_hi);
long long phi_row_shard_index(int T, int k_lo, int k_hi, int k, int j);
cudaError_t launch_phi_rows(const PhiRowsArgs& a, cudaStream_t stream, unsigned long long* launches);

// Margins (12d) on assembled operators (margins.cu)
struct MarginArgs {
  const float *phi_xw, *phi_uw, *phi_xe, *phi_ue, *Hx, *Hu, *w, *f;   // phi_uw / Hu and phi_xe / phi_ue may be null
  float* sigma;
  int batch, T, n, m, p, nc;
};
bool margins_supported(int n, int m, int T);
cudaError_t launch_operator_margins(const MarginArgs& a, cudaStream_t stream, unsigned long long* launches);

// Whole hot path of a small problem in one launch (fused_small.cu): n <= 64 and all of A in one SM's shared memory
struct FusedSmallArgs {
  const float *A, *B, *c, *x0, *u, *w, *g;
  float *x_out, *phi_out, *r_out, *lambda_out, *grad_u_out, *grad_x0_out;
  int batch, T, n, m, tube_mode;
};
bool fused_small_supported(int batch, int T, int n, int m);
cudaError_t launch_fused_small(const FusedSmallArgs& a, cudaStream_t stream, unsigned long long* launches);

// Cluster size (CTAs per item, 1..16, any integer) for the two vector kernels.  max_active[C] = clusters of C CTAs
// that can be resident at once (cudaOccupancyMaxActiveClusters; 0 = not launchable).  Minimises a simple
// time model over the waves of clusters: an SM streams ~70 GB/s, the device ~6.5 TB/s (both measured).
int pick_cluster_model(int batch, int n, const int* max_active, int sm_budget = 0);
// fills max_active[1..16] for `kernel` (any __global__ function pointer) at the given block size / dynamic smem
void query_max_active_clusters(const void* kernel, int threads, size_t smem, int* max_active);
// developer override LTV_SCAN_<name>=<int>, compiled in only with -DLTV_TUNING; the product build returns `dflt`
int env_int(const char* name, int dflt);
// value of a documented ltv_set_option knob (include/ltv_scan.h)
int option(int which);
// for entry points that live outside api.cu: add to the library's launch counter; record a failed CUDA call for
// ltv_last_cuda_error (clears the runtime's error state) and return LTV_ERR_CUDA
void count_launches(unsigned long long n);
int report_cuda_error(cudaError_t e);

// optional per-kernel timing (ltv_profile_enable): CUDA events recorded on the launch stream around a kernel
enum ProfClass { kProfRollout = 0, kProfAdjoint, kProfPhiLevel0, kProfPhiCombineTc, kProfPhiCombineSimt,
                 kProfPhiFinalize, kProfKalmanGemm, kProfKalmanSimt, kProfPhiRelayout, kProfVectorPair, kProfOfbSupport, kProfFusedSmall, kProfNumClasses };
struct ProfScope {
  ProfScope(int cls, cudaStream_t s);
  ~ProfScope();
  int slot;
  cudaStream_t stream;
  void* end_event;   // cudaEvent_t captured at construction
};

#ifdef LTV_TUNING
// developer builds: host-mapped record buffer of the spin-limit traps (ptx.cuh); device alias of the same memory
unsigned int* dbg_buffer_device();
#define LTV_DBG_INSTALL()                                                        \
  do {                                                                           \
    unsigned int* dbgp_ = dbg_buffer_device();                                   \
    cudaMemcpyToSymbolAsync(g_ltv_dbg, &dbgp_, sizeof(dbgp_), 0, cudaMemcpyHostToDevice, stream); \
  } while (0)
#else
#define LTV_DBG_INSTALL() do {} while (0)
#endif

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace ltv
