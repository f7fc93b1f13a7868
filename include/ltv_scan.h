/* ltv_scan.h - C ABI of the B200-native LTV-scan library (libltvscan.so).
 *
 * The data-parallel hot path of CORD-SLS (arxiv 2606.14188): the scan over the planning horizon of a
 * batched linear time-varying system
 *
 *     x_{t+1} = A_t x_t + B_t u_t + c_t ,   t = 0 .. T-1
 *
 * "linearizations of the dynamics ... about the nominal trajectory" (Sec. 4.2); "Both (13)
 * and (14) require dense matrix multiplications serially through the planning horizon.  As such, we use
 * parallel associative scans on the GPU"; "forward parallel associative scan"
 * (PAPER.md:177).  Three operations:
 *
 *   ltv_scan_rollout               x_1 .. x_T                       PAPER.md:53 eq.(2), :139 eq.(12b)
 *   ltv_scan_system_response_tube  Phi(t,s) = A_{t-1} ... A_s, s<t  PAPER.md:142 eq.(12c), Z of :150,
 *                                  (strictly-lower blocks of          recursion shape of :159 eq.(14)
 *                                  (I - Z A)^{-1}) fused with
 *                                  r_t = sum_{s<t} |Phi(t,s)| w_s   PAPER.md:147 eq.(12e), box form
 *   ltv_scan_adjoint               lam_t = A_t^T lam_{t+1} + g_t,   PAPER.md:106-110 eq.(10) chained
 *                                  dL/du_t = B_t^T lam_{t+1}          over the horizon
 *
 * Conventions common to all entry points
 *   - fp32, dense, contiguous, row-major, batch outermost.  A[b,t,i,j] = d x_{t+1,i} / d x_{t,j}.
 *   - Pointers documented "device" are CUDA device pointers of the current device, 16-byte aligned.
 *     Pointers documented "host" are ordinary host pointers (pinned memory recommended).
 *   - Ownership: the caller owns every buffer (inputs, outputs, workspace).  The library allocates no
 *     device memory, keeps no state across calls besides cached function attributes, enqueues its work on
 *     `cuda_stream` (a cudaStream_t passed as void*, NULL = legacy default stream) and returns WITHOUT
 *     synchronising.  Inputs are never modified; outputs and workspace must not alias inputs or each other.
 *   - Errors: every entry point returns an ltv_status.  Arguments are validated on the host before
 *     anything is enqueued (so a failed call has no side effects); nothing throws or aborts.  There is no
 *     CPU fallback: without an sm_100 device the calls return LTV_ERR_ARCH / LTV_ERR_CUDA.
 *   - Shape limits: batch, T, n >= 1; m >= 0; n % 4 == 0 (16-byte rows: TMA / 128-bit access); n <= 8192.
 *     Anything else is LTV_ERR_BAD_DIM (non-positive) or LTV_ERR_UNSUPPORTED_SHAPE.
 */
#ifndef LTV_SCAN_H_
#define LTV_SCAN_H_

#include <stddef.h>

#if defined(__GNUC__)
#define LTV_API __attribute__((visibility("default")))
#else
#define LTV_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  LTV_OK = 0,
  LTV_ERR_NULL_PTR = 1,            /* a required pointer is NULL                                     */
  LTV_ERR_BAD_DIM = 2,             /* batch, T, n < 1 or m < 0, or an unknown enum / flag value       */
  LTV_ERR_UNSUPPORTED_SHAPE = 3,   /* n % 4 != 0, n > 8192, index space overflow                      */
  LTV_ERR_ALIGNMENT = 4,           /* a device pointer is not 16-byte aligned                         */
  LTV_ERR_WORKSPACE_TOO_SMALL = 5, /* workspace_bytes < ltv_scan_workspace_bytes(...)                 */
  LTV_ERR_ARCH = 6,                /* current device is not compute capability 10.x                   */
  LTV_ERR_CUDA = 7,                /* a CUDA runtime / driver call failed: see ltv_last_cuda_error()  */
  LTV_ERR_STATIC_SCRATCH_LIMIT = 8 /* ltv_scan_system_response_tube_static: the problem needs more scratch than the
                                      library's fixed device array holds (ltv_static_scratch_bytes())      */
} ltv_status;

/* `op` argument of ltv_scan_workspace_bytes */
enum { LTV_OP_ROLLOUT = 0, LTV_OP_SYSTEM_RESPONSE_TUBE = 1, LTV_OP_ADJOINT = 2, LTV_OP_PIPELINE_HOST = 3,
       LTV_OP_PIPELINE_HOST_NO_PHI = 4 /* ltv_scan_pipeline_host with w_host == NULL: rollout + adjoint only */,
       LTV_OP_OBSERVER_RESPONSE = 5 /* ltv_scan_observer_response; pass p (rows of C) as `m` */,
       LTV_OP_KALMAN_GAINS = 6 /* ltv_scan_kalman_gains; pass p (rows of C) as `m` */,
       LTV_OP_CONSTRAINT_TIGHTENING = 7 /* ltv_scan_constraint_tightening; pass nc (constraint rows) as `m` */,
       LTV_OP_OUTPUT_FEEDBACK = 8 /* ltv_scan_output_feedback_response; `m` = max(m, p) of the call, or 0 = unknown */,
       LTV_OP_SYSTEM_RESPONSE_TUBE_RELAYOUT = 9 /* ltv_scan_system_response_tube with LTV_PHI_ROW_PACKED / _SQUARE_GRID */ };

/* `phi_layout` argument: where block (t,s), 0 <= s < t <= T-1, of one item sits in phi_out.  Blocks are contiguous
 * n x n row-major matrices in every layout; P = T(T-1)/2.
 *   LTV_PHI_ROW_PACKED (0)     phi_out[batch, P, n, n], block index p(t,s) = t(t-1)/2 + s: the block rows of the lower-
 *                              triangular operator one after the other, the order (12c)-(12e) index it in.
 *   LTV_PHI_SQUARE_GRID (1)    phi_out[batch, T, T, n, n], block (t,s) at grid cell t T + s; only cells with s < t are
 *                              written, the others are left untouched.
 *   LTV_PHI_COLUMN_PACKED (2)  phi_out[batch, P, n, n], block index q(t,s) = s(T-1) - s(s-1)/2 + (t-s-1)
 *                              (ltv_phi_block_index): column by column, so all blocks with the same s are one contiguous
 *                              tall (T-1-s)n x n row-major matrix.  This is the order the scan COMPUTES in - the
 *                              divide-and-conquer combine Phi(t,s) = Phi(t,mid) Phi(mid,s) streams its stacked left
 *                              operand and each output column as one matrix (128-row tiles run across block boundaries:
 *                              97-99 % tile fill instead of 78 % at n = 300) - and the FAST PATH: no extra pass.
 * With ROW_PACKED or SQUARE_GRID the scan runs column-packed inside the workspace (which must then also hold a
 * column-packed copy of Phi: op LTV_OP_SYSTEM_RESPONSE_TUBE_RELAYOUT) and one streaming block copy re-orders it into
 * phi_out at the end: + 8 n^2 bytes of HBM traffic per block (about + 3.5 ms on the 6 ms call at n = 300, T = 32,
 * batch 64).  ltv_scan_observer_response and ltv_scan_output_feedback_response accept LTV_PHI_COLUMN_PACKED only. */
enum { LTV_PHI_ROW_PACKED = 0, LTV_PHI_SQUARE_GRID = 1, LTV_PHI_COLUMN_PACKED = 2 };

/* `flags` bits of ltv_scan_system_response_tube / ltv_scan_observer_response. */
enum { LTV_TUBE_ROW_2NORM = 1,
       LTV_OBSERVER_SHIFTED_GAIN = 2 /* observer call only: PhiY(t,s) = PhiX(t,s) Lt_{s-1}, zero for s = 0 (see there) */ };

/* Block index q(t,s) of the COLUMN_PACKED layout; -1 if not 0 <= s < t <= T-1.  Pure host arithmetic. */
LTV_API long long ltv_phi_block_index(int T, int t, int s);
/* The same for any layout (ROW_PACKED: t(t-1)/2 + s; SQUARE_GRID: t T + s); -1 for a bad layout or index. */
LTV_API long long ltv_phi_block_index_layout(int T, int t, int s, int phi_layout);

/* Bytes of device workspace the given op needs for these sizes (0 is a valid answer; a NULL workspace is
 * then accepted).  Returns 0 for invalid arguments.  For LTV_OP_PIPELINE_HOST the figure covers device
 * staging copies of every input and output of ltv_scan_pipeline_host (including Phi). */
LTV_API size_t ltv_scan_workspace_bytes(int op, int batch, int T, int n, int m);

/* Rollout  x_{t+1} = A_t x_t + B_t u_t + c_t  (north_star (i)).
 *   A      device [batch,T,n,n]       required
 *   B      device [batch,T,n,m]       may be NULL (then u is ignored; the term is zero); also if m == 0
 *   c      device [batch,T,n]         may be NULL (zero)
 *   x0     device [batch,n]           required
 *   u      device [batch,T,m]         may be NULL (zero)
 *   x_out  device [batch,T,n]         x_out[b,t] = x_{t+1}
 * One thread-block cluster per item streams A_t through a shared-memory ring (HBM-bound GEMV chain);
 * the affine term b_t = B_t u_t + c_t is formed on the fly and never written. */
LTV_API int ltv_scan_rollout(const float* A, const float* B, const float* c, const float* x0, const float* u,
                     float* x_out, int batch, int T, int n, int m,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);

/* System response + reachable tube (north_star (ii); eq.(12c), :147 eq.(12e)).
 *   A        device [batch,T,n,n]     required; only A_0 .. A_{T-2} are read
 *   w        device [batch,T,n]       required; w_s >= 0, only s <= T-2 read
 *   phi_out  device [batch,P,n,n]     P = T(T-1)/2, or [batch,T,T,n,n] for LTV_PHI_SQUARE_GRID: layout `phi_layout`;
 *                                     Phi(t,t) = I is not stored
 *   r_out    device [batch,T,n]       r_0 = 0, r_t = sum_{s<t} |Phi(t,s)| w_s  (element-wise abs)
 *   flags    0, or LTV_TUBE_ROW_2NORM: r_t[i] = sum_{s<t} || row_i(Phi(t,s) diag(w_s)) ||_2, the row-wise two-norm
 *            tube of eq.(12e) as printed with the disturbance scaling E_s = diag(w_s)
 * T == 1 is valid: no blocks, r zero-filled.  Time-parallel schedule: level 0 copies the sub-diagonal
 * blocks Phi(s+1,s) = A_s; level l = 1..ceil(log2(T-1)) forms, for every aligned segment of 2^l steps with
 * midpoint mid, all Phi(t,s) = Phi(t,mid) Phi(mid,s), s < mid < t, as one stacked GEMM (3xTF32 on tcgen05
 * tensor cores for n >= 96, fp32 FMA below) whose epilogue also accumulates |Phi| w_s, so Phi is never
 * re-read for the tube.  The tube reduction is deterministic (fixed-order partial sums, no atomics). */
LTV_API int ltv_scan_system_response_tube(const float* A, const float* w, float* phi_out, float* r_out,
                                  int batch, int T, int n, int phi_layout, unsigned flags,
                                  void* workspace, size_t workspace_bytes, void* cuda_stream);

/* The same call for callers that cannot allocate device memory at all (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no workspace argument.  The scratch the call needs - the tube partial sums, exactly
 * ltv_scan_workspace_bytes(LTV_OP_SYSTEM_RESPONSE_TUBE, batch, T, n, 0) bytes - lives in a device array of FIXED size inside
 * the library: ltv_static_scratch_bytes() = 32 MiB, held by every GPU that loads the library until the process exits (enough
 * for BASELINE.json configs[0] whole, ~27 items of configs[1], 6 of configs[2], one of configs[3]).  Problems that need more
 * return LTV_ERR_STATIC_SCRATCH_LIMIT before anything is enqueued: split the batch, or use the regular call with a workspace.
 * The library calls no cudaMalloc, cudaFree or other allocating routine in this call.  Arguments, results and kernels are those
 * of ltv_scan_system_response_tube with phi_layout = LTV_PHI_COLUMN_PACKED (the only layout here: the others need a second
 * Phi-sized buffer).  SHARING: every call on a device uses the same array.  It keeps the previous call's contents, which is
 * harmless - each call writes every partial sum before it reads it, nothing needs to start at zero - but two calls that
 * overlap on the GPU (different streams without ordering between them) race on it; calls on one stream are safe. */
LTV_API size_t ltv_static_scratch_bytes(void);
LTV_API int ltv_scan_system_response_tube_static(const float* A, const float* w, float* phi_out, float* r_out,
                                                 int batch, int T, int n, unsigned flags, void* cuda_stream);

/* One SHARD of the system response of the same items (eq.(12c): the blocks of (I - Z A)^-1; tube rows :147
 * eq.(12e)): the block ROWS k_lo <= k < k_hi (1 <= k_lo < k_hi <= T) and their tube rows - what one GPU computes when single large items are split over several GPUs (optional; sharding.py has the
 * partition).  The split is by rows because a block row needs nothing outside itself, Phi(k,j) = Phi(k,j+1) A_j with
 * Phi(k,k) = I: every GPU holds A (replicated), no GPU reads another one's blocks, and r_k is COMPLETE on the GPU that owns row
 * k - no reduction over GPUs (summing the zero-initialised r of all shards, or gathering the rows, assembles r).
 *   A, w       as in ltv_scan_system_response_tube
 *   phi_rows_out device [batch,Ps,n,n]  Ps = ltv_phi_row_shard_blocks(T,k_lo,k_hi) = sum_{k=k_lo}^{k_hi-1} k; block (k,j), 0 <= j < k,
 *                                       at ltv_phi_row_shard_block_index(T,k_lo,k_hi,k,j): column by column (the shard's own
 *                                       column-packed order: column j holds k = max(k_lo, j+1) .. k_hi-1)
 *   r_out      device [batch,T,n]       rows k_lo .. k_hi-1 are written (and r_0 = 0 if k_lo == 1), the others left untouched
 *   flags      0 or LTV_TUBE_ROW_2NORM
 * k_hi - 1 backward steps over the columns, each one batched GEMM of the shard's stacked column j+1 with A_j (tcgen05 3xTF32
 * for n >= 96) plus a row kernel (block (j+1,j) = A_j, tube terms): one n^3 product per block as in the time-parallel scan, but
 * sequential in j - the price of a split with no communication.  k_lo = 1, k_hi = T is the whole response.  Deterministic.
 * No workspace.  batch <= 65535. */
LTV_API long long ltv_phi_row_shard_blocks(int T, int k_lo, int k_hi);
LTV_API long long ltv_phi_row_shard_block_index(int T, int k_lo, int k_hi, int k, int j);
LTV_API int ltv_scan_system_response_tube_rows(const float* A, const float* w, float* phi_rows_out, float* r_out,
                                               int batch, int T, int n, int k_lo, int k_hi, unsigned flags,
                                               void* cuda_stream);

/* Adjoint scan (north_star (iii); eq.(10) chained over the horizon) for
 * L = sum_{t=1}^{T} l_t(x_t), g_t = dl_t/dx_t, lam_{T+1} = 0:
 *     lam_T = g_T;  lam_t = A_t^T lam_{t+1} + g_t (t = T-1 .. 1);  grad_u[t] = B_t^T lam_{t+1} (t = 0 .. T-1);
 *     grad_x0 = A_0^T lam_1.
 *   A            device [batch,T,n,n]   required (A_0 is read only if grad_x0_out != NULL)
 *   B            device [batch,T,n,m]   required iff grad_u_out != NULL
 *   g            device [batch,T,n]     required; g[b,t-1] = g_t
 *   lambda_out   device [batch,T,n]     lambda_out[b,t-1] = lam_t
 *   grad_u_out   device [batch,T,m]     may be NULL
 *   grad_x0_out  device [batch,n]       may be NULL */
LTV_API int ltv_scan_adjoint(const float* A, const float* B, const float* g,
                     float* lambda_out, float* grad_u_out, float* grad_x0_out,
                     int batch, int T, int n, int m,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Rollout and adjoint scan of the same batch in ONE call (north_star (i) + (iii)): same arguments, results and
 * conventions as ltv_scan_rollout and ltv_scan_adjoint (the same kernels).  The two scans are independent - g is an
 * input - and each is a chain of T dependent steps per item.  A scan that alone occupies >= 80 % of the SMs with >= 128
 * rows per CTA already streams at 0.8-1.0 of the HBM peak; then each keeps its own configuration and the adjoint, enqueued on
 * the internal side stream, only takes the SMs the rollout leaves idle and fills in as its clusters finish (n = 300 x 64
 * items: 128 of 148 SMs each; 0.285 -> 0.270 ms against the two calls on one stream).  Otherwise (few
 * items, whose clusters cannot be wider than 16 CTAs; small systems, whose steps are too short to feed two CTAs per item)
 * the adjoint is enqueued on an internal side stream forked from and joined back into `cuda_stream` with events and the
 * two run CONCURRENTLY on half of the SMs each, with the widest clusters for which all clusters of both kernels are
 * resident at once (measured: n = 2400 x 4 items 0.631 -> 0.536 ms, n = 600 x 16 items 0.280 -> 0.215 ms, n = 180 x 64
 * items 0.262 -> 0.200 ms, n = 48 x 1 item 0.058 -> 0.030 ms).  Either way the call is stream-ordered like any other and
 * capturable in a CUDA graph.  The side stream and its two events are created once per host thread and device and kept. */
LTV_API int ltv_scan_rollout_adjoint(const float* A, const float* B, const float* c, const float* x0, const float* u,
                                     const float* g, float* x_out, float* lambda_out, float* grad_u_out,
                                     float* grad_x0_out, int batch, int T, int n, int m,
                                     void* workspace, size_t workspace_bytes, void* cuda_stream);

/* The whole hot path - north_star (i), (ii), (iii) - in one call on device buffers: every argument as in
 * ltv_scan_rollout, ltv_scan_system_response_tube and ltv_scan_adjoint (B, c, u, grad_u_out, grad_x0_out may be NULL as
 * there; flags: 0 or LTV_TUBE_ROW_2NORM; workspace: ltv_scan_workspace_bytes(LTV_OP_SYSTEM_RESPONSE_TUBE or
 * _RELAYOUT, ...)).  Two routes, same results up to the order of floating-point sums:
 *   small problems  n <= 64, T >= 2, phi_layout = LTV_PHI_COLUMN_PACKED and all of A_0 .. A_{T-1} fitting one SM's shared
 *                   memory (T n (n + 4) 4 bytes + ~40 KB <= 227 KB; BASELINE.json configs[0]: n = 48, T = 16): ONE
 *                   launch, one thread-block cluster per item - CTA r owns the block columns s = r, r + 15, .. of Phi as
 *                   chains Phi(t,s) = A_{t-1} Phi(t-1,s) that never leave its shared memory (fp32 FMA), the last CTA
 *                   runs rollout and adjoint side by side, one cluster barrier, tube rows summed over the columns
 *                   through distributed shared memory in fixed order (deterministic).  ltv_scan_all_is_fused tells.
 *   otherwise       ltv_scan_rollout_adjoint followed by ltv_scan_system_response_tube on `cuda_stream`. */
LTV_API int ltv_scan_all_is_fused(int batch, int T, int n, int m, int phi_layout);
LTV_API int ltv_scan_all(const float* A, const float* B, const float* c, const float* x0, const float* u, const float* w,
                         const float* g, float* x_out, float* phi_out, float* r_out, float* lambda_out,
                         float* grad_u_out, float* grad_x0_out, int batch, int T, int n, int m, int phi_layout,
                         unsigned flags, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Closed-loop observer propagation (eq.(14), :177), with gains that do not
 * depend on the injection step k (reading q15):
 *     Abar_j = A_j + Lt_j C_j,   PhiX(t,s) = Abar_{t-1} ... Abar_s,   PhiY(t,s) = PhiX(t,s) Lt_s,   0 <= s < t <= T-1
 * WARNING - which PhiY: by default PhiY follows eq.(14) AS PRINTED (the gain of step s beside PhiX(t,s)).  That is NOT
 * the Phihat^y that satisfies the second achievability identity of (12c) and that the assembly (15) needs (DESIGN.md
 * q20, q21, demonstrated by tests/test_oracle_pins_assembly.py): there the observation of step j-1 enters through
 * Phihat^y(k,j) = Phihat^x(k,j) Lt_{j-1}, j >= 1, and Phihat^y(k,0) = 0.  Pass LTV_OBSERVER_SHIFTED_GAIN in `flags` to
 * get that form (PhiY(t,s) = PhiX(t,s) Lt_{s-1}, zero blocks for s = 0); chaining ltv_scan_kalman_gains ->
 * ltv_scan_observer_response -> (15) without the flag gives a wrong Phi^xe.  ltv_scan_output_feedback_response uses
 * the shifted form internally.
 *   A        device [batch,T,n,n]     required; A_0 .. A_{T-2} are read
 *   Lt       device [batch,T,n,p]     required; Lt_j is the gain that multiplies C_j, Abar_j = A_j + Lt_j C_j: with
 *                                     the gains of (13) Lt_j = L_{j+1}^T, i.e. exactly the Lt_out array of
 *                                     ltv_scan_kalman_gains (DESIGN.md q17); 1 <= p <= 32
 *   C        device [batch,T,p,n]     required; observation Jacobians
 *   w        device [batch,T,n]       required; tube of PhiX exactly as in ltv_scan_system_response_tube
 *   phi_out  device [batch,P,n,nc]    nc = ltv_observer_row_floats(n,p) = n + 4*ceil(p/4); in every row, columns
 *                                     [0,n) hold PhiX(t,s), [n,n+p) PhiY(t,s), the rest zeros; block order `phi_layout`
 *   r_out    device [batch,T,n]       r_t = sum_{s<t} |PhiX(t,s)| w_s  (or the two-norm form with LTV_TUBE_ROW_2NORM)
 *   flags    0 or any of LTV_TUBE_ROW_2NORM, LTV_OBSERVER_SHIFTED_GAIN
 * The same time-parallel scan as above runs over the closed-loop matrices; PhiY rides along as p extra columns of
 * the right operand ([PhiX | PhiY](t,s) = PhiX(t,mid) [PhiX | PhiY](mid,s)), so it costs (n+p)/n of the products and
 * no second pass over Phi.  Level 0 forms Abar_s while A_s streams through, and PhiY(s+1,s) = Abar_s Lt_s.
 * Workspace: ltv_scan_workspace_bytes(LTV_OP_OBSERVER_RESPONSE, batch, T, n, p). */
LTV_API int ltv_observer_row_floats(int n, int p);
LTV_API int ltv_scan_observer_response(const float* A, const float* Lt, const float* C, const float* w,
                                       float* phi_out, float* r_out, int batch, int T, int n, int p, int phi_layout,
                                       unsigned flags, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Constraint-tightening margins (second form; eq.(12d)), process-disturbance term,
 * state part of the constraint rows, with the system response of (12c) and E_j = diag(w_j) (DESIGN.md q3b, q19):
 *     sigma_0 = 0;   sigma_k[i] = sum_{j=0}^{k-1} || c_{k,i}^T Phi(k,j) E_j ||_2,   k = 1 .. T-1,   c_{k,i}^T = Hc[b,k,i,:]
 *   A          device [batch,T,n,n]     required; A_0 .. A_{T-2} are read
 *   w          device [batch,T,n]       required; w_0 .. w_{T-2} are read
 *   Hc         device [batch,T,nc,n]    required; constraint rows per step (Hc[b,0] is not read), nc >= 1
 *   sigma_out  device [batch,T,nc]
 *   flags      must be 0
 * Phi is neither formed nor read: the rows Psi(k,j) = Hc_k Phi(k,j) obey Psi(k,j) = Psi(k,j+1) A_j, so one backward
 * sweep over j carries the stack of all rows with k > j through one batched GEMM per step ((T-1-j) nc rows; 3xTF32 on
 * tcgen05 for n >= 96, fp32 FMA below) and a row-norm kernel: 2 n^2 nc (T-1-j) flop per step, A read once.
 * Deterministic.  Workspace: ltv_scan_workspace_bytes(LTV_OP_CONSTRAINT_TIGHTENING, batch, T, n, nc). */
LTV_API int ltv_scan_constraint_tightening(const float* A, const float* w, const float* Hc, float* sigma_out,
                                           int batch, int T, int n, int nc, unsigned flags,
                                           void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Backward-Kalman recursion of the output-feedback stage (eq.(13)), with the
 * disturbance scalings taken diagonal, E_j = diag(e_j), F_j = diag(f_j) (readings q3b, q18):
 *     Pi_0 = Xi Xi^T (given);   for j = 0 .. T-1:
 *     L_{j+1}  = -(F_j F_j^T + C_j Pi_j C_j^T)^{-1} C_j Pi_j A_j^T
 *     Pi_{j+1} = E_j E_j^T + A_j Pi_j A_j^T + A_j Pi_j C_j^T L_{j+1}
 *   A        device [batch,T,n,n]      required
 *   C        device [batch,T,p,n]      required; observation Jacobians, 1 <= p <= 32
 *   e        device [batch,T,n]        required; process-disturbance scaling
 *   f        device [batch,T,p]        required; observation-disturbance scaling, every entry > 0 (F_j F_j^T must be
 *                                      positive definite; not checked)
 *   Pi0      device [batch,n,n]        required; symmetric positive semi-definite
 *   Lt_out   device [batch,T,n,p]      Lt_out[b,j] = L_{j+1}^T, the gain formed from (A_j, C_j, Pi_j): exactly the `Lt`
 *                                      array of ltv_scan_observer_response (A_j + Lt_j C_j closes the loop around A_j)
 *   Pi_out   device [batch,T+1,n,n]    Pi_out[b,j] = Pi_j (Pi_out[b,0] = Pi0)
 *   flags    0 or LTV_KALMAN_RECURSION: the recursion; LTV_KALMAN_SCAN: the paper's associative scan (not both)
 * Two device paths give the same Pi_j, L_j up to rounding on well-conditioned models:
 *   scan       PAPER.md:166-177: the associative elements (17) combined by rule (16) (re-derived, DESIGN.md q14) in a
 *              Sklansky prefix scan, ceil(log2(T+1)) launches with one CTA per combination (Gauss-Jordan with partial
 *              pivoting and the five products in shared memory), then the gains of all steps in one pass.  n <= 64
 *              (LTV_ERR_UNSUPPORTED_SHAPE beyond).  Logarithmic depth: the faster form for ONE small problem (n = 40, batch 1:
 *              417 vs 927 us at T = 32, 550 vs 3677 us at T = 128).  Runs only on request, because of its
 *              ACCURACY: the combination solves (I + D~ P~) X = [A~ | D~] in fp32, D~ = C^T (F F^T)^-1 C; its condition number
 *              grows like max(C^2 / f^2) ||Pi||.  Measured at n = 48 against the fp64 oracle: within 1e-4 for f >= 1e-3 with
 *              Pi0 ~ 1e-4 (the library's test models) and for f = 1e-2 with Pi0 = 0.01 I; gains off by 7.5e-3 at Pi0 = 0.01 I,
 *              f = 1e-3, by 2.5e-2 at Pi0 = I, f = 1e-2, NaN beyond - where the recursion, whose only inverse is the p x p
 *              innovation covariance, stays at 1e-5 .. 5e-4 (tests/test_gpu_kalman.py has the case).
 *   recursion  n <= 64: the whole recursion of an item in ONE CTA, one launch for the batch (Pi_j stays in shared memory, fp32 FMA;
 *              n = 40, batch 1: 363 us at T = 32 against 927 us for the batched form below).  Larger n: time-sequential, batch-parallel: per step one pass forms G = C Pi, the p x p innovation covariance (Cholesky), the
 * gain and the closed-loop matrix Abar_j = A_j + Lt_j C_j, then two batched 3xTF32 tcgen05 GEMMs form
 * Pi_{j+1} = A_j (Abar_j Pi_j)^T + E E^T (fp32 FMA for n < 96).  ~10x fewer flops than the scan: the faster form
 *              whenever one time step over the batch fills the machine.
 * Results are symmetric up to rounding.
 * Workspace: ltv_scan_workspace_bytes(LTV_OP_KALMAN_GAINS, batch, T, n, p). */
#define LTV_KALMAN_SCAN 1u
#define LTV_KALMAN_RECURSION 2u
LTV_API int ltv_scan_kalman_gains(const float* A, const float* C, const float* e, const float* f, const float* Pi0,
                                  float* Lt_out, float* Pi_out, int batch, int T, int n, int p, unsigned flags,
                                  void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Assembled output-feedback responses (first form; eq.(15)) and the reachable tube of
 * eq.(12e) (:147) with both of its terms, for a controller given by GAINS: state feedback u_k = Kfb_k xhat_k on the
 * estimate of the predictor-form observer xhat_{k+1} = A_k xhat_k + B_k u_k - Lt_k (y_k - C_k xhat_k), with Lt as
 * ltv_scan_kalman_gains returns it.  With Phibar = (I - Z(A + B Kfb))^-1, Phihat = (I - Z(A + Lt C))^-1 (DESIGN.md q20, q21):
 *     Phi^xw = Phibar^x + Phihat^x - Phibar^x M Phihat^x,      Phi^xe = Phihat^y - Phibar^x M Phihat^y,      M = I - Z A
 *     tau_0 = 0;  tau_k[i] = sum_{j<k} ||row_i(Phi^xw(k,j) diag(w_j))||_2 + sum_{1<=j<k} ||row_i(Phi^xe(k,j) diag(f_{j-1}))||_2
 *   A         device [batch,T,n,n]    required (A_0 .. A_{T-2} are read)
 *   B         device [batch,T,n,m]    required, m >= 1
 *   Kfb       device [batch,T,m,n]    required; state-feedback gains
 *   Lt        device [batch,T,n,p]    required; Lt_k = L_{k+1}^T, 1 <= p <= 32
 *   C         device [batch,T,p,n]    required
 *   w         device [batch,T,n]      required; process-disturbance scaling E_j = diag(w_j)
 *   f         device [batch,T,p]      required; observation-disturbance scaling; f_{j-1} scales the noise e~_j of the
 *                                     measurement of x_{j-1}
 *   phi_xw_out device [batch,P,n,n]   block (k,j), 0 <= j < k <= T-1, COLUMN_PACKED order (ltv_phi_block_index)
 *   phi_xe_out device [batch,P,n,p]   same block order; blocks with j = 0 are zero; may be NULL
 *   tau_out   device [batch,T,n]
 *   flags     must be 0
 * Method: the closed loop in (x, x - xhat) is the LTV system A_aug = [[A + B Kfb, -B Kfb], [0, A + Lt C]], and with
 * G = Phi_aug(k,j): Phi^xw = G11 + G12, Phi^xe = G12 Lt_{j-1}.  G is block upper triangular (G11 = Phibar^x,
 * G22 = Phihat^x).  For n < 96 the library runs the plain scan on the 2n x 2n Jacobians and one extraction pass.  For
 * n >= 96 one of two routes (LTV_OPT_OUTPUT_FEEDBACK_ROUTE; default: chosen by size):
 *   cross scan   G12(t,s) = G11(t,mid) G12(mid,s) + G12(t,mid) G22(mid,s): two n-state time-parallel scans and one cross scan
 *                whose combine accumulates both products in one tcgen05 K loop (4 n^3 products per block, log depth), then one
 *                pass that forms Phi^xw (in place over Phibar^x), Phi^xe and the tube;
 *   columns      (m, p <= 8) one scan for Phibar^x, then the backward recursion over the columns of
 *                ltv_scan_output_feedback_assemble carried on the difference D = G12 = Phi^xw - Phibar^x,
 *                    D(k,j) = D(k,j+1) Abar_j - [Phibar^x(k,j+1) B_j] Kfb_j,   D(k,k) = 0,   Abar_j = A_j + Lt_j C_j,
 *                    Phi^xw = Phibar^x + D,   Phi^xe(k,j) = D(k,j) Lt_{j-1}
 *                (2 n^3 products per block, T-1 sequential steps of one batched GEMM + one fused row kernel; no difference of
 *                nearly equal operators is formed, so small gains lose no digits; D lives in two column buffers).  C2 (batch
 *                64): 26 ms against 38 ms for the cross scan, workspace 14.5 against 24.5 GB; single large items 1.65x;
 *                small problems (a GEMM step below ~4 waves of tiles) stay on the log-depth route.
 * Both are deterministic.  The input-side operators Phi^uw, Phi^ue of (15) come from ltv_scan_output_feedback_constraints
 * (below).  n <= 4096.  Workspace: ltv_scan_workspace_bytes(LTV_OP_OUTPUT_FEEDBACK, batch, T, n, max(m, p)) - the last
 * argument may be 0 ("not known yet": room for either route); it must be asked AFTER LTV_OPT_OUTPUT_FEEDBACK_ROUTE is set. */
LTV_API int ltv_scan_output_feedback_response(const float* A, const float* B, const float* Kfb, const float* Lt,
                                              const float* C, const float* w, const float* f, float* phi_xw_out,
                                              float* phi_xe_out, float* tau_out, int batch, int T, int n, int m, int p,
                                              unsigned flags, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Input-side output-feedback responses of eq.(15) and the constraint-tightening margins of eq.(12d) with BOTH terms and
 * constraint rows on the stacked pair [z_k; v_k], for the same
 * gain-defined controller as ltv_scan_output_feedback_response (u_k = Kfb_k xhat_k, predictor-form observer):
 *     Phi^uw(k,j) = Kfb_k (Phi^xw(k,j) - Phihat^x(k,j)),    Phi^ue(k,j) = Kfb_k (Phi^xe(k,j) - Phihat^x(k,j) Lt_{j-1}),
 *     sigma_0 = 0;  sigma_k[i] = sum_{j<k} || c_{k,i}^T [Phi^xw; Phi^uw](k,j) diag(w_j) ||_2
 *                              + sum_{1<=j<k} || c_{k,i}^T [Phi^xe; Phi^ue](k,j) diag(f_{j-1}) ||_2,   c_{k,i}^T = [Hx[b,k,i,:], Hu[b,k,i,:]]
 * (0 <= j < k <= T-1; the blocks equal Phibar^u (I - M Phihat^x) and -Phibar^u M Phihat^y of (15): pinned in the oracle tests).
 *   A, B, Kfb, Lt, C, w, f   as in ltv_scan_output_feedback_response (all required, m >= 1, 1 <= p <= 32)
 *   Hx         device [batch,T,nc,n]   state part of the constraint rows (Hx[b,0] is not read); required iff nc > 0
 *   Hu         device [batch,T,nc,m]   input part of the constraint rows; required iff nc > 0
 *   phi_uw_out device [batch,P,m,n]    block (k,j) in COLUMN_PACKED order (ltv_phi_block_index); may be NULL
 *   phi_ue_out device [batch,P,m,p]    same order; blocks with j = 0 are zero; may be NULL
 *   sigma_out  device [batch,T,nc]     required iff nc > 0
 *   flags      must be 0
 * Method: a row s^T on xi = (x, x - xhat) propagates backwards as psi(k,j) = psi(k,j+1) A_aug,j with the augmented closed-
 * loop Jacobian A_aug = [[A + B Kfb, -B Kfb], [0, A + Lt C]]; constraint row i of step k starts from
 * [Hx + Hu Kfb_k | -Hu Kfb_k], row a of the input response from [Kfb_k[a] | -Kfb_k[a]]; then c^T Phi^w(k,j) = psi1 + psi2 and
 * c^T Phi^e(k,j) = psi2 Lt_{j-1}.  One backward sweep over j carries the stack of the rows of all k > j through one batched
 * GEMM per step ((T-1-j)(nc + m) rows of 2n floats; tcgen05 3xTF32 for 2n >= 96) - no Phi is formed or read.  Deterministic.
 * 2n <= 8192, batch <= 65535.  Workspace: ltv_scan_output_feedback_constraints_workspace_bytes(batch, T, n, m, nc). */
LTV_API size_t ltv_scan_output_feedback_constraints_workspace_bytes(int batch, int T, int n, int m, int nc);
LTV_API int ltv_scan_output_feedback_constraints(const float* A, const float* B, const float* Kfb, const float* Lt,
                                                 const float* C, const float* w, const float* f, const float* Hx,
                                                 const float* Hu, float* phi_uw_out, float* phi_ue_out, float* sigma_out,
                                                 int batch, int T, int n, int m, int p, int nc, unsigned flags,
                                                 void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Eq.(15) for a GENERAL state-feedback response: Phibar = (Phibar^x, Phibar^u) is given
 * as block operators - e.g. the solution of the state-feedback SLS problem - instead of being generated from gains; the
 * observer response Phihat is that of the gains of (13)/(14) as in ltv_scan_output_feedback_response (Phihat^x(k,j) =
 * Abar_{k-1} .. Abar_j, Abar_j = A_j + Lt_j C_j, Phihat^y(k,j) = Phihat^x(k,j) Lt_{j-1}; DESIGN.md q20, q21).  With M = I - Z A:
 *     Phi^xw = Phibar^x + Phihat^x - Phibar^x M Phihat^x,    Phi^uw = Phibar^u (I - M Phihat^x),
 *     Phi^xe = Phihat^y - Phibar^x M Phihat^y,               Phi^ue = -Phibar^u M Phihat^y,
 *     tau_0 = 0;  tau_k[i] = sum_{j<k} ||row_i(Phi^xw(k,j) diag(w_j))||_2 + sum_{1<=j<k} ||row_i(Phi^xe(k,j) diag(f_{j-1}))||_2
 *   A, Lt, C, w, f  as in ltv_scan_output_feedback_response (all required; 1 <= p <= 32)
 *   phibar_x   device [batch,P,n,n]     blocks (k,j), 0 <= j < k <= T-1, COLUMN_PACKED (ltv_phi_block_index); the diagonal
 *                                       blocks are NOT passed: Phibar^x(k,k) = I for every achievable response
 *   phibar_u   device [batch,P+T,m,n]   blocks (k,j), 0 <= j <= k <= T-1, INCLUDING the diagonal: column j holds its T - j
 *                                       blocks k = j .. T-1 one after the other, block index j T - j(j-1)/2 + (k - j);
 *                                       required iff phi_uw_out != NULL
 *   phi_xw_out device [batch,P,n,n]     COLUMN_PACKED, strictly-lower blocks (Phi^xw(k,k) = I)
 *   phi_xe_out device [batch,P,n,p]     same order; blocks with j = 0 are zero; may be NULL
 *   phi_uw_out device [batch,P,m,n]     same order (Phi^uw(k,k) = 0); may be NULL
 *   phi_ue_out device [batch,P,m,p]     same order, j = 0 zero (the diagonal blocks Phi^ue(k,k) = -Phibar^u(k,k) Lt_{k-1} are
 *                                       not part of the output); may be NULL; needs phi_uw_out
 *   tau_out    device [batch,T,n]       may be NULL
 *   flags      must be 0
 * Method: no block-operator product is formed.  M is block bidiagonal and Phihat^x(i,j) = Phihat^x(i,j+1) Abar_j, so
 *     Phi^xw(k,j) = Phi^xw(k,j+1) Abar_j - [Phibar^x(k,j+1) Lt_j] C_j  (Phi^xw(k,k) = I),   same for Phi^uw with Phibar^u (start 0),
 *     Phi^xe(k,j) = (Phi^xw - Phibar^x)(k,j) Lt_{j-1},   Phi^ue(k,j) = (Phi^uw - Phibar^u)(k,j) Lt_{j-1}
 * (pinned against the oracle's dense evaluation of (15)): one n^3 product per block - as many as the Phi scan - in T-1
 * backward steps, each one batched GEMM of the stacked column j+1 with Abar_j (tcgen05 3xTF32 for n >= 96) plus a fused row
 * kernel (rank-p correction, Phi^xe / Phi^ue, tube).  Deterministic.  batch <= 65535.
 * Workspace: ltv_scan_output_feedback_assemble_workspace_bytes(batch, T, n, m, p). */
LTV_API size_t ltv_scan_output_feedback_assemble_workspace_bytes(int batch, int T, int n, int m, int p);
LTV_API int ltv_scan_output_feedback_assemble(const float* A, const float* Lt, const float* C, const float* w,
                                              const float* f, const float* phibar_x, const float* phibar_u,
                                              float* phi_xw_out, float* phi_xe_out, float* phi_uw_out, float* phi_ue_out,
                                              float* tau_out, int batch, int T, int n, int m, int p, unsigned flags,
                                              void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Constraint-tightening margins of eq.(12d), both terms, constraint rows on [z_k; v_k], evaluated on
 * ASSEMBLED output-feedback operators - those of ltv_scan_output_feedback_assemble (general Phibar) or of the gain-defined calls:
 *     sigma_0 = 0;  sigma_k[i] = sum_{j<k}    || (Hx[b,k,i,:] Phi^xw(k,j) + Hu[b,k,i,:] Phi^uw(k,j)) diag(w_j) ||_2
 *                              + sum_{1<=j<k} || (Hx[b,k,i,:] Phi^xe(k,j) + Hu[b,k,i,:] Phi^ue(k,j)) diag(f_{j-1}) ||_2
 *   phi_xw   device [batch,P,n,n]   COLUMN_PACKED strictly-lower blocks; required
 *   phi_uw   device [batch,P,m,n]   may be NULL together with Hu (constraints on the state only)
 *   phi_xe   device [batch,P,n,p]   may be NULL (no observation term; f is then not read)
 *   phi_ue   device [batch,P,m,p]   may be NULL; needs phi_uw
 *   Hx       device [batch,T,nc,n]  required (Hx[b,0] is not read);   Hu  device [batch,T,nc,m]
 *   w        device [batch,T,n];    f  device [batch,T,p]
 *   sigma_out device [batch,T,nc]
 *   flags    must be 0
 * One CTA per (item, step k) walks j in order and keeps the nc sums: deterministic, no workspace, every operator block is
 * read once (HBM-bound).  n <= 512, p <= 32, batch <= 65535 (LTV_ERR_UNSUPPORTED_SHAPE beyond); any nc (8 rows per pass
 * over the operators). */
LTV_API int ltv_scan_operator_constraint_margins(const float* phi_xw, const float* phi_uw, const float* phi_xe,
                                                 const float* phi_ue, const float* Hx, const float* Hu, const float* w,
                                                 const float* f, float* sigma_out, int batch, int T, int n, int m, int p,
                                                 int nc, unsigned flags, void* cuda_stream);

/* One pass of the whole hot path from HOST buffers: copies A, B, c, x0, u, w, g host->device into
 * `workspace` (device, >= ltv_scan_workspace_bytes(LTV_OP_PIPELINE_HOST, ...)), runs the path (ltv_scan_rollout_adjoint, then
 * ltv_scan_system_response_tube)
 * on `cuda_stream`, copies x, r, lambda, grad_u, grad_x0 device->host and synchronises the stream before
 * returning.  Phi (11 GB at the benchmark sizes) stays in the workspace on the device, where its consumer
 * (the tube / constraint tightening) lives, unless phi_host != NULL, in which case it is copied back too.
 * All *_host pointers are host memory; B, c, u may be NULL as in ltv_scan_rollout; grad_x0_host and
 * phi_host may be NULL.  *phi_device_out (if not NULL) receives the device address of Phi inside workspace.
 * w_host == NULL skips the system-response / tube stage (rollout + adjoint only, BASELINE.json configs[4]): r_host
 * is then not written and may be NULL, and the workspace need is LTV_OP_PIPELINE_HOST_NO_PHI.
 * The batch is processed in up to sixteen chunks (LTV_OPT_PIPELINE_CHUNKS; multiples of 4 items): an internal non-blocking copy stream,
 * created and destroyed inside the call, uploads chunk i+1 while chunk i is computed on `cuda_stream` (items
 * are independent, so this changes no result); host buffers should be pinned for the copies to overlap. */
LTV_API int ltv_scan_pipeline_host(const float* A_host, const float* B_host, const float* c_host,
                           const float* x0_host, const float* u_host, const float* w_host,
                           const float* g_host,
                           float* x_host, float* phi_host, float* r_host, float* lambda_host,
                           float* grad_u_host, float* grad_x0_host,
                           int batch, int T, int n, int m,
                           void* workspace, size_t workspace_bytes, void* cuda_stream,
                           float** phi_device_out);

/* Process-wide options: plain ints, thread-safe, each with a sound default; none changes a result beyond the order of
 * floating-point sums.  The library reads NO environment variables (developer builds made with -DLTV_TUNING aside).
 *   LTV_OPT_VECTOR_CLUSTER   CTAs per batch item (thread-block cluster size) of the rollout and adjoint kernels:
 *                            0 (default) = chosen by an occupancy / bandwidth model, 1 .. 16 = forced (falls back to 1
 *                            if that cluster cannot be placed).  Used by the tests to cover every cluster size.
 *   LTV_OPT_PIPELINE_CHUNKS  number of batch chunks ltv_scan_pipeline_host overlaps upload and compute over:
 *                            1 .. 16, default 16 (1 = no overlap; C2: 16.0 ms with 4, 15.3 ms with 8, 15.1 ms with 16 - the upload at PCIe rates is the long leg, more chunks shorten the exposed last compute).
 *   LTV_OPT_OUTPUT_FEEDBACK_ROUTE  how ltv_scan_output_feedback_response evaluates (15) for n >= 96: 1 = cross scan (log depth,
 *                            4 n^3 products per block), 2 = column recursion (one scan for Phibar^x + the backward recursion
 *                            of ltv_scan_output_feedback_assemble: 2 n^3 products per block, T-1 sequential steps), 0
 *                            (default) = by size (2 once a step's GEMM fills the GPU).  Read by the call AND by
 *                            ltv_scan_workspace_bytes(LTV_OP_OUTPUT_FEEDBACK, ..): size the workspace after setting it.
 * ltv_set_option returns LTV_ERR_BAD_DIM for an unknown option or a value out of range; ltv_get_option returns -1 for
 * an unknown option. */
enum { LTV_OPT_VECTOR_CLUSTER = 0, LTV_OPT_PIPELINE_CHUNKS = 1, LTV_OPT_OUTPUT_FEEDBACK_ROUTE = 2, LTV_OPT_COUNT = 3 };
LTV_API int ltv_set_option(int option, int value);
LTV_API int ltv_get_option(int option);

/* Human-readable name of a status code (static storage). */
LTV_API const char* ltv_status_string(int status);
/* cudaError_t (as int) of the last failing CUDA call made by this library in this thread, 0 if none. */
LTV_API int ltv_last_cuda_error(void);
/* Library version, major*10000 + minor*100 + patch. */
LTV_API int ltv_version(void);
/* Number of kernel launches the library has enqueued since load (all threads); used by bench.py to report
 * `gpu_launches`. */
LTV_API unsigned long long ltv_launch_count(void);

/* Optional per-kernel timing for benchmarks.  While enabled, every kernel the library enqueues is bracketed by
 * CUDA events recorded on the launch stream (no synchronisation, no change to the kernels).
 * ltv_profile_collect waits for the recorded events, adds their elapsed times (milliseconds) and launch counts
 * per kernel class into the two caller arrays of LTV_PROFILE_CLASSES entries (host memory), and clears the
 * record.  Classes: 0 rollout, 1 adjoint, 2 Phi level 0 (copy + tube), 3 Phi combine (tcgen05 3xTF32),
 * 4 Phi combine (fp32 FMA, small n), 5 tube finalise, 6 batched GEMMs of the Kalman recursion and the constraint sweep
 * (tcgen05 3xTF32, or fp32 FMA for small n), 7 their fp32 support kernels (gain, closed loop, row norms), 8 the block
 * re-ordering copy of the non-native Phi layouts, 9-11 see ltv_profile_class_name. */
#define LTV_PROFILE_CLASSES 12
LTV_API int ltv_profile_enable(int on);
/* Short name of a profile class (static storage), NULL if cls is out of range. */
LTV_API const char* ltv_profile_class_name(int cls);
LTV_API int ltv_profile_collect(double* ms_by_class, unsigned long long* launches_by_class);

#ifdef __cplusplus
}
#endif
#endif /* LTV_SCAN_H_ */
