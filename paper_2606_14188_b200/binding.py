"""ctypes binding of libltvscan.so (include/ltv_scan.h).  Argument marshalling ONLY: every step of the path
runs in the library's CUDA kernels.  torch is used for device memory and the current stream.  There is no
CPU fallback: if the shared library is missing this module raises at import."""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libltvscan.so")

LTV_OK = 0
STATUS_NAMES = {
    0: "LTV_OK", 1: "LTV_ERR_NULL_PTR", 2: "LTV_ERR_BAD_DIM", 3: "LTV_ERR_UNSUPPORTED_SHAPE",
    4: "LTV_ERR_ALIGNMENT", 5: "LTV_ERR_WORKSPACE_TOO_SMALL", 6: "LTV_ERR_ARCH", 7: "LTV_ERR_CUDA",
    8: "LTV_ERR_STATIC_SCRATCH_LIMIT",
}
LTV_ERR_STATIC_SCRATCH_LIMIT = 8
LTV_OP_ROLLOUT, LTV_OP_SYSTEM_RESPONSE_TUBE, LTV_OP_ADJOINT, LTV_OP_PIPELINE_HOST = 0, 1, 2, 3
LTV_OP_PIPELINE_HOST_NO_PHI = 4
LTV_OP_OBSERVER_RESPONSE = 5
LTV_OP_KALMAN_GAINS = 6
LTV_OP_CONSTRAINT_TIGHTENING = 7
LTV_OP_OUTPUT_FEEDBACK = 8
LTV_TUBE_ROW_2NORM = 1
LTV_OBSERVER_SHIFTED_GAIN = 2
LTV_KALMAN_SCAN, LTV_KALMAN_RECURSION = 1, 2
LTV_PHI_ROW_PACKED, LTV_PHI_SQUARE_GRID, LTV_PHI_COLUMN_PACKED = 0, 1, 2
LTV_OP_SYSTEM_RESPONSE_TUBE_RELAYOUT = 9
LTV_OPT_VECTOR_CLUSTER, LTV_OPT_PIPELINE_CHUNKS, LTV_OPT_OUTPUT_FEEDBACK_ROUTE = 0, 1, 2

EXPORTS = (
    "ltv_phi_block_index", "ltv_phi_block_index_layout", "ltv_scan_workspace_bytes", "ltv_scan_rollout", "ltv_scan_system_response_tube",
    "ltv_scan_adjoint", "ltv_scan_pipeline_host", "ltv_status_string", "ltv_last_cuda_error", "ltv_version",
    "ltv_launch_count", "ltv_profile_enable", "ltv_profile_collect", "ltv_scan_observer_response",
    "ltv_observer_row_floats", "ltv_scan_kalman_gains",
    "ltv_scan_constraint_tightening", "ltv_scan_output_feedback_response", "ltv_set_option", "ltv_get_option",
    "ltv_profile_class_name", "ltv_scan_rollout_adjoint", "ltv_scan_all", "ltv_scan_all_is_fused", "ltv_scan_output_feedback_constraints", "ltv_scan_output_feedback_constraints_workspace_bytes",
    "ltv_static_scratch_bytes", "ltv_scan_system_response_tube_static",
    "ltv_scan_output_feedback_assemble", "ltv_scan_output_feedback_assemble_workspace_bytes",
    "ltv_scan_operator_constraint_margins",
    "ltv_phi_row_shard_blocks", "ltv_phi_row_shard_block_index", "ltv_scan_system_response_tube_rows",
)


class LtvError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {STATUS_NAMES.get(status, status)} (cuda error {lib.ltv_last_cuda_error()})")


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2606_14188_b200.build` "
            "(nvcc, sm_100a).  There is no CPU fallback.")
    L = ctypes.CDLL(LIB_PATH)
    vp, sz, i, fp = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int, ctypes.c_void_p
    L.ltv_phi_block_index.restype = ctypes.c_longlong
    L.ltv_phi_block_index.argtypes = [i, i, i]
    L.ltv_phi_block_index_layout.restype = ctypes.c_longlong
    L.ltv_phi_block_index_layout.argtypes = [i, i, i, i]
    L.ltv_scan_workspace_bytes.restype = sz
    L.ltv_scan_workspace_bytes.argtypes = [i, i, i, i, i]
    L.ltv_scan_rollout.restype = i
    L.ltv_scan_rollout.argtypes = [fp] * 6 + [i] * 4 + [vp, sz, vp]
    L.ltv_scan_system_response_tube.restype = i
    L.ltv_scan_system_response_tube.argtypes = [fp] * 4 + [i] * 4 + [ctypes.c_uint, vp, sz, vp]
    L.ltv_scan_output_feedback_assemble.restype = i
    L.ltv_scan_output_feedback_assemble.argtypes = [fp] * 12 + [i] * 5 + [ctypes.c_uint, vp, sz, vp]
    L.ltv_scan_output_feedback_assemble_workspace_bytes.restype = sz
    L.ltv_scan_output_feedback_assemble_workspace_bytes.argtypes = [i] * 5
    L.ltv_scan_operator_constraint_margins.restype = i
    L.ltv_scan_operator_constraint_margins.argtypes = [fp] * 9 + [i] * 6 + [ctypes.c_uint, vp]
    L.ltv_phi_row_shard_blocks.restype = ctypes.c_longlong
    L.ltv_phi_row_shard_blocks.argtypes = [i, i, i]
    L.ltv_phi_row_shard_block_index.restype = ctypes.c_longlong
    L.ltv_phi_row_shard_block_index.argtypes = [i] * 5
    L.ltv_scan_system_response_tube_rows.restype = i
    L.ltv_scan_system_response_tube_rows.argtypes = [fp] * 4 + [i] * 5 + [ctypes.c_uint, vp]
    L.ltv_static_scratch_bytes.restype = sz
    L.ltv_static_scratch_bytes.argtypes = []
    L.ltv_scan_system_response_tube_static.restype = i
    L.ltv_scan_system_response_tube_static.argtypes = [fp] * 4 + [i] * 3 + [ctypes.c_uint, vp]
    L.ltv_scan_adjoint.restype = i
    L.ltv_scan_adjoint.argtypes = [fp] * 6 + [i] * 4 + [vp, sz, vp]
    L.ltv_scan_rollout_adjoint.restype = i
    L.ltv_scan_rollout_adjoint.argtypes = [fp] * 10 + [i] * 4 + [vp, sz, vp]
    L.ltv_scan_all.restype = i
    L.ltv_scan_all.argtypes = [fp] * 13 + [i] * 5 + [ctypes.c_uint, vp, sz, vp]
    L.ltv_scan_all_is_fused.restype = i
    L.ltv_scan_all_is_fused.argtypes = [i] * 5
    L.ltv_scan_pipeline_host.restype = i
    L.ltv_scan_pipeline_host.argtypes = [fp] * 13 + [i] * 4 + [vp, sz, vp, ctypes.POINTER(ctypes.c_void_p)]
    L.ltv_scan_observer_response.restype = i
    L.ltv_scan_observer_response.argtypes = [fp] * 6 + [i] * 5 + [ctypes.c_uint, vp, sz, vp]
    L.ltv_scan_kalman_gains.restype = i
    L.ltv_scan_kalman_gains.argtypes = [fp] * 7 + [i] * 4 + [ctypes.c_uint, vp, sz, vp]
    L.ltv_scan_constraint_tightening.restype = i
    L.ltv_scan_constraint_tightening.argtypes = [fp] * 4 + [i] * 4 + [ctypes.c_uint, vp, sz, vp]
    L.ltv_scan_output_feedback_response.restype = i
    L.ltv_scan_output_feedback_response.argtypes = [fp] * 10 + [i] * 5 + [ctypes.c_uint, vp, sz, vp]
    L.ltv_scan_output_feedback_constraints.restype = i
    L.ltv_scan_output_feedback_constraints.argtypes = [fp] * 12 + [i] * 6 + [ctypes.c_uint, vp, sz, vp]
    L.ltv_scan_output_feedback_constraints_workspace_bytes.restype = sz
    L.ltv_scan_output_feedback_constraints_workspace_bytes.argtypes = [i] * 5
    L.ltv_observer_row_floats.restype = i
    L.ltv_observer_row_floats.argtypes = [i, i]
    L.ltv_set_option.restype = i
    L.ltv_set_option.argtypes = [i, i]
    L.ltv_get_option.restype = i
    L.ltv_get_option.argtypes = [i]
    L.ltv_status_string.restype = ctypes.c_char_p
    L.ltv_status_string.argtypes = [i]
    L.ltv_last_cuda_error.restype = i
    L.ltv_version.restype = i
    L.ltv_launch_count.restype = ctypes.c_ulonglong
    L.ltv_profile_enable.restype = i
    L.ltv_profile_enable.argtypes = [i]
    L.ltv_profile_collect.restype = i
    L.ltv_profile_collect.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_ulonglong)]
    return L


lib = _load()


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _dev(t, name, shape):
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise ValueError(f"{name}: need a contiguous fp32 CUDA tensor")
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: shape {tuple(t.shape)} != {tuple(shape)}")
    return t


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def ltv_phi_block_index(T: int, t: int, s: int) -> int:
    return int(lib.ltv_phi_block_index(T, t, s))


def ltv_scan_workspace_bytes(op: int, batch: int, T: int, n: int, m: int) -> int:
    return int(lib.ltv_scan_workspace_bytes(op, batch, T, n, m))


def ltv_set_option(option: int, value: int) -> None:
    st = lib.ltv_set_option(option, value)
    if st != LTV_OK:
        raise LtvError(st, "ltv_set_option")


def ltv_get_option(option: int) -> int:
    return int(lib.ltv_get_option(option))


def ltv_launch_count() -> int:
    return int(lib.ltv_launch_count())


lib.ltv_profile_class_name.restype = ctypes.c_char_p
lib.ltv_profile_class_name.argtypes = [ctypes.c_int]
PROFILE_CLASSES = tuple(lib.ltv_profile_class_name(i).decode() for i in range(12))


def ltv_profile_enable(on: bool) -> None:
    lib.ltv_profile_enable(1 if on else 0)


def ltv_profile_collect() -> dict:
    """{class: (total ms, launches)} of the kernels enqueued since the last collect / enable."""
    ms = (ctypes.c_double * len(PROFILE_CLASSES))()
    cnt = (ctypes.c_ulonglong * len(PROFILE_CLASSES))()
    st = lib.ltv_profile_collect(ms, cnt)
    if st != LTV_OK:
        raise LtvError(st, "ltv_profile_collect")
    return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(PROFILE_CLASSES)}


def ltv_scan_rollout(A, B, c, x0, u, x_out=None):
    """x_out[b,t] = x_{t+1};  A[batch,T,n,n], B[batch,T,n,m]|None, c[batch,T,n]|None, x0[batch,n], u[batch,T,m]|None."""
    batch, T, n, _ = A.shape
    m = 0 if B is None else B.shape[-1]
    _dev(A, "A", (batch, T, n, n)); _dev(B, "B", (batch, T, n, m)); _dev(c, "c", (batch, T, n))
    _dev(x0, "x0", (batch, n)); _dev(u, "u", (batch, T, m))
    if x_out is None:
        x_out = torch.empty((batch, T, n), device=A.device, dtype=torch.float32)
    _dev(x_out, "x_out", (batch, T, n))
    st = lib.ltv_scan_rollout(_ptr(A), _ptr(B), _ptr(c), _ptr(x0), _ptr(u), _ptr(x_out), batch, T, n, m,
                              None, 0, _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_rollout")
    return x_out


def ltv_phi_block_index_layout(T: int, t: int, s: int, layout: int) -> int:
    return int(lib.ltv_phi_block_index_layout(T, t, s, layout))


def ltv_scan_system_response_tube(A, w, phi_out=None, r_out=None, workspace=None, two_norm=False,
                                  layout=LTV_PHI_COLUMN_PACKED):
    """Returns (phi, r[batch,T,n]); phi[batch,P,n,n] in COLUMN_PACKED (default, the fast path) or ROW_PACKED order, or
    phi[batch,T,T,n,n] for LTV_PHI_SQUARE_GRID (cells with s >= t untouched).  `workspace`: optional uint8 CUDA tensor.
    two_norm=True: the row-wise two-norm tube of eq.(12e) with E_s = diag(w_s) instead of the box tube."""
    batch, T, n, _ = A.shape
    P = T * (T - 1) // 2
    shape = (batch, T, T, n, n) if layout == LTV_PHI_SQUARE_GRID else (batch, P, n, n)
    _dev(A, "A", (batch, T, n, n)); _dev(w, "w", (batch, T, n))
    if phi_out is None:
        phi_out = torch.empty(shape, device=A.device, dtype=torch.float32)
    if r_out is None:
        r_out = torch.empty((batch, T, n), device=A.device, dtype=torch.float32)
    _dev(phi_out, "phi_out", shape); _dev(r_out, "r_out", (batch, T, n))
    need = ltv_scan_workspace_bytes(LTV_OP_SYSTEM_RESPONSE_TUBE if layout == LTV_PHI_COLUMN_PACKED
                                    else LTV_OP_SYSTEM_RESPONSE_TUBE_RELAYOUT, batch, T, n, 0)
    if workspace is None:
        workspace = torch.empty(max(need, 16), device=A.device, dtype=torch.uint8)
    st = lib.ltv_scan_system_response_tube(_ptr(A), _ptr(w), _ptr(phi_out), _ptr(r_out), batch, T, n,
                                           layout, LTV_TUBE_ROW_2NORM if two_norm else 0,
                                           _ptr(workspace), workspace.numel(), _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_system_response_tube")
    return phi_out, r_out


def ltv_scan_output_feedback_assemble(A, Lt, C, w, f, phibar_x, phibar_u=None, want_xe=True, want_ue=True, want_tau=True,
                                      workspace=None):
    """Eq.(15) for a general Phibar: phibar_x[batch,P,n,n] (COLUMN_PACKED strictly-lower blocks, diagonal = I implied),
    phibar_u[batch,P+T,m,n] (blocks j <= k incl. the diagonal, column by column) or None.  Returns a dict with phi_xw
    [batch,P,n,n], phi_xe [batch,P,n,p] | None, phi_uw [batch,P,m,n] | None, phi_ue [batch,P,m,p] | None, tau [batch,T,n] | None."""
    batch, T, n, _ = A.shape
    p = C.shape[2]
    P = T * (T - 1) // 2
    m = 0 if phibar_u is None else phibar_u.shape[2]
    _dev(A, "A", (batch, T, n, n)); _dev(Lt, "Lt", (batch, T, n, p)); _dev(C, "C", (batch, T, p, n))
    _dev(w, "w", (batch, T, n)); _dev(f, "f", (batch, T, p)); _dev(phibar_x, "phibar_x", (batch, P, n, n))
    _dev(phibar_u, "phibar_u", (batch, P + T, m, n))
    mk = lambda *shape: torch.empty(shape, device=A.device, dtype=torch.float32)
    out = dict(phi_xw=mk(batch, P, n, n), phi_xe=mk(batch, P, n, p) if want_xe else None,
               phi_uw=mk(batch, P, m, n) if phibar_u is not None else None,
               phi_ue=mk(batch, P, m, p) if (phibar_u is not None and want_ue) else None,
               tau=mk(batch, T, n) if want_tau else None)
    need = int(lib.ltv_scan_output_feedback_assemble_workspace_bytes(batch, T, n, m, p))
    if workspace is None:
        workspace = torch.empty(max(need, 16), device=A.device, dtype=torch.uint8)
    st = lib.ltv_scan_output_feedback_assemble(_ptr(A), _ptr(Lt), _ptr(C), _ptr(w), _ptr(f), _ptr(phibar_x), _ptr(phibar_u),
                                               _ptr(out["phi_xw"]), _ptr(out["phi_xe"]), _ptr(out["phi_uw"]),
                                               _ptr(out["phi_ue"]), _ptr(out["tau"]), batch, T, n, m, p, 0,
                                               _ptr(workspace), workspace.numel(), _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_output_feedback_assemble")
    return out


def ltv_scan_operator_constraint_margins(phi_xw, Hx, w, phi_uw=None, Hu=None, phi_xe=None, phi_ue=None, f=None):
    """sigma[batch,T,nc] of eq.(12d), both terms, from assembled operators (COLUMN_PACKED strictly-lower blocks)."""
    batch, P, n, _ = phi_xw.shape
    T = w.shape[1]
    nc = Hx.shape[2]
    m = 0 if phi_uw is None else phi_uw.shape[2]
    p = 0 if phi_xe is None else phi_xe.shape[3]
    _dev(phi_xw, "phi_xw", (batch, P, n, n)); _dev(Hx, "Hx", (batch, T, nc, n)); _dev(w, "w", (batch, T, n))
    _dev(phi_uw, "phi_uw", (batch, P, m, n)); _dev(Hu, "Hu", (batch, T, nc, m))
    _dev(phi_xe, "phi_xe", (batch, P, n, p)); _dev(phi_ue, "phi_ue", (batch, P, m, p)); _dev(f, "f", (batch, T, p))
    sigma = torch.empty((batch, T, nc), device=phi_xw.device, dtype=torch.float32)
    st = lib.ltv_scan_operator_constraint_margins(_ptr(phi_xw), _ptr(phi_uw), _ptr(phi_xe), _ptr(phi_ue), _ptr(Hx), _ptr(Hu),
                                                  _ptr(w), _ptr(f), _ptr(sigma), batch, T, n, m, p, nc, 0, _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_operator_constraint_margins")
    return sigma


def ltv_phi_row_shard_blocks(T, k_lo, k_hi):
    return int(lib.ltv_phi_row_shard_blocks(T, k_lo, k_hi))


def ltv_phi_row_shard_block_index(T, k_lo, k_hi, k, j):
    return int(lib.ltv_phi_row_shard_block_index(T, k_lo, k_hi, k, j))


def ltv_scan_system_response_tube_rows(A, w, k_lo, k_hi, phi_rows_out=None, r_out=None, two_norm=False):
    """Block rows k_lo <= k < k_hi of the system response (one shard of items split over GPUs): returns (phi_rows
    [batch,Ps,n,n] in the shard's column-packed order, r[batch,T,n] with the shard's rows filled, zeros elsewhere if r_out
    is not given)."""
    batch, T, n, _ = A.shape
    Ps = ltv_phi_row_shard_blocks(T, k_lo, k_hi)
    if Ps < 0:
        raise ValueError("need 1 <= k_lo < k_hi <= T")
    _dev(A, "A", (batch, T, n, n)); _dev(w, "w", (batch, T, n))
    if phi_rows_out is None:
        phi_rows_out = torch.empty((batch, Ps, n, n), device=A.device, dtype=torch.float32)
    if r_out is None:
        r_out = torch.zeros((batch, T, n), device=A.device, dtype=torch.float32)
    _dev(phi_rows_out, "phi_rows_out", (batch, Ps, n, n)); _dev(r_out, "r_out", (batch, T, n))
    st = lib.ltv_scan_system_response_tube_rows(_ptr(A), _ptr(w), _ptr(phi_rows_out), _ptr(r_out), batch, T, n, k_lo, k_hi,
                                                LTV_TUBE_ROW_2NORM if two_norm else 0, _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_system_response_tube_rows")
    return phi_rows_out, r_out


def ltv_static_scratch_bytes():
    return int(lib.ltv_static_scratch_bytes())


def ltv_scan_system_response_tube_static(A, w, phi_out, r_out, two_norm=False):
    """ltv_scan_system_response_tube without any workspace: the library's fixed 32 MiB device array is the scratch, nothing is
    allocated by the library or by this binding (phi_out[batch,P,n,n] COLUMN_PACKED and r_out[batch,T,n] must be given).
    Raises LtvError(LTV_ERR_STATIC_SCRATCH_LIMIT) if the problem needs more scratch.  Calls that overlap on the GPU race on
    the shared array; calls on one stream are safe."""
    batch, T, n, _ = A.shape
    P = T * (T - 1) // 2
    _dev(A, "A", (batch, T, n, n)); _dev(w, "w", (batch, T, n))
    if phi_out is None or r_out is None:
        raise ValueError("ltv_scan_system_response_tube_static allocates nothing: pass phi_out and r_out")
    _dev(phi_out, "phi_out", (batch, P, n, n)); _dev(r_out, "r_out", (batch, T, n))
    st = lib.ltv_scan_system_response_tube_static(_ptr(A), _ptr(w), _ptr(phi_out), _ptr(r_out), batch, T, n,
                                                  LTV_TUBE_ROW_2NORM if two_norm else 0, _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_system_response_tube_static")
    return phi_out, r_out


def ltv_observer_row_floats(n, p):
    return int(lib.ltv_observer_row_floats(n, p))


def ltv_scan_observer_response(A, Lt, C, w, phi_out=None, r_out=None, workspace=None, two_norm=False, shifted_gain=False):
    """Closed-loop observer propagation (eq.(14)): returns (phi[batch,P,n,nc] COLUMN_PACKED with PhiX in columns
    [0,n) and PhiY in [n,n+p) of every row, r[batch,T,n]).  Lt[batch,T,n,p] (Lt_j closes the loop around A_j),
    C[batch,T,p,n].  shifted_gain=True: PhiY(t,s) = PhiX(t,s) Lt_{s-1} (the Phihat^y of (12c)/(15)) instead of the
    printed form of (14), PhiX(t,s) Lt_s."""
    batch, T, n, _ = A.shape
    p = Lt.shape[-1]
    P = T * (T - 1) // 2
    nc = ltv_observer_row_floats(n, p)
    _dev(A, "A", (batch, T, n, n)); _dev(Lt, "Lt", (batch, T, n, p)); _dev(C, "C", (batch, T, p, n))
    _dev(w, "w", (batch, T, n))
    if phi_out is None:
        phi_out = torch.empty((batch, P, n, nc), device=A.device, dtype=torch.float32)
    if r_out is None:
        r_out = torch.empty((batch, T, n), device=A.device, dtype=torch.float32)
    _dev(phi_out, "phi_out", (batch, P, n, nc)); _dev(r_out, "r_out", (batch, T, n))
    need = ltv_scan_workspace_bytes(LTV_OP_OBSERVER_RESPONSE, batch, T, n, p)
    if workspace is None:
        workspace = torch.empty(max(need, 16), device=A.device, dtype=torch.uint8)
    st = lib.ltv_scan_observer_response(_ptr(A), _ptr(Lt), _ptr(C), _ptr(w), _ptr(phi_out), _ptr(r_out), batch, T, n, p,
                                        LTV_PHI_COLUMN_PACKED,
                                        (LTV_TUBE_ROW_2NORM if two_norm else 0) | (LTV_OBSERVER_SHIFTED_GAIN if shifted_gain else 0),
                                        _ptr(workspace), workspace.numel(), _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_observer_response")
    return phi_out, r_out


def ltv_scan_constraint_tightening(A, w, Hc, sigma_out=None, workspace=None):
    """Constraint-tightening margins (eq.(12d)): sigma[batch,T,nc], sigma[b,k,i] = sum_{j<k} ||Hc[b,k,i] Phi(k,j) diag(w_j)||_2."""
    batch, T, n, _ = A.shape
    nc = Hc.shape[2]
    _dev(A, "A", (batch, T, n, n)); _dev(w, "w", (batch, T, n)); _dev(Hc, "Hc", (batch, T, nc, n))
    if sigma_out is None:
        sigma_out = torch.empty((batch, T, nc), device=A.device, dtype=torch.float32)
    _dev(sigma_out, "sigma_out", (batch, T, nc))
    need = ltv_scan_workspace_bytes(LTV_OP_CONSTRAINT_TIGHTENING, batch, T, n, nc)
    if workspace is None:
        workspace = torch.empty(max(need, 16), device=A.device, dtype=torch.uint8)
    st = lib.ltv_scan_constraint_tightening(_ptr(A), _ptr(w), _ptr(Hc), _ptr(sigma_out), batch, T, n, nc, 0,
                                            _ptr(workspace), workspace.numel(), _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_constraint_tightening")
    return sigma_out


def ltv_scan_output_feedback_response(A, B, Kfb, Lt, C, w, f, want_xe=True, workspace=None):
    """Assembled output-feedback responses (eq.(15)) for gain-defined controllers and the tube (12e): returns
    (phi_xw[batch,P,n,n], phi_xe[batch,P,n,p] | None, tau[batch,T,n]), blocks in COLUMN_PACKED order."""
    batch, T, n, _ = A.shape
    m, p = B.shape[-1], C.shape[2]
    P = T * (T - 1) // 2
    _dev(A, "A", (batch, T, n, n)); _dev(B, "B", (batch, T, n, m)); _dev(Kfb, "Kfb", (batch, T, m, n))
    _dev(Lt, "Lt", (batch, T, n, p)); _dev(C, "C", (batch, T, p, n)); _dev(w, "w", (batch, T, n)); _dev(f, "f", (batch, T, p))
    phi_xw = torch.empty((batch, P, n, n), device=A.device, dtype=torch.float32)
    phi_xe = torch.empty((batch, P, n, p), device=A.device, dtype=torch.float32) if want_xe else None
    tau = torch.empty((batch, T, n), device=A.device, dtype=torch.float32)
    need = ltv_scan_workspace_bytes(LTV_OP_OUTPUT_FEEDBACK, batch, T, n, max(m, p))
    if workspace is None:
        workspace = torch.empty(max(need, 16), device=A.device, dtype=torch.uint8)
    st = lib.ltv_scan_output_feedback_response(_ptr(A), _ptr(B), _ptr(Kfb), _ptr(Lt), _ptr(C), _ptr(w), _ptr(f),
                                               _ptr(phi_xw), _ptr(phi_xe), _ptr(tau), batch, T, n, m, p, 0,
                                               _ptr(workspace), workspace.numel(), _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_output_feedback_response")
    return phi_xw, phi_xe, tau


def ltv_scan_output_feedback_constraints(A, B, Kfb, Lt, C, w, f, Hx=None, Hu=None, want_inputs=True, workspace=None):
    """Input-side responses of eq.(15) and the closed-loop margins of eq.(12d), both terms, rows on [z; v]: returns
    (phi_uw[batch,P,m,n] | None, phi_ue[batch,P,m,p] | None, sigma[batch,T,nc] | None), blocks in COLUMN_PACKED order.
    Hx[batch,T,nc,n], Hu[batch,T,nc,m] (both or neither)."""
    batch, T, n, _ = A.shape
    m, p = B.shape[-1], C.shape[2]
    P = T * (T - 1) // 2
    nc = 0 if Hx is None else Hx.shape[2]
    _dev(A, "A", (batch, T, n, n)); _dev(B, "B", (batch, T, n, m)); _dev(Kfb, "Kfb", (batch, T, m, n))
    _dev(Lt, "Lt", (batch, T, n, p)); _dev(C, "C", (batch, T, p, n)); _dev(w, "w", (batch, T, n)); _dev(f, "f", (batch, T, p))
    _dev(Hx, "Hx", (batch, T, nc, n)); _dev(Hu, "Hu", (batch, T, nc, m))
    phi_uw = torch.empty((batch, P, m, n), device=A.device, dtype=torch.float32) if want_inputs else None
    phi_ue = torch.empty((batch, P, m, p), device=A.device, dtype=torch.float32) if want_inputs else None
    sigma = torch.empty((batch, T, nc), device=A.device, dtype=torch.float32) if nc > 0 else None
    need = int(lib.ltv_scan_output_feedback_constraints_workspace_bytes(batch, T, n, m, nc))
    if workspace is None:
        workspace = torch.empty(max(need, 16), device=A.device, dtype=torch.uint8)
    st = lib.ltv_scan_output_feedback_constraints(_ptr(A), _ptr(B), _ptr(Kfb), _ptr(Lt), _ptr(C), _ptr(w), _ptr(f), _ptr(Hx),
                                                  _ptr(Hu), _ptr(phi_uw), _ptr(phi_ue), _ptr(sigma), batch, T, n, m, p, nc, 0,
                                                  _ptr(workspace), workspace.numel(), _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_output_feedback_constraints")
    return phi_uw, phi_ue, sigma


def ltv_scan_kalman_gains(A, C, e, f, Pi0, Lt_out=None, Pi_out=None, workspace=None, mode=0):
    """Backward-Kalman recursion (eq.(13)): returns (Lt[batch,T,n,p] with Lt[b,j] = L_{j+1}^T, Pi[batch,T+1,n,n]).
    C[batch,T,p,n], e[batch,T,n], f[batch,T,p] (> 0), Pi0[batch,n,n] symmetric PSD.  mode: 0 the library picks,
    LTV_KALMAN_SCAN (associative scan (16)(17), n <= 64) or LTV_KALMAN_RECURSION."""
    batch, T, n, _ = A.shape
    p = C.shape[2]
    _dev(A, "A", (batch, T, n, n)); _dev(C, "C", (batch, T, p, n)); _dev(e, "e", (batch, T, n))
    _dev(f, "f", (batch, T, p)); _dev(Pi0, "Pi0", (batch, n, n))
    if Lt_out is None:
        Lt_out = torch.empty((batch, T, n, p), device=A.device, dtype=torch.float32)
    if Pi_out is None:
        Pi_out = torch.empty((batch, T + 1, n, n), device=A.device, dtype=torch.float32)
    _dev(Lt_out, "Lt_out", (batch, T, n, p)); _dev(Pi_out, "Pi_out", (batch, T + 1, n, n))
    need = ltv_scan_workspace_bytes(LTV_OP_KALMAN_GAINS, batch, T, n, p)
    if workspace is None:
        workspace = torch.empty(max(need, 16), device=A.device, dtype=torch.uint8)
    st = lib.ltv_scan_kalman_gains(_ptr(A), _ptr(C), _ptr(e), _ptr(f), _ptr(Pi0), _ptr(Lt_out), _ptr(Pi_out),
                                   batch, T, n, p, mode, _ptr(workspace), workspace.numel(), _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_kalman_gains")
    return Lt_out, Pi_out


def ltv_scan_adjoint(A, B, g, want_grad_x0=True, lambda_out=None, grad_u_out=None, grad_x0_out=None):
    """Returns (lam[batch,T,n] with lam[b,t-1] = lam_t, grad_u[batch,T,m]|None, grad_x0[batch,n]|None)."""
    batch, T, n, _ = A.shape
    m = 0 if B is None else B.shape[-1]
    _dev(A, "A", (batch, T, n, n)); _dev(B, "B", (batch, T, n, m)); _dev(g, "g", (batch, T, n))
    if lambda_out is None:
        lambda_out = torch.empty((batch, T, n), device=A.device, dtype=torch.float32)
    if grad_u_out is None and B is not None and m > 0:
        grad_u_out = torch.empty((batch, T, m), device=A.device, dtype=torch.float32)
    if grad_x0_out is None and want_grad_x0:
        grad_x0_out = torch.empty((batch, n), device=A.device, dtype=torch.float32)
    st = lib.ltv_scan_adjoint(_ptr(A), _ptr(B), _ptr(g), _ptr(lambda_out), _ptr(grad_u_out), _ptr(grad_x0_out),
                              batch, T, n, m, None, 0, _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_adjoint")
    return lambda_out, grad_u_out, grad_x0_out


def ltv_scan_rollout_adjoint(A, B, c, x0, u, g, want_grad_x0=True, x_out=None, lambda_out=None, grad_u_out=None,
                             grad_x0_out=None):
    """Rollout and adjoint of the same batch, concurrently (one call): returns (x, lam, grad_u | None, grad_x0 | None)
    with the conventions of ltv_scan_rollout / ltv_scan_adjoint."""
    batch, T, n, _ = A.shape
    m = 0 if B is None else B.shape[-1]
    _dev(A, "A", (batch, T, n, n)); _dev(B, "B", (batch, T, n, m)); _dev(c, "c", (batch, T, n))
    _dev(x0, "x0", (batch, n)); _dev(u, "u", (batch, T, m)); _dev(g, "g", (batch, T, n))
    mk = lambda *s: torch.empty(s, device=A.device, dtype=torch.float32)
    if x_out is None:
        x_out = mk(batch, T, n)
    if lambda_out is None:
        lambda_out = mk(batch, T, n)
    if grad_u_out is None and B is not None and m > 0:
        grad_u_out = mk(batch, T, m)
    if grad_x0_out is None and want_grad_x0:
        grad_x0_out = mk(batch, n)
    st = lib.ltv_scan_rollout_adjoint(_ptr(A), _ptr(B), _ptr(c), _ptr(x0), _ptr(u), _ptr(g), _ptr(x_out), _ptr(lambda_out),
                                      _ptr(grad_u_out), _ptr(grad_x0_out), batch, T, n, m, None, 0, _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_rollout_adjoint")
    return x_out, lambda_out, grad_u_out, grad_x0_out


def ltv_scan_all_is_fused(batch, T, n, m, layout=LTV_PHI_COLUMN_PACKED) -> bool:
    return bool(lib.ltv_scan_all_is_fused(batch, T, n, m, layout))


def ltv_scan_all(A, B, c, x0, u, w, g, want_grad_x0=True, two_norm=False, layout=LTV_PHI_COLUMN_PACKED, outs=None,
                 workspace=None):
    """The whole hot path in one call: returns dict(x, phi, r, lam, grad_u, grad_x0) of device tensors (conventions of the
    three single calls).  Small problems (ltv_scan_all_is_fused) run as ONE kernel launch."""
    batch, T, n, _ = A.shape
    m = 0 if B is None else B.shape[-1]
    P = T * (T - 1) // 2
    _dev(A, "A", (batch, T, n, n)); _dev(B, "B", (batch, T, n, m)); _dev(c, "c", (batch, T, n))
    _dev(x0, "x0", (batch, n)); _dev(u, "u", (batch, T, m)); _dev(w, "w", (batch, T, n)); _dev(g, "g", (batch, T, n))
    mk = lambda *s: torch.empty(s, device=A.device, dtype=torch.float32)
    if outs is None:
        outs = dict(x=mk(batch, T, n), phi=mk(*((batch, T, T, n, n) if layout == LTV_PHI_SQUARE_GRID else (batch, P, n, n))),
                    r=mk(batch, T, n), lam=mk(batch, T, n), grad_u=mk(batch, T, m) if (B is not None and m > 0) else None,
                    grad_x0=mk(batch, n) if want_grad_x0 else None)
    need = ltv_scan_workspace_bytes(LTV_OP_SYSTEM_RESPONSE_TUBE if layout == LTV_PHI_COLUMN_PACKED
                                    else LTV_OP_SYSTEM_RESPONSE_TUBE_RELAYOUT, batch, T, n, 0)
    if workspace is None:
        workspace = torch.empty(max(need, 16), device=A.device, dtype=torch.uint8)
    st = lib.ltv_scan_all(_ptr(A), _ptr(B), _ptr(c), _ptr(x0), _ptr(u), _ptr(w), _ptr(g), _ptr(outs["x"]), _ptr(outs["phi"]),
                          _ptr(outs["r"]), _ptr(outs["lam"]), _ptr(outs["grad_u"]), _ptr(outs["grad_x0"]), batch, T, n, m,
                          layout, LTV_TUBE_ROW_2NORM if two_norm else 0, _ptr(workspace), workspace.numel(), _stream())
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_all")
    return outs


def ltv_scan_pipeline_host(A, B, c, x0, u, w, g, workspace, want_grad_x0=True, phi_host=None, outs=None):
    """Whole path from HOST (CPU, ideally pinned) fp32 tensors; returns dict of host outputs and the device
    address of Phi inside `workspace` (a uint8 CUDA tensor of >= workspace_bytes(LTV_OP_PIPELINE_HOST)).
    w=None skips the Phi / tube stage (workspace need: LTV_OP_PIPELINE_HOST_NO_PHI)."""
    batch, T, n, _ = A.shape
    m = 0 if B is None else B.shape[-1]
    for name, t in (("A", A), ("B", B), ("c", c), ("x0", x0), ("u", u), ("w", w), ("g", g), ("phi_host", phi_host)):
        if t is not None and (t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous()):
            raise ValueError(f"{name}: need a contiguous fp32 host tensor")
    if outs is None:
        pin = torch.cuda.is_available()
        mk = lambda *s: torch.empty(s, dtype=torch.float32, pin_memory=pin)
        outs = dict(x=mk(batch, T, n), r=mk(batch, T, n) if w is not None else None, lam=mk(batch, T, n),
                    grad_u=mk(batch, T, m) if (B is not None and m > 0) else None,
                    grad_x0=mk(batch, n) if want_grad_x0 else None)
    phi_dev = ctypes.c_void_p(0)
    st = lib.ltv_scan_pipeline_host(_ptr(A), _ptr(B), _ptr(c), _ptr(x0), _ptr(u), _ptr(w), _ptr(g),
                                    _ptr(outs["x"]), _ptr(phi_host), _ptr(outs["r"]), _ptr(outs["lam"]),
                                    _ptr(outs["grad_u"]), _ptr(outs["grad_x0"]), batch, T, n, m,
                                    _ptr(workspace), workspace.numel(), _stream(), ctypes.byref(phi_dev))
    if st != LTV_OK:
        raise LtvError(st, "ltv_scan_pipeline_host")
    outs["phi_device_ptr"] = phi_dev.value
    return outs
