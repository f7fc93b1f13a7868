"""ltv_scan_output_feedback_assemble - eq.(15) and the tube (12e) for a GENERAL state-feedback response
Phibar given as block operators - against the pinned oracle's dense evaluation of (15), through the C-ABI binding.
Tolerance: max|err| / max|ref| <= 1e-4 per output tensor."""
import numpy as np
import pytest

from assembly_inputs import blk, general_phibar, observer_operators
from oracle import ltv_oracle as O

pytestmark = pytest.mark.gpu
TOL = 1e-4


@pytest.fixture(scope="module")
def L():
    import torch

    assert torch.cuda.is_available(), "GPU tests need a GPU (no CPU fallback)"
    import __graft_entry__ as G

    G.build()
    import paper_2606_14188_b200 as lib

    return lib


def _item(T, n, m, p, seed):
    rng = np.random.default_rng(seed)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    A = f32(np.eye(n)[None] + rng.normal(0.0, 0.4 / np.sqrt(n), (T, n, n)))
    B = f32(rng.normal(0.0, 1.0, (T, n, m)))
    C = f32(rng.normal(0.0, 1.0 / np.sqrt(n), (T, p, n)))
    Lt = f32(0.3 * rng.normal(0.0, 1.0, (T, n, p)))
    w = f32(rng.uniform(0.0, 1e-3, (T, n)))
    f = f32(rng.uniform(1e-3, 5e-3, (T, p)))
    PbX, PbU = general_phibar(A, B, seed=seed + 1)
    return A, C, Lt, w, f, f32(PbX), f32(PbU)      # the operators rounded to fp32 once: both sides start from these


def _pack(L, T, n, m, PbX, PbU):
    """dense fp32 operators -> the call's layouts: phibar_x [P,n,n] column-packed strictly lower, phibar_u [P+T,m,n] with diagonal."""
    P = T * (T - 1) // 2
    px = np.zeros((P, n, n), dtype=np.float32)
    pu = np.zeros((P + T, m, n), dtype=np.float32)
    for j in range(T):
        for k in range(j, T):
            pu[j * T - j * (j - 1) // 2 + (k - j)] = blk(PbU, k, j, m, n)
            if k > j:
                px[L.ltv_phi_block_index(T, k, j)] = blk(PbX, k, j, n, n)
    return px, pu


@pytest.mark.parametrize("n,T,m,p,batch", [(24, 6, 2, 3, 2),      # fp32-FMA products
                                           (48, 2, 3, 4, 1),      # T = 2: a single block, no GEMM
                                           (96, 7, 3, 4, 1),      # smallest tensor-core size
                                           (132, 5, 6, 6, 2),     # ragged tiles
                                           (100, 4, 1, 1, 1),     # single input, single output
                                           (64, 3, 4, 20, 1),     # wide observation
                                           (300, 6, 6, 6, 2),     # C2-size blocks: two n-tiles of 160, stacks across blocks
                                           (640, 3, 2, 6, 1),     # one-row shared-memory pipeline on the x side (two-row buffers do not fit)
                                           (1200, 3, 2, 6, 1)])   # rows too long for the shared-memory pipeline: register kernel
def test_general_assembly_against_the_oracle(L, n, T, m, p, batch):
    import torch

    items = [_item(T, n, m, p, seed=11 * n + T + 100 * b) for b in range(batch)]
    A, C, Lt, w, f = [np.stack([it[q] for it in items]) for q in range(5)]
    packed = [_pack(L, T, n, m, it[5], it[6]) for it in items]
    px = np.stack([q[0] for q in packed]); pu = np.stack([q[1] for q in packed])
    cu = lambda a: torch.from_numpy(a).cuda()
    out = L.ltv_scan_output_feedback_assemble(cu(A), cu(Lt), cu(C), cu(w), cu(f), cu(px), cu(pu))
    out2 = L.ltv_scan_output_feedback_assemble(cu(A), cu(Lt), cu(C), cu(w), cu(f), cu(px), None, want_xe=False, want_tau=False)
    torch.cuda.synchronize()
    assert out2["phi_uw"] is None and out2["phi_xe"] is None and torch.equal(out["phi_xw"], out2["phi_xw"])
    got = {k: v.cpu().numpy() for k, v in out.items()}
    ref = {k: np.zeros_like(v) for k, v in got.items()}
    for b, it in enumerate(items):
        A64 = it[0].astype(np.float64)
        PbX, PbU = it[5].astype(np.float64), it[6].astype(np.float64)
        for k in range(T):
            PbX[k * n:(k + 1) * n, k * n:(k + 1) * n] = np.eye(n)     # the call takes the diagonal of Phibar^x as I
            PbX[k * n:(k + 1) * n, (k + 1) * n:] = 0.0
        PhX, PhY = observer_operators(A64, it[2], it[1])
        Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A64, PbX, PbU, PhX, PhY)
        ref["tau"][b] = O.output_feedback_tube(Pxw, Pxe, it[3], it[4])
        for k in range(1, T):
            for j in range(k):
                q = L.ltv_phi_block_index(T, k, j)
                ref["phi_xw"][b, q] = blk(Pxw, k, j, n, n); ref["phi_xe"][b, q] = blk(Pxe, k, j, n, p)
                ref["phi_uw"][b, q] = blk(Puw, k, j, m, n); ref["phi_ue"][b, q] = blk(Pue, k, j, m, p)
    for key in ("phi_xw", "phi_xe", "phi_uw", "phi_ue", "tau"):
        assert np.all(np.isfinite(got[key])), key
        assert O.rel_err(got[key], ref[key]) <= TOL, (key, O.rel_err(got[key], ref[key]))


def test_general_assembly_reproduces_the_gain_defined_call(L):
    """Phibar generated from gains K (Phibar^x = response of A + B K, Phibar^u(k,j) = K_k Phibar^x(k,j)) must give what
    ltv_scan_output_feedback_response / _constraints return for the same controller."""
    import torch

    n, T, m, p, batch = 132, 6, 3, 4, 2
    rng = np.random.default_rng(9)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    A = f32(np.eye(n)[None, None] + rng.normal(0.0, 0.4 / np.sqrt(n), (batch, T, n, n)))
    B = f32(rng.normal(0.0, 1.0, (batch, T, n, m)))
    K = f32(0.3 * rng.normal(0.0, 1.0 / np.sqrt(n), (batch, T, m, n)))
    C = f32(rng.normal(0.0, 1.0 / np.sqrt(n), (batch, T, p, n)))
    Lt = f32(0.3 * rng.normal(0.0, 1.0, (batch, T, n, p)))
    w = f32(rng.uniform(0.0, 1e-3, (batch, T, n))); f = f32(rng.uniform(1e-3, 5e-3, (batch, T, p)))
    cu = lambda a: torch.from_numpy(a).cuda()
    xw, xe, tau = L.ltv_scan_output_feedback_response(cu(A), cu(B), cu(K), cu(Lt), cu(C), cu(w), cu(f))
    P = T * (T - 1) // 2
    px = np.zeros((batch, P, n, n), dtype=np.float32); pu = np.zeros((batch, P + T, m, n), dtype=np.float32)
    for b in range(batch):
        Atil = A[b].astype(np.float64) + B[b].astype(np.float64) @ K[b].astype(np.float64)
        blocks = O.system_response_item(Atil)
        for j in range(T):
            for k in range(j, T):
                Pkj = np.eye(n) if k == j else blocks[O.packed_index(k, j)]
                pu[b, j * T - j * (j - 1) // 2 + (k - j)] = K[b, k].astype(np.float64) @ Pkj
                if k > j:
                    px[b, L.ltv_phi_block_index(T, k, j)] = Pkj
    out = L.ltv_scan_output_feedback_assemble(cu(A), cu(Lt), cu(C), cu(w), cu(f), cu(px), cu(pu))
    torch.cuda.synchronize()
    rel = lambda a, b: float((a - b).abs().max() / b.abs().max())
    assert rel(out["phi_xw"], xw) <= TOL and rel(out["phi_xe"], xe) <= TOL and rel(out["tau"], tau) <= TOL


def test_general_assembly_validation(L):
    f = L.lib.ltv_scan_output_feedback_assemble
    assert L.lib.ltv_scan_output_feedback_assemble_workspace_bytes(2, 5, 48, 3, 4) >= 2 * 5 * 48 * 48 * 4
    assert L.lib.ltv_scan_output_feedback_assemble_workspace_bytes(2, 5, 48, 3, 33) == 0
    import ctypes
    buf = (ctypes.c_float * 64)()
    q = ctypes.cast(buf, ctypes.c_void_p)
    assert f(None, q, q, q, q, q, None, q, None, None, None, None, 1, 2, 4, 0, 1, 0, q, 1 << 20, None) == 1     # NULL A
    assert f(q, q, q, q, q, q, None, q, None, q, None, None, 1, 2, 4, 1, 1, 0, q, 1 << 20, None) == 1           # phi_uw without phibar_u
    assert f(q, q, q, q, q, q, None, q, None, None, None, None, 1, 2, 4, 0, 0, 0, q, 1 << 20, None) == 2        # p = 0
    assert f(q, q, q, q, q, q, None, q, None, None, None, None, 1, 2, 4, 0, 1, 1, q, 1 << 20, None) == 2        # flags
    assert f(q, q, q, q, q, q, None, q, None, None, None, None, 1, 2, 4, 0, 1, 0, q, 8, None) == 5              # workspace


def test_general_assembly_full_batch_c2_shape_sampled_items(L):
    """n = 300, batch 64 (BASELINE.json configs[1]: the launch configuration bench.py times) at a horizon the oracle's dense
    operators can hold (T = 12); two sampled items against the oracle, every item finite."""
    import torch

    n, T, m, p, batch = 300, 12, 6, 6, 64
    sample = (0, 37)
    rng = np.random.default_rng(2026)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    A = f32(np.eye(n)[None, None] + rng.normal(0.0, 0.4 / np.sqrt(n), (batch, T, n, n)))
    C = f32(rng.normal(0.0, 1.0 / np.sqrt(n), (batch, T, p, n)))
    Lt = f32(0.3 * rng.normal(0.0, 1.0, (batch, T, n, p)))
    w = f32(rng.uniform(0.0, 1e-3, (batch, T, n))); f = f32(rng.uniform(1e-3, 5e-3, (batch, T, p)))
    P = T * (T - 1) // 2
    px = f32(rng.normal(0.0, 0.3 / np.sqrt(n), (batch, P, n, n)))          # any operators with unit diagonal are valid inputs of (15)
    pu = f32(rng.normal(0.0, 0.3 / np.sqrt(n), (batch, P + T, m, n)))
    dense = {}
    for b in sample:
        B = rng.normal(0.0, 1.0, (T, n, m))
        PbX, PbU = general_phibar(A[b], B, seed=b + 3)
        px[b], pu[b] = _pack(L, T, n, m, f32(PbX), f32(PbU))
    cu = lambda a: torch.from_numpy(a).cuda()
    out = L.ltv_scan_output_feedback_assemble(cu(A), cu(Lt), cu(C), cu(w), cu(f), cu(px), cu(pu))
    torch.cuda.synchronize()
    for v in out.values():
        assert torch.isfinite(v).all()
    for b in sample:
        PbX = np.eye(T * n); PbU = np.zeros((T * m, T * n))
        for j in range(T):
            for k in range(j, T):
                PbU[k * m:(k + 1) * m, j * n:(j + 1) * n] = pu[b, j * T - j * (j - 1) // 2 + (k - j)]
                if k > j:
                    PbX[k * n:(k + 1) * n, j * n:(j + 1) * n] = px[b, L.ltv_phi_block_index(T, k, j)]
        PhX, PhY = observer_operators(A[b], Lt[b], C[b])
        Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A[b].astype(np.float64), PbX, PbU, PhX, PhY)
        tau = O.output_feedback_tube(Pxw, Pxe, w[b], f[b])
        ref = {k2: np.zeros_like(v[b].cpu().numpy()) for k2, v in out.items()}
        ref["tau"] = tau
        for k in range(1, T):
            for j in range(k):
                q = L.ltv_phi_block_index(T, k, j)
                ref["phi_xw"][q] = blk(Pxw, k, j, n, n); ref["phi_xe"][q] = blk(Pxe, k, j, n, p)
                ref["phi_uw"][q] = blk(Puw, k, j, m, n); ref["phi_ue"][q] = blk(Pue, k, j, m, p)
        for key in ref:
            assert O.rel_err(out[key][b].cpu().numpy(), ref[key]) <= TOL, (b, key)


@pytest.mark.parametrize("n,T,m,p,nc,batch", [(24, 6, 2, 3, 4, 2),      # fp32-FMA path of the assembly
                                              (132, 5, 6, 6, 3, 2),     # two column quads per lane, ragged
                                              (300, 6, 6, 6, 6, 2),     # C2-size blocks
                                              (96, 4, 3, 4, 11, 1),     # more than 8 constraint rows: two passes
                                              (48, 2, 1, 1, 1, 1)])     # T = 2: one block
def test_margins_on_assembled_operators_general_phibar(L, n, T, m, p, nc, batch):
    """Chain general assembly -> ltv_scan_operator_constraint_margins against the oracle's eq.(12d) (both terms, rows on
    [z; v]) evaluated on the oracle's own dense operators of eq.(15)."""
    import torch

    items = [_item(T, n, m, p, seed=13 * n + T + 100 * b) for b in range(batch)]
    A, C, Lt, w, f = [np.stack([it[q] for it in items]) for q in range(5)]
    packed = [_pack(L, T, n, m, it[5], it[6]) for it in items]
    px = np.stack([q[0] for q in packed]); pu = np.stack([q[1] for q in packed])
    rng = np.random.default_rng(n + nc)
    Hx = rng.normal(0.0, 1.0, (batch, T, nc, n)).astype(np.float32)
    Hu = rng.normal(0.0, 1.0, (batch, T, nc, m)).astype(np.float32)
    cu = lambda a: torch.from_numpy(a).cuda()
    out = L.ltv_scan_output_feedback_assemble(cu(A), cu(Lt), cu(C), cu(w), cu(f), cu(px), cu(pu))
    sig = L.ltv_scan_operator_constraint_margins(out["phi_xw"], cu(Hx), cu(w), phi_uw=out["phi_uw"], Hu=cu(Hu),
                                                 phi_xe=out["phi_xe"], phi_ue=out["phi_ue"], f=cu(f))
    sig_x = L.ltv_scan_operator_constraint_margins(out["phi_xw"], cu(Hx), cu(w))          # state rows, w term only
    torch.cuda.synchronize()
    ref = np.zeros((batch, T, nc)); ref_x = np.zeros((batch, T, nc))
    for b, it in enumerate(items):
        A64 = it[0].astype(np.float64)
        PbX, PbU = it[5].astype(np.float64), it[6].astype(np.float64)
        for k in range(T):
            PbX[k * n:(k + 1) * n, k * n:(k + 1) * n] = np.eye(n)
            PbX[k * n:(k + 1) * n, (k + 1) * n:] = 0.0
        PhX, PhY = observer_operators(A64, it[2], it[1])
        Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A64, PbX, PbU, PhX, PhY)
        ref[b] = O.output_feedback_constraint_tightening(Pxw, Puw, Pxe, Pue, it[3], it[4], Hx[b], Hu[b])
        ref_x[b] = O.output_feedback_constraint_tightening(Pxw, np.zeros_like(Puw), np.zeros_like(Pxe), np.zeros_like(Pue),
                                                           it[3], it[4], Hx[b], np.zeros_like(Hu[b]))
    assert np.all(sig.cpu().numpy()[:, 0] == 0.0)
    assert O.rel_err(sig.cpu().numpy(), ref) <= TOL, O.rel_err(sig.cpu().numpy(), ref)
    assert O.rel_err(sig_x.cpu().numpy(), ref_x) <= TOL


def test_margins_on_operators_equal_the_gain_defined_sweep(L):
    """For a gain-defined controller the margins computed from the assembled operators must equal those of
    ltv_scan_output_feedback_constraints (which never forms an operator block)."""
    import torch

    n, T, m, p, nc, batch = 132, 6, 3, 4, 5, 2
    rng = np.random.default_rng(19)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    A = f32(np.eye(n)[None, None] + rng.normal(0.0, 0.4 / np.sqrt(n), (batch, T, n, n)))
    B = f32(rng.normal(0.0, 1.0, (batch, T, n, m)))
    K = f32(0.3 * rng.normal(0.0, 1.0 / np.sqrt(n), (batch, T, m, n)))
    C = f32(rng.normal(0.0, 1.0 / np.sqrt(n), (batch, T, p, n)))
    Lt = f32(0.3 * rng.normal(0.0, 1.0, (batch, T, n, p)))
    w = f32(rng.uniform(0.0, 1e-3, (batch, T, n))); f = f32(rng.uniform(1e-3, 5e-3, (batch, T, p)))
    Hx = f32(rng.normal(0.0, 1.0, (batch, T, nc, n))); Hu = f32(rng.normal(0.0, 1.0, (batch, T, nc, m)))
    cu = lambda a: torch.from_numpy(a).cuda()
    xw, xe, _ = L.ltv_scan_output_feedback_response(cu(A), cu(B), cu(K), cu(Lt), cu(C), cu(w), cu(f))
    uw, ue, sig_ref = L.ltv_scan_output_feedback_constraints(cu(A), cu(B), cu(K), cu(Lt), cu(C), cu(w), cu(f), cu(Hx), cu(Hu))
    sig = L.ltv_scan_operator_constraint_margins(xw, cu(Hx), cu(w), phi_uw=uw, Hu=cu(Hu), phi_xe=xe, phi_ue=ue, f=cu(f))
    torch.cuda.synchronize()
    assert float((sig - sig_ref).abs().max() / sig_ref.abs().max()) <= TOL


def test_margins_validation(L):
    import ctypes
    g = L.lib.ltv_scan_operator_constraint_margins
    buf = (ctypes.c_float * 64)()
    q = ctypes.cast(buf, ctypes.c_void_p)
    assert g(q, None, None, None, None, None, q, None, q, 1, 2, 4, 0, 0, 1, 0, None) == 1      # NULL Hx
    assert g(q, q, None, None, q, None, q, None, q, 1, 2, 4, 1, 0, 1, 0, None) == 1            # phi_uw without Hu
    assert g(q, None, None, None, q, None, q, None, q, 1, 2, 4, 0, 0, 0, 0, None) == 2         # nc = 0
    assert g(q, None, None, None, q, None, q, None, q, 1, 2, 1028, 0, 0, 1, 0, None) == 3      # n > 512
