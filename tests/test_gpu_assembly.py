"""Eq.(15) on the device for controllers given by gains (first step): with u = K xhat and the
predictor-form observer, the output-feedback closed loop is the LTV system xi_{k+1} = [[A + B K, -B K], [0, A + Lt C]] xi_k
in xi = (x, x - xhat), so ONE call of ltv_scan_system_response_tube on the 2n-state augmented Jacobians yields every
block of Phi^xw, Phi^xe (and Phi^uw, Phi^ue after the feedback gain): Phi^xw(k,j) = G11 + G12, Phi^xe(k,j) = G12 Lt_{j-1}
with G = Phi_aug(k,j).  Checked against the pinned oracle assemble_output_feedback, which evaluates (15) as printed.
(The block extraction below is test code; a dedicated assembly call for general Phibar is not built - DESIGN.md.)"""
import numpy as np
import pytest

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


def _gains(T, n, m, p, seed):
    rng = np.random.default_rng(seed)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    A = f32(np.eye(n)[None] + rng.normal(0.0, 0.4 / np.sqrt(n), (T, n, n)))
    B = f32(rng.normal(0.0, 1.0, (T, n, m)))
    C = f32(rng.normal(0.0, 1.0 / np.sqrt(n), (T, p, n)))
    K = f32(0.3 * rng.normal(0.0, 1.0 / np.sqrt(n), (T, m, n)))
    Lt = f32(0.3 * rng.normal(0.0, 1.0, (T, n, p)))
    return A, B, C, K, Lt


def _dense(blocks, T, n):
    D = np.eye(T * n)
    for t in range(1, T):
        for s in range(t):
            D[t * n:(t + 1) * n, s * n:(s + 1) * n] = blocks[O.packed_index(t, s)]
    return D


@pytest.mark.parametrize("n,T,m,p", [(24, 6, 2, 3),      # 2n = 48: fp32-FMA combine
                                     (48, 7, 3, 4),      # 2n = 96: smallest tensor-core size
                                     (132, 5, 6, 6)])    # 2n = 264: two n-tiles, ragged k-block
def test_output_feedback_response_via_augmented_system(L, n, T, m, p):
    import torch

    A, B, C, K, Lt = _gains(T, n, m, p, seed=3 * n + T)
    A64, B64, C64, K64, Lt64 = [a.astype(np.float64) for a in (A, B, C, K, Lt)]
    # fp32 augmented Jacobians handed to the GPU (and, promoted, to the oracle operators below)
    Aaug = np.zeros((1, T, 2 * n, 2 * n), dtype=np.float32)
    BK = (B64 @ K64).astype(np.float32)
    Aaug[0, :, :n, :n] = A + BK
    Aaug[0, :, :n, n:] = -BK
    Aaug[0, :, n:, n:] = (A64 + Lt64 @ C64).astype(np.float32)
    w = np.ones((1, T, 2 * n), dtype=np.float32)
    phi, _ = L.ltv_scan_system_response_tube(torch.from_numpy(Aaug).cuda(), torch.from_numpy(w).cuda())
    torch.cuda.synchronize()
    phi = phi[0].cpu().numpy()

    # oracle: (15) as printed, on operators built from the SAME fp32 closed-loop matrices
    Atil, Abar = Aaug[0, :, :n, :n].astype(np.float64), Aaug[0, :, n:, n:].astype(np.float64)
    PbX = _dense(O.system_response_item(Atil), T, n)
    PbU = np.vstack([K64[k] @ PbX[k * n:(k + 1) * n] for k in range(T)])
    PhX = _dense(O.system_response_item(Abar), T, n)
    PhY = np.zeros((T * n, T * p))
    for j in range(1, T):
        PhY[:, j * p:(j + 1) * p] = PhX[:, j * n:(j + 1) * n] @ Lt64[j - 1]
    # M of (15) must be the open-loop I - Z A with A = Atil - B K = Abar - Lt C: use the fp32-consistent difference
    Aopen = Atil - (-Aaug[0, :, :n, n:].astype(np.float64))
    Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(Aopen, PbX, PbU, PhX, PhY)

    got_xw, ref_xw, got_xe, ref_xe, got_uw, ref_uw = [], [], [], [], [], []
    for k in range(1, T):
        for j in range(k):
            G = phi[L.ltv_phi_block_index(T, k, j)].astype(np.float64)
            got_xw.append(G[:n, :n] + G[:n, n:]); ref_xw.append(Pxw[k * n:(k + 1) * n, j * n:(j + 1) * n])
            got_uw.append(K64[k] @ (G[:n, :n] + G[:n, n:] - G[n:, :n] - G[n:, n:]))
            ref_uw.append(Puw[k * m:(k + 1) * m, j * n:(j + 1) * n])
            if j >= 1:
                got_xe.append(G[:n, n:] @ Lt64[j - 1]); ref_xe.append(Pxe[k * n:(k + 1) * n, j * p:(j + 1) * p])
            assert np.all(G[n:, :n] == 0.0)        # block-triangular structure survives the scan exactly
    assert O.rel_err(np.stack(got_xw), np.stack(ref_xw)) <= TOL
    assert O.rel_err(np.stack(got_uw), np.stack(ref_uw)) <= TOL
    assert O.rel_err(np.stack(got_xe), np.stack(ref_xe)) <= TOL


def _oracle_ofb(A, B, C, K, Lt, w, f):
    """(15) + (12e) from the oracle, on operators built from the fp32 inputs promoted to fp64 (one item)."""
    A, B, C, K, Lt = [a.astype(np.float64) for a in (A, B, C, K, Lt)]
    T, n, _ = A.shape
    m, p = B.shape[2], C.shape[1]
    PbX = _dense(O.system_response_item(A + B @ K), T, n)
    PbU = np.vstack([K[k] @ PbX[k * n:(k + 1) * n] for k in range(T)])
    PhX = _dense(O.observer_response_item(A, Lt, C)[0], T, n)
    PhY = np.zeros((T * n, T * p))
    for j in range(1, T):
        PhY[:, j * p:(j + 1) * p] = PhX[:, j * n:(j + 1) * n] @ Lt[j - 1]
    Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A, PbX, PbU, PhX, PhY)
    return Pxw, Pxe, O.output_feedback_tube(Pxw, Pxe, w, f)


@pytest.mark.parametrize("n,T,m,p,batch", [(24, 6, 2, 3, 2),      # 2n = 48: fp32-FMA combine
                                           (48, 7, 3, 4, 1),      # 2n = 96: smallest tensor-core size
                                           (132, 5, 6, 6, 2),     # ragged tiles
                                           (100, 4, 1, 1, 1),     # single input, single output
                                           (64, 3, 4, 20, 1),     # wide observation (three groups of 8)
                                           (300, 5, 3, 5, 2),     # column route: two-row kernel, m < p (zero-padded vectors)
                                           (164, 4, 7, 2, 1),     # column route: two-row kernel, m > p, ragged tiles
                                           (640, 4, 3, 5, 1),     # column route: one-row shared-memory pipeline in difference mode
                                           (800, 3, 2, 2, 1),     # column route: register kernel in difference mode
                                           (96, 2, 2, 2, 1),      # T = 2: a single block, no product in either route
                                           (100, 3, 2, 3, 2),     # T = 3: one product step
                                           (132, 4, 12, 3, 1)])   # m > 8: the column route is not available, both settings take the cross scan
@pytest.mark.parametrize("route", [1, 2])                         # n >= 96: cross scan / column recursion (LTV_OPT_OUTPUT_FEEDBACK_ROUTE)
def test_output_feedback_response_call(L, n, T, m, p, batch, route):
    """ltv_scan_output_feedback_response (n < 96: augmented Jacobians, Phi scan on 2n states, extraction + tube; n >= 96: both
    structured routes; all on the device) against eq.(15) and (12e) evaluated by the oracle."""
    import torch

    if n < 96 and route == 2:
        pytest.skip("one route below n = 96")
    L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, route)
    try:
        _response_call_case(L, n, T, m, p, batch)
    finally:
        L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, 0)


def _response_call_case(L, n, T, m, p, batch):
    import torch

    items = [_gains(T, n, m, p, seed=7 * n + T + b) for b in range(batch)]
    A, B, C, K, Lt = [np.stack([it[q] for it in items]) for q in range(5)]
    rng = np.random.default_rng(n)
    w = rng.uniform(0.1, 1.0, (batch, T, n)).astype(np.float32)
    f = rng.uniform(0.1, 1.0, (batch, T, p)).astype(np.float32)
    d = [torch.from_numpy(a).cuda() for a in (A, B, K, Lt, C, w, f)]
    xw, xe, tau = L.ltv_scan_output_feedback_response(*d)
    torch.cuda.synchronize()
    xw, xe, tau = xw.cpu().numpy(), xe.cpu().numpy(), tau.cpu().numpy()
    for b in range(batch):
        Pxw, Pxe, tau_ref = _oracle_ofb(A[b], B[b], C[b], K[b], Lt[b], w[b], f[b])
        ref_w = np.stack([Pxw[k * n:(k + 1) * n, j * n:(j + 1) * n] for j in range(T - 1) for k in range(j + 1, T)])
        ref_e = np.stack([Pxe[k * n:(k + 1) * n, j * p:(j + 1) * p] for j in range(T - 1) for k in range(j + 1, T)])
        assert O.rel_err(xw[b], ref_w) <= TOL
        assert O.rel_err(xe[b], ref_e) <= TOL
        assert O.rel_err(tau[b], tau_ref) <= TOL
        assert np.all(tau[b, 0] == 0.0)
        assert np.all(xe[b, :T - 1] == 0.0)      # column j = 0: no measurement precedes step 0


def test_kalman_gains_to_output_feedback_tube_pipeline(L):
    """Stage 3 end to end on the device: gains of (13) -> responses (15) -> tube (12e); oracle: the same chain in fp64."""
    import torch
    from workloads import dense_random, observation_model

    n, T, batch, m, p = 64, 6, 2, 3, 4
    W = dense_random(batch, T, n, m, seed=31, scale=0.4)
    M = observation_model(batch, T, n, p, seed=32, kind="dense")
    K = (0.2 * np.random.default_rng(33).normal(0.0, 1.0 / np.sqrt(n), (batch, T, m, n))).astype(np.float32)
    w1 = (1e3 * W.w).astype(np.float32)
    dA, dB = torch.from_numpy(W.A).cuda(), torch.from_numpy(W.B).cuda()
    dC, de, df, dP = [torch.from_numpy(M[k]).cuda() for k in ("C", "e", "f", "Pi0")]
    Lt, _ = L.ltv_scan_kalman_gains(dA, dC, de, df, dP)
    xw, xe, tau = L.ltv_scan_output_feedback_response(dA, dB, torch.from_numpy(K).cuda(), Lt, dC,
                                                      torch.from_numpy(w1).cuda(), df)
    torch.cuda.synchronize()
    _, Lt_ref = O.kalman_recursion(W.A, M["C"], M["e"], M["f"], M["Pi0"])
    for b in range(batch):
        _, _, tau_ref = _oracle_ofb(W.A[b], W.B[b], M["C"][b], K[b], Lt_ref[b], w1[b], M["f"][b])
        assert O.rel_err(tau[b].cpu().numpy(), tau_ref) <= TOL


def _oracle_all_four(A, B, C, K, Lt):
    A, B, C, K, Lt = [a.astype(np.float64) for a in (A, B, C, K, Lt)]
    T, n, _ = A.shape
    p = C.shape[1]
    PbX = _dense(O.system_response_item(A + B @ K), T, n)
    PbU = np.vstack([K[k] @ PbX[k * n:(k + 1) * n] for k in range(T)])
    PhX = _dense(O.observer_response_item(A, Lt, C)[0], T, n)
    PhY = np.zeros((T * n, T * p))
    for j in range(1, T):
        PhY[:, j * p:(j + 1) * p] = PhX[:, j * n:(j + 1) * n] @ Lt[j - 1]
    return O.assemble_output_feedback(A, PbX, PbU, PhX, PhY)


@pytest.mark.parametrize("n,T,m,p,nc,batch", [(24, 6, 2, 3, 3, 2),     # 2n = 48: fp32-FMA GEMMs
                                              (48, 7, 3, 4, 5, 1),     # 2n = 96: smallest tensor-core size
                                              (132, 5, 6, 6, 4, 2),    # ragged tiles
                                              (100, 4, 1, 1, 1, 1),    # single input / output / constraint
                                              (64, 9, 4, 20, 2, 1),    # wide observation, longer horizon (parity of the ping-pong)
                                              (300, 4, 6, 6, 6, 1)])   # C2 state size
def test_output_feedback_constraints_call(L, n, T, m, p, nc, batch):
    """ltv_scan_output_feedback_constraints: Phi^uw, Phi^ue of eq.(15) and the margins of eq.(12d) with both terms and
    rows on [z; v], against the oracle (assemble_output_feedback as printed + output_feedback_constraint_tightening)."""
    import torch

    items = [_gains(T, n, m, p, seed=11 * n + T + b) for b in range(batch)]
    A, B, C, K, Lt = [np.stack([it[q] for it in items]) for q in range(5)]
    rng = np.random.default_rng(n + 1)
    w = rng.uniform(0.1, 1.0, (batch, T, n)).astype(np.float32)
    f = rng.uniform(0.1, 1.0, (batch, T, p)).astype(np.float32)
    Hx = rng.normal(0.0, 1.0, (batch, T, nc, n)).astype(np.float32)
    Hu = rng.normal(0.0, 1.0, (batch, T, nc, m)).astype(np.float32)
    d = [torch.from_numpy(a).cuda() for a in (A, B, K, Lt, C, w, f, Hx, Hu)]
    uw, ue, sig = L.ltv_scan_output_feedback_constraints(*d)
    _, _, sig_only = L.ltv_scan_output_feedback_constraints(*d, want_inputs=False)
    uw2, ue2, none = L.ltv_scan_output_feedback_constraints(*d[:7])
    torch.cuda.synchronize()
    assert none is None and torch.equal(uw, uw2) and torch.equal(ue, ue2) and torch.equal(sig, sig_only)
    uw, ue, sig = uw.cpu().numpy(), ue.cpu().numpy(), sig.cpu().numpy()
    for b in range(batch):
        Pxw, Puw, Pxe, Pue = _oracle_all_four(A[b], B[b], C[b], K[b], Lt[b])
        ref_uw = np.stack([Puw[k * m:(k + 1) * m, j * n:(j + 1) * n] for j in range(T - 1) for k in range(j + 1, T)])
        ref_ue = np.stack([Pue[k * m:(k + 1) * m, j * p:(j + 1) * p] for j in range(T - 1) for k in range(j + 1, T)])
        assert O.rel_err(uw[b], ref_uw) <= TOL
        assert O.rel_err(ue[b], ref_ue) <= TOL
        assert np.all(ue[b, :T - 1] == 0.0)      # column j = 0: no measurement precedes step 0
        ref_sig = O.output_feedback_constraint_tightening(Pxw, Puw, Pxe, Pue, w[b], f[b], Hx[b], Hu[b])
        assert O.rel_err(sig[b], ref_sig) <= TOL
        assert np.all(sig[b, 0] == 0.0)


def test_output_feedback_constraints_identity_rows_equal_the_tube_call(L):
    """Identity state rows, no input part: the margins are the output-feedback tube of (12e) - the two device calls
    (forward structured scan + extraction vs backward sweep) must agree to rounding."""
    import torch

    n, T, m, p = 96, 6, 3, 4
    A, B, C, K, Lt = [a[None] for a in _gains(T, n, m, p, seed=5)]
    rng = np.random.default_rng(6)
    w = rng.uniform(0.1, 1.0, (1, T, n)).astype(np.float32)
    f = rng.uniform(0.1, 1.0, (1, T, p)).astype(np.float32)
    Hx = np.ascontiguousarray(np.broadcast_to(np.eye(n, dtype=np.float32), (1, T, n, n)))
    Hu = np.zeros((1, T, n, m), dtype=np.float32)
    d = [torch.from_numpy(a).cuda() for a in (A, B, K, Lt, C, w, f)]
    _, _, tau = L.ltv_scan_output_feedback_response(*d)
    _, _, sig = L.ltv_scan_output_feedback_constraints(*d, torch.from_numpy(Hx).cuda(), torch.from_numpy(Hu).cuda(),
                                                       want_inputs=False)
    torch.cuda.synchronize()
    assert O.rel_err(sig.cpu().numpy(), tau.cpu().numpy()) <= TOL


@pytest.mark.parametrize("route", [1, 2])
def test_output_feedback_response_single_step_horizon(L, route):
    """T = 1: no block exists, tau_0 = 0, nothing is written to the (empty) operator arrays - on both routes."""
    import torch

    n, m, p, batch = 96, 2, 3, 2
    A, B, C, K, Lt = [np.stack([q for q in x]) for x in zip(*[_gains(1, n, m, p, seed=5 + b) for b in range(batch)])]
    w = np.ones((batch, 1, n), np.float32); f = np.ones((batch, 1, p), np.float32)
    L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, route)
    try:
        xw, xe, tau = L.ltv_scan_output_feedback_response(*[torch.from_numpy(a).cuda() for a in (A, B, K, Lt, C, w, f)])
        torch.cuda.synchronize()
    finally:
        L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, 0)
    assert xw.shape[1] == 0 and bool(torch.all(tau == 0))


@pytest.mark.parametrize("route", [1, 2])
def test_output_feedback_response_without_phi_xe(L, route):
    """phi_xe_out = NULL: Phi^xw and the tube (which still contains the observation term) are unchanged - on both routes."""
    import torch

    n, T, m, p, batch = 132, 5, 3, 4, 2
    items = [_gains(T, n, m, p, seed=40 + b) for b in range(batch)]
    A, B, C, K, Lt = [np.stack([it[q] for it in items]) for q in range(5)]
    rng = np.random.default_rng(8)
    w = rng.uniform(0.1, 1.0, (batch, T, n)).astype(np.float32)
    f = rng.uniform(0.1, 1.0, (batch, T, p)).astype(np.float32)
    d = [torch.from_numpy(a).cuda() for a in (A, B, K, Lt, C, w, f)]
    L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, route)
    try:
        xw, xe, tau = L.ltv_scan_output_feedback_response(*d)
        xw2, xe2, tau2 = L.ltv_scan_output_feedback_response(*d, want_xe=False)
        torch.cuda.synchronize()
    finally:
        L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, 0)
    assert xe is not None and xe2 is None
    assert torch.equal(xw, xw2) and torch.equal(tau, tau2)      # deterministic: bitwise the same
