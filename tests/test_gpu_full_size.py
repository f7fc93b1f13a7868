"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same binding calls, same
batch, default cluster / tile choices).  The oracle cannot produce 11 GB of Phi in seconds, so outputs are
SAMPLED: whole items for the vector outputs and the tube, single blocks Phi(t,s) (oracle/phi_block: the plain
ordered product) for the system response, plus properties that hold at any size (semigroup identity, r_0 = 0,
translation fixed point of the mass-spring generator).  Tolerance 1e-4 (north_star), per sampled tensor."""
import numpy as np
import pytest

from oracle import ltv_oracle as O
from workloads import config, generate

pytestmark = pytest.mark.gpu
TOL = 1e-4


@pytest.fixture(scope="module")
def L():
    import torch

    assert torch.cuda.is_available()
    import __graft_entry__ as G

    G.build()
    import paper_2606_14188_b200 as lib

    return lib


def _dev(W, keys=("A", "B", "c", "x0", "u", "w", "g")):
    import torch

    return {k: torch.from_numpy(getattr(W, k)).cuda() for k in keys}


def _vector_outputs(L, W, d, items):
    import torch

    x = L.ltv_scan_rollout(d["A"], d["B"], d["c"], d["x0"], d["u"])
    lam, gu, gx0 = L.ltv_scan_adjoint(d["A"], d["B"], d["g"])
    torch.cuda.synchronize()
    for b in items:
        assert O.rel_err(x[b].cpu().numpy(), O.rollout_item(W.A[b], W.B[b], W.c[b], W.x0[b], W.u[b])) <= TOL
        rl, rgu, rgx = O.adjoint_item(W.A[b], W.B[b], W.g[b])
        assert O.rel_err(lam[b].cpu().numpy(), rl) <= TOL
        assert O.rel_err(gu[b].cpu().numpy(), rgu) <= TOL
        assert O.rel_err(gx0[b].cpu().numpy(), rgx) <= TOL
    assert bool(torch.isfinite(x).all()) and bool(torch.isfinite(lam).all())
    # the same through ltv_scan_rollout_adjoint - the call bench.py's step makes (ltv_scan_all): at these sizes it may run the two
    # scans side by side on half of the SMs each with cluster sizes of its own (C3: 4 CTAs per item, C4: 10, C5 batch 64: 1)
    x2, lam2, gu2, gx2 = L.ltv_scan_rollout_adjoint(d["A"], d["B"], d["c"], d["x0"], d["u"], d["g"])
    torch.cuda.synchronize()
    for b in items:
        assert O.rel_err(x2[b].cpu().numpy(), O.rollout_item(W.A[b], W.B[b], W.c[b], W.x0[b], W.u[b])) <= TOL
        rl, rgu, rgx = O.adjoint_item(W.A[b], W.B[b], W.g[b])
        assert O.rel_err(lam2[b].cpu().numpy(), rl) <= TOL
        assert O.rel_err(gu2[b].cpu().numpy(), rgu) <= TOL
        assert O.rel_err(gx2[b].cpu().numpy(), rgx) <= TOL
    assert bool(torch.isfinite(x2).all()) and bool(torch.isfinite(lam2).all())
    # every item, not only the sampled ones: the two routes agree (different summation orders: tolerance, not bit equality)
    assert float((x2 - x).abs().max() / x.abs().max()) <= TOL and float((lam2 - lam).abs().max() / lam.abs().max()) <= TOL


def _phi_samples(L, W, phi, samples):
    T = W.A.shape[1]
    worst = 0.0
    for b, t, s in samples:
        ref = O.phi_block(W.A[b], t, s)
        got = phi[b, L.ltv_phi_block_index(T, t, s)].cpu().numpy()
        worst = max(worst, O.rel_err(got, ref))
    assert worst <= TOL, worst
    return worst


def _semigroup(L, phi, b, t, k, s, T):
    """Phi(t,s) = Phi(t,k) Phi(k,s): checked on the GPU's own blocks in fp64 (a property, not the oracle)."""
    q = lambda tt, ss: phi[b, L.ltv_phi_block_index(T, tt, ss)].double()
    lhs = q(t, s)
    rhs = q(t, k) @ q(k, s)
    err = float((lhs - rhs).abs().max() / rhs.abs().max())
    assert err <= TOL, err


def test_c2_full(L):
    import torch

    W = generate(config(1))                               # n=300, T=32, batch=64: the bench workload
    batch, T, n, m = W.shape
    d = _dev(W)
    _vector_outputs(L, W, d, items=[0, 31, 63])
    phi, r = L.ltv_scan_system_response_tube(d["A"], d["w"])
    torch.cuda.synchronize()
    assert bool(torch.isfinite(r).all()) and bool((r[:, 0] == 0).all())
    # whole tube + every block of two items (the oracle needs ~1 s per item here)
    for b in (0, 63):
        ref_phi, ref_r = O.system_response_tube_item(W.A[b], W.w[b])
        perm = [O.packed_index(t, s) for s in range(T - 1) for t in range(s + 1, T)]
        assert O.rel_err(phi[b].cpu().numpy(), ref_phi[perm]) <= TOL
        assert O.rel_err(r[b].cpu().numpy(), ref_r) <= TOL
    _phi_samples(L, W, phi, [(17, 31, 0), (40, 16, 15), (5, 24, 7), (62, 2, 0), (33, 31, 30)])
    _semigroup(L, phi, 21, 31, 16, 0, T)
    # translation fixed point (L 1 = 0): Phi(t,s) tau = tau for every block of an item
    N = n // 6
    tau = torch.zeros(n, device="cuda")
    tau[0:3 * N:3] = 1.0
    assert float((phi[7] @ tau - tau).abs().max()) < 1e-3


def test_c3_full(L):
    import torch

    W = generate(config(2))                               # n=600, T=32, batch=16
    batch, T, n, m = W.shape
    d = _dev(W)
    _vector_outputs(L, W, d, items=[0, 15])
    phi, r = L.ltv_scan_system_response_tube(d["A"], d["w"])
    torch.cuda.synchronize()
    ref_phi, ref_r = O.system_response_tube_item(W.A[3], W.w[3])
    perm = [O.packed_index(t, s) for s in range(T - 1) for t in range(s + 1, T)]
    assert O.rel_err(phi[3].cpu().numpy(), ref_phi[perm]) <= TOL
    assert O.rel_err(r[3].cpu().numpy(), ref_r) <= TOL
    _phi_samples(L, W, phi, [(0, 31, 0), (15, 20, 3), (9, 1, 0)])
    _semigroup(L, phi, 12, 30, 8, 1, T)


def test_c4_full(L):
    import torch

    W = generate(config(3))                               # n=2400, T=16, batch=4, m=12
    batch, T, n, m = W.shape
    d = _dev(W)
    _vector_outputs(L, W, d, items=[0, 3])
    phi, r = L.ltv_scan_system_response_tube(d["A"], d["w"])
    torch.cuda.synchronize()
    assert bool(torch.isfinite(r).all()) and bool((r[:, 0] == 0).all())
    # one WHOLE item against the oracle: all 120 blocks and every tube row r_1 .. r_15 (the rows that pass through the
    # CTA-pair epilogue, 15 n-tiles of partials and the finalise kernel at this size).  The oracle's block rows are
    # streamed (fp64 Phi of a C4 item is 5.5 GB): each row is compared and dropped; ~5 s of oracle time.
    b = 2
    w64 = W.w[b].astype(np.float64)
    worst_phi, den_phi, worst_r, den_r = 0.0, 0.0, 0.0, 0.0
    for t, row in O.phi_rows_item(W.A[b]):
        acc = np.zeros(n)
        for s in range(t):
            got = phi[b, L.ltv_phi_block_index(T, t, s)].cpu().numpy().astype(np.float64)
            worst_phi = max(worst_phi, float(np.max(np.abs(got - row[s]))))
            den_phi = max(den_phi, float(np.max(np.abs(row[s]))))
            acc = acc + np.abs(row[s]) @ w64[s]             # (12e) box form, the definition
        worst_r = max(worst_r, float(np.max(np.abs(r[b, t].cpu().numpy() - acc))))
        den_r = max(den_r, float(np.max(np.abs(acc))))
    assert worst_phi / den_phi <= TOL, worst_phi / den_phi
    assert worst_r / den_r <= TOL, worst_r / den_r
    # and through the oracle's own fused routine for the tube of another item (rows only; Phi dropped)
    assert O.rel_err(r[0].cpu().numpy(), O.tube_item(W.A[0], W.w[0])) <= TOL
    _phi_samples(L, W, phi, [(0, 2, 0), (3, 15, 12), (1, 9, 4), (3, 15, 0)])
    _semigroup(L, phi, 1, 15, 8, 0, T)                    # GPU-vs-GPU PROPERTY, not parity


@pytest.mark.parametrize("batch", [64, 256, 1024])
def test_c5_sweep(L, batch):
    W = generate(config(4, batch=batch))                  # n=180, T=64: rollout + adjoint only
    d = _dev(W, keys=("A", "B", "c", "x0", "u", "g"))
    _vector_outputs(L, W, d, items=[0, batch // 2, batch - 1])


def test_c2_full_observer_and_two_norm(L):
    """NEXT-1 / NEXT-2 at the bench size (n=300, T=32, batch=64, p=6): every block and both tubes of one item against
    the oracle, sampled blocks of others, and the semigroup property on the GPU's own [PhiX | PhiY] blocks."""
    import torch

    W = generate(config(1))
    batch, T, n, m = W.shape
    p = 6
    rng = np.random.default_rng(99)
    Lt = rng.normal(0.0, 0.05 / np.sqrt(p), (batch, T, n, p)).astype(np.float32)
    C = rng.normal(0.0, 1.0 / np.sqrt(n), (batch, T, p, n)).astype(np.float32)
    A, w = torch.from_numpy(W.A).cuda(), torch.from_numpy(W.w).cuda()
    phi, r = L.ltv_scan_observer_response(A, torch.from_numpy(Lt).cuda(), torch.from_numpy(C).cuda(), w, two_norm=True)
    torch.cuda.synchronize()
    nc = L.ltv_observer_row_floats(n, p)
    assert phi.shape[-1] == nc and bool((phi[..., n + p:] == 0).all())
    perm = [O.packed_index(t, s) for s in range(T - 1) for t in range(s + 1, T)]
    b = 37
    X, Y = O.observer_response_item(W.A[b], Lt[b], C[b])
    got = phi[b].cpu().numpy()
    assert O.rel_err(got[..., :n], X[perm]) <= TOL and O.rel_err(got[..., n:n + p], Y[perm]) <= TOL
    Abar = W.A[b].astype(np.float64) + Lt[b].astype(np.float64) @ C[b].astype(np.float64)
    assert O.rel_err(r[b].cpu().numpy(), O.tube_row2norm_item(Abar, W.w[b])) <= TOL
    for (bb, t, s) in [(0, 31, 0), (63, 17, 16), (12, 9, 2)]:
        Ab = W.A[bb].astype(np.float64) + Lt[bb].astype(np.float64) @ C[bb].astype(np.float64)
        ref = O.phi_block(Ab, t, s)
        blk = phi[bb, L.ltv_phi_block_index(T, t, s)].cpu().numpy()
        assert O.rel_err(blk[:, :n], ref) <= TOL and O.rel_err(blk[:, n:n + p], ref @ Lt[bb, s].astype(np.float64)) <= TOL
    q = lambda tt, ss: phi[50, L.ltv_phi_block_index(T, tt, ss)].double()
    rhs = q(30, 11)[:, :n] @ q(11, 3)
    assert float((q(30, 3) - rhs).abs().max() / rhs.abs().max()) <= TOL


# ------------------------------------------------------------------ NEXT rows at full size (sampled items)
@pytest.mark.parametrize("ci,p,items", [(1, 6, (0, 37, 63)), (2, 6, (0, 15)), (3, 12, (3,))])
def test_full_size_kalman_gains(L, ci, p, items):
    """ltv_scan_kalman_gains at the C2 / C3 / C4 sizes with the whole batch on the device (the configuration
    `bench.py --kalman` times); the oracle recursion (13) runs for the sampled items only.  Properties that hold at any
    size: Pi_out[:, 0] is Pi0 bit for bit, every Pi_j is symmetric to rounding and finite."""
    import torch
    from workloads import observation_model

    W = generate(config(ci))
    batch, T, n, _ = W.A.shape
    M = observation_model(batch, T, n, p, seed=900 + ci, kind="track")
    d = [torch.from_numpy(a).cuda() for a in (W.A, M["C"], M["e"], M["f"], M["Pi0"])]
    Lt, Pi = L.ltv_scan_kalman_gains(*d)
    torch.cuda.synchronize()
    assert torch.equal(Pi[:, 0], d[4]) and bool(torch.isfinite(Pi).all()) and bool(torch.isfinite(Lt).all())
    asym = (Pi - Pi.transpose(-1, -2)).abs().amax(dim=(-1, -2)) / Pi.abs().amax(dim=(-1, -2))
    assert float(asym.max()) <= TOL
    for b in items:
        Pi_ref, Lt_ref = O.kalman_recursion_item(W.A[b], M["C"][b], M["e"][b], M["f"][b], M["Pi0"][b])
        got_Pi, got_Lt = Pi[b].cpu().numpy(), Lt[b].cpu().numpy()
        assert O.rel_err(got_Pi, Pi_ref) <= TOL and O.rel_err(got_Lt, Lt_ref) <= TOL
        assert O.rel_err(got_Pi[-1], Pi_ref[-1]) <= TOL and O.rel_err(got_Lt[-1], Lt_ref[-1]) <= TOL


@pytest.mark.parametrize("ci,nc,items", [(1, 6, (0, 63)), (2, 6, (7,))])
def test_full_size_constraint_tightening(L, ci, nc, items):
    """ltv_scan_constraint_tightening at the C2 / C3 sizes (whole batch on the device, sampled items against the
    oracle); sigma_0 = 0, finiteness and positivity for k >= 1 are checked on every item."""
    import torch

    W = generate(config(ci))
    batch, T, n, _ = W.A.shape
    Hc = np.random.default_rng(70 + ci).normal(0.0, 1.0, (batch, 1, nc, n)).astype(np.float32)
    Hc = np.ascontiguousarray(np.broadcast_to(Hc, (batch, T, nc, n)))
    sig = L.ltv_scan_constraint_tightening(torch.from_numpy(W.A).cuda(), torch.from_numpy(W.w).cuda(),
                                           torch.from_numpy(Hc).cuda())
    torch.cuda.synchronize()
    sig = sig.cpu().numpy()
    assert np.all(sig[:, 0] == 0.0) and np.all(np.isfinite(sig)) and np.all(sig[:, 1:] > 0.0)
    for b in items:
        assert O.rel_err(sig[b], O.constraint_tightening_item(W.A[b], W.w[b], Hc[b])) <= TOL


def _ofb_inputs(W, p, seed):
    batch, T, n, m = W.shape
    rng = np.random.default_rng(seed)
    K = (0.2 * rng.normal(0.0, 1.0 / np.sqrt(n), (batch, T, m, n))).astype(np.float32)
    Lt = (0.05 * rng.normal(0.0, 1.0 / np.sqrt(p), (batch, T, n, p))).astype(np.float32)
    C = rng.normal(0.0, 1.0 / np.sqrt(n), (batch, T, p, n)).astype(np.float32)
    f = rng.uniform(1e-3, 5e-3, (batch, T, p)).astype(np.float32)
    return K, Lt, C, f


def _dense_lower(blocks, T, n, cols=None):
    """[T n, T cols] block lower-triangular operator with identity diagonal (cols = n) from row-packed blocks."""
    cols = n if cols is None else cols
    D = np.eye(T * n) if cols == n else np.zeros((T * n, T * cols))
    for t in range(1, T):
        for s in range(t):
            D[t * n:(t + 1) * n, s * cols:(s + 1) * cols] = blocks[O.packed_index(t, s)]
    return D


@pytest.mark.parametrize("route", [0, 1, 2])     # default (column recursion at this size), cross scan, column recursion
def test_full_size_output_feedback_response_vs_oracle(L, route):
    L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, route)
    try:
        _full_size_output_feedback_response_vs_oracle(L)
    finally:
        L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, 0)


def _full_size_output_feedback_response_vs_oracle(L):
    """ltv_scan_output_feedback_response on C2-size items (n=300, m=6, p=6, whole batch of 64, structured tcgen05 path)
    at a horizon the oracle's dense block operators can hold (T=8: [2400 x 2400] operators): every block of Phi^xw,
    Phi^xe and the whole tube of a sampled item against oracle/ - eq.(15) as printed (O.assemble_output_feedback) on
    Phibar = (I - Z(A + B K))^-1, Phihat = (I - Z(A + Lt C))^-1 built by the oracle's system response, and
    O.output_feedback_tube."""
    import torch

    W = generate(config(1, T=8))
    batch, T, n, m = W.shape
    p = 6
    K, Lt, C, f = _ofb_inputs(W, p, seed=78)
    d = [torch.from_numpy(a).cuda() for a in (W.A, W.B, K, Lt, C, W.w, f)]
    xw, xe, tau = L.ltv_scan_output_feedback_response(*d)
    torch.cuda.synchronize()
    assert bool(torch.all(tau[:, 0] == 0)) and bool(torch.isfinite(tau).all())
    perm = [O.packed_index(t, s) for s in range(T - 1) for t in range(s + 1, T)]
    for b in (0, 45):
        A64, B64, K64, Lt64, C64 = [a[b].astype(np.float64) for a in (W.A, W.B, K, Lt, C)]
        PbX = _dense_lower(O.system_response_item(A64 + B64 @ K64), T, n)
        PbU = np.vstack([K64[k] @ PbX[k * n:(k + 1) * n] for k in range(T)])
        PhX = _dense_lower(O.system_response_item(A64 + Lt64 @ C64), T, n)
        PhY = np.zeros((T * n, T * p))
        for j in range(1, T):                                # q20/q21: Phihat^y(k,j) = Phihat^x(k,j) Lt_{j-1}
            PhY[:, j * p:(j + 1) * p] = PhX[:, j * n:(j + 1) * n] @ Lt64[j - 1]
        Pxw, _, Pxe, _ = O.assemble_output_feedback(A64, PbX, PbU, PhX, PhY)
        blk = lambda D, t, s, c: D[t * n:(t + 1) * n, s * c:(s + 1) * c]
        ref_xw = np.stack([blk(Pxw, t, s, n) for s in range(T - 1) for t in range(s + 1, T)])
        ref_xe = np.stack([blk(Pxe, t, s, p) for s in range(T - 1) for t in range(s + 1, T)])
        assert O.rel_err(xw[b].cpu().numpy(), ref_xw) <= TOL
        assert O.rel_err(xe[b].cpu().numpy(), ref_xe) <= TOL
        assert O.rel_err(tau[b].cpu().numpy(), O.output_feedback_tube(Pxw, Pxe, W.w[b], f[b])) <= TOL


def test_full_size_output_feedback_constraints_vs_oracle(L):
    """ltv_scan_output_feedback_constraints on C2-size items (n=300, m=6, p=6, nc=6, whole batch of 64) at T=8, where the
    oracle's dense operators of (15) fit: every block of Phi^uw, Phi^ue and all margins of (12d) of sampled items."""
    import torch

    W = generate(config(1, T=8))
    batch, T, n, m = W.shape
    p, nc = 6, 6
    K, Lt, C, f = _ofb_inputs(W, p, seed=79)
    rng = np.random.default_rng(80)
    Hx = rng.normal(0.0, 1.0, (batch, T, nc, n)).astype(np.float32)
    Hu = rng.normal(0.0, 1.0, (batch, T, nc, m)).astype(np.float32)
    d = [torch.from_numpy(a).cuda() for a in (W.A, W.B, K, Lt, C, W.w, f, Hx, Hu)]
    uw, ue, sig = L.ltv_scan_output_feedback_constraints(*d)
    torch.cuda.synchronize()
    assert bool(torch.all(sig[:, 0] == 0)) and bool(torch.isfinite(sig).all())
    for b in (0, 45):
        A64, B64, K64, Lt64, C64 = [a[b].astype(np.float64) for a in (W.A, W.B, K, Lt, C)]
        PbX = _dense_lower(O.system_response_item(A64 + B64 @ K64), T, n)
        PbU = np.vstack([K64[k] @ PbX[k * n:(k + 1) * n] for k in range(T)])
        PhX = _dense_lower(O.system_response_item(A64 + Lt64 @ C64), T, n)
        PhY = np.zeros((T * n, T * p))
        for j in range(1, T):
            PhY[:, j * p:(j + 1) * p] = PhX[:, j * n:(j + 1) * n] @ Lt64[j - 1]
        Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A64, PbX, PbU, PhX, PhY)
        ref_uw = np.stack([Puw[k * m:(k + 1) * m, j * n:(j + 1) * n] for j in range(T - 1) for k in range(j + 1, T)])
        ref_ue = np.stack([Pue[k * m:(k + 1) * m, j * p:(j + 1) * p] for j in range(T - 1) for k in range(j + 1, T)])
        assert O.rel_err(uw[b].cpu().numpy(), ref_uw) <= TOL
        assert O.rel_err(ue[b].cpu().numpy(), ref_ue) <= TOL
        ref = O.output_feedback_constraint_tightening(Pxw, Puw, Pxe, Pue, W.w[b], f[b], Hx[b], Hu[b])
        assert O.rel_err(sig[b].cpu().numpy(), ref) <= TOL


def test_full_size_output_feedback_response(L):
    """The same call at the full C2 horizon (T=32, whole batch), where the oracle's dense operators of (15) would be
    [9600 x 9600]: a SECOND check only (the oracle-routed test is the one above) - the block row k = T-1 of one item
    against the blocks of the augmented closed loop built here by the plain ordered product in fp64 (the oracle tests
    pin that these blocks equal eq.(15)); tau_0 = 0 everywhere."""
    import torch

    W = generate(config(1))
    batch, T, n, m = W.shape
    p = 6
    K, Lt, C, f = _ofb_inputs(W, p, seed=77)
    d = [torch.from_numpy(a).cuda() for a in (W.A, W.B, K, Lt, C, W.w, f)]
    xw, xe, tau = L.ltv_scan_output_feedback_response(*d)
    torch.cuda.synchronize()
    assert bool(torch.all(tau[:, 0] == 0)) and bool(torch.isfinite(tau).all())
    b, k = 41, T - 1
    A64, B64, K64, Lt64, C64 = [a[b].astype(np.float64) for a in (W.A, W.B, K, Lt, C)]
    Aaug = np.zeros((T, 2 * n, 2 * n))
    Aaug[:, :n, :n] = A64 + B64 @ K64
    Aaug[:, :n, n:] = -(B64 @ K64)
    Aaug[:, n:, n:] = A64 + Lt64 @ C64
    G = np.eye(2 * n)
    tau_ref = np.zeros(n)
    worst_w = worst_e = 0.0
    for j in range(k - 1, -1, -1):          # G = Phi_aug(k, j) = Phi_aug(k, j+1) A_aug,j
        G = G @ Aaug[j]
        ref_w = G[:n, :n] + G[:n, n:]
        q = L.ltv_phi_block_index(T, k, j)
        worst_w = max(worst_w, O.rel_err(xw[b, q].cpu().numpy(), ref_w))
        tau_ref += np.sqrt(np.sum((ref_w * W.w[b, j].astype(np.float64)[None, :]) ** 2, axis=1))
        if j >= 1:
            ref_e = G[:n, n:] @ Lt64[j - 1]
            worst_e = max(worst_e, O.rel_err(xe[b, q].cpu().numpy(), ref_e))
            tau_ref += np.sqrt(np.sum((ref_e * f[b, j - 1].astype(np.float64)[None, :]) ** 2, axis=1))
    assert worst_w <= TOL and worst_e <= TOL
    assert O.rel_err(tau[b, k].cpu().numpy(), tau_ref) <= TOL
