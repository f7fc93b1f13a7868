"""Parity of the CUDA path (through the C-ABI binding) against the fp64 oracle, element by element, on the
same seeded inputs.  Tolerance: north_star's max|err| / max|ref| <= 1e-4 per output tensor (fp32 / 3xTF32);
integer-valued inputs must be reproduced EXACTLY (all partial sums < 2^24)."""
import numpy as np
import pytest

from oracle import ltv_oracle as O
from workloads import config, dense_random, generate, small_integer

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


def _dev(W):
    import torch

    return {k: torch.from_numpy(getattr(W, k)).cuda() for k in ("A", "B", "c", "x0", "u", "w", "g")}


def _col_perm(T):
    """oracle row-packed index of every block, in COLUMN_PACKED order"""
    return [O.packed_index(t, s) for s in range(T - 1) for t in range(s + 1, T)]


def _run_all(L, W, phi=True):
    import torch

    d = _dev(W)
    out = {}
    out["x"] = L.ltv_scan_rollout(d["A"], d["B"], d["c"], d["x0"], d["u"])
    if phi:
        out["phi"], out["r"] = L.ltv_scan_system_response_tube(d["A"], d["w"])
    out["lam"], out["grad_u"], out["grad_x0"] = L.ltv_scan_adjoint(d["A"], d["B"], d["g"])
    torch.cuda.synchronize()
    return {k: (None if v is None else v.cpu().numpy()) for k, v in out.items()}


def _ref_all(W, phi=True):
    ref = {"x": O.rollout(W.A, W.B, W.c, W.x0, W.u)}
    if phi:
        T = W.A.shape[1]
        perm = _col_perm(T)
        pr = [O.system_response_tube_item(W.A[b], W.w[b]) for b in range(W.A.shape[0])]
        ref["phi"] = np.stack([p[0][perm] for p in pr]) if perm else np.zeros((W.A.shape[0], 0) + W.A.shape[2:])
        ref["r"] = np.stack([p[1] for p in pr])
    ref["lam"], ref["grad_u"], ref["grad_x0"] = O.adjoint(W.A, W.B, W.g)
    return ref


def _check(got, ref, exact=False):
    errs = {}
    for k, r in ref.items():
        if r is None:
            continue
        assert got[k].shape == r.shape, k
        assert np.all(np.isfinite(got[k])), k
        if exact:
            assert np.array_equal(got[k].astype(np.float64), r), k
        errs[k] = O.rel_err(got[k], r)
        assert errs[k] <= TOL, (k, errs)
    return errs


# ------------------------------------------------------------------ the five configs (C2-C5 at reduced batch / T
# so the oracle finishes in seconds; full sizes are sampled in test_gpu_full_size.py)
@pytest.mark.parametrize("k,over", [
    (0, {}),                                   # C1 exactly: n=48 (fp32-FMA Phi path), T=16, batch 1
    (1, dict(batch=3, T=9)),                   # C2 shape: n=300 -> two 160-wide n-tiles, ragged m-tiles
    (1, dict(batch=2, T=32)),                  # C2 full horizon (5 levels)
    (2, dict(batch=2, T=6)),                   # C3: n=600
    (4, dict(batch=5, T=64)),                  # C5: n=180, long horizon
])
def test_configs(L, k, over):
    W = generate(config(k, **over))
    errs = _check(_run_all(L, W), _ref_all(W))
    print(config(k, **over)["name"], errs)


def test_config4_large_cloth_small_T(L):
    W = generate(config(3, batch=1, T=4))      # n=2400, m=12
    _check(_run_all(L, W), _ref_all(W))


@pytest.mark.parametrize("n,T,batch,m", [(128, 5, 2, 3), (256, 16, 2, 4), (96, 3, 1, 0), (100, 7, 3, 2),
                                         (32, 12, 4, 5), (4, 3, 2, 1), (420, 4, 1, 7)])
def test_dense_random(L, n, T, batch, m):
    """Dense Jacobians (PAPER.md:166 'dense matrix multiplications'): no kernel may rely on sparsity."""
    W = dense_random(batch, T, n, max(m, 1), seed=100 + n)
    if m == 0:
        W.B = None
        W.u = None
        d = _dev_partial(W)
        import torch

        x = L.ltv_scan_rollout(d["A"], None, d["c"], d["x0"], None)
        lam, gu, gx0 = L.ltv_scan_adjoint(d["A"], None, d["g"])
        phi, r = L.ltv_scan_system_response_tube(d["A"], d["w"])
        torch.cuda.synchronize()
        assert gu is None
        assert O.rel_err(x.cpu().numpy(), O.rollout(W.A, None, W.c, W.x0, None)) <= TOL
        rl, _, rgx = O.adjoint(W.A, None, W.g)
        assert O.rel_err(lam.cpu().numpy(), rl) <= TOL and O.rel_err(gx0.cpu().numpy(), rgx) <= TOL
        assert O.rel_err(r.cpu().numpy(), O.tube(W.A, W.w)) <= TOL
        return
    _check(_run_all(L, W), _ref_all(W))


def _dev_partial(W):
    import torch

    return {k: torch.from_numpy(getattr(W, k)).cuda() for k in ("A", "c", "x0", "w", "g")}


@pytest.mark.parametrize("n,T", [(64, 9), (160, 9), (288, 6)])
def test_integer_inputs_are_exact(L, n, T):
    """SURVEY 8c pin (vii): with small-integer data every product and partial sum is exactly representable, so
    fp32 FMA and the 3xTF32 split (hi carries everything, lo = 0) must match the fp64 oracle bit for bit."""
    W = small_integer(2, T, n, 3, seed=n + T)
    ref = _ref_all(W)
    assert max(np.abs(v).max() for v in ref.values()) < 2 ** 22
    _check(_run_all(L, W), ref, exact=True)


def test_edge_T1_and_T2(L):
    for T in (1, 2):
        W = dense_random(2, T, 128, 2, seed=T)
        got = _run_all(L, W)
        ref = _ref_all(W)
        _check(got, ref)
        assert np.all(got["r"][:, 0] == 0)


def test_null_optional_outputs_and_determinism(L):
    import torch

    W = dense_random(3, 10, 192, 4, seed=9)
    d = _dev(W)
    lam, gu, gx0 = L.ltv_scan_adjoint(d["A"], d["B"], d["g"], want_grad_x0=False)
    assert gx0 is None
    rl, rgu, _ = O.adjoint(W.A, W.B, W.g)
    assert O.rel_err(lam.cpu().numpy(), rl) <= TOL and O.rel_err(gu.cpu().numpy(), rgu) <= TOL
    p1, r1 = L.ltv_scan_system_response_tube(d["A"], d["w"])
    p2, r2 = L.ltv_scan_system_response_tube(d["A"], d["w"])
    torch.cuda.synchronize()
    assert torch.equal(p1, p2) and torch.equal(r1, r2)          # fixed-order tube reduction, no atomics


def test_inputs_not_modified_and_no_overrun(L):
    import torch

    W = dense_random(2, 6, 132, 3, seed=11)
    d = _dev(W)
    keep = {k: v.clone() for k, v in d.items()}
    batch, T, n, m = W.shape
    P = T * (T - 1) // 2
    guard = 1024
    phi = torch.full((batch * P * n * n + guard,), 7.0, device="cuda")
    r = torch.full((batch * T * n + guard,), 7.0, device="cuda")
    L.ltv_scan_system_response_tube(d["A"], d["w"], phi[:batch * P * n * n].view(batch, P, n, n),
                                    r[:batch * T * n].view(batch, T, n))
    L.ltv_scan_rollout(d["A"], d["B"], d["c"], d["x0"], d["u"])
    L.ltv_scan_adjoint(d["A"], d["B"], d["g"])
    torch.cuda.synchronize()
    assert torch.all(phi[-guard:] == 7.0) and torch.all(r[-guard:] == 7.0)
    for k in d:
        assert torch.equal(d[k], keep[k]), k


def test_pipeline_host_matches_device_calls(L):
    import torch

    W = generate(config(1, batch=2, T=6))
    batch, T, n, m = W.shape
    need = L.ltv_scan_workspace_bytes(L.LTV_OP_PIPELINE_HOST, batch, T, n, m)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    h = {k: torch.from_numpy(getattr(W, k)).pin_memory() for k in ("A", "B", "c", "x0", "u", "w", "g")}
    P = T * (T - 1) // 2
    phi_host = torch.empty((batch, P, n, n), dtype=torch.float32).pin_memory()
    outs = L.ltv_scan_pipeline_host(h["A"], h["B"], h["c"], h["x0"], h["u"], h["w"], h["g"], ws, phi_host=phi_host)
    got = dict(x=outs["x"].numpy(), r=outs["r"].numpy(), lam=outs["lam"].numpy(), grad_u=outs["grad_u"].numpy(),
               grad_x0=outs["grad_x0"].numpy(), phi=phi_host.numpy())
    _check(got, _ref_all(W))
    assert outs["phi_device_ptr"] != 0


@pytest.mark.gpu
def test_pipeline_host_chunked_and_without_phi(L):
    """batch 12 is uploaded and computed in chunks (4 + 4 + 4); w=None runs rollout + adjoint only."""
    import torch

    W = generate(config(0, batch=12, T=5))
    batch, T, n, m = W.shape
    ref = _ref_all(W)
    h = {k: torch.from_numpy(getattr(W, k)).pin_memory() for k in ("A", "B", "c", "x0", "u", "w", "g")}
    ws = torch.empty(L.ltv_scan_workspace_bytes(L.LTV_OP_PIPELINE_HOST, batch, T, n, m), dtype=torch.uint8, device="cuda")
    P = T * (T - 1) // 2
    phi_host = torch.empty((batch, P, n, n), dtype=torch.float32).pin_memory()
    outs = L.ltv_scan_pipeline_host(h["A"], h["B"], h["c"], h["x0"], h["u"], h["w"], h["g"], ws, phi_host=phi_host)
    _check(dict(x=outs["x"].numpy(), r=outs["r"].numpy(), lam=outs["lam"].numpy(), grad_u=outs["grad_u"].numpy(),
                grad_x0=outs["grad_x0"].numpy(), phi=phi_host.numpy()), ref)
    need = L.ltv_scan_workspace_bytes(L.LTV_OP_PIPELINE_HOST_NO_PHI, batch, T, n, m)
    assert 0 < need < ws.numel()
    ws2 = torch.empty(need, dtype=torch.uint8, device="cuda")
    o2 = L.ltv_scan_pipeline_host(h["A"], h["B"], h["c"], h["x0"], h["u"], None, h["g"], ws2)
    assert o2["r"] is None and o2["phi_device_ptr"] in (0, None)
    _check(dict(x=o2["x"].numpy(), lam=o2["lam"].numpy(), grad_u=o2["grad_u"].numpy(), grad_x0=o2["grad_x0"].numpy()),
           {k: ref[k] for k in ("x", "lam", "grad_u", "grad_x0")})


@pytest.mark.parametrize("cluster", [1, 2, 3, 5, 6, 7, 9, 10, 16])
def test_vector_scans_any_cluster_size(L, cluster):
    """Rollout and adjoint give the same answer for every cluster size the model may pick (ltv_set_option
    LTV_OPT_VECTOR_CLUSTER forces it): bands of 4-row multiples, last band blocks with fewer rows than m, clusters wider than 8."""
    import torch

    W = dense_random(2, 7, 640 if cluster == 16 else 300, 6, seed=40 + cluster)
    d = {k: torch.from_numpy(getattr(W, k)).cuda() for k in ("A", "B", "c", "x0", "u", "g")}
    L.ltv_set_option(L.LTV_OPT_VECTOR_CLUSTER, cluster)
    try:
        assert L.ltv_get_option(L.LTV_OPT_VECTOR_CLUSTER) == cluster
        x = L.ltv_scan_rollout(d["A"], d["B"], d["c"], d["x0"], d["u"])
        lam, gu, gx0 = L.ltv_scan_adjoint(d["A"], d["B"], d["g"])
        torch.cuda.synchronize()
    finally:
        L.ltv_set_option(L.LTV_OPT_VECTOR_CLUSTER, 0)
    rl, rgu, rgx = O.adjoint(W.A, W.B, W.g)
    _check(dict(x=x.cpu().numpy(), lam=lam.cpu().numpy(), grad_u=gu.cpu().numpy(), grad_x0=gx0.cpu().numpy()),
           dict(x=O.rollout(W.A, W.B, W.c, W.x0, W.u), lam=rl, grad_u=rgu, grad_x0=rgx))


@pytest.mark.parametrize("n,T,batch,m", [(644, 3, 2, 6),      # first size of the column-split (wide) rollout mode
                                         (1200, 4, 3, 12),    # 4-row chunks, 16-byte state exchange
                                         (4096, 3, 1, 6),     # 2-row chunks (4 rows exceed a ring stage)
                                         (8192, 2, 1, 3),     # maximum n: one row per chunk
                                         (180, 130, 2, 6),    # long horizon: many wraps of every ring / parity bit
                                         (36, 5, 150, 6)])    # more items than resident clusters, tiny n
def test_vector_scans_edge_sizes(L, n, T, batch, m):
    """Rollout + adjoint only (no Phi: the oracle's n^3 products would dominate) at the extremes of n, T, batch."""
    import torch

    W = dense_random(batch, T, n, m, seed=7 * n + T, scale=0.3)
    d = {k: torch.from_numpy(getattr(W, k)).cuda() for k in ("A", "B", "c", "x0", "u", "g")}
    x = L.ltv_scan_rollout(d["A"], d["B"], d["c"], d["x0"], d["u"])
    lam, gu, gx0 = L.ltv_scan_adjoint(d["A"], d["B"], d["g"])
    torch.cuda.synchronize()
    rl, rgu, rgx = O.adjoint(W.A, W.B, W.g)
    _check(dict(x=x.cpu().numpy(), lam=lam.cpu().numpy(), grad_u=gu.cpu().numpy(), grad_x0=gx0.cpu().numpy()),
           dict(x=O.rollout(W.A, W.B, W.c, W.x0, W.u), lam=rl, grad_u=rgu, grad_x0=rgx))


@pytest.mark.parametrize("n,T,batch", [(96, 4, 2),     # smallest tensor-core size: one 96-wide n-tile
                                       (164, 5, 1),    # two n-tiles, the second 4 columns wide
                                       (1000, 3, 1),   # K = 31.25 k-blocks: ragged last k-block
                                       (320, 20, 1),   # T-1 = 19: last segments ragged on every level
                                       (128, 3, 5)])   # T = 3: a single level-1 product per item
def test_phi_tube_shapes(L, n, T, batch):
    import torch

    W = dense_random(batch, T, n, 1, seed=3 * n + T, scale=0.4)
    A, w = torch.from_numpy(W.A).cuda(), torch.from_numpy(W.w).cuda()
    phi, r = L.ltv_scan_system_response_tube(A, w)
    torch.cuda.synchronize()
    ref = _ref_all(W)
    _check(dict(phi=phi.cpu().numpy(), r=r.cpu().numpy()), dict(phi=ref["phi"], r=ref["r"]))


@pytest.mark.parametrize("k,over", [(0, {}), (1, dict(batch=2, T=9)), (2, dict(batch=1, T=5))])
def test_row_two_norm_tube_configs(L, k, over):
    """flags = LTV_TUBE_ROW_2NORM: eq.(12e) as printed (row-wise two-norm, E_s = diag(w_s)); Phi itself is unchanged."""
    import torch

    W = generate(config(k, **over))
    A, w = torch.from_numpy(W.A).cuda(), torch.from_numpy(W.w).cuda()
    phi, r = L.ltv_scan_system_response_tube(A, w, two_norm=True)
    phi1, r1 = L.ltv_scan_system_response_tube(A, w)
    torch.cuda.synchronize()
    assert torch.equal(phi, phi1)
    ref = O.tube_row2norm(W.A, W.w)
    assert O.rel_err(r.cpu().numpy(), ref) <= TOL
    assert O.rel_err(r1.cpu().numpy(), O.tube(W.A, W.w)) <= TOL
    assert O.rel_err(r.cpu().numpy(), O.tube(W.A, W.w)) > 10 * TOL      # and it is not the box tube


@pytest.mark.parametrize("n,T,batch", [(164, 6, 2), (128, 3, 3), (420, 4, 1)])
def test_row_two_norm_tube_dense(L, n, T, batch):
    import torch

    W = dense_random(batch, T, n, 1, seed=11 * n + T, scale=0.4)
    phi, r = L.ltv_scan_system_response_tube(torch.from_numpy(W.A).cuda(), torch.from_numpy(W.w).cuda(), two_norm=True)
    torch.cuda.synchronize()
    assert O.rel_err(r.cpu().numpy(), O.tube_row2norm(W.A, W.w)) <= TOL


def _observer_inputs(batch, T, n, p, seed):
    rng = np.random.default_rng(seed)
    W = dense_random(batch, T, n, 1, seed=seed, scale=0.4)
    Lt = rng.normal(0.0, 0.3 / np.sqrt(p), (batch, T, n, p)).astype(np.float32)
    C = rng.normal(0.0, 1.0 / np.sqrt(n), (batch, T, p, n)).astype(np.float32)
    return W, Lt, C


@pytest.mark.parametrize("n,T,batch,p", [(48, 6, 2, 3),      # fp32-FMA path, nc = 52
                                         (128, 5, 2, 6),     # tensor-core path, nc = 136: second n-tile is PhiY only
                                         (300, 9, 2, 6),     # C2 shape: nc = 308 fits the padding of two 160-wide tiles
                                         (164, 4, 1, 32),    # widest gain block
                                         (132, 5, 2, 12),    # wide path (p > 8): transposed gains, two column groups
                                         (300, 4, 1, 20),    # wide path, three column groups (nc = 320)
                                         (100, 3, 3, 1)])
def test_observer_response(L, n, T, batch, p):
    """NEXT-1, eq.(14): PhiX over the closed-loop matrices A + Lt C, PhiY = PhiX Lt riding along as extra columns;
    the oracle multiplies on the RIGHT in the paper's order, the GPU runs the divide-and-conquer scan."""
    import torch

    W, Lt, C = _observer_inputs(batch, T, n, p, seed=5 * n + p)
    d = [torch.from_numpy(a).cuda() for a in (W.A, Lt, C, W.w)]
    phi, r = L.ltv_scan_observer_response(*d)
    torch.cuda.synchronize()
    nc = L.ltv_observer_row_floats(n, p)
    assert phi.shape == (batch, T * (T - 1) // 2, n, nc)
    phi = phi.cpu().numpy()
    X, Y = O.observer_response(W.A, Lt, C)
    perm = _col_perm(T)
    assert O.rel_err(phi[..., :n], X[:, perm]) <= TOL
    assert O.rel_err(phi[..., n:n + p], Y[:, perm]) <= TOL
    assert np.all(phi[..., n + p:] == 0.0)
    # tube of PhiX: the box-tube oracle applied to the closed-loop matrices (float64 Abar is not an fp32 input of
    # the GPU, so this check carries the rounding of forming Abar in fp32: still far inside TOL)
    Abar = W.A.astype(np.float64) + Lt.astype(np.float64) @ C.astype(np.float64)
    assert O.rel_err(r.cpu().numpy(), O.tube(Abar, W.w)) <= TOL


@pytest.mark.parametrize("n,T,batch,p", [(48, 6, 2, 3), (300, 9, 2, 6), (132, 5, 2, 12)])
def test_observer_response_shifted_gain(L, n, T, batch, p):
    """LTV_OBSERVER_SHIFTED_GAIN: PhiY(t,s) = PhiX(t,s) Lt_{s-1} (zero for s = 0), the Phihat^y of (12c)/(15) (DESIGN.md
    q20, q21); PhiX and the tube are unchanged.  SIMT, fused (p <= 8) and wide (p > 8) level-0 kernels."""
    import torch

    W, Lt, C = _observer_inputs(batch, T, n, p, seed=7 * n + p)
    d = [torch.from_numpy(a).cuda() for a in (W.A, Lt, C, W.w)]
    phi, r = L.ltv_scan_observer_response(*d, shifted_gain=True)
    phi_p, r_p = L.ltv_scan_observer_response(*d)
    torch.cuda.synchronize()
    assert torch.equal(phi[..., :n], phi_p[..., :n]) and torch.equal(r, r_p)
    phi = phi.cpu().numpy()
    X, Y = O.observer_response(W.A, Lt, C, shifted_gain=True)
    perm = _col_perm(T)
    assert O.rel_err(phi[..., :n], X[:, perm]) <= TOL
    assert O.rel_err(phi[..., n:n + p], Y[:, perm]) <= TOL
    assert np.all(phi[..., n + p:] == 0.0)
    assert np.all(phi[:, :T - 1, :, n:] == 0.0)          # column s = 0: blocks q = 0 .. T-2 of the column-packed order


def test_observer_zero_gain_is_the_open_loop_response(L):
    import torch

    W, Lt, C = _observer_inputs(2, 6, 132, 4, seed=3)
    A, w = torch.from_numpy(W.A).cuda(), torch.from_numpy(W.w).cuda()
    phi, r = L.ltv_scan_observer_response(A, torch.zeros_like(torch.from_numpy(Lt)).cuda(), torch.from_numpy(C).cuda(), w)
    phi0, r0 = L.ltv_scan_system_response_tube(A, w)
    torch.cuda.synchronize()
    assert torch.equal(phi[..., :132], phi0) and torch.equal(r, r0) and torch.all(phi[..., 132:] == 0)


def test_sharded_device_views_with_odd_item_size(L):
    """Device shards of a batch whose per-item sizes are not multiples of 4 floats (T m = 15, T p = 9): shard_arrays must
    hand the library 16-byte aligned tensors, and the shards must reproduce the whole batch bit for bit."""
    import torch

    from paper_2606_14188_b200.sharding import shard_arrays

    W = dense_random(5, 3, 36, 5, seed=91)
    d = {k: torch.from_numpy(getattr(W, k)).cuda() for k in ("A", "B", "c", "x0", "u", "g")}
    x = L.ltv_scan_rollout(d["A"], d["B"], d["c"], d["x0"], d["u"])
    lam, gu, _ = L.ltv_scan_adjoint(d["A"], d["B"], d["g"])
    xs, gus = [], []
    for rank in range(2):
        m = shard_arrays(d, rank, 2)
        assert all(v.data_ptr() % 16 == 0 for v in m.values())
        xs.append(L.ltv_scan_rollout(m["A"], m["B"], m["c"], m["x0"], m["u"]))
        gus.append(L.ltv_scan_adjoint(m["A"], m["B"], m["g"])[1])
    torch.cuda.synchronize()
    assert torch.equal(torch.cat(xs), x) and torch.equal(torch.cat(gus), gu)


@pytest.mark.parametrize("n,T,batch", [(48, 6, 2),       # fp32-FMA combine
                                       (132, 7, 3),      # tcgen05 combine, ragged k-block and m-tile
                                       (300, 4, 1)])
def test_phi_layouts_of_the_survey_boundary(L, n, T, batch):
    """phi_layout = ROW_PACKED (block index t(t-1)/2 + s, the oracle's own order: no permutation in the
    test) and SQUARE_GRID ([batch,T,T,n,n], only s < t written).  Both must hold exactly the COLUMN_PACKED result
    (the re-ordering is a copy) and match the oracle; r is the same in every layout."""
    import torch

    W = dense_random(batch, T, n, 1, seed=13 * n + T, scale=0.4)
    A, w = torch.from_numpy(W.A).cuda(), torch.from_numpy(W.w).cuda()
    P = T * (T - 1) // 2
    phi_c, r_c = L.ltv_scan_system_response_tube(A, w)
    phi_r, r_r = L.ltv_scan_system_response_tube(A, w, layout=L.LTV_PHI_ROW_PACKED)
    grid = torch.full((batch, T, T, n, n), 777.0, device="cuda")
    phi_g, r_g = L.ltv_scan_system_response_tube(A, w, phi_out=grid, layout=L.LTV_PHI_SQUARE_GRID)
    torch.cuda.synchronize()
    ref = O.system_response(W.A)                                # row-packed
    assert O.rel_err(phi_r.cpu().numpy(), ref) <= TOL
    assert torch.equal(r_c, r_r) and torch.equal(r_c, r_g)
    assert O.rel_err(r_c.cpu().numpy(), O.tube(W.A, W.w)) <= TOL
    g = phi_g.cpu().numpy()
    for t in range(T):
        for s in range(T):
            if s < t:
                assert L.ltv_phi_block_index_layout(T, t, s, L.LTV_PHI_SQUARE_GRID) == t * T + s
                assert L.ltv_phi_block_index_layout(T, t, s, L.LTV_PHI_ROW_PACKED) == O.packed_index(t, s)
                assert L.ltv_phi_block_index_layout(T, t, s, L.LTV_PHI_COLUMN_PACKED) == L.ltv_phi_block_index(T, t, s)
                assert np.array_equal(g[:, t, s], phi_c[:, L.ltv_phi_block_index(T, t, s)].cpu().numpy())
                assert np.array_equal(g[:, t, s], phi_r[:, O.packed_index(t, s)].cpu().numpy())
            else:
                assert np.all(g[:, t, s] == 777.0)               # untouched
    assert L.ltv_phi_block_index_layout(T, 0, 0, L.LTV_PHI_ROW_PACKED) == -1
    assert L.ltv_phi_block_index_layout(T, 1, 0, 7) == -1


def test_phi_layout_validation(L):
    import torch

    W = dense_random(1, 3, 48, 1, seed=5)
    A, w = torch.from_numpy(W.A).cuda(), torch.from_numpy(W.w).cuda()
    with pytest.raises(L.LtvError) as e:
        L.ltv_scan_system_response_tube(A, w, layout=3)
    assert e.value.status == 2
    ws = torch.empty(max(16, L.ltv_scan_workspace_bytes(L.LTV_OP_SYSTEM_RESPONSE_TUBE, 1, 3, 48, 0)), dtype=torch.uint8, device="cuda")
    with pytest.raises(L.LtvError) as e:      # the native workspace is too small for a re-ordered layout
        L.ltv_scan_system_response_tube(A, w, workspace=ws, layout=L.LTV_PHI_ROW_PACKED)
    assert e.value.status == 5


@pytest.mark.parametrize("n,T,batch,m", [(48, 16, 1, 6), (300, 9, 5, 6), (180, 20, 70, 6), (644, 3, 2, 4), (1200, 4, 3, 12),
                                         (180, 12, 64, 6), (300, 6, 32, 6), (180, 8, 32, 6)])   # the last three: few items of a
def test_rollout_adjoint_pair(L, n, T, batch, m):                                                # small system, side by side on half
                                                                                                 # the machine each (second rule)
    """ltv_scan_rollout_adjoint (both scans concurrently, half of the SMs each) against the oracle and the single calls."""
    import torch

    W = dense_random(batch, T, n, m, seed=3 * n + batch, scale=0.3)
    d = {k: torch.from_numpy(getattr(W, k)).cuda() for k in ("A", "B", "c", "x0", "u", "g")}
    for rep in range(2):                                   # twice: the cached side stream / events are reused
        x, lam, gu, gx0 = L.ltv_scan_rollout_adjoint(d["A"], d["B"], d["c"], d["x0"], d["u"], d["g"])
    x1 = L.ltv_scan_rollout(d["A"], d["B"], d["c"], d["x0"], d["u"])
    torch.cuda.synchronize()
    assert torch.equal(x, x1)
    rl, rgu, rgx = O.adjoint(W.A, W.B, W.g)
    _check(dict(x=x.cpu().numpy(), lam=lam.cpu().numpy(), grad_u=gu.cpu().numpy(), grad_x0=gx0.cpu().numpy()),
           dict(x=O.rollout(W.A, W.B, W.c, W.x0, W.u), lam=rl, grad_u=rgu, grad_x0=rgx))
    # optional outputs absent
    x2, lam2, gu2, gx2 = L.ltv_scan_rollout_adjoint(d["A"], None, d["c"], d["x0"], None, d["g"], want_grad_x0=False)
    torch.cuda.synchronize()
    assert gu2 is None and gx2 is None
    assert O.rel_err(x2.cpu().numpy(), O.rollout(W.A, None, W.c, W.x0, None)) <= TOL
    assert O.rel_err(lam2.cpu().numpy(), rl) <= TOL


@pytest.mark.parametrize("n,batch,cluster", [(1536, 48, 4), (2400, 16, 8), (2432, 8, 16)])
def test_vector_scans_many_ctas_large_n_repeatable(L, n, batch, cluster):
    """Regression test of the ring bug of round 2: big matrices on >= ~100 CTAs, more clusters than fit
    at once, both scans also on two streams at the same time.  With an odd shared-memory ring these shapes died with
    'unspecified launch failure' within 1-30 launches; now every repeat must reproduce the first result bit for bit and
    item 0 must match the oracle."""
    import torch

    T, m = 6, 12
    g = torch.Generator(device="cuda").manual_seed(n + batch)
    A = torch.randn((batch, T, n, n), device="cuda", generator=g) * (0.3 / n ** 0.5)
    A += torch.eye(n, device="cuda")
    B = torch.randn((batch, T, n, m), device="cuda", generator=g) * 0.1
    c = torch.randn((batch, T, n), device="cuda", generator=g) * 0.01
    x0 = torch.randn((batch, n), device="cuda", generator=g)
    u = torch.randn((batch, T, m), device="cuda", generator=g) * 0.1
    gg = torch.randn((batch, T, n), device="cuda", generator=g)
    side = torch.cuda.Stream()
    L.ltv_set_option(L.LTV_OPT_VECTOR_CLUSTER, cluster)
    try:
        first = None
        for rep in range(25):
            x = L.ltv_scan_rollout(A, B, c, x0, u)
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                lam, gu, gx0 = L.ltv_scan_adjoint(A, B, gg)
                lam_b, _, _ = L.ltv_scan_adjoint(A, B, gg)       # a second adjoint right behind: clusters of two launches overlap
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            got = (x, lam, gu, gx0)
            assert torch.equal(lam, lam_b)
            if first is None:
                first = [t.clone() for t in got]
            else:
                for a, b in zip(first, got):
                    assert torch.equal(a, b)
    finally:
        L.ltv_set_option(L.LTV_OPT_VECTOR_CLUSTER, 0)
    A0, B0 = A[0].cpu().numpy(), B[0].cpu().numpy()
    rl, rgu, rgx = O.adjoint_item(A0, B0, gg[0].cpu().numpy())
    _check(dict(x=first[0][0].cpu().numpy(), lam=first[1][0].cpu().numpy(), grad_u=first[2][0].cpu().numpy(), grad_x0=first[3][0].cpu().numpy()),
           dict(x=O.rollout_item(A0, B0, c[0].cpu().numpy(), x0[0].cpu().numpy(), u[0].cpu().numpy()), lam=rl, grad_u=rgu, grad_x0=rgx))


def _all_vs_oracle(L, W, two_norm=False, exact=False, layout=None):
    import torch

    d = {k: torch.from_numpy(getattr(W, k)).cuda() for k in ("A", "B", "c", "x0", "u", "w", "g")}
    kw = {} if layout is None else dict(layout=layout)
    o = L.ltv_scan_all(d["A"], d["B"], d["c"], d["x0"], d["u"], d["w"], d["g"], two_norm=two_norm, **kw)
    torch.cuda.synchronize()
    T = W.A.shape[1]
    rl, rgu, rgx = O.adjoint(W.A, W.B, W.g)
    phi_ref = O.system_response(W.A)
    if layout is None:
        phi_ref = phi_ref[:, _col_perm(T)]
    ref = dict(x=O.rollout(W.A, W.B, W.c, W.x0, W.u), phi=phi_ref,
               r=(O.tube_row2norm(W.A, W.w) if two_norm else O.tube(W.A, W.w)), lam=rl, grad_u=rgu, grad_x0=rgx)
    return _check({k: v.cpu().numpy() for k, v in o.items() if v is not None}, ref, exact=exact)


@pytest.mark.parametrize("n,T,batch,m", [(48, 16, 1, 6),      # C1 exactly (shape)
                                         (48, 16, 20, 6),     # more clusters than fit at once
                                         (64, 8, 3, 5),       # largest n, two k groups
                                         (32, 20, 2, 3),      # T - 1 = 19 columns over 15 column CTAs (two slots)
                                         (4, 3, 2, 1), (16, 2, 1, 2), (36, 5, 4, 0), (60, 9, 2, 12)])
def test_scan_all_fused_small(L, n, T, batch, m):
    """ltv_scan_all on shapes that take the single-launch route, against the oracle (both tube forms)."""
    assert L.ltv_scan_all_is_fused(batch, T, n, m)
    W = dense_random(batch, T, n, max(m, 1), seed=17 * n + T, scale=0.4)
    if m == 0:
        import torch

        d = {k: torch.from_numpy(getattr(W, k)).cuda() for k in ("A", "c", "x0", "w", "g")}
        o = L.ltv_scan_all(d["A"], None, d["c"], d["x0"], None, d["w"], d["g"])
        torch.cuda.synchronize()
        assert o["grad_u"] is None
        assert O.rel_err(o["x"].cpu().numpy(), O.rollout(W.A, None, W.c, W.x0, None)) <= TOL
        assert O.rel_err(o["r"].cpu().numpy(), O.tube(W.A, W.w)) <= TOL
        assert O.rel_err(o["phi"].cpu().numpy(), O.system_response(W.A)[:, _col_perm(T)]) <= TOL
        rl, _, rgx = O.adjoint(W.A, None, W.g)
        assert O.rel_err(o["lam"].cpu().numpy(), rl) <= TOL and O.rel_err(o["grad_x0"].cpu().numpy(), rgx) <= TOL
        return
    _all_vs_oracle(L, W)
    _all_vs_oracle(L, W, two_norm=True)


def test_scan_all_config1_and_integer_exact(L):
    """BASELINE.json configs[0] through the single launch; small-integer inputs must come out bit-exact."""
    from workloads import small_integer

    W = generate(config(0))
    assert L.ltv_scan_all_is_fused(*W.shape)
    print("C1 fused", _all_vs_oracle(L, W))
    _all_vs_oracle(L, small_integer(2, 9, 48, 3, seed=12), exact=True)


def test_scan_all_generic_route_and_layouts(L):
    """Shapes that do not fit the single launch go through ltv_scan_rollout_adjoint + ltv_scan_system_response_tube;
    a non-native layout forces the generic route even for a small problem."""
    assert not L.ltv_scan_all_is_fused(2, 5, 132, 3)
    assert not L.ltv_scan_all_is_fused(1, 64, 64, 3)          # A does not fit one SM's shared memory
    _all_vs_oracle(L, dense_random(2, 5, 132, 3, seed=77, scale=0.4))
    assert not L.ltv_scan_all_is_fused(2, 6, 48, 3, L.LTV_PHI_ROW_PACKED)
    _all_vs_oracle(L, dense_random(2, 6, 48, 3, seed=78, scale=0.4), layout=L.LTV_PHI_ROW_PACKED)
