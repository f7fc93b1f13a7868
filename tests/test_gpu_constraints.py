"""GPU parity of ltv_scan_constraint_tightening (eq.(12d), SURVEY 8f NEXT-2 second form) against the pinned fp64
oracle, through the C-ABI binding; tolerance max|err| / max|ref| <= 1e-4 as for the rest of the path."""
import numpy as np
import pytest

from oracle import ltv_oracle as O
from workloads import config, dense_random, generate

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


def _rows(batch, T, nc, n, seed):
    return np.random.default_rng(seed).normal(0.0, 1.0, (batch, T, nc, n)).astype(np.float32)


def _gpu(L, A, w, Hc):
    import torch

    s = L.ltv_scan_constraint_tightening(*[torch.from_numpy(a).cuda() for a in (A, w, Hc)])
    torch.cuda.synchronize()
    return s.cpu().numpy()


@pytest.mark.parametrize("n,T,batch,nc", [(48, 6, 2, 3),      # fp32-FMA products
                                          (48, 16, 1, 8),     # C1 shape
                                          (128, 5, 3, 4),     # stack of 4 .. 16 rows: one ragged m-tile
                                          (132, 9, 2, 20),    # stack grows past 128 rows: two m-tiles, ragged k-block
                                          (300, 8, 2, 40),    # C2 width, 280 rows at the last step: CTA-pair tiles
                                          (164, 3, 1, 1),     # a single constraint row
                                          (600, 4, 2, 6)])
def test_constraint_tightening_dense(L, n, T, batch, nc):
    W = dense_random(batch, T, n, 1, seed=13 * n + nc, scale=0.4)
    Hc = _rows(batch, T, nc, n, seed=n + nc)
    got = _gpu(L, W.A, W.w, Hc)
    ref = O.constraint_tightening(W.A, W.w, Hc)
    assert got.shape == ref.shape == (batch, T, nc)
    assert np.all(got[:, 0] == 0.0)
    assert O.rel_err(got, ref) <= TOL
    for k in range(1, T):
        assert O.rel_err(got[:, k], ref[:, k]) <= TOL, k


@pytest.mark.parametrize("ci,T", [(0, 16), (1, 7), (2, 4)])
def test_constraint_tightening_mass_spring(L, ci, T):
    W = generate(config(ci, batch=2 if ci else 1, T=T))
    batch, _, n, _ = W.A.shape
    Hc = _rows(batch, T, 6, n, seed=50 + ci)
    assert O.rel_err(_gpu(L, W.A, W.w, Hc), O.constraint_tightening(W.A, W.w, Hc)) <= TOL


def test_identity_rows_reproduce_the_row2norm_tube_of_the_phi_call(L):
    """Two independent device paths (backward row sweep vs the Phi scan's fused two-norm epilogue) agree."""
    import torch

    n, T, batch = 132, 6, 2
    W = dense_random(batch, T, n, 1, seed=21, scale=0.4)
    Hc = np.ascontiguousarray(np.broadcast_to(np.eye(n, dtype=np.float32), (batch, T, n, n)))
    sig = _gpu(L, W.A, W.w, Hc)
    _, r = L.ltv_scan_system_response_tube(torch.from_numpy(W.A).cuda(), torch.from_numpy(W.w).cuda(), two_norm=True)
    torch.cuda.synchronize()
    assert O.rel_err(sig, r.cpu().numpy()) <= 1e-5


def test_T1_and_argument_errors(L):
    import torch

    A = torch.zeros((2, 1, 48, 48), device="cuda")
    s = L.ltv_scan_constraint_tightening(A, torch.ones((2, 1, 48), device="cuda"), torch.ones((2, 1, 3, 48), device="cuda"))
    torch.cuda.synchronize()
    assert s.shape == (2, 1, 3) and torch.all(s == 0)
    A = torch.zeros((1, 3, 48, 48), device="cuda")
    with pytest.raises(L.LtvError) as ei:
        L.ltv_scan_constraint_tightening(A, torch.ones((1, 3, 48), device="cuda"), torch.ones((1, 3, 2, 48), device="cuda"),
                                         workspace=torch.empty(256, device="cuda", dtype=torch.uint8))
    assert ei.value.status == 5
