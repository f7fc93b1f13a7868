"""ltv_scan_system_response_tube_static: the system response + tube call for callers that cannot allocate device memory
(its scratch is a fixed 32 MiB device array inside the library) against the regular call with a caller-provided workspace.
Collected LAST on purpose (file name): the suite runs with `pytest -x`, a failure here must not hide other tests.
Passes alone in a fresh process and after the other tests (it shares no state with them but the library)."""
import pytest

from workloads import config, dense_random, generate

pytestmark = pytest.mark.gpu
TOL = 1e-4   # max|a - b| / max|b| per output tensor: the tolerance of the other parity tests (here the kernels are the same)


@pytest.fixture(scope="module")
def L():
    import torch

    assert torch.cuda.is_available(), "GPU tests need a GPU (no CPU fallback)"
    import __graft_entry__ as G

    G.build()
    import paper_2606_14188_b200 as lib

    return lib


def _rel(a, b):
    return float((a - b).abs().max() / b.abs().max().clamp_min(1e-30))


def _both(L, W, two_norm=False):
    import torch

    batch, T, n, _ = W.shape
    P = T * (T - 1) // 2
    A = torch.from_numpy(W.A).cuda()
    w = torch.from_numpy(W.w).cuda()
    phi_ref, r_ref = L.ltv_scan_system_response_tube(A, w, two_norm=two_norm)          # existing path, torch workspace
    phi = torch.full((batch, P, n, n), float("nan"), device="cuda")
    r = torch.full((batch, T, n), float("nan"), device="cuda")
    before = torch.cuda.memory_allocated()
    L.ltv_scan_system_response_tube_static(A, w, phi, r, two_norm=two_norm)
    assert torch.cuda.memory_allocated() == before                                      # the binding allocated nothing either
    torch.cuda.synchronize()
    assert torch.isfinite(phi).all() and torch.isfinite(r).all()
    assert _rel(phi, phi_ref) <= TOL and _rel(r, r_ref) <= TOL
    return phi, r


def test_static_scratch_matches_workspace_path_two_calls_in_a_row(L):
    """Two calls in a row on one stream, the second on a smaller problem with another tile geometry, so that it runs on top of
    the first call's left-over partial sums: nothing needs to start at zero.  Then the first problem again."""
    assert L.ltv_static_scratch_bytes() == 32 << 20
    W1 = dense_random(3, 9, 300, 4, seed=501)           # tcgen05 path, two n-tiles of 160 columns, ragged m-tiles
    W2 = generate(config(0))                            # BASELINE.json configs[0]: n = 48, fp32-FMA path
    W3 = dense_random(2, 6, 132, 4, seed=502)           # one ragged n-tile
    p1, r1 = _both(L, W1)
    _both(L, W2)
    _both(L, W3, two_norm=True)
    p1b, r1b = _both(L, W1)                             # same inputs, scratch now holds other problems' sums
    import torch

    assert torch.equal(p1, p1b) and torch.equal(r1, r1b)   # deterministic: bit for bit


def test_static_scratch_limit_is_an_error_not_an_overrun(L):
    import torch

    n, T = 300, 32                                       # configs[1]: 1.19 MB of scratch per item
    per_item = L.ltv_scan_workspace_bytes(L.LTV_OP_SYSTEM_RESPONSE_TUBE, 1, T, n, 0)
    too_many = L.ltv_static_scratch_bytes() // per_item + 2
    A = torch.zeros((too_many, T, n, n), device="cuda")
    w = torch.zeros((too_many, T, n), device="cuda")
    phi = torch.zeros((1,), device="cuda").expand(0)    # never touched: the call must fail before anything is enqueued
    l0 = L.ltv_launch_count()
    st = L.lib.ltv_scan_system_response_tube_static(A.data_ptr(), w.data_ptr(), A.data_ptr(), w.data_ptr(), too_many, T, n, 0, None)
    assert st == L.LTV_ERR_STATIC_SCRATCH_LIMIT and L.ltv_launch_count() == l0
    assert L.lib.ltv_status_string(st) == b"LTV_ERR_STATIC_SCRATCH_LIMIT"
    assert L.lib.ltv_scan_system_response_tube_static(None, w.data_ptr(), A.data_ptr(), w.data_ptr(), 1, T, n, 0, None) == 1
    assert L.lib.ltv_scan_system_response_tube_static(A.data_ptr(), w.data_ptr(), A.data_ptr(), w.data_ptr(), 1, T, n, 4, None) == 2
    del phi
