"""ltv_scan_system_response_tube_rows - the block rows of the system response that one GPU computes when single items are split
over GPUs (optional) - against the oracle, shard by shard, on ONE GPU: the shards of a partition are run one after
the other and must assemble to the whole response and tube."""
import numpy as np
import pytest

from oracle import ltv_oracle as O
from paper_2606_14188_b200.sharding import row_shard_range
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


def _check_partition(L, W, world, two_norm=False, by_time_model=False):
    import torch

    batch, T, n, _ = W.shape
    A = torch.from_numpy(W.A).cuda(); w = torch.from_numpy(W.w).cuda()
    ref = [O.system_response_tube_item(W.A[b], W.w[b]) for b in range(batch)]
    ref_r = np.stack([O.tube_row2norm_item(W.A[b], W.w[b]) for b in range(batch)]) if two_norm else np.stack([q[1] for q in ref])
    r_sum = torch.zeros((batch, T, n), device="cuda")
    seen = set()
    for rank in range(world):
        k_lo, k_hi = row_shard_range(T, rank, world, n=n if by_time_model else None)
        if k_lo == k_hi:
            continue
        phi, r = L.ltv_scan_system_response_tube_rows(A, w, k_lo, k_hi, two_norm=two_norm)
        torch.cuda.synchronize()
        assert phi.shape[1] == sum(range(k_lo, k_hi)) == L.ltv_phi_row_shard_blocks(T, k_lo, k_hi)
        got = phi.cpu().numpy()
        want = np.zeros_like(got)
        idx = set()
        for k in range(k_lo, k_hi):
            for j in range(k):
                q = L.ltv_phi_row_shard_block_index(T, k_lo, k_hi, k, j)
                idx.add(q)
                seen.add((k, j))
                for b in range(batch):
                    want[b, q] = ref[b][0][O.packed_index(k, j)]
        assert idx == set(range(phi.shape[1]))                       # the shard's index map is a bijection
        assert O.rel_err(got, want) <= TOL
        rr = r.cpu().numpy()
        mask = np.zeros(T, dtype=bool); mask[k_lo:k_hi] = True
        assert np.all(rr[:, ~mask] == 0.0)                           # rows of other shards are not touched
        assert O.rel_err(rr[:, mask], ref_r[:, mask]) <= TOL
        r_sum += r
    assert seen == {(k, j) for k in range(1, T) for j in range(k)}   # the shards cover every block exactly once
    assert O.rel_err(r_sum.cpu().numpy(), ref_r) <= TOL


@pytest.mark.parametrize("n,T,batch,world", [(48, 16, 1, 1),      # C1 shape, the whole response through the row route
                                             (48, 16, 2, 4),      # fp32-FMA products
                                             (132, 9, 2, 3),      # tensor cores, ragged tiles
                                             (300, 7, 3, 2),      # C2-size blocks, stacks across block boundaries
                                             (96, 3, 1, 4)])      # more ranks than rows: empty shards
def test_row_shards_assemble_to_the_oracle_response(L, n, T, batch, world):
    _check_partition(L, dense_random(batch, T, n, 2, seed=n + T + world), world)


def test_row_shards_of_the_time_model_partition(L):
    """The partition balanced by modelled time (row_shard_range with the state dimension given) assembles to the same response."""
    _check_partition(L, dense_random(1, 12, 164, 2, seed=31), 3, by_time_model=True)
    _check_partition(L, dense_random(2, 7, 300, 2, seed=32), 4, by_time_model=True)


def test_row_shards_two_norm_tube_and_config1(L):
    _check_partition(L, generate(config(0)), 3)
    _check_partition(L, dense_random(2, 6, 132, 2, seed=5), 2, two_norm=True)


def test_row_shard_equals_the_scan_at_c4_block_size(L):
    """One C4-size item (n = 2400, T = 6 to keep the oracle out of it): the row route on two shards against the library's own
    time-parallel scan (GPU-vs-GPU PROPERTY: different order of the products, same blocks), and one block row against the oracle."""
    import torch

    W = generate(config(3, batch=1))
    A = torch.from_numpy(W.A[:, :6].copy()).cuda(); w = torch.from_numpy(W.w[:, :6].copy()).cuda()
    T = 6
    phi, r = L.ltv_scan_system_response_tube(A, w)
    r_sum = torch.zeros_like(r)
    for rank in range(2):
        k_lo, k_hi = row_shard_range(T, rank, 2)
        ps, rs = L.ltv_scan_system_response_tube_rows(A, w, k_lo, k_hi)
        r_sum += rs
        for k in range(k_lo, k_hi):
            for j in range(k):
                a = ps[0, L.ltv_phi_row_shard_block_index(T, k_lo, k_hi, k, j)]
                b = phi[0, L.ltv_phi_block_index(T, k, j)]
                assert float((a - b).abs().max() / b.abs().max()) <= TOL
        if rank == 1:
            k = k_hi - 1
            ref = O.phi_block(W.A[0, :6], k, 0)
            assert O.rel_err(ps[0, L.ltv_phi_row_shard_block_index(T, k_lo, k_hi, k, 0)].cpu().numpy(), ref) <= TOL
    torch.cuda.synchronize()
    assert float((r_sum - r).abs().max() / r.abs().max()) <= TOL


def test_row_shard_validation(L):
    import ctypes
    g = L.lib.ltv_scan_system_response_tube_rows
    buf = (ctypes.c_float * 64)()
    q = ctypes.cast(buf, ctypes.c_void_p)
    assert g(None, q, q, q, 1, 4, 4, 1, 4, 0, None) == 1
    assert g(q, q, q, q, 1, 4, 4, 0, 4, 0, None) == 2          # k_lo < 1
    assert g(q, q, q, q, 1, 4, 4, 2, 2, 0, None) == 2          # empty range
    assert g(q, q, q, q, 1, 4, 4, 1, 5, 0, None) == 2          # k_hi > T
    assert L.ltv_phi_row_shard_blocks(8, 3, 6) == 3 + 4 + 5 and L.ltv_phi_row_shard_blocks(8, 3, 3) == -1
    assert L.ltv_phi_row_shard_block_index(8, 3, 6, 2, 0) == -1 and L.ltv_phi_row_shard_block_index(8, 3, 6, 3, 0) == 0
