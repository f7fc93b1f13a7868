"""N > 1 host logic on CPU: world_size-2 gloo.  Shards partition the batch, every rank generates exactly the
items of the unsharded workload it owns, the oracle on the shards equals the oracle on the whole batch (no
collective is needed on the data path), and the timing reduction is a max over ranks."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

from paper_2606_14188_b200.sharding import shard_range


def test_shard_range_partitions():
    for gb in (0, 1, 5, 64, 1023):
        for world in (1, 2, 3, 8):
            r = [shard_range(gb, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == gb
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1


def test_shard_arrays_returns_16_byte_aligned_slices():
    """A slice starting at an odd item of an array with T*m (or T*p) not a multiple of 4 floats is not 16-byte aligned
    (the library would answer LTV_ERR_ALIGNMENT): shard_arrays hands out an aligned copy with the same content."""
    import torch

    from paper_2606_14188_b200.sharding import shard_arrays

    batch, T, p, n = 5, 6, 3, 8
    base = np.zeros(batch * T * p + 4, dtype=np.float32)
    off = (-base.ctypes.data // 4) % 4                       # make f itself 16-byte aligned
    f = base[off:off + batch * T * p].reshape(batch, T, p)
    f[:] = np.arange(f.size, dtype=np.float32).reshape(f.shape)
    A = np.zeros((batch, T, n, n), dtype=np.float32)
    for world in (2, 3):
        for rank in range(world):
            b0, b1 = shard_range(batch, rank, world)
            mine = shard_arrays(dict(A=A, f=f, none=None), rank, world)
            assert mine["none"] is None and np.array_equal(mine["f"], f[b0:b1])
            assert mine["f"].ctypes.data % 16 == 0 and mine["A"].ctypes.data % 16 == 0
            tm = shard_arrays(dict(f=torch.from_numpy(f)), rank, world)["f"]
            assert tm.data_ptr() % 16 == 0 and torch.equal(tm, torch.from_numpy(f)[b0:b1])


def _worker(rank, world, port, q):
    import torch.distributed as dist

    from oracle import ltv_oracle as O
    from paper_2606_14188_b200.sharding import reduce_max, reduce_sum, shard_arrays
    from workloads import config, generate, observation_model

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = config(0, batch=5, T=6)
    b0, b1 = shard_range(cfg["batch"], rank, world)
    W = generate(cfg, item_range=(b0, b1))
    X = O.rollout(W.A, W.B, W.c, W.x0, W.u)
    r = O.tube(W.A, W.w)
    # the next rows shard the same way: observation model generated for the whole batch, sliced per rank
    Wall = generate(cfg)
    M = observation_model(cfg["batch"], cfg["T"], Wall.A.shape[-1], 3, seed=9, kind="track")
    Hc = np.random.default_rng(4).normal(size=(cfg["batch"], cfg["T"], 2, Wall.A.shape[-1])).astype(np.float32)
    mine = shard_arrays(dict(A=Wall.A, w=Wall.w, Hc=Hc, **M), rank, world)
    assert np.array_equal(mine["A"], W.A)
    Pi, Lt = O.kalman_recursion(mine["A"], mine["C"], mine["e"], mine["f"], mine["Pi0"])
    sig = O.constraint_tightening(mine["A"], mine["w"], mine["Hc"])
    t_max = reduce_max(1.0 + rank)              # "time" of this rank
    units = reduce_sum(float(b1 - b0))
    q.put((rank, b0, b1, X, r, t_max, units, Pi, Lt, sig))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_batch_sharding_gloo():
    from oracle import ltv_oracle as O
    from workloads import config, generate

    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    world = 2
    procs = [ctx.Process(target=_worker, args=(k, world, port, q)) for k in range(world)]
    for p in procs:
        p.start()
    got = sorted([q.get(timeout=120) for _ in range(world)], key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    W = generate(config(0, batch=5, T=6))
    X = O.rollout(W.A, W.B, W.c, W.x0, W.u)
    r = O.tube(W.A, W.w)
    assert np.array_equal(np.concatenate([g[3] for g in got]), X)
    assert np.array_equal(np.concatenate([g[4] for g in got]), r)
    from workloads import observation_model
    M = observation_model(5, 6, W.A.shape[-1], 3, seed=9, kind="track")
    Hc = np.random.default_rng(4).normal(size=(5, 6, 2, W.A.shape[-1])).astype(np.float32)
    Pi, Lt = O.kalman_recursion(W.A, M["C"], M["e"], M["f"], M["Pi0"])
    assert np.array_equal(np.concatenate([g[7] for g in got]), Pi)
    assert np.array_equal(np.concatenate([g[8] for g in got]), Lt)
    assert np.array_equal(np.concatenate([g[9] for g in got]), O.constraint_tightening(W.A, W.w, Hc))
    assert all(g[5] == 2.0 for g in got)        # max over ranks
    assert all(g[6] == 5.0 for g in got)        # units of all ranks


def test_row_shard_range_partitions_the_block_rows():
    from paper_2606_14188_b200.sharding import row_shard_range

    for T in (1, 2, 3, 16, 32, 65):
        for world in (1, 2, 3, 8):
            r = [row_shard_range(T, k, world) for k in range(world)]
            assert r[0][0] == 1 and r[-1][1] == max(T, 1)
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))        # contiguous, disjoint, covering 1 .. T-1
            assert all(a <= b for a, b in r)
            blocks = [sum(range(a, b)) for a, b in r]
            assert sum(blocks) == T * (T - 1) // 2
            if T >= 16:                                                        # balanced by BLOCKS up to one row (<= T-1 blocks)
                assert max(blocks) - T * (T - 1) / 2 / world <= T


def test_row_shard_range_balanced_by_the_time_model():
    """With the state dimension given the partition is balanced by modelled time, not block count: still contiguous, disjoint
    and covering, the same on every rank, and its slowest shard is modelled no slower than the block-count partition's."""
    from paper_2606_14188_b200.sharding import row_shard_cost, row_shard_range

    for n, T in ((2400, 16), (1200, 32), (300, 32), (132, 9)):
        for world in (2, 3, 8):
            r = [row_shard_range(T, k, world, n=n) for k in range(world)]
            assert r[0][0] == 1 and r[-1][1] == T
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1)) and all(a <= b for a, b in r)
            assert sum(sum(range(a, b)) for a, b in r) == T * (T - 1) // 2
            old = [row_shard_range(T, k, world) for k in range(world)]
            worst = lambda part: max(row_shard_cost(T, a, b, n) for a, b in part)
            assert worst(r) <= worst(old) * (1 + 1e-9)
    assert row_shard_range(16, 1, 2, n=48) == row_shard_range(16, 1, 2)      # below the tensor-core path: block count


def _row_worker(rank, world, port, q):
    """One item split over the ranks by block rows: each rank computes ITS rows with the oracle's row recursion (what
    ltv_scan_system_response_tube_rows does on a GPU), the tube is assembled by the one all-reduce of the row-sharded path."""
    import torch
    import torch.distributed as dist

    from oracle import ltv_oracle as O
    from paper_2606_14188_b200.sharding import assemble_tube_rows, row_shard_range
    from workloads import config, generate

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    W = generate(config(0, batch=2, T=9))                    # A is replicated: every rank generates the same items
    batch, T, n, _ = W.shape
    k_lo, k_hi = row_shard_range(T, rank, world)
    r_local = torch.zeros((batch, T, n), dtype=torch.float64)
    mine = {}
    for b in range(batch):
        for t, row in O.phi_rows_item(W.A[b]):               # block rows of the oracle, in order
            if k_lo <= t < k_hi:
                acc = np.zeros(n)
                for s in range(t):
                    acc = acc + np.abs(row[s]) @ W.w[b, s].astype(np.float64)
                    mine[(b, t, s)] = row[s].copy()
                r_local[b, t] = torch.from_numpy(acc)
    own = r_local.clone()
    r_all = assemble_tube_rows(r_local)
    q.put((rank, k_lo, k_hi, own.numpy(), r_all.numpy(), sorted(mine.keys())))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_row_sharding_of_single_items_gloo():
    from oracle import ltv_oracle as O
    from workloads import config, generate

    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    world = 2
    procs = [ctx.Process(target=_row_worker, args=(k, world, port, q)) for k in range(world)]
    for p in procs:
        p.start()
    got = sorted([q.get(timeout=120) for _ in range(world)], key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    W = generate(config(0, batch=2, T=9))
    T = W.A.shape[1]
    r = O.tube(W.A, W.w)
    assert got[0][1] == 1 and got[0][2] == got[1][1] and got[1][2] == T
    for g in got:
        assert np.allclose(g[4], r, rtol=1e-12, atol=0.0)                     # every rank ends up with the complete tube
        mask = np.zeros(T, dtype=bool); mask[g[1]:g[2]] = True
        assert np.all(g[3][:, ~mask] == 0.0) and np.allclose(g[3][:, mask], r[:, mask], rtol=1e-12)   # its own rows were complete
    keys = got[0][5] + got[1][5]
    assert len(keys) == len(set(keys)) == 2 * T * (T - 1) // 2                # every block on exactly one rank
