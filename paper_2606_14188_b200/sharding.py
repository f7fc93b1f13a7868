"""Batch sharding for N > 1 GPUs: the LTV path has no data-path collective (items are independent), so a
rank just owns a contiguous range of batch items; timing is reduced with a MAX over ranks."""
from __future__ import annotations


def shard_range(global_batch: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced [b0, b1) of `global_batch` items for `rank` of `world` (sizes differ by <= 1)."""
    if not (0 <= rank < world) or global_batch < 0:
        raise ValueError("bad rank/world/batch")
    base, rem = divmod(global_batch, world)
    b0 = rank * base + min(rank, rem)
    return b0, b0 + base + (1 if rank < rem else 0)


def row_shard_cost(T: int, k_lo: int, k_hi: int, n: int, sms: int = 148) -> float:
    """Modelled seconds of ltv_scan_system_response_tube_rows for the rows [k_lo, k_hi) of one item on one B200: per column
    step j a batched tcgen05 GEMM of the shard's cn(j) = k_hi - max(k_lo, j+2) blocks, counted in ROUNDS of tiles over the
    SMs (128 x 160 tiles on all SMs, or 256 x 160 CTA-pair tiles on half as many - whichever the library's own rule picks), a
    fixed launch cost, and the row kernel's pass over the column.  Fitted once against measured shard times (n = 2400, T = 16:
    within 5 % for 1-8 shards; n = 1200: 25 % low but in the right order) - a load-balancing model, not a timing claim."""
    import numpy as np

    if k_hi <= k_lo:
        return 0.0
    j = np.arange(0, k_hi - 1)
    nt = -(-n // 160)
    tile_s = 2.0 * 128 * 160 * n * 3 / 6.7e12                       # one round of 128-row 3xTF32 tiles
    cn = np.maximum(k_hi - np.maximum(k_lo, j + 2), 0)
    r1 = np.ceil(np.ceil(cn * n / 128) * nt / sms)
    r2 = np.ceil(np.ceil(cn * n / 256) * nt / (sms // 2))
    gemm = np.where(cn > 0, np.minimum(1.25 * r2, 1.54 * r1), 0.0) * tile_s
    rows = (k_hi - np.maximum(k_lo, j + 1)) * float(n) * n * 8 / 6.0e12
    return float(np.sum(gemm + rows + 5e-6))


def row_shard_range(T: int, rank: int, world: int, n: int | None = None, sms: int = 148) -> tuple[int, int]:
    """Block rows [k_lo, k_hi) of the system response Phi(k,j), 1 <= k <= T-1, for `rank` of `world` when ONE item (or a
    batch too small to shard) is split over the GPUs (ltv_scan_system_response_tube_rows, optional).  Ranges are
    contiguous, disjoint and cover 1 .. T-1; a rank may get an empty range (k_lo == k_hi) when there are more ranks than
    rows.  Nothing is exchanged on the data path: every rank holds A, computes its rows alone, and owns the complete tube
    rows r_k of its range.
    Balance: without `n`, by block count (row k has k blocks).  With the state dimension `n` (>= 96, the tensor-core path),
    by the modelled time row_shard_cost - the last rows are long chains of small GEMMs that fill the GPU badly, so equal
    block counts leave the last ranks 1.3x slower: the partition minimises the slowest rank's modelled time (every rank
    computes the same partition: a pure function of T, world, n, sms)."""
    if not (0 <= rank < world) or T < 1:
        raise ValueError("bad rank/world/T")
    if n is not None and n >= 96 and world > 1 and T > 2:
        cost = lambda a, b: row_shard_cost(T, a, b, n, sms)

        def cut(bound):   # greedy: every rank takes rows while its modelled time stays within `bound`
            bounds, lo = [1], 1
            for _ in range(world):
                a, b = lo, T                                    # largest hi in [lo, T] with cost(lo, hi) <= bound (cost grows with hi)
                while a < b:
                    mid = (a + b + 1) // 2
                    if cost(lo, mid) <= bound:
                        a = mid
                    else:
                        b = mid - 1
                lo = a
                bounds.append(lo)
            return bounds

        lo_b, hi_b = 0.0, cost(1, T)
        for _ in range(40):                                     # smallest bound that lets `world` ranks cover all rows
            mid_b = 0.5 * (lo_b + hi_b)
            if cut(mid_b)[-1] >= T:
                hi_b = mid_b
            else:
                lo_b = mid_b
        bounds = cut(hi_b)
        bounds[-1] = T
        return bounds[rank], bounds[rank + 1]
    total = T * (T - 1) // 2                       # blocks of all rows
    bounds = [1]
    k = 1
    acc = 0
    for r in range(1, world):
        target = total * r / world
        while k < T and abs(acc + k - target) <= abs(acc - target):  # take row k while that brings the block count closer to the target
            acc += k
            k += 1
        bounds.append(k)
    bounds.append(T)
    return bounds[rank], bounds[rank + 1]


def assemble_tube_rows(r_local, device=None):
    """Sum over ranks of the zero-initialised r[batch,T,n] arrays of the row shards = the complete tube (every row is
    non-zero on exactly one rank; identity without torch.distributed).  The only exchange of the row-sharded path, and not
    on its data path: T n floats per item."""
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(r_local, op=dist.ReduceOp.SUM)
    return r_local


def shard_arrays(arrays: dict, rank: int, world: int) -> dict:
    """The items [b0, b1) of this rank of every batch-leading array in `arrays` (None entries pass through): all calls of
    the library - rollout, system response, adjoint, observer response, Kalman gains, constraint margins, output-feedback
    responses - treat batch items independently, so this is the whole distribution scheme."""
    sizes = {v.shape[0] for v in arrays.values() if v is not None}
    if len(sizes) != 1:
        raise ValueError("arrays disagree on the batch size")
    b0, b1 = shard_range(sizes.pop(), rank, world)
    return {k: (None if v is None else _aligned(v[b0:b1])) for k, v in arrays.items()}


def _aligned(view):
    """The library wants 16-byte aligned device pointers (LTV_ERR_ALIGNMENT otherwise).  A slice that starts at an
    arbitrary item of an array whose per-item size is not a multiple of 4 floats (u[T,m], f[T,p], grad_u with odd T m)
    is not: such views are returned as fresh contiguous copies, all others as views."""
    if hasattr(view, "data_ptr"):                      # torch tensor
        return view if (view.data_ptr() % 16 == 0 and view.is_contiguous()) else view.clone(
            memory_format=__import__("torch").contiguous_format)
    ptr = view.__array_interface__["data"][0]          # numpy array
    return view if (ptr % 16 == 0 and view.flags["C_CONTIGUOUS"]) else view.copy()


def reduce_max(value: float, device=None) -> float:
    """max over ranks of a python float (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def reduce_sum(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
