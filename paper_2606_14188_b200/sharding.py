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


def row_shard_range(T: int, rank: int, world: int) -> tuple[int, int]:
    """Block rows [k_lo, k_hi) of the system response Phi(k,j), 1 <= k <= T-1, for `rank` of `world` when ONE item (or a
    batch too small to shard) is split over the GPUs (ltv_scan_system_response_tube_rows, optional).  Row k has
    k blocks, so the ranges are balanced by block count, not by row count: contiguous, disjoint, covering 1 .. T-1; a rank
    may get an empty range (k_lo == k_hi) when there are more ranks than rows.  Nothing is exchanged on the data path: every
    rank holds A, computes its rows alone, and owns the complete tube rows r_k of its range."""
    if not (0 <= rank < world) or T < 1:
        raise ValueError("bad rank/world/T")
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
