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
