"""Element sharding across ranks: contiguous ranges, no data-path collective.
Pure host logic (no CUDA): used by bench.py and covered by a world_size-2 gloo test on CPU."""
from __future__ import annotations


def shard_range(total: int, rank: int, world: int, align: int = 32):
    """(first, count) of rank's contiguous element range; boundaries are multiples of `align` (one warp tile)
    except the end of the tensor.  The ranges of ranks 0..world-1 partition [0, total)."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    tiles = (total + align - 1) // align
    base, extra = divmod(tiles, world)
    t0 = rank * base + min(rank, extra)
    t1 = t0 + base + (1 if rank < extra else 0)
    first, last = min(total, t0 * align), min(total, t1 * align)
    return first, last - first


def max_over_ranks(value: float, group=None) -> float:
    """max of a python float over the process group (device timing is reduced this way); identity without dist."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return value
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    t = torch.tensor([value], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
