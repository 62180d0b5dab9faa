"""Host-side helpers for running the TNRD path on several GPUs (one process per GPU).

The method has no exchange step when images are independent (every operation is local to
one image), so the data path uses NO collective: a batch is split across ranks, each rank runs libtnrd on its
share.  torch.distributed is used only for the barrier and for the max-over-ranks of the measured time.
"""
from __future__ import annotations


def shard_range(n_items: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [lo, hi) share of n_items for `rank`; sizes differ by at most one, earlier ranks get the extra."""
    if world < 1 or not (0 <= rank < world) or n_items < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_items, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar (elapsed time); identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """SUM all-reduce of a scalar (units processed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def slab_bounds(H: int, rank: int, world: int, T: int, ksize: int) -> tuple[int, int, int, int]:
    """Row slab of ONE large image for `rank`: returns (lo, hi, src_lo, src_hi).

    Rows [lo, hi) are the rank's share of the output; rows [src_lo, src_hi) of f and u0 are what it must process to get
    them right.  Every stage reaches 2r rows (r = (ksize - 1) / 2: k_i * u, then kbar_i * phi), so u_T on [lo, hi)
    depends on rows within 2 r T of it; the margin is cut off only at the true image border, where the
    slab's own mirror extension IS the image's.  No exchange between ranks: a 2 r T overlap instead (every
    operation is local)."""
    lo, hi = shard_range(H, rank, world)
    m = (ksize - 1) * T
    return lo, hi, max(0, lo - m), min(H, hi + m)
