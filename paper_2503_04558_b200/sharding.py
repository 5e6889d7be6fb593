"""Multi-GPU decomposition of the hot path (partitioning A): particles are
independent given the fields, so they are sharded by contiguous
index range, one process per GPU; the grid is replicated.  Push+deposit needs no data-path
collective; a coupled loop sums the per-rank fluxes with ONE all-reduce of the contiguous
three-array flux block before the (replicated) field step."""


def shard_range(n, rank, world):
    """contiguous [lo, hi) of `n` items owned by `rank` of `world` (sizes differ by <= 1)."""
    base, rem = divmod(int(n), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def allreduce_flux(flux):
    """sum the flux arrays over ranks (torch.distributed; NCCL on GPUs, gloo on CPU).
    `flux` is the contiguous block [3, rows, pitch] (one collective) or a list of arrays that
    are views of one such block; separate arrays fall back to one collective each."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1):
        return flux
    if isinstance(flux, torch.Tensor):
        dist.all_reduce(flux, op=dist.ReduceOp.SUM)
        return flux
    base = getattr(flux[0], "_base", None)
    if base is not None and base.is_contiguous() and all(getattr(t, "_base", None) is base for t in flux) \
            and sum(t.numel() for t in flux) == base.numel():
        dist.all_reduce(base, op=dist.ReduceOp.SUM)
    else:
        for t in flux:
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return flux
