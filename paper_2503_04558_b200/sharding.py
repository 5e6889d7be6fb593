"""Multi-GPU decomposition of the hot path (partitioning A): particles are
independent given the fields, so they are sharded by contiguous
index range, one process per GPU; the grid is replicated.  Push+deposit needs no data-path
collective; a coupled loop sums the per-rank fluxes with one all-reduce before the
(replicated) field step."""


def shard_range(n, rank, world):
    """contiguous [lo, hi) of `n` items owned by `rank` of `world` (sizes differ by <= 1)."""
    base, rem = divmod(int(n), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def allreduce_flux(flux_tensors):
    """sum the three flux arrays over ranks (torch.distributed; NCCL on GPUs, gloo on CPU)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        for t in flux_tensors:
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return flux_tensors
