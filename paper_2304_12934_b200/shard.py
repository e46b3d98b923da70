"""z-sharding for N > 1 GPUs: the path partitions by slice -- forward and adjoint are independent
per slice, so ranks take contiguous z-ranges with no data-path collective ("weak" replicas of the slab pipeline).
MBIR's 26-neighbour prior would need a one-slice halo exchange per iteration; that is SURVEY 8(f) #3, not built."""


def shard_slices(n_slices, rank, world):
    """contiguous [lo, hi) of rank; sizes differ by at most one group of 8 slices."""
    groups = (n_slices + 7) // 8
    base, extra = divmod(groups, world)
    glo = rank * base + min(rank, extra)
    ghi = glo + base + (1 if rank < extra else 0)
    return min(glo * 8, n_slices), min(ghi * 8, n_slices)


def max_over_ranks(seconds, device="cuda"):
    import torch, torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(seconds)
    t = torch.tensor([float(seconds)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
