"""z-sharding for N > 1 GPUs: the path partitions by slice.

Forward and adjoint are independent per slice, so ranks take contiguous z-ranges with no data-path collective (bench.py --gpus N:
"weak" replicas of the slab pipeline).  MBIR couples slices only through the prior's neighbourhood and three global scalars:
`TorchComm` is the transport `tc_mbir_sharded` asks for (include/tc.h: tc_comm) -- one halo slice to each z-neighbour and one
all-reduce of four doubles per iteration -- on torch.distributed (NCCL point-to-point over NVLink on GPUs; gloo on CPU for tests).
No arithmetic of the method lives here.
"""


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


class TorchComm:
    """Halo exchange and scalar all-reduce between z-neighbours rank - 1 (down) and rank + 1 (up) of the default process group.
    send_down / send_up / recv_down / recv_up are (n, n) float32 tensors on `device`, None where there is no neighbour."""

    def __init__(self, n, device="cuda", rank=None, world=None):
        import torch, torch.distributed as dist
        self.dist, self.torch = dist, torch
        self.rank = dist.get_rank() if rank is None else rank
        self.world = dist.get_world_size() if world is None else world
        self.device = device
        mk = lambda: torch.zeros((n, n), dtype=torch.float32, device=device)
        self.send_down, self.recv_down = (mk(), mk()) if self.rank > 0 else (None, None)
        self.send_up, self.recv_up = (mk(), mk()) if self.rank < self.world - 1 else (None, None)

    def exchange(self):
        d, ops = self.dist, []
        if self.rank > 0:
            ops += [d.P2POp(d.isend, self.send_down, self.rank - 1), d.P2POp(d.irecv, self.recv_down, self.rank - 1)]
        if self.rank < self.world - 1:
            ops += [d.P2POp(d.isend, self.send_up, self.rank + 1), d.P2POp(d.irecv, self.recv_up, self.rank + 1)]
        if ops:
            for r in d.batch_isend_irecv(ops):
                r.wait()
        if self.device != "cpu":
            self.torch.cuda.synchronize()

    def allreduce(self, vals):
        t = self.torch.tensor(list(vals), dtype=self.torch.float64, device=self.device)
        self.dist.all_reduce(t)
        return t.tolist()
