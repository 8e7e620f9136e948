"""Multi-GPU plumbing shared by both modes of `bench.py --gpus N`.

Default mode = replicas: N GPUs run N independent lattices (north_star keeps the path on one GPU), no data-path
collective.  The sharded alternative (one lattice cut into T-slabs with a face exchange per application) lives in
slab.py and uses the same Group.  This module holds the cross-rank logic both need -- rendezvous, barrier,
max-over-ranks of the device time, whole-job throughput -- on torch.distributed (NCCL on GPUs, gloo in the CPU tests).
"""
import os


def env_ranks():
    """(rank, world_size, local_rank) from the torchrun environment (1-process defaults)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0")))


class Group:
    """Process group wrapper; a no-op for world_size 1."""

    def __init__(self, backend="nccl", device=None):
        self.rank, self.world, self.local = env_ranks()
        self.device = device
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            kwargs = {}
            if backend == "nccl" and device is not None:
                kwargs["device_id"] = device
            dist.init_process_group(backend, **kwargs)
            self.dist = dist

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max_over_ranks(self, value: float) -> float:
        if self.dist is None:
            return float(value)
        import torch
        t = torch.tensor([float(value)], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()
            self.dist = None


def whole_job_rate(units_per_rank: float, world: int, max_ms: float) -> float:
    """units of all ranks / max-over-ranks time, in units per second (weak scaling)."""
    return units_per_rank * world / (max_ms * 1e-3)
