"""Multi-GPU plumbing of the "replicas only" mode: one process per GPU, each advancing its own coil.

The hot path has no data-path collective (north_star fixes one GPU per simulation).  What N > 1 ranks share is the
measurement protocol: a barrier on both sides of the timed region, the MAX over ranks of the device time, and a
whole-job aggregate.  These helpers hold that host logic so that it can be exercised on CPU with the gloo backend
(tests/test_replicas.py); bench.py uses them with nccl.
"""
from __future__ import annotations

import os


def env_rank():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of the per-cell Jc0 perturbation of replica `rank`: rank 0 keeps the config's seed."""
    return base_seed + 100 * rank


class Group:
    """Thin wrapper over torch.distributed for the three things the replicas need."""

    def __init__(self, backend: str | None = None, device=None):
        self.rank, self.local_rank, self.world = env_rank()
        self.dist = None
        self.device = device
        if self.world > 1:
            import torch.distributed as dist
            if not dist.is_initialized():
                kw = {}
                if backend == "nccl" and device is not None:
                    kw["device_id"] = device
                dist.init_process_group(backend or "gloo", **kw)
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

    def aggregate_rate(self, units_per_rank: float, seconds_this_rank: float) -> float:
        """Whole-job throughput: units of all ranks divided by the slowest rank's time."""
        return self.world * units_per_rank / self.max_over_ranks(seconds_this_rank)

    def close(self):
        if self.dist is not None and self.dist.is_initialized():
            self.dist.destroy_process_group()
