"""Host-side logic of the N > 1 launch ("replicas only").

The path of BASELINE.json's north_star runs on one GPU, so N ranks are N independent replicas of the
workload (seeds differ, no data-path collective).  The only inter-rank traffic is the timing protocol of
bench.py: a barrier on both sides of the timed region and the MAX over ranks of the device time.
torch.distributed provides it (NCCL on the GPUs, gloo in the CPU tests); nothing here touches the fields.
"""
from __future__ import annotations

import os


def rank_info():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) without one."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of rank's replica: distinct per rank, rank 0 keeps the configuration's own seed."""
    return base_seed + 100 * rank


class Replicas:
    """Barrier, max-over-ranks and whole-job throughput for `world` independent replicas."""

    def __init__(self, dist=None, device=None):
        self.dist = dist                      # an initialised torch.distributed module, or None for one rank
        self.device = device
        self.world = dist.get_world_size() if dist is not None else 1
        self.rank = dist.get_rank() if dist is not None else 0

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        if self.dist is None:
            return float(x)
        import torch
        t = torch.tensor([float(x)], dtype=torch.float64, device=self.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, x: float) -> float:
        if self.dist is None:
            return float(x)
        import torch
        t = torch.tensor([float(x)], dtype=torch.float64, device=self.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return float(t.item())

    def throughput(self, units_this_rank: float, ms_this_rank: float) -> float:
        """Whole-job units per second: the units all ranks processed / the slowest rank's time."""
        return self.sum_over_ranks(units_this_rank) / (self.max_over_ranks(ms_this_rank) * 1e-3)
