"""Multi-GPU plumbing: replicas only.

The path shards with NO exchange step (pages are independent; under tensor parallelism every
rank's pool holds its own head partition of every page, "head partitions"), so N
GPUs run N independent replicas of the same calls.  The
only collective is the timing reduction of the bench: barrier, max over ranks of the device-timed
interval, and the sum of units all ranks processed.  Backend: nccl on GPUs, gloo in the CPU tests.
"""
from __future__ import annotations

import os


class Replicas:
    def __init__(self, backend: str | None = None):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.dist = None
        self.device = None
        if self.world > 1:
            import torch
            import torch.distributed as dist

            if backend is None:
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            kw = {}
            if backend == "nccl":
                self.device = torch.device("cuda", self.local_rank)
                kw["device_id"] = self.device
            dist.init_process_group(backend, **kw)
            self.dist = dist

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        """Every multi-GPU time is the max over ranks of a device-timed interval."""
        if self.dist is None:
            return float(x)
        import torch

        t = torch.tensor([float(x)], dtype=torch.float64, device=self.device or "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, x: float) -> float:
        if self.dist is None:
            return float(x)
        import torch

        t = torch.tensor([float(x)], dtype=torch.float64, device=self.device or "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return float(t.item())

    def whole_job_rate(self, units_this_rank: float, seconds_this_rank: float) -> float:
        """Aggregate throughput of N independent replicas: all units / slowest rank's time."""
        return self.sum_over_ranks(units_this_rank) / self.max_over_ranks(seconds_this_rank)

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()
            self.dist = None
