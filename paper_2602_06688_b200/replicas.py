"""Host-side plumbing for running N independent replicas of the path, one process per GPU.

The path does not shard (BASELINE.json:north_star: one GPU, no sharding, no collectives;
DESIGN.md "Multi-GPU: replicas only"): every rank runs the whole path on its own sources.
The only cross-rank traffic is measurement plumbing -- a barrier around the timed region and
a max-reduction of the measured time -- through ``torch.distributed`` (NCCL on GPUs, gloo in
the CPU tests).  There is no data-path collective.
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


class Replicas:
    def __init__(self, backend: str | None = None, device: torch.device | None = None):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device if device is not None else torch.device("cpu")
        self.owns_group = False
        if self.world > 1 and not dist.is_initialized():
            kw = {}
            if backend == "nccl":
                kw["device_id"] = self.device
            dist.init_process_group(backend or "gloo", **kw)
            self.owns_group = True

    @property
    def distributed(self) -> bool:
        return self.world > 1

    def barrier(self) -> None:
        if self.distributed:
            dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        """The slowest rank's time: multi-GPU numbers are the max over ranks, never a mean."""
        if not self.distributed:
            return float(x)
        t = torch.tensor([float(x)], dtype=torch.float64, device=self.device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, x: float) -> float:
        if not self.distributed:
            return float(x)
        t = torch.tensor([float(x)], dtype=torch.float64, device=self.device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    def seed_offset(self) -> int:
        """Each replica works on different sources: offset added to the synthetic-input seed."""
        return 10000 * self.rank

    def whole_job_throughput(self, units_this_rank: float, seconds_this_rank: float) -> float:
        """Units all ranks processed / the slowest rank's time (bench.py's ``value``)."""
        return self.sum_over_ranks(units_this_rank) / self.max_over_ranks(seconds_this_rank)

    def close(self) -> None:
        if self.owns_group and dist.is_initialized():
            dist.destroy_process_group()
            self.owns_group = False
