"""Rank plumbing for `bench.py --gpus N`: replicas only.

Every reference voxel is independent (section 1), and one case is tens of microseconds on one B200,
so a case is never sharded: every rank runs whole cases on its own GPU and there is NO data-path collective.  The
only exchanges are the barrier around the timed region and the max-over-ranks of the device time, both through
`torch.distributed` (nccl on the GPU box, gloo in the CPU tests).  Nothing of the method's arithmetic is here.
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


class Replicas:
    """One process per GPU.  `backend=None` picks nccl when CUDA is there, else gloo."""

    def __init__(self, backend: str | None = None, device: torch.device | None = None):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device if device is not None else torch.device("cpu")
        self.owns_group = False
        if self.world > 1 and not dist.is_initialized():
            backend = backend or ("nccl" if self.device.type == "cuda" else "gloo")
            kw = {"device_id": self.device} if backend == "nccl" else {}
            dist.init_process_group(backend, rank=self.rank, world_size=self.world, **kw)
            self.owns_group = True

    def barrier(self) -> None:
        if self.world > 1:
            dist.barrier()
        if self.device.type == "cuda":
            torch.cuda.synchronize(self.device)

    def max_over_ranks(self, x: float) -> float:
        """The job's time is the slowest rank's."""
        if self.world == 1:
            return float(x)
        t = torch.tensor([x], dtype=torch.float64, device=self.device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, x: float) -> float:
        """Units processed by the whole job (each replica counts its own)."""
        if self.world == 1:
            return float(x)
        t = torch.tensor([x], dtype=torch.float64, device=self.device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    def job_rate(self, units_this_rank: float, seconds_this_rank: float) -> float:
        """Whole-job throughput: units all ranks processed / max-over-ranks time."""
        return self.sum_over_ranks(units_this_rank) / self.max_over_ranks(seconds_this_rank)

    def close(self) -> None:
        if self.owns_group and dist.is_initialized():
            dist.destroy_process_group()
            self.owns_group = False
