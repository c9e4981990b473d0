"""Multi-GPU plumbing of the benchmark: replicas only.

The encoder has no exchange step, so N GPUs run N independent replicas of the same workload; the only
communication is a barrier around the timed region and a MAX reduction of the per-rank device times.
Backend "nccl" on GPUs (one process per GPU under torchrun), "gloo" in the CPU tests.
"""
from __future__ import annotations

import os
from typing import Optional

import torch


class Replicas:
    def __init__(self, backend: Optional[str] = None, device: Optional[torch.device] = None):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            if not dist.is_initialized():
                backend = backend or ("nccl" if torch.cuda.is_available() else "gloo")
                kw = {}
                if backend == "nccl" and device is not None:
                    kw["device_id"] = device
                dist.init_process_group(backend, **kw)
            self.dist = dist

    def barrier(self) -> None:
        """Device sync + rank barrier + device sync: both sides of a timed region."""
        if torch.cuda.is_available():
            torch.cuda.synchronize()
        if self.dist is not None:
            self.dist.barrier()
        if torch.cuda.is_available():
            torch.cuda.synchronize()

    def max_over_ranks(self, value: float) -> float:
        if self.dist is None:
            return float(value)
        dev = self.device if (self.device is not None and self.dist.get_backend() == "nccl") else "cpu"
        t = torch.tensor([value], dtype=torch.float64, device=dev)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def whole_job_rate(self, units_per_rank: int, ms_local: float) -> tuple[float, float]:
        """-> (units per second over ALL ranks, max-over-ranks ms): weak scaling, every rank did
        `units_per_rank` units in at most the slowest rank's time."""
        ms = self.max_over_ranks(ms_local)
        return units_per_rank * self.world / (ms * 1e-3), ms

    @property
    def is_reporter(self) -> bool:
        return self.rank == 0

    def close(self) -> None:
        if self.dist is not None and self.dist.is_initialized():
            self.dist.destroy_process_group()
            self.dist = None
