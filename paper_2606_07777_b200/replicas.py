"""Multi-GPU plumbing for the measurement harness: REPLICAS ONLY.

BASELINE.json's north_star keeps the whole path on one GPU ("no sharding across GPUs, no NCCL"), so N > 1 means
N independent copies of the single-GPU job, one process per GPU.  Nothing on the data path crosses ranks; the
only exchanges are the timing barrier and the max-over-ranks of the measured time, which this module provides
over `torch.distributed` (backend "nccl" on GPUs; "gloo" in the CPU tests).
"""
from __future__ import annotations

import os


class Replicas:
    """One process per replica, launched by torchrun (RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* in the env)."""

    def __init__(self, backend: str | None = None):
        import torch
        self.torch = torch
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.backend = backend or ("nccl" if torch.cuda.is_available() else "gloo")
        self.dist = None
        self.device = torch.device("cuda", self.local_rank) if self.backend == "nccl" else torch.device("cpu")
        if self.backend == "nccl":
            torch.cuda.set_device(self.local_rank)
        if self.world > 1:
            import torch.distributed as dist
            kw = {"device_id": self.device} if self.backend == "nccl" else {}
            dist.init_process_group(backend=self.backend, **kw)
            self.dist = dist

    def barrier(self):
        """All replicas arrive, and (on GPUs) all queued device work has finished."""
        if self.dist is not None:
            self.dist.barrier()
        if self.backend == "nccl":
            self.torch.cuda.synchronize()

    def max_over_ranks(self, value: float) -> float:
        """The slowest replica's time: multi-GPU numbers are the max over ranks, never a mean or rank 0's."""
        t = self.torch.tensor([float(value)], dtype=self.torch.float64, device=self.device)
        if self.dist is not None:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def aggregate_throughput(self, units_per_replica: float, seconds_this_rank: float) -> float:
        """Whole-job throughput of N replicas: all units processed / the slowest replica's time (weak scaling)."""
        return self.world * units_per_replica / self.max_over_ranks(seconds_this_rank)

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()
            self.dist = None
