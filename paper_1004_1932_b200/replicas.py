"""Rank plumbing for bench.py: the path does not shard ("replicas only"),
so N GPUs run N independent replicas of the workload, one process per GPU, and the only
cross-rank traffic is the barrier around the timed region and the reduction of the timings.
No data-path collective exists.  Works with backend "nccl" (GPU box) and "gloo" (CPU tests).

Holds no arithmetic of the method.
"""
import os

import torch
import torch.distributed as dist


class Ranks:
    """World of one process per GPU read from the torchrun environment; world_size 1 needs no
    process group at all."""

    def __init__(self, backend=None):
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.backend = backend
        self._own_pg = False
        if self.world > 1 and not dist.is_initialized():
            if backend is None:
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            kw = {}
            if backend == "nccl":
                kw["device_id"] = torch.device("cuda", self.local_rank)
            dist.init_process_group(backend=backend, rank=self.rank, world_size=self.world, **kw)
            self.backend = backend
            self._own_pg = True
        elif self.world > 1:
            self.backend = dist.get_backend()

    def _dev(self):
        return torch.device("cuda", self.local_rank) if self.backend == "nccl" else torch.device("cpu")

    def barrier(self):
        if self.world > 1:
            if self.backend == "nccl":
                dist.barrier(device_ids=[self.local_rank])
            else:
                dist.barrier()

    def max(self, x: float) -> float:
        """Max over ranks (timings: the job is as slow as its slowest replica)."""
        if self.world == 1:
            return float(x)
        t = torch.tensor([float(x)], dtype=torch.float64, device=self._dev())
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum(self, x: float) -> float:
        """Sum over ranks (units of work processed by the whole job)."""
        if self.world == 1:
            return float(x)
        t = torch.tensor([float(x)], dtype=torch.float64, device=self._dev())
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    def throughput(self, local_units: float, local_seconds: float) -> float:
        """Whole-job throughput of independent replicas: all ranks' units / the slowest rank's time."""
        return self.sum(local_units) / self.max(local_seconds)

    def close(self):
        if self._own_pg and dist.is_initialized():
            dist.destroy_process_group()
            self._own_pg = False
