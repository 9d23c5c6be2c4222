"""Multi-GPU plumbing of bench.py: "replicas only".

The paper's method is single-GPU and BASELINE.json's north_star runs everything on one GPU,
so N > 1 means N independent replicas of the workload, one process per GPU, with NO data-path collective: the only
communication is the timing protocol (barrier on both sides of the timed region, maximum of the device times over
the ranks, rank 0 reports).  This module holds that protocol so that it can be exercised on CPU with the gloo
backend (tests/test_replicas.py); it contains none of the method's arithmetic.
"""
from __future__ import annotations

import os


def env_rank():
    """(rank, local_rank, world_size) as torchrun exports them; (0, 0, 1) for a plain `python bench.py`."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


class Replicas:
    """One replica per rank.  backend: "nccl" on GPUs, "gloo" on CPU (tests)."""

    def __init__(self, backend="nccl", device=None):
        self.rank, self.local_rank, self.world = env_rank()
        self.device = device
        self.dist = None
        if self.world > 1:
            import torch
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            kw = {}
            if backend == "nccl" and device is not None:
                kw["device_id"] = torch.device(device)
            if not dist.is_initialized():
                dist.init_process_group(backend, **kw)
            self.dist = dist

    def barrier(self):
        """all ranks reach this point (and, on a GPU, their queued work has finished)"""
        if self.dist is not None:
            self.dist.barrier()
        if self.device is not None and str(self.device).startswith("cuda"):
            import torch
            torch.cuda.synchronize()

    def max_over_ranks(self, x: float) -> float:
        """the slowest replica's time: the job is done when the last rank is"""
        if self.dist is None:
            return float(x)
        import torch
        t = torch.tensor([x], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def whole_job_rate(self, units_per_rank: float, seconds_this_rank: float) -> float:
        """units all ranks processed / the slowest rank's time ("scaling": "weak": per-rank work is fixed)"""
        return units_per_rank * self.world / self.max_over_ranks(seconds_this_rank)

    def close(self):
        if self.dist is not None and self.dist.is_initialized():
            self.dist.destroy_process_group()
            self.dist = None
