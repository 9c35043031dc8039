"""Rank plumbing for `bench.py --gpus N`: the path does not shard ("replicas only"), so every rank
runs an independent replica; the only cross-rank operations are the timing barrier and the max-over-ranks
reduction of the device time.  No data-path collective.  Backend "nccl" on GPUs, "gloo" in the CPU tests."""
from __future__ import annotations

import os


def dist_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


class Ranks:
    def __init__(self, backend: str = "nccl", device=None):
        self.rank, self.world, self.local = dist_env()
        self.device = device
        self._dist = None
        if self.world > 1:
            import torch.distributed as dist
            kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
            dist.init_process_group(backend, **kw)
            self._dist = dist

    def barrier(self):
        if self._dist is not None:
            self._dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        if self._dist is None:
            return float(x)
        import torch
        t = torch.tensor([float(x)], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self._dist.all_reduce(t, op=self._dist.ReduceOp.MAX)
        return float(t.item())

    def whole_job_rate(self, units_per_rank: float, seconds_this_rank: float) -> float:
        """units all ranks processed / max-over-ranks time (every rank processes the same number of units)."""
        return self.world * units_per_rank / self.max_over_ranks(seconds_this_rank)

    def close(self):
        if self._dist is not None:
            self._dist.destroy_process_group()
            self._dist = None
