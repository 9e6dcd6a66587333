"""Multi-GPU plumbing for the bench: REPLICAS ONLY.

BASELINE.json fixes one GPU, no sharding and no collectives for this path, so N GPUs run N independent replicas of
the same workload, one process per GPU.  torch.distributed is used only for the barrier around the timed region and
for the max-over-ranks of the device time; no data-path collective exists.  Backend "nccl" on GPUs, "gloo" in the
CPU tests (tests/test_replicas_gloo.py, world_size 2).
"""
from __future__ import annotations

import os


class Replicas:
    def __init__(self, backend: str | None = None, device=None):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device
        self._dist = None
        if self.world > 1:
            import torch.distributed as dist
            self._dist = dist
            if not dist.is_initialized():
                kw = {}
                if backend == "nccl" and device is not None:
                    kw["device_id"] = device
                dist.init_process_group(backend or "nccl", **kw)

    def barrier(self):
        if self._dist is not None:
            self._dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        """max of a per-rank scalar (the device time of the timed region)."""
        if self._dist is None:
            return float(x)
        import torch
        t = torch.tensor([float(x)], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self._dist.all_reduce(t, op=self._dist.ReduceOp.MAX)
        return float(t.item())

    def aggregate_rate(self, units_per_rank_step: float, steps: int, t_ms_local: float):
        """Whole-job throughput: units all ranks processed / max-over-ranks time.  Returns (value, t_ms_max)."""
        t_ms = self.max_over_ranks(t_ms_local)
        return self.world * steps * units_per_rank_step / (t_ms * 1e-3), t_ms

    def is_reporter(self) -> bool:
        return self.rank == 0

    def close(self):
        if self._dist is not None and self._dist.is_initialized():
            self._dist.destroy_process_group()
