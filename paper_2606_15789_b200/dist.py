"""Multi-GPU plumbing for bench.py: the path shards by independent batches (one replica of the layer and one
batch per GPU, weak scaling, NO data-path collective — DESIGN.md §10 "Multi-GPU").  torch.distributed is used only for the
timing contract: a barrier on both sides of the timed region and the MAX over ranks of the measured time."""
from __future__ import annotations

import os


class Ranks:
    def __init__(self, backend: str | None = None, device=None):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.dist = None
        self.device = device
        if self.world > 1:
            import torch.distributed as dist
            kw = {}
            if backend == "nccl" and device is not None:
                kw["device_id"] = device
            dist.init_process_group(backend or "gloo", **kw)
            self.dist = dist

    def batch_seed(self, base: int) -> int:
        """Every rank draws its own activations (its own batch of requests)."""
        return base + 97 * self.rank

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max_over_ranks(self, value: float) -> float:
        if self.dist is None:
            return float(value)
        import torch
        t = torch.tensor([float(value)], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def aggregate(self, units_per_rank: float, seconds_this_rank: float) -> float:
        """Whole-job throughput: units all ranks processed / the slowest rank's time."""
        return self.world * units_per_rank / self.max_over_ranks(seconds_this_rank)

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()
