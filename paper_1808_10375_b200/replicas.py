"""Multi-GPU plumbing of bench.py: independent replicas, one reconstruction per rank.

north_star fixes the path to one GPU (no sharding, no collective on the data path), so N GPUs
run N independent DM reconstructions.  torch.distributed is used for
exactly two things: a barrier around the timed region and the max-over-ranks of the device
time.  Backend "nccl" on the GPUs, "gloo" in the CPU tests (tests/test_replicas.py).
"""
from __future__ import annotations

import os


class ReplicaGroup:
    def __init__(self, backend: str = "nccl", device=None):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.backend, self.device, self._dist = backend, device, None
        if self.world > 1:
            import torch.distributed as dist
            kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
            dist.init_process_group(backend, **kw)
            self._dist = dist

    @property
    def seed(self) -> int:
        """Every replica reconstructs its own synthetic data set."""
        return self.rank

    def _sync_device(self):
        if self.backend == "nccl":
            import torch
            torch.cuda.synchronize()

    def barrier(self):
        self._sync_device()
        if self._dist is not None:
            self._dist.barrier()
        self._sync_device()

    def max_over_ranks(self, x: float) -> float:
        if self._dist is None:
            return float(x)
        import torch
        dev = self.device if self.backend == "nccl" else "cpu"
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        self._dist.all_reduce(t, op=self._dist.ReduceOp.MAX)
        return float(t.item())

    def aggregate(self, units_per_rank_per_step: int, steps: int, ms_max: float) -> float:
        """Whole-job throughput: the units all ranks processed / the slowest rank's time (weak scaling)."""
        return self.world * units_per_rank_per_step * steps / (ms_max * 1e-3)

    def close(self):
        if self._dist is not None:
            self._dist.destroy_process_group()
            self._dist = None
