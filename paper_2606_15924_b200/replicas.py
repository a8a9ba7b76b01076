"""Replica plumbing for N > 1 (replicas only).

The views of one TurboGS iteration are independent (Alg. 1 step 2), so the hot path has no
exchange step: every rank runs the whole five-call step on its own view and nothing crosses the
interconnect in the data path.  What N ranks do share is the MEASUREMENT: a barrier on both sides of the
timed region, the max over ranks of the device time and the sum over ranks of the units processed.
``torch.distributed`` is used for exactly that (backend "nccl" on GPUs, "gloo" in the CPU tests).
"""
from __future__ import annotations

import os


class Replicas:
    def __init__(self, backend: str = "nccl", device=None):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device if device is not None else torch.device("cpu")
        self._own = False
        if self.world > 1 and not dist.is_initialized():
            kw = {"device_id": self.device} if backend == "nccl" else {}
            dist.init_process_group(backend, **kw)
            self._own = True

    # one view per rank: the index of rank r's view (the scene is replicated, the view differs; bench.py hands it to
    # workloads.orbit_view, rank 0 keeps the config's own camera)
    def view_seed(self, base_seed: int) -> int:
        return int(base_seed) + self.rank

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        if self.device.type == "cuda":
            self.torch.cuda.synchronize(self.device)

    def _reduce(self, value: float, op) -> float:
        if self.world == 1:
            return float(value)
        t = self.torch.tensor([float(value)], dtype=self.torch.float64, device=self.device)
        self.dist.all_reduce(t, op=op)
        return float(t.item())

    def max_over_ranks(self, value: float) -> float:
        """Timed regions are reported as the slowest rank's device time."""
        return self._reduce(value, self.dist.ReduceOp.MAX)

    def sum_over_ranks(self, value: float) -> float:
        """Units processed by the whole job (value = whole-job throughput numerator)."""
        return self._reduce(value, self.dist.ReduceOp.SUM)

    def throughput(self, units_this_rank: float, steps: int, ms_this_rank: float) -> float:
        """Whole-job units/s: all ranks' units divided by the slowest rank's time."""
        ms = self.max_over_ranks(ms_this_rank)
        units = self.sum_over_ranks(units_this_rank)
        return units * steps / (ms * 1e-3)

    def close(self):
        if self._own and self.dist.is_initialized():
            self.dist.destroy_process_group()
            self._own = False
