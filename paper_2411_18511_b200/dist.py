"""Multi-GPU plumbing for bench.py.  The path does not exchange data between GPUs (BASELINE.json north_star:
"no MPI and no collectives"): every rank applies the operators to its own lattice replica, so the
only collectives are the barrier and the max/sum over ranks of the timing — torch.distributed over NCCL on GPUs,
gloo on CPU (tests)."""
from __future__ import annotations

import os


class Ranks:
    """One process per GPU; a single process when WORLD_SIZE is unset or 1."""

    def __init__(self, backend=None, device=None):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device
        self.dist = None
        if self.world > 1:
            import torch
            import torch.distributed as dist
            if backend is None:
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            if not dist.is_initialized():
                os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
                os.environ.setdefault("MASTER_PORT", "29533")
                kw = {}
                if backend == "nccl":
                    kw["device_id"] = torch.device("cuda", self.local_rank)
                dist.init_process_group(backend=backend, rank=self.rank, world_size=self.world, **kw)
            self.dist = dist
            self.backend = backend
            if self.device is None:
                self.device = "cuda:%d" % self.local_rank if backend == "nccl" else "cpu"

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def _reduce(self, value, op):
        if self.dist is None:
            return float(value)
        import torch
        t = torch.tensor([float(value)], dtype=torch.float64, device=self.device)
        self.dist.all_reduce(t, op=op)
        return float(t.item())

    def max(self, value):
        return self._reduce(value, self.dist.ReduceOp.MAX if self.dist else None)

    def sum(self, value):
        return self._reduce(value, self.dist.ReduceOp.SUM if self.dist else None)

    def close(self):
        if self.dist is not None and self.dist.is_initialized():
            self.dist.destroy_process_group()


def whole_job_throughput(ranks: Ranks, units_this_rank: float, seconds_this_rank: float):
    """value = units all ranks processed / max over ranks of the time (bench.py contract)."""
    t = ranks.max(seconds_this_rank)
    u = ranks.sum(units_this_rank)
    return u / t, t
