"""Multi-GPU plumbing: N independent replicas, one process per GPU (replicas only).

The path has no exchange step -- units (segment, layer, kv head, token) are independent (PAPER.md:131 is a
per-token re-rotation; BASELINE.json north_star: "one GPU, no sharding, no collectives") -- so no data-path
collective exists.  torch.distributed is used for exactly two control-plane things: a barrier around the timed
region and the max-over-ranks / sum-over-ranks reduction of the timing and token counts.  Works with the
`nccl` backend on GPUs and with `gloo` on CPU (tests/test_replicas.py, world_size 2).
"""
import os

import torch
import torch.distributed as dist


class Replicas:
    def __init__(self, backend=None, device=None):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device
        self.backend = backend
        self._own = False
        if self.world > 1 and not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            backend = backend or ("nccl" if torch.cuda.is_available() else "gloo")
            kw = {}
            if backend == "nccl" and device is not None:
                kw["device_id"] = torch.device(device)
            dist.init_process_group(backend=backend, rank=self.rank, world_size=self.world, **kw)
            self.backend = backend
            self._own = True

    def _t(self, x, dtype):
        dev = self.device if (self.backend == "nccl" and self.device is not None) else "cpu"
        return torch.tensor([x], dtype=dtype, device=dev)

    def barrier(self):
        if self.world > 1:
            dist.barrier()

    def max(self, x: float) -> float:
        if self.world == 1:
            return float(x)
        t = self._t(x, torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum(self, x: int) -> int:
        if self.world == 1:
            return int(x)
        t = self._t(x, torch.int64)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return int(t.item())

    def close(self):
        if self._own and dist.is_initialized():
            dist.destroy_process_group()
            self._own = False


def aggregate_throughput(rep: Replicas, units_this_rank: int, seconds_this_rank: float) -> dict:
    """Whole-job throughput of N replicas: all units processed / the slowest rank's time."""
    total = rep.sum(units_this_rank)
    t = rep.max(seconds_this_rank)
    return {"units": total, "seconds": t, "per_second": (total / t) if t > 0 else float("inf")}
