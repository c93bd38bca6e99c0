"""Replica plumbing for ``bench.py --gpus N`` — rendezvous, barrier and whole-job aggregation.

The D-instance KV path shards by request with no exchange step inside it (DESIGN.md §8,
SURVEY §8(e): independent D-instances behind the Router), so N GPUs are N
independent replicas, one process each.  ``torch.distributed`` serves only

  * the barrier that brackets the timed region,
  * MAX over ranks of the device time (the job is as slow as its slowest replica),
  * SUM over ranks of the units processed (whole-job throughput = sum units / max time).

No KV byte, query or output ever crosses ranks.  The same code runs over NCCL on the GPU box
and over gloo on CPU (``tests/test_multirank_cpu.py``, world size 2).
"""
from __future__ import annotations

import os
from dataclasses import dataclass

import torch
import torch.distributed as dist


@dataclass
class Replicas:
    rank: int
    world: int
    local_rank: int
    device: torch.device       # where the reduction tensors live (cuda:<local> for nccl, cpu for gloo)
    backend: str | None        # None: single process, no process group

    @property
    def salt(self) -> int:
        """Per-rank salt of the seeded workload: every replica draws its OWN requests (weak scaling)."""
        return self.rank

    def barrier(self) -> None:
        if self.world > 1:
            if self.backend == "nccl":
                dist.barrier(device_ids=[self.local_rank])
            else:
                dist.barrier()
        if self.device.type == "cuda":
            torch.cuda.synchronize(self.device)

    def _reduce(self, x: float, op) -> float:
        if self.world == 1:
            return float(x)
        t = torch.tensor([x], dtype=torch.float64, device=self.device)
        dist.all_reduce(t, op=op)
        return float(t.item())

    def max(self, x: float) -> float:
        return self._reduce(x, dist.ReduceOp.MAX)

    def sum(self, x: float) -> float:
        return self._reduce(x, dist.ReduceOp.SUM)

    def throughput(self, units_this_rank: float, ms_this_rank: float) -> tuple[float, float]:
        """(whole-job units per second, max-over-ranks milliseconds)."""
        ms = self.max(ms_this_rank)
        return self.sum(units_this_rank) / (ms * 1e-3), ms

    def close(self) -> None:
        if self.world > 1 and dist.is_initialized():
            dist.destroy_process_group()


def init(backend: str | None = None) -> Replicas:
    """Read RANK / LOCAL_RANK / WORLD_SIZE (torchrun's env) and join the process group if WORLD_SIZE > 1.
    backend: "nccl" (default when CUDA is available) or "gloo"."""
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if backend is None:
        backend = "nccl" if torch.cuda.is_available() else "gloo"
    if backend == "nccl":
        torch.cuda.set_device(local)
        device = torch.device("cuda", local)
    else:
        device = torch.device("cpu")
    if world == 1:
        return Replicas(rank, world, local, device, None)
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    if backend == "nccl":
        dist.init_process_group("nccl", device_id=device)
    else:
        dist.init_process_group("gloo")
    return Replicas(rank, world, local, device, backend)
