"""Host-side plumbing for `bench.py --gpus N`: independent replicas, one process per GPU.

DESIGN.md section 8: the north star drops the paper's inter-GPU layer (PAPER.md L192-230:
halo exchange, migration, the Allreduce of the time step), so the hot path has no data-path
collective.  Additional GPUs step independent replicas of the same workload ("replicas only",
weak scaling).  What is left for `torch.distributed` is the measurement protocol: a barrier on
both sides of the timed region, the MAX over ranks of the device-timed duration, and the SUM of
the units processed.  Nothing here touches particle data.

Works with the `nccl` backend (GPU box) and with `gloo` (CPU tests, world size 2).
"""
from __future__ import annotations

import os
from dataclasses import dataclass

import torch
import torch.distributed as dist


@dataclass
class Replica:
    rank: int
    world: int
    local_rank: int
    backend: str | None      # None: single process, no process group

    @property
    def is_root(self) -> bool:
        return self.rank == 0


def env_rank() -> tuple[int, int, int]:
    """(RANK, WORLD_SIZE, LOCAL_RANK) as torchrun exports them; (0, 1, 0) without torchrun."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str | None = None) -> Replica:
    """Join the process group when WORLD_SIZE > 1.  backend = None picks nccl when CUDA is
    available, else gloo.  MASTER_ADDR / MASTER_PORT come from the launcher (127.0.0.1)."""
    rank, world, local = env_rank()
    if world == 1:
        return Replica(0, 1, local, None)
    if backend is None:
        backend = "nccl" if torch.cuda.is_available() else "gloo"
    if backend == "nccl":
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        dist.init_process_group(backend)
    return Replica(rank, world, local, backend)


def _reduce_device(r: Replica) -> torch.device:
    return torch.device("cuda", r.local_rank) if r.backend == "nccl" else torch.device("cpu")


def barrier(r: Replica) -> None:
    """Device-complete on this rank, then all ranks, then device-complete again (the bracket
    the bench contract asks for around the timed region)."""
    if torch.cuda.is_available():
        torch.cuda.synchronize()
    if r.world > 1:
        dist.barrier()
        if torch.cuda.is_available():
            torch.cuda.synchronize()


def max_over_ranks(r: Replica, x: float) -> float:
    """Slowest rank's value of a duration (every rank gets the result)."""
    if r.world == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=_reduce_device(r))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(r: Replica, x: float) -> float:
    """Whole-job total of a count (units processed by all replicas)."""
    if r.world == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=_reduce_device(r))
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_rate(r: Replica, units_local: float, ms_local: float) -> tuple[float, float]:
    """(whole-job units per second, max-over-ranks milliseconds): total units of all replicas
    divided by the slowest replica's time - the value bench.py reports at N GPUs."""
    ms = max_over_ranks(r, ms_local)
    units = sum_over_ranks(r, units_local)
    return units / (ms * 1e-3), ms


def finalize(r: Replica) -> None:
    if r.world > 1 and dist.is_initialized():
        dist.destroy_process_group()
