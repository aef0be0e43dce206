"""Multi-GPU plumbing: one process per GPU, rows sharded with NO data-path collective.

The K parameter rows of a batch are independent (the paper evaluates one
row per iteration and has no multi-GPU path), so scaling out is "each rank evaluates
its own rows against a replica of the observation".  torch.distributed is used only for the
rendezvous, the barrier around the timed region, the max-over-ranks of the device time and the
sum of the rows processed.  Backend: nccl on GPUs, gloo in the CPU tests.
"""
from __future__ import annotations

import os
from dataclasses import dataclass


@dataclass
class Ranks:
    rank: int = 0
    world: int = 1
    local_rank: int = 0
    backend: str = ""

    @property
    def is_main(self) -> bool:
        return self.rank == 0


def init_from_env(backend: str = "nccl") -> Ranks:
    """Reads RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* (set by torch.distributed.run).  Without them
    (plain `python bench.py`) this is a single-rank job and torch.distributed is not touched."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world <= 1:
        return Ranks()
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29500")
    rank = int(os.environ["RANK"])
    local_rank = int(os.environ.get("LOCAL_RANK", rank))
    if backend == "nccl":
        import torch
        torch.cuda.set_device(local_rank)
    if not dist.is_initialized():
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return Ranks(rank, world, local_rank, backend)


def _tensor(r: Ranks, value: float):
    import torch
    dev = "cuda" if r.backend == "nccl" else "cpu"
    return torch.tensor([float(value)], dtype=torch.float64, device=dev)


def barrier(r: Ranks) -> None:
    if r.world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(r: Ranks, value: float) -> float:
    """Slowest rank's time: every multi-GPU number is the max over ranks, never a wall clock."""
    if r.world == 1:
        return float(value)
    import torch.distributed as dist
    t = _tensor(r, value)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(r: Ranks, value: float) -> float:
    if r.world == 1:
        return float(value)
    import torch.distributed as dist
    t = _tensor(r, value)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(r: Ranks, units_this_rank: float, seconds_this_rank: float) -> tuple:
    """(whole-job units / s, slowest rank's seconds): sum of units over ranks / max of time."""
    tmax = max_over_ranks(r, seconds_this_rank)
    units = sum_over_ranks(r, units_this_rank)
    return (units / tmax if tmax > 0 else float("nan")), tmax


def finalize(r: Ranks) -> None:
    if r.world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()
