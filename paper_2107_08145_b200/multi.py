"""N > 1 plumbing of bench.py (host logic only; no kernel).

Two ways to use several GPUs ("Multi-GPU"):
  weak    independent problems: as in the paper's weak-scaling runs (one 288^3 block per GPU, PAPER.md:297,
          sec. 6.4) every rank owns one block-local atmosphere and solves it on its own GPU; the only
          communication is the timing reduction (max over ranks);
  strong  ONE box sharded by band x octant: the sweep units are dealt round
          robin to the ranks (rts_set_shard), every rank sweeps its own units, and ONE sum all-reduce
          completes Q_rad and I_top (`allreduce_sum`).
Works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import os
from typing import Optional, Tuple


def env_ranks() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) without it."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def rank_seed_offset(rank: int) -> int:
    """Each rank's block is its own seeded atmosphere of the same recipe and size."""
    return 1000 * rank


def max_over_ranks(x: float, world: int, device: Optional[str] = None) -> float:
    """MAX all-reduce of one scalar (the slowest rank defines the step time)."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate(local_ms: float, local_units: float, world: int, device: Optional[str] = None) -> dict:
    """Whole-job throughput: units processed by all ranks / the slowest rank's time."""
    t = max_over_ranks(local_ms, world, device)
    return {"ms": t, "value": world * local_units / (t * 1e-3)}


def reference_arm_runs_here(rank: int) -> bool:
    """`bench.py --impl reference`: rank 0 alone runs and prints; the others exit 0."""
    return rank == 0


def shard_units(n_units: int, rank: int, nranks: int) -> list:
    """The sweep units (in the library's unit order) that rank `rank` of `nranks` sweeps: round robin,
    the rule of rts_set_shard."""
    if nranks < 1 or not (0 <= rank < nranks):
        raise ValueError("need 0 <= rank < nranks")
    return [u for u in range(n_units) if u % nranks == rank]


def allreduce_sum(world: int, *tensors):
    """The one data-path collective of the strong-scaling mode: sum over ranks of the partial Q_rad / I_top
    (in place; no-op for one rank)."""
    if world == 1:
        return
    import torch.distributed as dist
    for t in tensors:
        if t is not None:
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
