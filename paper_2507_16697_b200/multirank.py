"""Host-side rank logic for `bench.py --gpus N` (one process per GPU, no data-path collective).

The RingX hot path on one node has no exchange step (the north_star excludes collectives): batch x heads are
independent units, so every rank runs the workload on its own seeded batch ("weak" scaling) and the
only communication is a barrier and a MAX-reduction of the timed region.  `shard_units` is the partition a
strong-scaling caller would use to split B*H heads over ranks with no communication.
"""
from __future__ import annotations

import dataclasses

import torch


def rank_config(cfg, rank: int):
    """The per-rank workload: same shapes, its own seed (so ranks do not share inputs)."""
    return dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank)


def shard_units(n_units: int, world: int, rank: int) -> range:
    """Contiguous, balanced partition of `n_units` independent (batch, head) units: covers every unit exactly once,
    sizes differ by at most one."""
    base, rem = divmod(n_units, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX-reduce a per-rank timing (milliseconds or seconds) over the process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_tflops(world: int, flops_per_rank_step: float, ms_per_step: float) -> float:
    """Whole-job throughput: the units all ranks processed divided by the max-over-ranks time."""
    return world * flops_per_rank_step / (ms_per_step * 1e-3) / 1e12
