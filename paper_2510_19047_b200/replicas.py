"""Replica plumbing for ``bench.py --gpus N`` ("replicas only").

Templates are independent (one tile per GPU, no communication) and
BASELINE.json fixes a single-GPU path, so there is NO data-path collective here: every rank
runs the whole hot path on its own context and its own slice of the seeded template bank.
``torch.distributed`` is used for exactly two things: the barrier around the timed region and
the max-over-ranks of the measured time.  Works with ``nccl`` (GPU box) and ``gloo`` (CPU tests).
"""
from __future__ import annotations

import os
from dataclasses import dataclass


@dataclass(frozen=True)
class RankInfo:
    rank: int
    world: int
    local_rank: int

    @staticmethod
    def from_env(env=None) -> "RankInfo":
        e = os.environ if env is None else env
        return RankInfo(int(e.get("RANK", "0")), int(e.get("WORLD_SIZE", "1")), int(e.get("LOCAL_RANK", "0")))


def bank_seed(base_seed: int, rank: int) -> int:
    """Seed of rank r's template bank: disjoint streams, rank 0 identical to the 1-GPU run."""
    return base_seed + 7919 * rank


def init(info: RankInfo, backend: str, device=None):
    """Join the process group (no-op for world == 1).  Rendezvous comes from MASTER_ADDR/PORT."""
    if info.world == 1:
        return None
    import torch.distributed as dist
    if not dist.is_initialized():
        kw = {}
        if backend == "nccl" and device is not None:
            kw["device_id"] = device
        dist.init_process_group(backend, rank=info.rank, world_size=info.world, **kw)
    return dist


def barrier(info: RankInfo):
    if info.world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value: float, info: RankInfo, device="cpu") -> float:
    """Max of a per-rank scalar (the timed region's duration) over all ranks."""
    if info.world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank: int, seconds_max: float, info: RankInfo) -> float:
    """Whole-job throughput: units all ranks processed / slowest rank's time."""
    return info.world * units_per_rank / seconds_max


def finish(info: RankInfo):
    if info.world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()
