"""Multi-GPU plumbing for the Pici hot path: REPLICAS ONLY.

Every kernel of the path is rank-local and the north-star keeps all P logical ranks of a collective inside
one GPU's HBM, so there is no data-path collective between GPUs.  With N processes (one per GPU) each
process runs the same per-GPU workload on its own buffers, drawn from rank-specific seeds ("each process
uses a distinct pseudorandom seed").  torch.distributed is used only to agree on the timing
(max over ranks) and to sum the units processed.  Works with the nccl backend on GPUs and with gloo on CPU
(tests/test_replicas_gloo.py, world_size 2).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def world() -> tuple[int, int]:
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def rank_seeds(config_seed: int, rank: int, k: int) -> list[int]:
    """k distinct stream seeds for replica `rank` of a config with seed S.  Logical rank j of the config uses
    stream S*1000 + j (workloads.py, j < 999); replica r > 0 moves to its own block of 1 000 000 seeds, so replica 1
    of seed 0 can never equal replica 0 of seed 1 (replica 0 keeps the config's own streams)."""
    assert 0 <= config_seed < 1000 and 0 <= k < 999
    return [rank * 1_000_000 + config_seed * 1000 + j for j in range(k)]


def max_over_ranks(value: float, device="cpu") -> float:
    """Timing rule: a multi-GPU number is the MAX over ranks of the device-measured time."""
    _, w = world()
    if w == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    _, w = world()
    if w == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_throughput(units_this_rank: float, ms_this_rank: float, device="cpu") -> tuple[float, float]:
    """(units per second over all ranks, max-over-ranks ms): value = sum(units) / max(time)."""
    ms = max_over_ranks(ms_this_rank, device)
    units = sum_over_ranks(units_this_rank, device)
    return units / (ms * 1e-3), ms
