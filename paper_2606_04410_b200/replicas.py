"""Multi-GPU host logic: replicas only.

The chunk-decode path has no exchange step (single GPU, sequential chunk by chunk; BASELINE.json's configs
carry no temporal context), so N GPUs = N independent decoders.  The only collectives are the timing barrier and the
max-over-ranks of the elapsed time; chunks of a job are dealt round-robin.  Works on any torch.distributed backend
(nccl on the GPU box, gloo in the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def world() -> tuple[int, int]:
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def shard_chunks(n_chunks_total: int, rank: int, world_size: int) -> list[int]:
    """Indices of the chunks rank `rank` decodes: round-robin, no communication needed."""
    return list(range(rank, n_chunks_total, world_size))


def max_over_ranks(value: float, device: torch.device | str = "cpu") -> float:
    """Whole-job time = the slowest rank's time."""
    rank, ws = world()
    if ws == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank_step: int, steps: int, elapsed_ms_this_rank: float, device="cpu") -> float:
    """Aggregate units/s of the whole job: units all ranks processed / max-over-ranks time (weak scaling)."""
    _, ws = world()
    total_ms = max_over_ranks(elapsed_ms_this_rank, device)
    return ws * units_per_rank_step * steps / (total_ms / 1e3)
