"""Multi-GPU plumbing.  The path shards with NO data-path collective: every (sequence, kv-head) unit is independent
through summarize -> select -> decode, so N GPUs run N replicas, each on its own batch slice and page
pool ("replicas only", weak scaling).  torch.distributed is used for the barrier and the max-over-ranks timing only."""
from __future__ import annotations

import os
from typing import List, Tuple

import torch
import torch.distributed as dist


def env_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1-process defaults)."""
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def init(backend: str) -> Tuple[int, int, int]:
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    if dist.is_initialized():
        dist.barrier()


def replica_seed(base_seed: int, rank: int) -> int:
    """Every replica draws its own batch (different lengths, page tables, K/V)."""
    return base_seed + 7 * rank


def shard_sequences(n_seq_total: int, rank: int, world: int) -> List[int]:
    """Strong-scaling helper: contiguous, balanced slice of a global batch for this rank."""
    base, rem = divmod(n_seq_total, world)
    lo = rank * base + min(rank, rem)
    return list(range(lo, lo + base + (1 if rank < rem else 0)))


def max_over_ranks(x: float, device="cpu") -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, device="cpu") -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_throughput(units_this_rank: float, seconds_this_rank: float, device="cpu") -> Tuple[float, float]:
    """(units all ranks processed / max-over-ranks time, that time)."""
    t = max_over_ranks(seconds_this_rank, device)
    u = sum_over_ranks(units_this_rank, device)
    return u / t, t
