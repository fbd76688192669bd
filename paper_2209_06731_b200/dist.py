"""Multi-GPU plumbing for the bench: the E×B term is diagonal in species and Hermite index
 and pointwise in z, so it shards over (s, m, z) with NO data-path collective
(the paper's own decomposition is species, then Hermite blocks: line 503).  Weak scaling: each rank
owns one Hermite block of Nm moments of a problem with Nm*world moments; phi and the tables are
replicated.  torch.distributed is used only for the barrier and the max-over-ranks of the time.
"""
from __future__ import annotations

import os


def env_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def hermite_block(Nm_per_rank: int, rank: int, world: int) -> tuple[int, int, int]:
    """(m_start, m_stop, Nm_global) of this rank's contiguous Hermite block (weak scaling)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return rank * Nm_per_rank, (rank + 1) * Nm_per_rank, Nm_per_rank * world


def init(backend: str):
    import torch.distributed as dist
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29533")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(units_this_rank: float, seconds_this_rank: float, device="cpu") -> tuple[float, float]:
    """Whole-job throughput = units all ranks processed / max-over-ranks time. -> (value, seconds)."""
    sec = max_over_ranks(seconds_this_rank, device)
    units = sum_over_ranks(units_this_rank, device)
    return units / sec, sec


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
