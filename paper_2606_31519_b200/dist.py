"""Multi-GPU plumbing of the RaBitQCache path (host logic only; torch.distributed for the plumbing).

The path shards with NO data-path collective: every (sequence, KV-head group) is independent end to
end; BASELINE.json fixes the build to one GPU, so `bench.py --gpus N` runs N independent
layer replicas (weak scaling) and only the timing is reduced (max over ranks).  `kv_head_shard` is the
partition a tensor-parallel deployment would use (each rank owns a contiguous block of KV heads and
their G query heads; the only exchange would be an all-gather of the [B][Hq][D] outputs).
"""
from __future__ import annotations

import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init_process_group(backend: str):
    """Initialise torch.distributed from MASTER_ADDR / MASTER_PORT (127.0.0.1 rendezvous) when WORLD_SIZE > 1."""
    import torch.distributed as dist
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    """MAX all-reduce of a scalar (device timing is reported as the max over ranks)."""
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


def shard_range(n_units: int, rank: int, world: int):
    """Contiguous, balanced [lo, hi) of `n_units` independent units for `rank` (first n % world ranks get one more)."""
    if world <= 0 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n_units, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def kv_head_shard(n_kv_heads: int, n_q_heads: int, rank: int, world: int):
    """KV heads [g0, g1) and their query heads [h0, h1) owned by `rank`."""
    if n_q_heads % n_kv_heads:
        raise ValueError("n_q_heads must be a multiple of n_kv_heads")
    G = n_q_heads // n_kv_heads
    g0, g1 = shard_range(n_kv_heads, rank, world)
    return (g0, g1), (g0 * G, g1 * G)
