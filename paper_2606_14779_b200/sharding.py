"""Host-side helpers for running the path on more than one GPU.

The path shards with no data-path collective: tensor-parallel ranks own disjoint KV heads of every block,
data-parallel ranks own disjoint requests, and placement is a pure function of (weights, K_l) so every rank
derives the same map on its own.  torch.distributed is used only for the bench's barrier / max-over-ranks
timing and, optionally, to agree on measured bandwidths.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple


def shard_heads(n_kv_heads: int, tp: int, rank: int) -> Tuple[int, int]:
    """(first head, number of heads) owned by tensor-parallel `rank`; heads must divide evenly."""
    if tp <= 0 or not 0 <= rank < tp:
        raise ValueError("bad tp / rank")
    if n_kv_heads % tp:
        raise ValueError(f"{n_kv_heads} KV heads do not divide over tp={tp}")
    per = n_kv_heads // tp
    return rank * per, per


def shard_requests(n_requests: int, world: int, rank: int) -> List[int]:
    """Requests owned by data-parallel `rank` (round-robin)."""
    if world <= 0 or not 0 <= rank < world:
        raise ValueError("bad world / rank")
    return list(range(rank, n_requests, world))


def max_over_ranks(values: Sequence[float], device=None) -> List[float]:
    """Element-wise max over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]


def agree_on_bandwidth(bandwidth_gbps: Sequence[float], device=None) -> List[float]:
    """Optional: make every rank use rank 0's measured bandwidths so that all ranks place identically."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in bandwidth_gbps]
    t = torch.tensor(list(bandwidth_gbps), dtype=torch.float64, device=device)
    dist.broadcast(t, src=0)
    return [float(x) for x in t.tolist()]
