"""Multi-GPU plumbing: which rank owns which streams, and the over-ranks reductions of bench.py.

Streams are independent units (the paper scales by replicating servers and
splitting data into time-contiguous segments) and one stream's updates are strictly serial
(PAPER.md:174), so the path shards by stream and has NO data-path collective (DESIGN.md "Multi-GPU",
SURVEY.md 8(e)): every GPU holds the rings, overlap-add state and a full copy of the weights for its own
streams.  What crosses ranks is bookkeeping only: the max-over-ranks timing and, when one consumer
wants them, the per-stream scores gathered to rank 0.  No arithmetic of the method lives here.
"""
from __future__ import annotations

from typing import List, Sequence


def streams_of_rank(n_total: int, world: int, rank: int) -> List[int]:
    """Global stream ids owned by `rank`: stream i lives on GPU i mod world."""
    if world < 1 or not 0 <= rank < world or n_total < 0:
        raise ValueError(f"bad partition request: n_total={n_total} world={world} rank={rank}")
    return list(range(rank, n_total, world))


def rank_of_stream(i: int, world: int) -> int:
    return i % world


def local_index(i: int, world: int) -> int:
    """Position of global stream i inside its owner's batch (the row of that rank's [n][C][S] input)."""
    return i // world


def stream_seed(seed: int, i: int) -> int:
    """Stream i's input seed is seed + i, whichever rank owns it: results of
    a stream do not depend on how streams are spread over GPUs."""
    return seed + i


def max_over_ranks(value: float, device=None) -> float:
    """The timing rule of bench.py: a multi-GPU number is the MAX over ranks (collective on the default
    process group; identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_scores(local_scores: Sequence[float], n_total: int, device=None):
    """Per-stream scores of every rank, in GLOBAL stream order, on rank 0 (None elsewhere).  Not on the
    data path: one small gather per update for a single consumer."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return list(map(float, local_scores))
    world, rank = dist.get_world_size(), dist.get_rank()
    per = (n_total + world - 1) // world
    mine = torch.full((per,), float("nan"), dtype=torch.float32, device=device)
    own = streams_of_rank(n_total, world, rank)
    if len(local_scores) != len(own):
        raise ValueError(f"rank {rank} owns {len(own)} streams but holds {len(local_scores)} scores")
    if own:
        mine[:len(own)] = torch.as_tensor(list(local_scores), dtype=torch.float32, device=device)
    bufs = [torch.empty_like(mine) for _ in range(world)] if rank == 0 else None
    dist.gather(mine, bufs, dst=0)
    if rank != 0:
        return None
    out = [float("nan")] * n_total
    for r in range(world):
        for j, i in enumerate(streams_of_rank(n_total, world, r)):
            out[i] = float(bufs[r][j])
    return out
