"""Multi-GPU sharding of an hsg job: by disorder sample, with no data-path collective.

PAPER.md:115: "completely independent simulations of different disorder realizations are easily
parallelized also over different GPU devices".  Parallel tempering couples only the temperatures of one
(sample, replica) and the overlaps only the replicas of one sample, so a rank that owns a contiguous
block of samples never talks to another rank while sweeping.  ``hsg_desc.sample_offset`` keys every
random stream by the GLOBAL sample id, which makes a G-rank run reproduce the 1-rank run bit for bit.

This module holds only the shard arithmetic and the gather of per-sample observables (index and
communication plumbing; no method arithmetic).  It works with any ``torch.distributed`` backend
(``nccl`` on GPUs, ``gloo`` in the CPU tests).
"""
from __future__ import annotations

from typing import List, Sequence, Tuple


def shard_bounds(n_samples: int, world_size: int) -> List[Tuple[int, int]]:
    """[(sample_offset, count)] per rank: contiguous blocks, the first ``n_samples % world_size`` ranks
    own one sample more.  Ranks beyond the number of samples own an empty block."""
    if n_samples < 0 or world_size < 1:
        raise ValueError("shard_bounds: n_samples >= 0 and world_size >= 1 required")
    base, extra = divmod(n_samples, world_size)
    out, off = [], 0
    for r in range(world_size):
        cnt = base + (1 if r < extra else 0)
        out.append((off, cnt))
        off += cnt
    return out


def shard_of_rank(n_samples: int, world_size: int, rank: int) -> Tuple[int, int]:
    """(sample_offset, count) of ``rank``: pass them to ``hsg_create(..., n_samples=count, sample_offset=offset)``.
    count == 0 (more ranks than samples): the rank creates no engine (``hsg_create`` refuses an empty context) and passes a
    zero-length tensor to ``gather_by_sample``."""
    if not 0 <= rank < world_size:
        raise ValueError("shard_of_rank: rank out of range")
    return shard_bounds(n_samples, world_size)[rank]


def owner_of_sample(n_samples: int, world_size: int, d: int) -> Tuple[int, int]:
    """(rank, local index) of global sample ``d``."""
    if not 0 <= d < n_samples:
        raise ValueError("owner_of_sample: sample out of range")
    for r, (off, cnt) in enumerate(shard_bounds(n_samples, world_size)):
        if off <= d < off + cnt:
            return r, d - off
    raise AssertionError("unreachable")


def gather_by_sample(local, n_samples: int, group=None):
    """All-gather per-sample observables: ``local`` is this rank's tensor [count, ...] (leading index = local
    sample); returns the tensor [n_samples, ...] in global sample order on every rank.  Shards may differ in
    size by one sample (``shard_bounds``); the exchange pads to the largest shard.  This is the ONLY
    communication of a sharded job and it is outside the hot path (a few kB per measurement)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        if local.shape[0] != n_samples:
            raise ValueError("gather_by_sample: single process must hold every sample")
        return local
    world = dist.get_world_size(group)
    bounds = shard_bounds(n_samples, world)
    rank = dist.get_rank(group)
    if local.shape[0] != bounds[rank][1]:
        raise ValueError(f"gather_by_sample: rank {rank} holds {local.shape[0]} samples, expected {bounds[rank][1]}")
    cap = max(c for _, c in bounds)
    tail = tuple(local.shape[1:])
    padded = torch.zeros((cap,) + tail, dtype=local.dtype, device=local.device)
    padded[: local.shape[0]] = local
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded.contiguous(), group=group)
    return torch.cat([p[:c] for p, (_, c) in zip(parts, bounds)], dim=0)


def max_over_ranks(values: Sequence[float], device=None, group=None) -> List[float]:
    """MAX all-reduce of a few timings (bench.py: a multi-GPU time is the slowest rank's)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return [float(v) for v in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return t.tolist()
