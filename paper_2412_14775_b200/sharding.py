"""Multi-GPU plumbing: one process per GPU, baselines partitioned across ranks, no data-path collective.

Every (baseline, channel) stream is mitigated separately, so the path shards by baseline (or by
subband / time chunk) with no exchange step: each rank runs the same kernel on its own slice and writes its own
slice of the outputs.  The only collectives are bookkeeping: the max-over-ranks of a device-measured time and the
sum of the per-set confusion counters against an injected ground truth (PAPER.md:235 definitions).  Both are
plain `torch.distributed` all-reduces and work on the nccl (GPU) and gloo (CPU tests) backends alike.
This module holds none of the method's arithmetic.
"""
from __future__ import annotations

from typing import Optional, Tuple

import torch


def shard_baselines(n_baselines: int, world_size: int, rank: int) -> Tuple[int, int]:
    """Contiguous balanced partition: (b_first, b_count) of `rank`; the first n % world ranks get one more."""
    if not (0 <= rank < world_size) or n_baselines < 0:
        raise ValueError("bad rank / world_size")
    q, r = divmod(n_baselines, world_size)
    first = rank * q + min(rank, r)
    return first, q + (1 if rank < r else 0)


def rank_work(n_baselines: int, world_size: int, rank: int, scaling: str = "weak", base_seed: int = 1234) -> dict:
    """What `rank` processes in bench.py --gpus N.
    weak:   every rank owns its own subband chunk (all baselines, seed base+rank) -- per-GPU work fixed.
    strong: ONE chunk (seed base, the same on every rank) partitioned by baseline -- total work fixed; the rank's plan
            is restricted with rfi_plan_set_baseline_shard(b_first, b_count).  world_size 1 is never sharded."""
    if scaling not in ("weak", "strong"):
        raise ValueError("scaling must be 'weak' or 'strong'")
    if scaling == "strong" and world_size > 1:
        b0, bc = shard_baselines(n_baselines, world_size, rank)
        if bc < 1:
            raise ValueError("more ranks than baselines")
        return {"sharded": True, "b_first": b0, "b_count": bc, "seed": base_seed}
    if not (0 <= rank < world_size):
        raise ValueError("bad rank / world_size")
    return {"sharded": False, "b_first": 0, "b_count": n_baselines, "seed": base_seed + rank}


def sum_scalar_over_ranks(value, device=None, group=None) -> float:
    """SUM all-reduce of a scalar (samples or bytes processed by each rank)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return float(t.item())


def max_over_ranks(value: float, device=None, group=None) -> float:
    """MAX all-reduce of a scalar (e.g. milliseconds measured with CUDA events on each rank)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def confusion_counts(flags: torch.Tensor, truth: torch.Tensor) -> torch.Tensor:
    """int64 [K, 4]: per threshold set (false alarms, clean windows, missed detections, RFI windows) of this
    rank's slice.  flags bool [K, n_win, cells]; truth bool [n_win, cells].  Harness bookkeeping, not the method."""
    f = flags.bool()
    t = truth.bool().unsqueeze(0)
    return torch.stack([(f & ~t).flatten(1).sum(1), (~t).expand_as(f).flatten(1).sum(1),
                        (~f & t).flatten(1).sum(1), t.expand_as(f).flatten(1).sum(1)], 1).to(torch.int64)


def sum_over_ranks(counts: torch.Tensor, group=None) -> torch.Tensor:
    """SUM all-reduce (in place) of the K x 4 confusion counters: the one exchange the sweep needs."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(counts, op=dist.ReduceOp.SUM, group=group)
    return counts


def rates(counts: torch.Tensor):
    """(false-alarm probability, missed-detection probability) per set from summed counters."""
    c = counts.to(torch.float64)
    return c[:, 0] / c[:, 1].clamp(min=1), c[:, 2] / c[:, 3].clamp(min=1)
