"""Host-side logic of the multi-GPU path.

Inference shards by queries: rank r owns a contiguous block of the query rows, the projection P and
the class hypervectors C are replicated, and no collective sits on the data path.  The only
exchanges are the ones a driver needs around the kernels: the max-over-ranks of a device time and
(optionally) collecting the label shards on rank 0.  Works on any torch.distributed backend (nccl on
the GPUs, gloo in the CPU tests); holds no arithmetic of the method.
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple

import torch
import torch.distributed as dist


def shard_bounds(n: int, world: int, rank: int) -> Tuple[int, int]:
    """Rows [lo, hi) of rank `rank` when n rows are split over `world` ranks: contiguous blocks, the
    first n % world ranks get one row more (every row owned exactly once, blocks in rank order)."""
    if world < 1 or not 0 <= rank < world or n < 0:
        raise ValueError("bad shard arguments")
    q, r = divmod(n, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def max_over_ranks(value: float, device: Optional[torch.device] = None) -> float:
    """The largest `value` any rank holds (a step time is the slowest rank's)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_labels(local: torch.Tensor, n_total: int) -> Optional[torch.Tensor]:
    """Collects the per-rank label shards (shard_bounds order) into one [n_total] int32 tensor on
    rank 0; other ranks get None.  Shards may differ in length by one row (ragged gather through
    padding to the longest shard)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        assert local.numel() == n_total
        return local
    world, rank = dist.get_world_size(), dist.get_rank()
    longest = -(-n_total // world)
    pad = torch.full((longest,), -1, dtype=torch.int32, device=local.device)
    pad[: local.numel()] = local.to(torch.int32)
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    if rank != 0:
        return None
    out = torch.empty(n_total, dtype=torch.int32, device=local.device)
    for r in range(world):
        lo, hi = shard_bounds(n_total, world, r)
        out[lo:hi] = parts[r][: hi - lo]
    return out


def classify_sharded(classify_rows: Callable[[int, int], torch.Tensor], n_total: int) -> Optional[torch.Tensor]:
    """Runs `classify_rows(lo, hi)` (labels of query rows [lo, hi), e.g. hdc_encode_rp + hdc_classify
    on this rank's GPU) on this rank's shard and gathers the labels on rank 0."""
    world = dist.get_world_size() if dist.is_initialized() else 1
    rank = dist.get_rank() if dist.is_initialized() else 0
    lo, hi = shard_bounds(n_total, world, rank)
    local = classify_rows(lo, hi)
    assert local.numel() == hi - lo
    return gather_labels(local, n_total)


def train_epoch_sharded(delta_fn: Callable[[int, int], torch.Tensor], apply_fn: Callable[[torch.Tensor], None],
                        n_total: int, batch: int = 0) -> None:
    """One data-parallel retraining epoch: the samples of every mini-batch are
    split over the ranks (shard_bounds inside the mini-batch), `delta_fn(lo, hi)` returns this rank's
    int32 class update of global samples [lo, hi) against the current accumulators (hdc_train_delta),
    the deltas are summed over the ranks with ONE all-reduce per mini-batch, and `apply_fn(delta)`
    applies the sum (hdc_train_apply).  Integer addition commutes, so every rank applies the same
    delta and the replicas of the class accumulators stay bit-identical to a single-GPU epoch."""
    world = dist.get_world_size() if dist.is_initialized() else 1
    rank = dist.get_rank() if dist.is_initialized() else 0
    B = n_total if batch in (0, None) or batch > n_total else int(batch)
    for b0 in range(0, n_total, B):
        nb = min(B, n_total - b0)
        lo, hi = shard_bounds(nb, world, rank)
        delta = delta_fn(b0 + lo, b0 + hi)
        if world > 1:
            dist.all_reduce(delta, op=dist.ReduceOp.SUM)
        apply_fn(delta)
