"""The N > 1 path on CPU: two gloo ranks run the host-side sharding logic that bench.py and a
multi-GPU caller use (paper_2606_26547_b200/shard.py).  The per-shard `classify_rows` is a stand-in
that labels a row by a function of its global index, so that a wrong bound, a dropped row or a
shard stitched in the wrong place shows up in the gathered result.  No method arithmetic here."""
from __future__ import annotations

import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_26547_b200 import shard


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


@pytest.mark.parametrize("n,world", [(10, 2), (11, 2), (1, 2), (0, 3), (7, 7), (5, 8), (131072, 8)])
def test_shard_bounds_partition(n, world):
    prev = 0
    sizes = []
    for r in range(world):
        lo, hi = shard.shard_bounds(n, world, r)
        assert lo == prev and hi >= lo
        prev = hi
        sizes.append(hi - lo)
    assert prev == n
    assert max(sizes) - min(sizes) <= 1
    assert sizes == sorted(sizes, reverse=True)


def test_shard_bounds_rejects_bad_arguments():
    for args in ((4, 0, 0), (4, 2, 2), (4, 2, -1), (-1, 2, 0)):
        with pytest.raises(ValueError):
            shard.shard_bounds(*args)


def _worker(rank: int, world: int, port: int, n_total: int, out_dir: str):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seen = []

        def classify_rows(lo, hi):
            seen.append((lo, hi))
            idx = torch.arange(lo, hi, dtype=torch.int64)
            return ((idx * 7 + 3) % 26).to(torch.int32)

        labels = shard.classify_sharded(classify_rows, n_total)
        assert seen == [shard.shard_bounds(n_total, world, rank)]
        slow = shard.max_over_ranks(1.0 + rank)
        assert slow == float(world)
        if rank == 0:
            torch.save(labels, os.path.join(out_dir, "labels.pt"))
        else:
            assert labels is None
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_total", [1559, 2, 1])
def test_two_gloo_ranks_gather_every_label_once(tmp_path, n_total):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), n_total, str(tmp_path)), nprocs=world, join=True)
    labels = torch.load(os.path.join(str(tmp_path), "labels.pt"))
    idx = torch.arange(n_total, dtype=torch.int64)
    assert labels.dtype == torch.int32 and labels.shape == (n_total,)
    assert torch.equal(labels, ((idx * 7 + 3) % 26).to(torch.int32))


def test_single_process_paths_need_no_group():
    lab = shard.classify_sharded(lambda lo, hi: torch.arange(lo, hi, dtype=torch.int32), 5)
    assert lab.tolist() == [0, 1, 2, 3, 4]
    assert shard.max_over_ranks(2.5) == 2.5


def _train_worker(rank: int, world: int, port: int, out_dir: str):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n_total, batch = 103, 40
        state = {"C": torch.zeros(4, dtype=torch.int64), "calls": []}

        def delta_fn(lo, hi):                      # stand-in for hdc_train_delta: depends on the rows and on C
            state["calls"].append((lo, hi))
            idx = torch.arange(lo, hi, dtype=torch.int64)
            d = torch.zeros(4, dtype=torch.int64)
            d.index_add_(0, idx % 4, idx + state["C"].sum())
            return d

        def apply_fn(d):                           # stand-in for hdc_train_apply
            state["C"] = state["C"] + d

        shard.train_epoch_sharded(delta_fn, apply_fn, n_total, batch)
        torch.save((state["C"], state["calls"]), os.path.join(out_dir, f"train_{rank}.pt"))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_train_epoch_all_reduces_one_delta_per_mini_batch(tmp_path):
    world = 2
    mp.spawn(_train_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    C0, calls0 = torch.load(os.path.join(str(tmp_path), "train_0.pt"))
    C1, calls1 = torch.load(os.path.join(str(tmp_path), "train_1.pt"))
    assert torch.equal(C0, C1)                                         # identical replicas
    # single-process run of the same stand-ins
    state = {"C": torch.zeros(4, dtype=torch.int64)}

    def delta_fn(lo, hi):
        idx = torch.arange(lo, hi, dtype=torch.int64)
        d = torch.zeros(4, dtype=torch.int64)
        d.index_add_(0, idx % 4, idx + state["C"].sum())
        return d

    def apply_fn(d):
        state["C"] = state["C"] + d

    shard.train_epoch_sharded(delta_fn, apply_fn, 103, 40)
    assert torch.equal(state["C"], C0)
    # each mini-batch was split in two contiguous shards that tile it
    assert calls0 == [(0, 20), (40, 60), (80, 92)] and calls1 == [(20, 40), (60, 80), (92, 103)]
