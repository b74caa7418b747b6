"""The N > 1 path on CPU: world_size 2 over gloo.  Streams shard by rank with no data-path collective
(DESIGN.md "Multi-GPU"); what is tested here is the host logic that surrounds the kernels: the
stream -> rank partition, per-stream seeding independent of the partition, the max-over-ranks timing
reduction bench.py uses, and the gather of per-stream scores in global order."""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2108_12430_b200 import shard
from paper_2108_12430_b200 import specs as S
from paper_2108_12430_b200 import synth


def test_partition_covers_every_stream_once():
    for n in (0, 1, 2, 7, 128, 513):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                own = shard.streams_of_rank(n, world, r)
                assert all(shard.rank_of_stream(i, world) == r for i in own)
                assert [shard.local_index(i, world) for i in own] == list(range(len(own)))
                seen += own
            assert sorted(seen) == list(range(n))
            sizes = [len(shard.streams_of_rank(n, world, r)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def test_partition_rejects_bad_arguments():
    with pytest.raises(ValueError):
        shard.streams_of_rank(4, 0, 0)
    with pytest.raises(ValueError):
        shard.streams_of_rank(4, 2, 2)


def test_single_process_reductions_are_identities():
    assert shard.max_over_ranks(3.5) == 3.5
    assert shard.gather_scores([0.25, 0.5], 2) == [0.25, 0.5]


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, n_total: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        own = shard.streams_of_rank(n_total, world, rank)
        # every rank synthesises only its own streams; stream i's samples depend on i alone
        sp = S.StreamSpec(len(own), 2, 4096, 256, 64)
        one = S.StreamSpec(1, 2, 4096, 256, 64)
        x = np.stack([synth.stream_channels(shard.stream_seed(11, i), one, 128) for i in own]) if own else \
            np.zeros((0, one.channels, 128), np.float32)
        assert x.shape == (len(own), sp.channels, 128)
        # stand-in "score" per stream: a checksum of its input (the kernels need a GPU; the plumbing does not)
        local = [float(np.float32(x[j].astype(np.float64).sum() % 1.0)) for j in range(len(own))]
        allsc = shard.gather_scores(local, n_total)
        t = shard.max_over_ranks(1.0 + rank)
        ids = [None] * world
        dist.all_gather_object(ids, own)
        if rank == 0:
            assert t == float(world)
            assert sorted(i for part in ids for i in part) == list(range(n_total))
            np.save(os.path.join(out_dir, "scores.npy"), np.asarray(allsc, dtype=np.float64))
        else:
            assert allsc is None and t == float(world)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_total", [5, 8])
def test_world2_gloo_partition_gather_and_max(tmp_path, n_total):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), n_total, str(tmp_path)), nprocs=world, join=True)
    got = np.load(tmp_path / "scores.npy")
    one = S.StreamSpec(1, 2, 4096, 256, 64)
    want = [float(np.float32(synth.stream_channels(shard.stream_seed(11, i), one, 128).astype(np.float64).sum() % 1.0))
            for i in range(n_total)]
    # global order restored, and identical to what a single process computes for the same streams
    assert np.array_equal(got, np.asarray(want))


def test_bench_reference_arm_runs_only_on_rank0(monkeypatch, capsys):
    """Under torchrun the reference arm prints from rank 0 alone; other ranks exit without work."""
    import importlib
    bench = importlib.import_module("bench")
    monkeypatch.setenv("RANK", "1")
    ns = type("A", (), dict(streams=1, stride=512, dtype="fp16", warmup=0, steps=1, reference_budget=1.0, gpus=2))
    bench.run_reference(ns)
    assert capsys.readouterr().out == ""
