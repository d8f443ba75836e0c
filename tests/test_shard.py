"""Host logic of the data-parallel path: token-balanced document shards, no data-path
collective, scores concatenated afterwards.  Runs on CPU: the N > 1 path is exercised with two gloo processes,
each scoring its shard with the fp64 oracle (test infrastructure) in place of the CUDA call."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2606_26439_b200 import shard, synth


def test_bounds_partition_all_documents_and_balance_tokens():
    lens = synth.lognormal_lengths(10_000, seed=1)
    off = synth.offsets_from_lengths(lens)
    for world in (1, 2, 3, 8):
        b = shard.shard_bounds(off, world)
        assert b[0] == 0 and b[-1] == 10_000 and np.all(np.diff(b) >= 0)
        tokens = off[b[1:]] - off[b[:-1]]
        assert tokens.sum() == off[-1]
        assert np.abs(tokens - off[-1] / world).max() <= 180  # one document of slack (lengths are clipped at 180)


def test_shard_documents_rebases_offsets():
    off = synth.offsets_from_lengths(np.array([3, 0, 5, 2, 0, 7], dtype=np.int64))
    seen = []
    for r in range(3):
        b_lo, b_hi, t_lo, t_hi, local = shard.shard_documents(off, 3, r)
        assert local[0] == 0 and local[-1] == t_hi - t_lo
        assert np.array_equal(np.diff(local), np.diff(off[b_lo:b_hi + 1]))
        seen += list(range(b_lo, b_hi))
    assert seen == list(range(6))


def test_degenerate_shards():
    off = synth.offsets_from_lengths(np.array([5], dtype=np.int64))
    b = shard.shard_bounds(off, 4)  # more ranks than documents: some shards are empty
    assert b[0] == 0 and b[-1] == 1 and np.all(np.diff(b) >= 0)
    assert shard.max_over_ranks(3.5) == 3.5 and shard.sum_over_ranks(2.0) == 2.0  # no process group: identity


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q, D, off, ref, out):
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        b_lo, b_hi, t_lo, t_hi, local = shard.shard_documents(off, world, rank)
        local_scores = torch.from_numpy(oracle.maxsim(q, D[t_lo:t_hi], local))  # stands in for tms_maxsim on this rank
        full = shard.gather_scores(local_scores, world)
        ok = bool(np.array_equal(full.numpy(), ref))
        slowest = shard.max_over_ranks(float(rank + 1))
        total = shard.sum_over_ranks(float(b_hi - b_lo))
        out.put((rank, ok, slowest, total))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_two_ranks_score_their_shards_and_concatenate():
    world = 2
    lens = np.concatenate([[0, 1, 300], synth.lognormal_lengths(397, seed=3)])
    off = synth.offsets_from_lengths(lens)
    q = synth.unit_tokens(2 * 8, 32, torch.float32, seed=4).view(2, 8, 32)
    D = synth.unit_tokens(int(off[-1]), 32, torch.float32, seed=5)
    ref = oracle.maxsim(q, D, off)
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q, D, off, ref, out)) for r in range(world)]
    for p in procs:
        p.start()
    results = sorted(out.get(timeout=150) for _ in range(world))
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    for rank, ok, slowest, total in results:
        assert ok, f"rank {rank}: gathered scores differ from the single-process result"
        assert slowest == float(world) and total == float(len(lens))
