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


def _bench_rank_worker(rank, world, port, out):
    """The rank logic of bench.py (shard.rank_seed, shard.aggregate_throughput) on two gloo processes."""
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        B = 1000
        seed = shard.rank_seed(7, rank)
        lens = synth.lognormal_lengths(B, seed=seed)  # every rank draws its own shard, as bench.py does
        local_ms = 2.0 + 3.0 * rank                    # rank 1 is the slow one
        value, ms = shard.aggregate_throughput(B, local_ms)
        out.put((rank, seed, int(lens.sum()), value, ms))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_bench_rank_logic_on_two_gloo_ranks():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_bench_rank_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    results = sorted(out.get(timeout=150) for _ in range(world))
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    (r0, s0, t0, v0, ms0), (r1, s1, t1, v1, ms1) = results
    assert (s0, s1) == (7, 1007) and t0 != t1, "ranks must own different shards"
    assert ms0 == ms1 == 5.0, "the job's time is the slowest rank's"
    assert v0 == v1 == pytest.approx(2 * 1000 / 5.0e-3), "value is the whole-job aggregate"
    assert shard.aggregate_throughput(1000, 4.0) == (pytest.approx(250000.0), 4.0)  # one process: identity


def test_bench_gpus_flag_spawns_its_own_ranks():
    """`python bench.py --gpus N` must start N ranks itself (no launcher): checked on the command it builds."""
    import importlib.util
    import sys
    from unittest import mock

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(root, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    seen = {}

    class FakeRanks:  # stands in for the torchrun child: NCCL chatter before AND after rank 0's JSON line
        def __init__(self, cmd, env=None, **kw):
            seen["cmd"], seen["env"] = cmd, env
            self.stdout = iter(["rank 1 NCCL INFO Init START\n", '{"metric": "m", "value": 1}\n',
                                "rank 3 NCCL INFO comm destroyed\n"])

        def wait(self):
            return 0

    argv = ["bench.py", "--gpus", "4", "--steps", "2", "--warmup", "3"]
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "NCCL_DEBUG")}
    import io
    out = io.StringIO()
    with mock.patch.object(sys, "argv", argv), mock.patch("subprocess.Popen", FakeRanks), \
            mock.patch.object(sys, "stdout", out), \
            mock.patch.dict(os.environ, env, clear=True), pytest.raises(SystemExit) as e:
        bench.main()
    assert e.value.code == 0
    cmd = seen["cmd"]
    assert "torch.distributed.run" in cmd and "--nproc-per-node=4" in cmd and "127.0.0.1" in cmd
    assert cmd[-6:] == argv[1:]
    # communicator lines are on by default (the driver's rank check reads them) ...
    assert seen["env"]["NCCL_DEBUG"] == "INFO" and seen["env"]["NCCL_DEBUG_SUBSYS"] == "INIT"
    # ... and rank 0's JSON line is still the LAST line of stdout
    lines = out.getvalue().splitlines()
    assert len(lines) == 3 and lines[-1].startswith('{"metric"') and "comm destroyed" in lines[1]
