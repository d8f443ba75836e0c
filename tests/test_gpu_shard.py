"""NEXT-3 on the GPU ("splitting the candidate batch evenly across GPUs ... only a final
concatenation of per-shard scores"): a ragged store is cut with shard_documents, every shard is scored through the C
ABI, and the concatenation must equal the unsharded call bit for bit and the oracle within tolerance; per-shard top-k
lists merged with tms_topk_merge must equal oracle.topk over all scores.  Runs on ONE GPU (shards in sequence)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_26439_b200 import shard, synth, tms

pytestmark = pytest.mark.gpu
DEV = "cuda"
RAGGED = np.array([5, 128, 1, 0, 300, 127, 129, 64, 0, 0, 17, 256, 8, 1, 1, 1000, 33], dtype=np.int64)


def _store(n_docs, seed):
    lens = np.concatenate([RAGGED, synth.lognormal_lengths(n_docs, seed=seed), RAGGED[::-1]])
    return synth.offsets_from_lengths(lens)


@pytest.mark.parametrize("G", [2, 3, 8])
@pytest.mark.parametrize("dtype", [torch.bfloat16, torch.float32])
def test_dense_shards_concatenate_to_the_unsharded_result(G, dtype):
    off = _store(3000, seed=G)
    Q, Nq, d = 8, 32, 128
    q = synth.unit_tokens(Q * Nq, d, dtype, seed=1).view(Q, Nq, d)
    D = synth.unit_tokens(int(off[-1]), d, dtype, seed=2)
    qd, Dd = q.to(DEV), D.to(DEV)
    whole = tms.tms_maxsim(qd, Dd, torch.from_numpy(off).to(DEV))
    parts, covered = [], 0
    for r in range(G):
        b_lo, b_hi, t_lo, t_hi, local = shard.shard_documents(off, G, r)
        assert b_lo == covered
        covered = b_hi
        parts.append(tms.tms_maxsim(qd, Dd[t_lo:t_hi], torch.from_numpy(local).to(DEV)))
    assert covered == len(off) - 1
    cat = torch.cat(parts, dim=1)
    assert torch.equal(cat, whole), "sharded scores must be bit-identical to the unsharded call"
    ref = oracle.maxsim(q, D, off)
    inf = np.isneginf(ref)
    got = cat.cpu().numpy().astype(np.float64)
    assert np.array_equal(np.isneginf(got), inf)
    assert np.abs(got[~inf] - ref[~inf]).max() <= (1e-5 if dtype == torch.float32 else 2e-3) * Nq


@pytest.mark.parametrize("G", [2, 3, 8])
def test_pq_shards_concatenate_to_the_unsharded_result(G):
    off = _store(2500, seed=10 + G)
    Q, Nq, T = 8, 32, int(off[-1])
    q = synth.unit_tokens(Q * Nq, 128, torch.bfloat16, seed=3).view(Q, Nq, 128)
    C = synth.pq_codebooks(16, 256, 8, seed=4)
    codes = synth.pq_codes(T, 16, seed=5)
    qd, Cd, cd = q.to(DEV), C.to(DEV), codes.to(DEV)
    lut = tms.tms_pq_build_lut(qd, Cd)  # replicated on every rank (queries and tables are small)
    whole = tms.tms_pq_maxsim(lut, cd, torch.from_numpy(off).to(DEV))
    whole_dec = tms.tms_pq_maxsim_decode(qd, Cd, cd, torch.from_numpy(off).to(DEV))
    parts, parts_dec = [], []
    for r in range(G):
        b_lo, b_hi, t_lo, t_hi, local = shard.shard_documents(off, G, r)
        od = torch.from_numpy(local).to(DEV)
        parts.append(tms.tms_pq_maxsim(lut, cd[t_lo:t_hi], od))
        parts_dec.append(tms.tms_pq_maxsim_decode(qd, Cd, cd[t_lo:t_hi], od))
    assert torch.equal(torch.cat(parts, dim=1), whole)
    assert torch.equal(torch.cat(parts_dec, dim=1), whole_dec)
    ref = oracle.pq_maxsim(q, C, codes, off)
    inf = np.isneginf(ref)
    for got in (whole, whole_dec):
        g = got.cpu().numpy().astype(np.float64)
        assert np.array_equal(np.isneginf(g), inf) and np.abs(g[~inf] - ref[~inf]).max() <= 2e-3 * Nq


@pytest.mark.parametrize("G,k", [(2, 100), (3, 17), (8, 100), (8, 1024)])
def test_per_shard_topk_and_merge_equal_the_global_topk(G, k):
    off = _store(12000, seed=20 + G)
    B = len(off) - 1
    Q, Nq, d = 4, 32, 64
    q = synth.unit_tokens(Q * Nq, d, torch.bfloat16, seed=6).view(Q, Nq, d)
    D = synth.unit_tokens(int(off[-1]), d, torch.bfloat16, seed=7)
    qd, Dd = q.to(DEV), D.to(DEV)
    whole = tms.tms_maxsim(qd, Dd, torch.from_numpy(off).to(DEV))
    vals, idxs, bases = [], [], []
    for r in range(G):
        b_lo, b_hi, t_lo, t_hi, local = shard.shard_documents(off, G, r)
        s = tms.tms_maxsim(qd, Dd[t_lo:t_hi], torch.from_numpy(local).to(DEV))
        v, i = tms.tms_topk(s, min(k, b_hi - b_lo))
        assert v.shape[1] == k, "test sizes keep every shard larger than k"
        vals.append(v)
        idxs.append(i)
        bases.append(b_lo)
    mv, mi = tms.tms_topk_merge(torch.stack(vals), torch.stack(idxs), bases, k)
    ref_v, ref_i = oracle.topk(whole.cpu().numpy(), k)  # oracle's ranking of the very same fp32 scores
    assert np.array_equal(mi.cpu().numpy(), ref_i), "merged indices must equal the global top-k, ties included"
    assert np.array_equal(mv.cpu().numpy(), ref_v)
    gv, gi = tms.tms_topk(whole, k)
    assert torch.equal(gv, mv) and torch.equal(gi, mi)


def test_topk_merge_ties_and_minus_infinity():
    # two shards full of ties: equal scores rank by GLOBAL index, -inf last
    v = torch.tensor([[[1.0, 1.0, float("-inf")]], [[1.0, 0.5, float("-inf")]]], dtype=torch.float32, device=DEV)
    i = torch.tensor([[[0, 2, 1]], [[1, 0, 2]]], dtype=torch.int64, device=DEV)
    mv, mi = tms.tms_topk_merge(v, i, [0, 10], 6)
    assert mi.cpu().tolist() == [[0, 2, 11, 10, 1, 12]]
    assert mv.cpu().tolist()[0][:4] == [1.0, 1.0, 1.0, 0.5] and all(np.isneginf(mv.cpu().numpy()[0, 4:]))
