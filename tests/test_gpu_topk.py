"""GPU parity for tms_topk: index work, so the bar is bit-exact -- the indices must be
the oracle's (score descending, ties by lower index first) and the values exact copies of the scores."""
import numpy as np
import pytest
import torch

import oracle
import planting
from paper_2606_26439_b200 import synth, tms

pytestmark = pytest.mark.gpu
DEV = "cuda"


def check(scores_np, k):
    s = torch.from_numpy(scores_np.astype(np.float32)).to(DEV)
    vals, idx = tms.tms_topk(s, k)
    torch.cuda.synchronize()
    ref_v, ref_i = oracle.topk(scores_np.astype(np.float32), k)
    assert np.array_equal(idx.cpu().numpy(), ref_i)
    assert np.array_equal(vals.cpu().numpy().astype(np.float64), ref_v)


@pytest.mark.parametrize("B,k", [(1, 1), (5, 5), (100, 7), (4096, 100), (4097, 100), (10_000, 1000), (123_457, 1024),
                                 (500_000, 100)])
def test_random_scores(B, k):
    rng = np.random.default_rng(B + k)
    check(rng.standard_normal((3, B)), k)


@pytest.mark.parametrize("k", [1, 2, 3, 64, 100, 127, 128, 129])  # k <= 128: the warp-resident kernel; 129: the sorting one
@pytest.mark.parametrize("B", [130, 4095, 4096, 4097, 50_000, 1_048_577])  # one chunk, chunk edges, two / three levels
def test_both_level_kernels_around_their_switch_point(B, k):
    if k > B:
        pytest.skip("k <= B")
    rng = np.random.default_rng(1000 * k + B % 997)
    s = rng.standard_normal((2, B))
    s[:, rng.integers(0, B, size=B // 5)] = -np.inf   # empty documents
    s[0, : min(B, 300)] = 1.0                         # a long tie at the top: lower index first
    check(s, k)


def test_ties_and_neg_inf_follow_the_index_rule():
    rng = np.random.default_rng(5)
    s = rng.integers(-2, 3, size=(4, 20_000)).astype(np.float64)  # five distinct values: thousands of ties
    s[:, ::7] = -np.inf
    check(s, 1000)
    check(np.full((2, 9000), -np.inf), 10)  # nothing but empty documents: the first k indices


def test_topk_of_real_scores_equals_topk_of_oracle_scores_on_planted_documents():
    Q, Nq, d, B = 8, 32, 128, 20_000
    off = synth.uniform_offsets(B, 64)
    q = synth.unit_tokens(Q * Nq, d, torch.bfloat16, seed=1).view(Q, Nq, d)
    D = synth.unit_tokens(int(off[-1]), d, torch.bfloat16, seed=2)
    ids = planting.plant_relevant(q, D, off, seed=3)
    scores = tms.tms_maxsim(q.to(DEV), D.to(DEV), torch.from_numpy(off).to(DEV))
    vals, idx = tms.tms_topk(scores, 100)
    assert np.array_equal(idx.cpu().numpy(), ids[:, :100])  # planted documents, in order (gaps twice the tolerance)
    ref_v, ref_i = oracle.topk(scores.cpu().numpy(), 100)  # and exactly the plain definition on the same scores
    assert np.array_equal(idx.cpu().numpy(), ref_i) and np.array_equal(vals.cpu().numpy().astype(np.float64), ref_v)


def test_argument_errors():
    s = torch.zeros((2, 100), device=DEV)
    with pytest.raises(RuntimeError, match="invalid"):
        tms.tms_topk(s, 101)
    with pytest.raises(RuntimeError, match="unsupported"):
        tms.tms_topk(torch.zeros((1, 5000), device=DEV), 2000)
