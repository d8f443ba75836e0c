"""Pins for the fp64 oracle (no GPU needed).

Each test ties oracle/oracle.c to something other than itself: the literal definition written a
second way (numpy float64), closed forms and invariants of Eq. 1, the ADC identity of
Eq. 8-9, and library routines the special cases reduce to.  Numbering P1..P15
follows SURVEY.md 8(c).
"""
import math

import numpy as np
import pytest
import torch

import oracle
import planting
from paper_2606_26439_b200 import synth

DTYPES = [torch.float32, torch.float16, torch.bfloat16]


def np_maxsim(q64: np.ndarray, D64: np.ndarray, off: np.ndarray) -> np.ndarray:
    """Eq. 1 with numpy: S = Q D^T (einsum), per-document segment max, sum over query tokens."""
    Q, Nq, _ = q64.shape
    B = len(off) - 1
    S = np.einsum("qid,jd->qij", q64, D64)  # [Q, Nq, T]
    out = np.empty((Q, B))
    for b in range(B):
        seg = S[:, :, off[b]:off[b + 1]]
        out[:, b] = seg.max(axis=2).sum(axis=1) if seg.shape[2] else -np.inf
    return out


def f64(t: torch.Tensor) -> np.ndarray:
    return t.to(torch.float64).numpy()


# ---- P1: brute force == numpy definition == transposed/parallel oracle ---------------------------------------------

@pytest.mark.parametrize("dtype", DTYPES)
def test_p1_bruteforce_matches_numpy_definition(dtype):
    g = torch.Generator().manual_seed(1)
    Q, Nq, d = 2, 4, 8
    lens = [3, 1, 5, 2, 4]
    off = synth.offsets_from_lengths(lens)
    q = torch.randn((Q, Nq, d), generator=g).to(dtype)
    D = torch.randn((int(off[-1]), d), generator=g).to(dtype)
    ref = np_maxsim(f64(q), f64(D), off)
    got = oracle.bruteforce(q, D, off)
    np.testing.assert_allclose(got, ref, rtol=0, atol=1e-12)
    got2 = oracle.maxsim(q, D, off, threads=3)
    assert np.array_equal(got, got2), "transposed oracle must be bit-identical to the brute force"


@pytest.mark.parametrize("dtype", DTYPES)
def test_p1_oracle_bitidentical_to_bruteforce_ragged(dtype):
    lens = synth.lognormal_lengths(40, seed=3, median=20, lo=1, hi=70)
    lens[7] = 0  # an empty document in the middle
    off = synth.offsets_from_lengths(lens)
    q = synth.unit_tokens(3 * 5, 24, dtype, seed=5).view(3, 5, 24)
    D = synth.unit_tokens(int(off[-1]), 24, dtype, seed=6)
    a = oracle.bruteforce(q, D, off)
    b = oracle.maxsim(q, D, off)
    assert np.array_equal(a, b)
    np.testing.assert_allclose(a, np_maxsim(f64(q), f64(D), off), rtol=0, atol=1e-12)
    assert np.all(np.isneginf(a[:, 7])), "empty document scores -inf (reading A2, Alg. 3 line 4)"


def test_element_decoding_every_fp16_and_bf16_bit_pattern():
    bits = np.arange(65536, dtype=np.uint16)
    finite16 = np.isfinite(bits.view(np.float16))
    hb, bb = bits[finite16], bits[np.isfinite(f64(torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16)))]
    for arr, name, ref in (
        (hb, "f16", hb.view(np.float16).astype(np.float64)),
        (bb, "bf16", f64(torch.from_numpy(bb.view(np.int16)).view(torch.bfloat16))),
    ):
        # one query token e_0 (the value 1.0 in storage bits), one single-element document per pattern, d = 1
        one = np.array([[[0x3C00 if name == "f16" else 0x3F80]]], dtype=np.uint16)
        docs = arr.reshape(-1, 1)
        off = np.arange(len(arr) + 1, dtype=np.int64)
        got = oracle.maxsim(one, docs, off, dtype=name)[0]
        assert np.array_equal(got, ref), name


# ---- P2: self-retrieval ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("dtype", DTYPES)
def test_p2_self_retrieval_scores_sum_of_squared_norms(dtype):
    Nq, d, Nd, B = 32, 128, 64, 6
    q = synth.unit_tokens(Nq, d, dtype, seed=11).view(1, Nq, d)
    D = synth.unit_tokens(B * Nd, d, dtype, seed=12)
    perm = torch.randperm(Nd, generator=torch.Generator().manual_seed(0))[:Nq]
    D[2 * Nd + perm] = q[0]  # document 2 contains the query's own tokens, scattered
    s = oracle.maxsim(q, D, synth.uniform_offsets(B, Nd))[0]
    expect = float((f64(q[0]) ** 2).sum())
    assert abs(s[2] - expect) < 1e-12
    tol = {torch.float32: 1e-5, torch.float16: 3e-3, torch.bfloat16: 2e-2}[dtype]
    assert abs(s[2] - Nq) < tol * Nq  # = Nq for unit norm, up to storage rounding of the norms
    assert np.argmax(s) == 2


# ---- P3: permutation invariance -------------------------------------------------------------------------------------

def test_p3_permuting_tokens_within_documents_and_documents():
    lens = np.array([5, 9, 1, 17, 8])
    off = synth.offsets_from_lengths(lens)
    q = synth.unit_tokens(8, 16, torch.float32, seed=1).view(2, 4, 16)
    D = synth.unit_tokens(int(off[-1]), 16, torch.float32, seed=2)
    base = oracle.maxsim(q, D, off)
    rng = np.random.default_rng(0)
    D2 = D.clone()
    for b in range(len(lens)):
        p = rng.permutation(lens[b]) + off[b]
        D2[off[b]:off[b + 1]] = D[torch.from_numpy(p)]
    assert np.array_equal(oracle.maxsim(q, D2, off), base), "max over j is order-free, bit for bit"
    order = rng.permutation(len(lens))
    D3 = torch.cat([D[off[b]:off[b + 1]] for b in order])
    off3 = synth.offsets_from_lengths(lens[order])
    assert np.array_equal(oracle.maxsim(q, D3, off3), base[:, order])


# ---- P4 / P15: bound and sanity range on unit-norm data --------------------------------------------------------------

def test_p4_bound_and_p15_typical_value():
    Nq, d, Nd, B = 32, 128, 128, 300
    q = synth.unit_tokens(2 * Nq, d, torch.float32, seed=0).view(2, Nq, d)
    D = synth.unit_tokens(B * Nd, d, torch.float32, seed=1)
    s = oracle.maxsim(q, D, synth.uniform_offsets(B, Nd))
    assert np.all(np.abs(s) <= Nq * (1 + 1e-6))
    # E[max of 128 N(0,1/128)] * 32 ~ 7.28 (SURVEY App. A Monte-Carlo); catches a missing normalisation or wrong Nd
    assert 7.0 < s.mean() < 7.6 and 0.1 < s.std() < 0.35


# ---- P6: one-hot queries -> sum of column maxima ---------------------------------------------------------------------

@pytest.mark.parametrize("dtype", DTYPES)
def test_p6_onehot_queries_give_sum_of_column_maxima(dtype):
    Q, Nq, d = 2, 6, 32
    q, pi = synth.onehot_queries(Q, Nq, d, dtype, seed=4)
    lens = [7, 3, 12]
    off = synth.offsets_from_lengths(lens)
    D = torch.randn((int(off[-1]), d), generator=torch.Generator().manual_seed(9)).to(dtype)
    s = oracle.maxsim(q, D, off)
    D64 = f64(D)
    for b in range(len(lens)):
        colmax = D64[off[b]:off[b + 1]].max(axis=0)
        for qq in range(Q):
            assert s[qq, b] == sum(colmax[pi[qq, i]] for i in range(Nq)), "exact: products by 1.0, sums of <= 6 terms"


# ---- P8: single-token documents reduce to a GEMV ---------------------------------------------------------------------

def test_p8_single_token_documents_are_a_gemv():
    Q, Nq, d, B = 2, 5, 16, 50
    q = synth.unit_tokens(Q * Nq, d, torch.float32, seed=3).view(Q, Nq, d)
    D = synth.unit_tokens(B, d, torch.float32, seed=4)
    s = oracle.maxsim(q, D, synth.uniform_offsets(B, 1))
    ref = f64(D) @ f64(q).sum(axis=1).T  # D @ (sum_i q_i): library matmul
    np.testing.assert_allclose(s, ref.T, rtol=0, atol=1e-13)


# ---- P9: additivity over query tokens --------------------------------------------------------------------------------

def test_p9_additive_over_query_tokens():
    q = synth.unit_tokens(2 * 12, 32, torch.float16, seed=1).view(2, 12, 32)
    off = synth.offsets_from_lengths([9, 14, 2, 30])
    D = synth.unit_tokens(int(off[-1]), 32, torch.float16, seed=2)
    full = oracle.maxsim(q, D, off)
    a = oracle.maxsim(q[:, :5].contiguous(), D, off)
    b = oracle.maxsim(q[:, 5:].contiguous(), D, off)
    np.testing.assert_allclose(full, a + b, rtol=0, atol=1e-13)


# ---- P10: monotone under appended tokens, unchanged under duplicated tokens ------------------------------------------

def test_p10_append_never_lowers_and_duplicate_changes_nothing():
    q = synth.unit_tokens(8, 16, torch.float32, seed=1).view(1, 8, 16)
    D = synth.unit_tokens(10, 16, torch.float32, seed=2)
    s = [oracle.maxsim(q, D[:n].contiguous(), np.array([0, n]))[0, 0] for n in range(1, 11)]
    assert all(s[i + 1] >= s[i] for i in range(9))
    dup = torch.cat([D, D[3:4], D[7:8]])
    assert oracle.maxsim(q, dup, np.array([0, 12]))[0, 0] == s[-1]


# ---- P11: zero-padding and consistent permutation of the embedding dimension -----------------------------------------

@pytest.mark.parametrize("dpad", [256, 768])
def test_p11_zero_padded_dimensions_leave_scores_unchanged(dpad):
    Nq, d, B, Nd = 8, 128, 5, 20
    q = synth.unit_tokens(Nq, d, torch.bfloat16, seed=1).view(1, Nq, d)
    D = synth.unit_tokens(B * Nd, d, torch.bfloat16, seed=2)
    off = synth.uniform_offsets(B, Nd)
    base = oracle.maxsim(q, D, off)
    qp = torch.zeros((1, Nq, dpad), dtype=torch.bfloat16)
    Dp = torch.zeros((B * Nd, dpad), dtype=torch.bfloat16)
    qp[..., :d], Dp[:, :d] = q, D
    assert np.array_equal(oracle.maxsim(qp, Dp, off), base)  # adding +0.0 terms is exact
    perm = torch.randperm(d, generator=torch.Generator().manual_seed(3))
    np.testing.assert_allclose(oracle.maxsim(q[..., perm].contiguous(), D[:, perm].contiguous(), off), base,
                               rtol=0, atol=1e-13)


# ---- P12: positive homogeneity ---------------------------------------------------------------------------------------

def test_p12_scaling_queries_by_two_doubles_the_score_exactly():
    q = synth.unit_tokens(6, 16, torch.float16, seed=1).view(1, 6, 16)
    D = synth.unit_tokens(30, 16, torch.float16, seed=2)
    off = synth.uniform_offsets(3, 10)
    assert np.array_equal(oracle.maxsim(q * 2, D, off), 2 * oracle.maxsim(q, D, off))


# ---- P5 / P13: PQ ----------------------------------------------------------------------------------------------------

def _pq_case(seed, Q=2, Nq=6, M=4, K=16, dsub=4, lens=(5, 1, 9, 0, 12)):
    d = M * dsub
    q = synth.unit_tokens(Q * Nq, d, torch.bfloat16, seed=seed).view(Q, Nq, d)
    C = synth.pq_codebooks(M, K, dsub, seed=seed + 1)
    off = synth.offsets_from_lengths(lens)
    codes = synth.pq_codes(int(off[-1]), M, seed=seed + 2, K=K)
    return q, C, codes, off


def test_p5_lut_sum_equals_decompressed_dot_product():
    """Eq. 8-9: sum_m T[i,m,c_jm] == q_i . dhat_j; the oracle decompresses, this test builds T in numpy fp64."""
    q, C, codes, off = _pq_case(7)
    got = oracle.pq_maxsim(q, C, codes, off)
    Q, Nq, d = q.shape
    M, K, dsub = C.shape
    T = np.einsum("qims,mks->qimk", f64(q).reshape(Q, Nq, M, dsub), f64(C))  # Eq. 8
    cd = codes.numpy()
    sim = np.zeros((Q, Nq, cd.shape[0]))
    for m in range(M):
        sim += T[:, :, m, cd[:, m]]  # Eq. 9
    ref = np.empty((Q, len(off) - 1))
    for b in range(len(off) - 1):
        seg = sim[:, :, off[b]:off[b + 1]]
        ref[:, b] = seg.max(axis=2).sum(axis=1) if seg.shape[2] else -np.inf
    np.testing.assert_allclose(got, ref, rtol=0, atol=1e-13)
    assert np.all(np.isneginf(got[:, 3]))


def test_p13_pq_oracle_equals_dense_oracle_on_explicitly_decompressed_vectors():
    q, C, codes, off = _pq_case(21, M=8, K=256, dsub=8, lens=(40, 3, 17))
    M, K, dsub = C.shape
    dhat = torch.stack([C[m, codes[:, m].long()] for m in range(M)], dim=1).reshape(codes.shape[0], M * dsub)
    dense = oracle.maxsim(q.to(torch.float32), dhat, off)  # bf16 queries up-converted exactly to fp32
    assert np.array_equal(oracle.pq_maxsim(q, C, codes, off), dense)


def test_pq_config5_score_range():
    """Reading A12: N(0, var 1/8) codebooks give ||dhat|| ~ 4 and scores ~ 29.5 +- 0.8."""
    Nq, M, K, dsub, B, Nd = 32, 16, 256, 8, 64, 128
    q = synth.unit_tokens(Nq, M * dsub, torch.bfloat16, seed=0).view(1, Nq, M * dsub)
    C = synth.pq_codebooks(M, K, dsub, seed=1)
    codes = synth.pq_codes(B * Nd, M, seed=2)
    s = oracle.pq_maxsim(q, C, codes, synth.uniform_offsets(B, Nd))
    assert 27.5 < s.mean() < 31.5


# ---- input recipe ----------------------------------------------------------------------------------------------------

def test_lognormal_length_recipe_matches_config3():
    lens = synth.lognormal_lengths(200000, seed=0)
    assert lens.min() >= 8 and lens.max() == 180
    assert abs(np.median(lens) - 64) <= 1 and 70.5 < lens.mean() < 73.0
    assert 0.015 < (lens == 180).mean() < 0.025


def test_unit_tokens_are_unit_norm_after_rounding():
    for dtype, tol in ((torch.float32, 1e-6), (torch.float16, 2e-4), (torch.bfloat16, 1.2e-3)):
        x = synth.unit_tokens(1000, 128, dtype, seed=0)
        n = np.linalg.norm(f64(x), axis=1)
        assert np.abs(n - 1).max() < tol
    a = synth.unit_tokens(100, 64, torch.bfloat16, seed=5)
    b = synth.unit_tokens(100, 64, torch.bfloat16, seed=5)
    assert torch.equal(a, b)


def test_planted_documents_rank_first_in_order():
    Q, Nq, d, B, Nd = 2, 32, 128, 600, 64
    q = synth.unit_tokens(Q * Nq, d, torch.bfloat16, seed=1).view(Q, Nq, d)
    D = synth.unit_tokens(B * Nd, d, torch.bfloat16, seed=2)
    off = synth.uniform_offsets(B, Nd)
    ids = planting.plant_relevant(q, D, off, seed=3, per_query=50)
    s = oracle.maxsim(q, D, off)
    for qq in range(Q):
        top = np.argsort(-s[qq], kind="stable")[:50]
        assert np.array_equal(top, ids[qq])
        gaps = -np.diff(s[qq, top])
        assert gaps.min() > 0.2  # Nq * 0.5 / 49 = 0.33 nominal, far above 2e-3*Nq = 0.064
        assert math.isclose(s[qq, top[0]], 0.95 * Nq, rel_tol=5e-3)


# ---- top-k (NEXT-2): the oracle's plain definition against a brute-force selection ------------------------------------

def test_topk_matches_bruteforce_selection_with_ties_and_neg_inf():
    rng = np.random.default_rng(11)
    s = rng.integers(-3, 4, size=(3, 40)).astype(np.float64)  # few distinct values: many ties
    s[0, 5] = s[1, 0] = s[2, 39] = -np.inf
    for k in (1, 7, 40):
        vals, idx = oracle.topk(s, k)
        for q in range(3):
            left = list(range(40))
            for r in range(k):  # repeatedly pick the best remaining document: highest score, then lowest index
                best = max(left, key=lambda b: (s[q, b], -b))
                left.remove(best)
                assert idx[q, r] == best and vals[q, r] == s[q, best]
    vals, idx = oracle.topk(np.array([[1.0, 3.0, 3.0, 2.0]]), 3)
    assert idx.tolist() == [[1, 2, 3]] and vals.tolist() == [[3.0, 3.0, 2.0]]
