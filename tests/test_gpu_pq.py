"""GPU parity for the PQ path: tms_pq_build_lut (Eq. 8) and tms_pq_maxsim (Eq. 9) against the oracle's
explicit decompress-then-score.  Queries are bf16, so the tolerance is 2e-3*Nq."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_26439_b200 import synth, tms

pytestmark = pytest.mark.gpu
DEV = "cuda"


def pq_case(Q, Nq, M, K, dsub, off, seed, q_dtype=torch.bfloat16):
    d = M * dsub
    q = synth.unit_tokens(Q * Nq, d, q_dtype, seed=seed).view(Q, Nq, d)
    C = synth.pq_codebooks(M, K, dsub, seed=seed + 1)
    codes = synth.pq_codes(int(off[-1]), M, seed=seed + 2, K=K)
    return q, C, codes


def run_pq(q, C, codes, off, variant="auto"):
    lut = tms.tms_pq_build_lut(q.to(DEV), C.to(DEV))
    out = tms.tms_pq_maxsim(lut, codes.to(DEV), torch.from_numpy(off).to(DEV), variant=variant)
    torch.cuda.synchronize()
    return lut.cpu().numpy(), out.cpu().numpy().astype(np.float64)


def assert_close(got, ref, atol):
    inf = np.isneginf(ref)
    assert np.array_equal(np.isneginf(got), inf)
    err = np.abs(got[~inf] - ref[~inf])
    assert err.size == 0 or err.max() <= atol, f"max |dscore| = {err.max():.3e} > {atol:.3e}"


@pytest.mark.parametrize("q_dtype", [torch.bfloat16, torch.float16, torch.float32])
def test_lut_matches_eq8_in_fp64(q_dtype):
    off = synth.uniform_offsets(1, 1)
    q, C, codes = pq_case(8, 32, 16, 256, 8, off, seed=1, q_dtype=q_dtype)
    lut, _ = run_pq(q, C, codes, off)
    ref = np.einsum("qims,mks->qimk", q.to(torch.float64).numpy().reshape(8, 32, 16, 8), C.to(torch.float64).numpy())
    assert np.abs(lut - ref).max() < 2e-6  # fp32 FMA chain of 8 terms, |terms| < 1


@pytest.mark.parametrize("variant", ["simt", "pq_smem", "pq_smem_f16"])
def test_config4_shape_small(variant):
    off = synth.uniform_offsets(3000, 128)
    q, C, codes = pq_case(8, 32, 16, 256, 8, off, seed=3)
    _, got = run_pq(q, C, codes, off, variant)
    assert_close(got, oracle.pq_maxsim(q, C, codes, off), 2e-3 * 32)
    assert 28.0 < got.mean() < 31.0


@pytest.mark.parametrize("variant", ["simt", "pq_smem", "pq_smem_f16"])
def test_ragged_documents(variant):
    lens = np.concatenate([[5, 128, 1, 0, 300, 16, 17, 15, 0, 0, 33, 1000],
                           synth.lognormal_lengths(2000, seed=2, median=40, lo=0, hi=200)])
    off = synth.offsets_from_lengths(lens)
    q, C, codes = pq_case(3, 32, 16, 256, 8, off, seed=5)
    _, got = run_pq(q, C, codes, off, variant)
    assert_close(got, oracle.pq_maxsim(q, C, codes, off), 2e-3 * 32)


@pytest.mark.parametrize("Q,Nq,M,K,dsub", [(2, 12, 8, 64, 4), (1, 32, 32, 256, 4), (5, 7, 16, 256, 8)])
def test_general_shapes_take_the_general_kernel(Q, Nq, M, K, dsub):
    off = synth.offsets_from_lengths(synth.lognormal_lengths(300, seed=4, median=30, lo=0, hi=100))
    q, C, codes = pq_case(Q, Nq, M, K, dsub, off, seed=7)
    _, got = run_pq(q, C, codes, off, "auto")
    assert_close(got, oracle.pq_maxsim(q, C, codes, off), 2e-3 * Nq)


def test_smem_and_general_kernels_agree_and_are_reproducible():
    off = synth.offsets_from_lengths(synth.lognormal_lengths(5000, seed=9))
    q, C, codes = pq_case(8, 32, 16, 256, 8, off, seed=11)
    _, a = run_pq(q, C, codes, off, "pq_smem")
    _, a2 = run_pq(q, C, codes, off, "pq_smem")
    _, b = run_pq(q, C, codes, off, "simt")
    assert np.array_equal(a, a2)
    assert np.abs(a - b).max() < 1e-4  # same fp32 terms, different summation order over m


def test_f16_table_entries_stay_well_inside_the_16_bit_tolerance():
    """TMS_VARIANT_PQ_SMEM_F16 rounds each stored table entry to fp16 (after a power-of-two block scale) and adds in
    fp32: measured against the fp64 oracle and against the fp32-entry kernel on config 4's distribution."""
    off = synth.offsets_from_lengths(synth.lognormal_lengths(5000, seed=9))
    q, C, codes = pq_case(8, 32, 16, 256, 8, off, seed=11)
    ref = oracle.pq_maxsim(q, C, codes, off)
    _, h = run_pq(q, C, codes, off, "pq_smem_f16")
    _, h2 = run_pq(q, C, codes, off, "pq_smem_f16")
    _, f = run_pq(q, C, codes, off, "pq_smem")
    assert np.array_equal(h, h2)
    assert np.abs(h - ref).max() <= 0.25 * 2e-3 * 32   # a quarter of the north_star tolerance
    assert np.abs(h - f).max() <= 0.25 * 2e-3 * 32


@pytest.mark.parametrize("scale", [1e-6, 1.0, 3e5])
def test_f16_table_is_block_scaled(scale):
    """The fp16 table is scaled by a power of two taken from max|lut|: codebooks of any magnitude neither overflow fp16
    (3e5 * entries ~ 1e5 > 65504) nor fall into its subnormals (1e-6); the error stays relative to the scores."""
    off = synth.offsets_from_lengths(synth.lognormal_lengths(1500, seed=21, lo=0))
    q, C, codes = pq_case(4, 16, 16, 256, 8, off, seed=23)
    C = (C * scale).contiguous()
    ref = oracle.pq_maxsim(q, C, codes, off)
    _, h = run_pq(q, C, codes, off, "pq_smem_f16")
    assert_close(h / scale, ref / scale, 0.25 * 2e-3 * 16)


@pytest.mark.parametrize("q_dtype", [torch.float32, torch.bfloat16, torch.float16])
@pytest.mark.parametrize("Nq", [32, 48, 20])  # 16-row slices possible / 8-row slices only / the general kernel
def test_auto_keeps_the_fp32_table_whatever_it_was_built_from(q_dtype, Nq):
    """tms_pq_maxsim sees only `lut`, not the queries' dtype, so its default must hold the tightest bound an input class
    carries: 1e-5*Nq for fp32 queries (north_star; scaled by max|dhat| as in test_p13), 2e-3*Nq for 16-bit ones.  The
    paper's table is fp32; fp16 entries are opt-in and are NOT inside the fp32 bound on this data."""
    lens = np.concatenate([[5, 128, 1, 0, 300, 16, 17, 15, 0, 0, 33, 1000],
                           synth.lognormal_lengths(3000, seed=31, median=60, lo=0, hi=200)])
    off = synth.offsets_from_lengths(lens)
    q, C, codes = pq_case(8, Nq, 16, 256, 8, off, seed=33, q_dtype=q_dtype)
    ref = oracle.pq_maxsim(q, C, codes, off)
    dhat_norm = float(np.sqrt((C.double().numpy() ** 2).sum(-1).max(-1).sum()))  # max over codes of ||dhat||
    _, auto = run_pq(q, C, codes, off)  # TMS_VARIANT_AUTO
    want = "pq_smem" if Nq % 8 == 0 else "simt"
    assert tms.tms_pq_maxsim_variant_used(8, Nq, 16, 256) == want
    _, named = run_pq(q, C, codes, off, want)
    assert np.array_equal(auto, named)
    assert_close(auto, ref, 1e-5 * Nq * max(1.0, dhat_norm))   # the fp32 bound holds for EVERY query dtype
    tol_16 = 2e-3 * Nq
    assert_close(auto, ref, tol_16)
    if Nq % 16 == 0:  # the opt-in: inside the 16-bit bound, outside the fp32 one (which is why it is not the default)
        _, h = run_pq(q, C, codes, off, "pq_smem_f16")
        assert_close(h, ref, tol_16)
        fin = np.isfinite(ref)
        assert np.abs(h[fin] - ref[fin]).max() > 1e-5 * Nq  # several times the plain fp32 bound of north_star


def test_f16_table_needs_whole_16_row_slices():
    off = synth.uniform_offsets(50, 20)
    q, C, codes = pq_case(2, 24, 16, 256, 8, off, seed=25)   # Nq = 24: fine for the fp32 table (8-row slices) only
    run_pq(q, C, codes, off, "pq_smem")
    with pytest.raises(RuntimeError):
        run_pq(q, C, codes, off, "pq_smem_f16")


def test_p13_lossless_codes_reproduce_the_dense_path():
    """Documents whose sub-vectors ARE centroids: the PQ score equals the dense fp32 score of those vectors."""
    M, K, dsub, B, Nd = 16, 256, 8, 400, 64
    off = synth.uniform_offsets(B, Nd)
    q, C, codes = pq_case(4, 32, M, K, dsub, off, seed=13, q_dtype=torch.float32)
    dhat = torch.stack([C[m, codes[:, m].long()] for m in range(M)], dim=1).reshape(B * Nd, M * dsub)
    _, pq = run_pq(q, C, codes, off, "pq_smem")
    dense = tms.tms_maxsim(q.to(DEV), dhat.to(DEV), torch.from_numpy(off).to(DEV)).cpu().numpy()
    assert np.abs(pq - dense).max() < 1e-5 * 32 * 4  # |dhat| ~ 4: scale the fp32 tolerance by the score magnitude


def test_host_entry_point():
    off = synth.offsets_from_lengths(synth.lognormal_lengths(6000, seed=15))
    q, C, codes = pq_case(8, 32, 16, 256, 8, off, seed=17)
    _, ref = run_pq(q, C, codes, off)
    scores = torch.empty((8, 6000), dtype=torch.float32).pin_memory()
    need = tms.tms_pq_maxsim_host_workspace_min_bytes(8, 32, 128, torch.bfloat16, 16, 256, 180)
    ws = torch.empty(need + (2 << 20), dtype=torch.uint8, device=DEV)  # ~1 MB per chunk buffer: several chunks
    tms.tms_pq_maxsim_host(q, C, codes.pin_memory(), torch.from_numpy(off), scores, ws)
    assert np.array_equal(scores.numpy().astype(np.float64), ref)


# ---- NEXT-4: decode-and-contract variant (codebook resident in shared memory, tensor cores) ---------------------------

def run_decode(q, C, codes, off):
    out = tms.tms_pq_maxsim_decode(q.to(DEV), C.to(DEV), codes.to(DEV), torch.from_numpy(off).to(DEV))
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("q_dtype", [torch.bfloat16, torch.float16, torch.float32])
@pytest.mark.parametrize("Q", [1, 8, 11])
def test_decode_variant_matches_the_oracle_and_the_lut_path(q_dtype, Q):
    lens = np.concatenate([[5, 128, 1, 0, 300, 16, 17, 15, 0, 0, 33, 1000],
                           synth.lognormal_lengths(1500, seed=Q, median=60, lo=0, hi=200)])
    off = synth.offsets_from_lengths(lens)
    q, C, codes = pq_case(Q, 32, 16, 256, 8, off, seed=20 + Q, q_dtype=q_dtype)
    got = run_decode(q, C, codes, off)
    ref = oracle.pq_maxsim(q, C, codes, off)
    assert_close(got, ref, 2e-3 * 32)
    fin = np.isfinite(ref)
    assert np.abs(got[fin] - ref[fin]).max() < 2e-4  # hi/lo split: far inside the tolerance
    _, lut_scores = run_pq(q, C, codes, off, "pq_smem")       # the LUT kernel over fp32 table entries
    assert np.abs(got[fin] - lut_scores[fin]).max() < 2e-4
    _, auto_scores = run_pq(q, C, codes, off)                 # what tms_pq_maxsim runs by default: the same fp32 entries
    assert np.array_equal(auto_scores, lut_scores)
    _, f16_scores = run_pq(q, C, codes, off, "pq_smem_f16")   # the opt-in fp16 entries
    assert np.abs(got[fin] - f16_scores[fin]).max() <= 0.25 * 2e-3 * 32


def test_decode_variant_exact_on_integer_codebooks():
    off = synth.offsets_from_lengths(synth.lognormal_lengths(800, seed=4))
    Q, Nq = 4, 32
    q = synth.small_int_tokens(Q * Nq, 128, torch.bfloat16, seed=1).view(Q, Nq, 128)
    C = torch.randint(-2, 3, (16, 256, 8), generator=torch.Generator().manual_seed(3)).to(torch.float32)
    codes = synth.pq_codes(int(off[-1]), 16, seed=5)
    assert np.array_equal(run_decode(q, C, codes, off), oracle.pq_maxsim(q, C, codes, off))


def test_decode_variant_rejects_other_shapes():
    off = synth.uniform_offsets(4, 8)
    q, C, codes = pq_case(1, 8, 8, 64, 4, off, seed=1)
    with pytest.raises(RuntimeError, match="unsupported"):
        tms.tms_pq_maxsim_decode(q.to(DEV), C.to(DEV), codes.to(DEV), torch.from_numpy(off).to(DEV))


def test_decode_fp16_operands_within_the_16_bit_tolerance():
    """TMS_PQ_FP16: queries and centroids rounded to fp16, one MMA per product.  Must stay inside 2e-3*Nq of the oracle
    (which decompresses the fp32 codebooks exactly), and much closer in practice; exact on integer codebooks."""
    lens = np.concatenate([[5, 128, 1, 0, 300, 127, 129, 64, 0, 17], synth.lognormal_lengths(3000, seed=11)])
    off = synth.offsets_from_lengths(lens)
    Q, Nq, T = 8, 32, int(off[-1])
    q = synth.unit_tokens(Q * Nq, 128, torch.bfloat16, seed=51).view(Q, Nq, 128)
    C = synth.pq_codebooks(16, 256, 8, seed=52)
    codes = synth.pq_codes(T, 16, seed=53)
    ref = oracle.pq_maxsim(q, C, codes, off)
    od = torch.from_numpy(off).to(DEV)
    got = tms.tms_pq_maxsim_decode(q.to(DEV), C.to(DEV), codes.to(DEV), od, precision="fp16").cpu().numpy().astype(np.float64)
    inf = np.isneginf(ref)
    assert np.array_equal(np.isneginf(got), inf)
    err = np.abs(got[~inf] - ref[~inf]).max()
    assert err <= 1e-3 * Nq, f"max |dscore| = {err:.3e}"
    # integer queries and centroids are exact in fp16: bit-exact scores
    qi = synth.small_int_tokens(Q * Nq, 128, torch.float16, seed=54).view(Q, Nq, 128)
    Ci = synth.small_int_tokens(16 * 256, 8, torch.float32, seed=55).view(16, 256, 8)
    refi = oracle.pq_maxsim(qi, Ci, codes, off)
    goti = tms.tms_pq_maxsim_decode(qi.to(DEV), Ci.to(DEV), codes.to(DEV), od, precision="fp16").cpu().numpy().astype(np.float64)
    assert np.array_equal(goti, refi)
