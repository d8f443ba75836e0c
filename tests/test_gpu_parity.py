"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the same
seeded inputs.  Sizes span several 128-token tiles, ragged tails and several CTAs; the oracle finishes
each case in seconds.  Full BASELINE.json sizes are in test_gpu_fullsize.py.

Tolerances (BASELINE.json north_star): |dscore| <= 1e-5*Nq for fp32 inputs, <= 2e-3*Nq for bf16/fp16
inputs with fp32 accumulation; exact-integer inputs must match with d = 0.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_26439_b200 import synth, tms

pytestmark = pytest.mark.gpu
DEV = "cuda"


def tol(dtype, Nq):
    return (1e-5 if dtype == torch.float32 else 2e-3) * Nq


def run_dense(q, D, off, variant="auto"):
    out = tms.tms_maxsim(q.to(DEV), D.to(DEV), torch.from_numpy(off).to(DEV), variant=variant)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


def assert_close(got, ref, atol):
    inf = np.isneginf(ref)
    assert np.array_equal(np.isneginf(got), inf), "-inf (empty documents) must match exactly"
    err = np.abs(got[~inf] - ref[~inf])
    assert err.size == 0 or err.max() <= atol, f"max |dscore| = {err.max():.3e} > {atol:.3e}"


def unit_case(Q, Nq, d, dtype, off, seed):
    q = synth.unit_tokens(Q * Nq, d, dtype, seed=seed).view(Q, Nq, d)
    D = synth.unit_tokens(int(off[-1]), d, dtype, seed=seed + 1)
    return q, D


# ---- configs[0]: the tiny fp32 case, exactly as BASELINE.json states it ---------------------------------------------

def test_config0_tiny_fp32():
    off = synth.uniform_offsets(1000, 128)
    q, D = unit_case(1, 32, 128, torch.float32, off, seed=0)
    got = run_dense(q, D, off)
    assert_close(got, oracle.maxsim(q, D, off), tol(torch.float32, 32))
    assert 7.0 < got.mean() < 7.6


# ---- both kernels, all dtypes, uniform and ragged documents ---------------------------------------------------------

RAGGED = np.array([5, 128, 1, 0, 300, 127, 129, 64, 0, 0, 17, 256, 8, 1, 1, 1000, 33], dtype=np.int64)


@pytest.mark.parametrize("variant", ["simt", "tcgen05"])
@pytest.mark.parametrize("dtype", [torch.bfloat16, torch.float16])
def test_uniform_colbert_shape(variant, dtype):
    off = synth.uniform_offsets(2500, 128)  # 320,000 tokens: ~17 tiles per CTA on 148 SMs
    q, D = unit_case(8, 32, 128, dtype, off, seed=3)
    assert_close(run_dense(q, D, off, variant), oracle.maxsim(q, D, off), tol(dtype, 32))


@pytest.mark.parametrize("variant", ["simt", "tcgen05"])
def test_lognormal_lengths(variant):
    off = synth.offsets_from_lengths(synth.lognormal_lengths(6000, seed=1))
    q, D = unit_case(8, 32, 128, torch.bfloat16, off, seed=5)
    assert_close(run_dense(q, D, off, variant), oracle.maxsim(q, D, off), tol(torch.bfloat16, 32))


@pytest.mark.parametrize("variant", ["simt", "tcgen05"])
@pytest.mark.parametrize("dtype", [torch.bfloat16, torch.float16])
def test_ragged_with_empty_single_token_and_long_documents(variant, dtype):
    lens = np.concatenate([RAGGED, synth.lognormal_lengths(400, seed=2, median=30, lo=0, hi=400), RAGGED[::-1]])
    off = synth.offsets_from_lengths(lens)
    q, D = unit_case(3, 32, 128, dtype, off, seed=7)
    assert_close(run_dense(q, D, off, variant), oracle.maxsim(q, D, off), tol(dtype, 32))


@pytest.mark.parametrize("variant", ["simt", "tcgen05"])
@pytest.mark.parametrize("lens", [[1], [128], [129], [7, 0], [0, 0, 3], [2000], [0, 0]])
def test_degenerate_batches(variant, lens):
    off = synth.offsets_from_lengths(lens)
    q, D = unit_case(2, 32, 128, torch.bfloat16, off, seed=9)
    if off[-1] == 0:  # nothing to stream: the tensor-core path declines, the dispatcher takes the general kernel
        D, variant = torch.zeros((0, 128), dtype=torch.bfloat16), "auto"
    assert_close(run_dense(q, D, off, variant), oracle.maxsim(q, D, off), tol(torch.bfloat16, 32))


@pytest.mark.parametrize("lens", [[1], [128], [129], [7, 0], [0, 0, 3], [2000], [0, 5, 0, 0], [64, 64, 1]])
@pytest.mark.parametrize("Nq", [32, 64])
def test_degenerate_batches_as_cta_pairs(lens, Nq):
    """The same corner cases through the CTA-pair kernel (d = 512, 256 query rows): one pair, one tile, empty documents;
    Nq = 64 adds the two-part long-query scratch on top."""
    off = synth.offsets_from_lengths(lens)
    q, D = unit_case(8 if Nq == 32 else 5, Nq, 512, torch.float16, off, seed=19)
    assert_close(run_dense(q, D, off, "tcgen05"), oracle.maxsim(q, D, off), tol(torch.float16, Nq))


def test_all_single_token_documents():
    off = synth.uniform_offsets(5000, 1)
    q, D = unit_case(4, 32, 128, torch.float16, off, seed=11)
    assert_close(run_dense(q, D, off, "tcgen05"), oracle.maxsim(q, D, off), tol(torch.float16, 32))


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_fp32_and_generic_shapes_on_the_simt_kernel(dtype):
    off = synth.offsets_from_lengths(synth.lognormal_lengths(300, seed=4, median=40, lo=0, hi=200))
    q, D = unit_case(3, 20, 96, dtype, off, seed=13)  # Nq not a power of two, d not a multiple of 64
    assert_close(run_dense(q, D, off, "simt"), oracle.maxsim(q, D, off), tol(dtype, 20))
    assert_close(run_dense(q, D, off, "auto"), oracle.maxsim(q, D, off), tol(dtype, 20))


# ---- pins P7 / P6 on the GPU: exact-integer inputs and one-hot queries must match with d = 0 -------------------------

@pytest.mark.parametrize("d", [64, 128, 256, 384, 512, 768])
@pytest.mark.parametrize("Q,Nq", [(1, 32), (4, 32), (8, 32), (5, 16), (3, 20), (16, 8)])
def test_exact_integer_inputs_are_bit_exact(d, Q, Nq):
    dtype = torch.bfloat16 if (d // 64 + Q) % 2 else torch.float16
    lens = np.concatenate([RAGGED, np.full(300, 128), synth.lognormal_lengths(300, seed=d + Q)])
    off = synth.offsets_from_lengths(lens)
    q = synth.small_int_tokens(Q * Nq, d, dtype, seed=1).view(Q, Nq, d)
    D = synth.small_int_tokens(int(off[-1]), d, dtype, seed=2)
    try:
        got = run_dense(q, D, off, "tcgen05")
    except RuntimeError as e:
        if "unsupported" in str(e):
            pytest.skip(f"tcgen05 path does not take Q={Q} Nq={Nq} d={d}")
        raise
    ref = oracle.maxsim(q, D, off)
    assert np.array_equal(got, ref), f"max |d| = {np.abs(got[np.isfinite(ref)] - ref[np.isfinite(ref)]).max()}"


@pytest.mark.parametrize("dtype", [torch.bfloat16, torch.float16])
def test_onehot_queries_pick_column_maxima(dtype):
    Q, Nq, d = 4, 32, 128
    q, pi = synth.onehot_queries(Q, Nq, d, dtype, seed=4)
    off = synth.offsets_from_lengths(synth.lognormal_lengths(500, seed=8))
    D = synth.unit_tokens(int(off[-1]), d, dtype, seed=6)
    got = run_dense(q, D, off, "tcgen05")
    D64 = D.to(torch.float64).numpy()
    ref = np.stack([[sum(D64[off[b]:off[b + 1], pi[qq, i]].max() for i in range(Nq)) for b in range(500)]
                    for qq in range(Q)])
    np.testing.assert_allclose(got, ref, rtol=0, atol=1e-5)  # products by 1.0; only the fp32 sum of 32 terms rounds


# ---- configs[3]: the dimension sweep (d > 128 accumulates 128-wide chunks before the max) ----------------------------

@pytest.mark.parametrize("d", [64, 256, 512, 768])
@pytest.mark.parametrize("variant", ["auto", "simt"])
def test_dimension_sweep(d, variant):
    off = synth.uniform_offsets(1200 if variant == "auto" else 300, 128)
    q, D = unit_case(4, 32, d, torch.bfloat16, off, seed=d)
    assert_close(run_dense(q, D, off, variant), oracle.maxsim(q, D, off), tol(torch.bfloat16, 32))


@pytest.mark.parametrize("d", [320, 384, 512, 768])
@pytest.mark.parametrize("Q", [5, 8, 11])
def test_two_query_blocks_at_large_d_run_as_cta_pairs(d, Q):
    """d*sizeof > 512 bytes leaves tensor memory room for ONE 128-row query block per SM; 256 rows then run as clusters
    of two CTAs that share every document tile by TMA multicast.  Same arithmetic per row as the
    single-CTA kernel, so scoring the queries four at a time (one block, no pairs) must give identical bits."""
    lens = np.concatenate([RAGGED, np.full(200, 128), synth.lognormal_lengths(700, seed=d + Q)])
    off = synth.offsets_from_lengths(lens)
    q, D = unit_case(Q, 32, d, torch.bfloat16, off, seed=d + 3 * Q)
    got = run_dense(q, D, off, "tcgen05")
    assert_close(got, oracle.maxsim(q, D, off), tol(torch.bfloat16, 32))
    parts = [run_dense(q[i:i + 4], D, off, "tcgen05") for i in range(0, Q, 4)]
    assert np.array_equal(got, np.concatenate(parts, axis=0))
    again = run_dense(q, D, off, "tcgen05")
    assert np.array_equal(got, again)


def test_p11_zero_padded_dimensions_tie_the_tiled_variant_to_d128():
    off = synth.offsets_from_lengths(synth.lognormal_lengths(800, seed=3))
    q, D = unit_case(4, 32, 128, torch.bfloat16, off, seed=21)
    base = run_dense(q, D, off, "tcgen05")
    for dpad in (256, 512):
        qp = torch.zeros((4, 32, dpad), dtype=torch.bfloat16)
        Dp = torch.zeros((D.shape[0], dpad), dtype=torch.bfloat16)
        qp[..., :128], Dp[:, :128] = q, D
        assert np.array_equal(run_dense(qp, Dp, off, "tcgen05"), base)


# ---- NEXT-1 shapes: the paper's Nq sweep (Table 10) and Nd sweep (Table 11) -----------------

@pytest.mark.parametrize("Nq", [8, 16, 37, 48, 64, 96])
def test_query_length_sweep(Nq):
    off = synth.offsets_from_lengths(np.concatenate([RAGGED, synth.lognormal_lengths(1500, seed=Nq)]))
    q, D = unit_case(3, Nq, 128, torch.bfloat16, off, seed=40 + Nq)
    ref = oracle.maxsim(q, D, off)
    assert_close(run_dense(q, D, off, "tcgen05"), ref, tol(torch.bfloat16, Nq))
    qi = synth.small_int_tokens(3 * Nq, 128, torch.bfloat16, seed=3).view(3, Nq, 128)
    Di = synth.small_int_tokens(int(off[-1]), 128, torch.bfloat16, seed=4)
    assert np.array_equal(run_dense(qi, Di, off, "tcgen05"), oracle.maxsim(qi, Di, off))


@pytest.mark.parametrize("Nd", [32, 64, 256, 512])
def test_document_length_sweep(Nd):
    off = synth.uniform_offsets(1000, Nd)
    q, D = unit_case(2, 32, 128, torch.float16, off, seed=60 + Nd)
    assert_close(run_dense(q, D, off, "tcgen05"), oracle.maxsim(q, D, off), tol(torch.float16, 32))


def test_fp32_inputs_on_the_tensor_cores_stay_within_1e5_nq():
    off = synth.offsets_from_lengths(np.concatenate([RAGGED, synth.lognormal_lengths(6000, seed=9)]))
    q, D = unit_case(8, 32, 128, torch.float32, off, seed=71)
    got, ref = run_dense(q, D, off, "tcgen05"), oracle.maxsim(q, D, off)
    assert_close(got, ref, tol(torch.float32, 32))
    fin = np.isfinite(ref)
    assert np.abs(got[fin] - ref[fin]).max() <= 5e-5  # measured ~1e-5: a sixth of the 3.2e-4 tolerance


# ---- properties at any size -------------------------------------------------------------------------------------------

def test_run_to_run_bit_reproducible_and_scores_overwritten():
    off = synth.offsets_from_lengths(synth.lognormal_lengths(20000, seed=5))
    q, D = unit_case(8, 32, 128, torch.bfloat16, off, seed=31)
    qd, Dd, od = q.to(DEV), D.to(DEV), torch.from_numpy(off).to(DEV)
    out = torch.full((8, 20000), float("nan"), device=DEV)
    a = tms.tms_maxsim(qd, Dd, od, scores=out).clone()
    b = tms.tms_maxsim(qd, Dd, od, scores=out)
    assert torch.equal(a, b) and bool(torch.isfinite(a).all())


def test_tcgen05_and_simt_kernels_agree():
    off = synth.offsets_from_lengths(synth.lognormal_lengths(4000, seed=6))
    q, D = unit_case(8, 32, 128, torch.float16, off, seed=33)
    a, b = run_dense(q, D, off, "tcgen05"), run_dense(q, D, off, "simt")
    assert np.abs(a - b).max() < 1e-4


def test_launch_counter_counts_kernels():
    off = synth.uniform_offsets(64, 128)
    q, D = unit_case(1, 32, 128, torch.bfloat16, off, seed=1)
    n0 = tms.tms_launch_count()
    run_dense(q, D, off)
    assert tms.tms_launch_count() == n0 + 1


# ---- host-buffer entry point -------------------------------------------------------------------------------------------

def test_host_entry_point_streams_chunks():
    off = synth.offsets_from_lengths(synth.lognormal_lengths(5000, seed=7))
    q, D = unit_case(8, 32, 128, torch.bfloat16, off, seed=35)
    scores = torch.empty((8, 5000), dtype=torch.float32).pin_memory()
    ws = torch.empty(8 << 20, dtype=torch.uint8, device=DEV)  # 8 MB: forces ~25 chunks over the 92 MB store
    tms.tms_maxsim_host(q, D.pin_memory(), torch.from_numpy(off), scores, ws)
    ref = run_dense(q, D, off)
    assert np.array_equal(scores.numpy().astype(np.float64), ref)
    small = torch.empty(1 << 16, dtype=torch.uint8, device=DEV)
    with pytest.raises(RuntimeError, match="workspace"):
        tms.tms_maxsim_host(q, D, torch.from_numpy(off), scores, small)


@pytest.mark.parametrize("d", [8, 32, 48, 80, 96, 160, 200])
def test_dimensions_that_are_not_whole_128_byte_blocks(d):
    off = synth.offsets_from_lengths(np.concatenate([RAGGED, synth.lognormal_lengths(700, seed=d)]))
    q, D = unit_case(5, 32, d, torch.bfloat16, off, seed=80 + d)
    assert_close(run_dense(q, D, off, "tcgen05"), oracle.maxsim(q, D, off), tol(torch.bfloat16, 32))
    qi = synth.small_int_tokens(5 * 32, d, torch.float16, seed=5).view(5, 32, d)
    Di = synth.small_int_tokens(int(off[-1]), d, torch.float16, seed=6)
    assert np.array_equal(run_dense(qi, Di, off, "tcgen05"), oracle.maxsim(qi, Di, off))


# ---- randomised shapes: every path of the tcgen05 kernel against the oracle --------------------------------------------

def _fuzz_lengths(rng, B):
    kind = rng.integers(0, 5)
    if kind == 0:   # tiny documents: several boundaries per 8-column chunk, many empties
        return rng.integers(0, 6, size=B)
    if kind == 1:   # single-token documents and empties only
        return rng.integers(0, 2, size=B)
    if kind == 2:   # the config-2 recipe
        return synth.lognormal_lengths(B, seed=int(rng.integers(1 << 30)))
    if kind == 3:   # a few very long documents among short ones
        lens = rng.integers(1, 40, size=B)
        lens[rng.integers(0, B, size=max(1, B // 50))] = rng.integers(500, 3000)
        return lens
    return np.full(B, int(rng.integers(1, 300)))  # uniform, any length


@pytest.mark.parametrize("seed", range(48))
def test_fuzz_shapes_against_the_oracle(seed):
    rng = np.random.default_rng(1000 + seed)
    dtype = [torch.bfloat16, torch.float16, torch.float32][seed % 3]
    # 16-bit d > 256 with more than 128 query rows runs as CTA pairs (TMA multicast); d = 320 has an odd block count
    d = int(rng.choice([64, 128, 192, 256, 320, 384, 512, 768] if dtype != torch.float32 else [64, 128, 256, 384]))
    Nq = int(rng.choice([1, 2, 3, 5, 8, 13, 16, 20, 31, 32, 64]))
    Q = int(rng.integers(1, 21))  # up to 20 queries: several query groups when Q*Nq > 256
    B = int(rng.integers(1, 1500))
    lens = _fuzz_lengths(rng, B).astype(np.int64)
    if lens.sum() == 0:
        lens[0] = 1
    off = synth.offsets_from_lengths(lens)
    q, D = unit_case(Q, Nq, d, dtype, off, seed=seed)
    ref = oracle.maxsim(q, D, off)
    assert_close(run_dense(q, D, off, "tcgen05"), ref, tol(dtype, Nq))
    qi = synth.small_int_tokens(Q * Nq, d, dtype, seed=seed + 1).view(Q, Nq, d)
    Di = synth.small_int_tokens(int(off[-1]), d, dtype, seed=seed + 2)
    assert np.array_equal(run_dense(qi, Di, off, "tcgen05"), oracle.maxsim(qi, Di, off))


# ---- parked documents outlive the ordinal ring (DOCRING wrap) ---------------------------------------------
# A warp of two epilogue sets parks only the documents that end in ITS columns (column halves) or ITS tiles (alternate
# tiles), up to 16 before it writes their scores, while the ordinal -> document ring (1024 entries) counts every document
# of the CTA.  The periodic stores below make one set park a single document per tile (or per two tiles) while > 64
# ordinals go by, so the 16 it holds span more than 1024 ordinals: the document index must have been resolved when the
# document was parked, not when the buffer is drained.  Every CTA starts on a period boundary (the token count is a
# multiple of 128 * SM count) and walks >= 24 tiles.

def _periodic_offsets(block, periods):
    return synth.offsets_from_lengths(np.tile(np.asarray(block, dtype=np.int64), periods))


@pytest.mark.parametrize("Q", [4, 8])  # one and two query blocks per CTA
def test_column_half_sets_with_one_long_and_64_single_token_documents_per_tile(Q):
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    off = _periodic_offsets([64] + [1] * 64, 24 * sms)
    q, D = unit_case(Q, 32, 128, torch.bfloat16, off, seed=61)
    assert_close(run_dense(q, D, off, "tcgen05"), oracle.maxsim(q, D, off), tol(torch.bfloat16, 32))
    # the mirrored tile: the set of the upper columns is the one that parks one document per tile
    off = _periodic_offsets([1] * 64 + [64], 24 * sms)
    q, D = unit_case(Q, 32, 128, torch.bfloat16, off, seed=63)
    assert_close(run_dense(q, D, off, "tcgen05"), oracle.maxsim(q, D, off), tol(torch.bfloat16, 32))


def test_alternate_tile_sets_with_a_128_token_document_then_128_single_token_documents():
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    # the periodic part first (CTA 0 starts at token 0 and takes T / SMs tokens of it), then long documents that lift
    # the mean length over 100 tokens, which is what selects the alternate-tile sets for one query block
    periodic = np.tile(np.asarray([128] + [1] * 128, dtype=np.int64), 64)
    n_long = 2 * sms
    long_len = 128 * (-(-(100 * (periodic.size + n_long)) // (128 * n_long)))  # whole tiles: later CTAs stay aligned
    lens = np.concatenate([periodic, np.full(n_long, long_len, dtype=np.int64)])
    off = synth.offsets_from_lengths(lens)
    assert off[-1] >= 100 * (off.size - 1) and off[-1] // sms >= 40 * 128
    q, D = unit_case(4, 32, 64, torch.bfloat16, off, seed=65)
    assert_close(run_dense(q, D, off, "tcgen05"), oracle.maxsim(q, D, off), tol(torch.bfloat16, 32))
