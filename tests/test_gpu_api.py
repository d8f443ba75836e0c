"""GPU tests of the boundary's behaviour (include/tms.h): which kernel AUTO runs, scratch errors instead of silent
fall-backs, the all-empty store, and the host-buffer entry points against the ORACLE (not against the device path)."""
import ctypes

import numpy as np
import pytest
import torch

import oracle
from paper_2606_26439_b200 import synth, tms

pytestmark = pytest.mark.gpu
DEV = "cuda"
RAGGED = np.array([5, 128, 1, 0, 300, 127, 129, 64, 0, 0, 17, 256, 8, 1, 1, 1000, 33], dtype=np.int64)


def tol(dtype, Nq):
    return (1e-5 if dtype == torch.float32 else 2e-3) * Nq


def assert_close(got, ref, atol):
    inf = np.isneginf(ref)
    assert np.array_equal(np.isneginf(got), inf)
    err = np.abs(got[~inf] - ref[~inf])
    assert err.size == 0 or err.max() <= atol, f"max |dscore| = {err.max():.3e} > {atol:.3e}"


# ---- which kernel runs -----------------------------------------------------------------------------------------------

@pytest.mark.parametrize("Q,Nq,d,dtype,want", [
    (8, 32, 128, torch.bfloat16, "tcgen05"), (1, 32, 128, torch.float32, "tcgen05"), (4, 32, 768, torch.float16, "tcgen05"),
    (8, 64, 128, torch.bfloat16, "tcgen05"), (3, 37, 96, torch.bfloat16, "tcgen05"), (8, 32, 384, torch.float32, "tcgen05"),
    (2, 32, 1024, torch.bfloat16, "simt"), (2, 32, 96, torch.float32, "simt"), (2, 32, 512, torch.float32, "simt"),
])
def test_variant_used_is_a_pure_function_of_the_shape(Q, Nq, d, dtype, want):
    B, T = 1000, 128000
    assert tms.tms_maxsim_variant_used(Q, Nq, d, B, T, dtype) == want
    # and AUTO computes what that variant computes, bit for bit
    off = synth.offsets_from_lengths(np.concatenate([RAGGED, np.full(40, 128)]))
    q = synth.unit_tokens(Q * Nq, d, dtype, seed=1).view(Q, Nq, d).to(DEV)
    D = synth.unit_tokens(int(off[-1]), d, dtype, seed=2).to(DEV)
    od = torch.from_numpy(off).to(DEV)
    assert torch.equal(tms.tms_maxsim(q, D, od), tms.tms_maxsim(q, D, od, variant=want))


def test_variant_used_for_huge_and_degenerate_stores():
    assert tms.tms_maxsim_variant_used(8, 32, 8, 1 << 20, (1 << 31) + 5, torch.bfloat16) == "tcgen05"  # token segments
    assert tms.tms_maxsim_variant_used(8, 32, 128, 0, 0, torch.bfloat16) == "auto"
    assert tms.tms_maxsim_variant_used(8, 32, 128, 10, 0, torch.bfloat16) == "auto"


# ---- scratch for long queries is never optional ------------------------------------------------------------------------

def _raw_maxsim(q, D, od, scores, ws_ptr, ws_len, variant=0):
    lib = tms.load()
    Q, Nq, d = q.shape
    return lib.tms_maxsim_variant(q.data_ptr(), Q, Nq, d, D.data_ptr(), od.data_ptr(), od.numel() - 1, D.shape[0],
                                  tms._DTYPES[q.dtype], scores.data_ptr(), ws_ptr, ws_len,
                                  torch.cuda.current_stream().cuda_stream, variant)


def test_missing_short_or_misaligned_workspace_is_an_error_not_a_slower_kernel():
    off = synth.uniform_offsets(300, 100)
    q = synth.unit_tokens(2 * 64, 128, torch.bfloat16, seed=1).view(2, 64, 128).to(DEV)
    D = synth.unit_tokens(int(off[-1]), 128, torch.bfloat16, seed=2).to(DEV)
    od = torch.from_numpy(off).to(DEV)
    scores = torch.empty((2, 300), dtype=torch.float32, device=DEV)
    need = tms.tms_maxsim_workspace_bytes(2, 64, 128, 300, torch.bfloat16)
    assert need == 2 * 2 * 300 * 4
    ws = torch.empty(need + 64, dtype=torch.uint8, device=DEV)
    n0 = tms.tms_launch_count()
    assert _raw_maxsim(q, D, od, scores, None, 0) == 4                      # TMS_ERR_WORKSPACE
    assert _raw_maxsim(q, D, od, scores, ws.data_ptr(), need - 1) == 4
    assert _raw_maxsim(q, D, od, scores, ws.data_ptr() + 4, need) == 3      # TMS_ERR_ALIGNMENT
    assert tms.tms_launch_count() == n0, "an error must not launch anything"
    assert _raw_maxsim(q, D, od, scores, ws.data_ptr(), need) == 0
    torch.cuda.synchronize()
    assert tms.tms_launch_count() == n0 + 2                                  # scoring + sum of the parts
    assert_close(scores.cpu().numpy().astype(np.float64), oracle.maxsim(q.cpu(), D.cpu(), off), tol(torch.bfloat16, 64))
    # the CUDA-core kernel needs no scratch and says so by running
    assert _raw_maxsim(q, D, od, scores, None, 0, variant=1) == 0


# ---- a store whose documents are all empty ------------------------------------------------------------------------------

@pytest.mark.parametrize("variant", ["auto", "tcgen05", "simt"])
def test_all_documents_empty(variant):
    B = 77
    od = torch.zeros(B + 1, dtype=torch.int64, device=DEV)
    q = synth.unit_tokens(3 * 32, 128, torch.bfloat16, seed=1).view(3, 32, 128).to(DEV)
    D = torch.empty((0, 128), dtype=torch.bfloat16, device=DEV)
    s = tms.tms_maxsim(q, D, od, variant=variant)
    assert s.shape == (3, B) and bool(torch.isneginf(s).all())


def test_all_documents_empty_pq_decode():
    B = 33
    od = torch.zeros(B + 1, dtype=torch.int64, device=DEV)
    q = synth.unit_tokens(2 * 32, 128, torch.bfloat16, seed=1).view(2, 32, 128).to(DEV)
    C = synth.pq_codebooks(16, 256, 8, seed=3).to(DEV)
    codes = torch.empty((0, 16), dtype=torch.uint8, device=DEV)
    assert bool(torch.isneginf(tms.tms_pq_maxsim_decode(q, C, codes, od)).all())


# ---- host-buffer entry points against the oracle ---------------------------------------------------------------------------

@pytest.mark.parametrize("Nq,dtype,Q,d", [(32, torch.bfloat16, 4, 128), (64, torch.float16, 4, 128), (48, torch.bfloat16, 4, 128),
                                          (32, torch.bfloat16, 8, 512)])  # the last one: CTA pairs through the host call
def test_host_entry_point_against_the_oracle(Nq, dtype, Q, d):
    lens = np.concatenate([RAGGED, synth.lognormal_lengths(1500, seed=7)])
    off = synth.offsets_from_lengths(lens)
    B = len(lens)
    q = synth.unit_tokens(Q * Nq, d, dtype, seed=35).view(Q, Nq, d)
    D = synth.unit_tokens(int(off[-1]), d, dtype, seed=36)
    scores = torch.empty((Q, B), dtype=torch.float32).pin_memory()
    ws = torch.empty(4 << 20, dtype=torch.uint8, device=DEV)  # forces several chunks
    assert tms.tms_maxsim_variant_used(Q, Nq, d, B, int(off[-1]), dtype) == "tcgen05"
    n0 = tms.tms_launch_count()
    tms.tms_maxsim_host(q, D.pin_memory(), torch.from_numpy(off), scores, ws)
    assert tms.tms_launch_count() - n0 >= 4, "several chunks expected"
    assert_close(scores.numpy().astype(np.float64), oracle.maxsim(q, D, off), tol(dtype, Nq))
    # same bits as the device entry point: the host call runs the same kernel
    dev = tms.tms_maxsim(q.to(DEV), D.to(DEV), torch.from_numpy(off).to(DEV)).cpu()
    assert torch.equal(dev, scores)


def test_pq_host_entry_points_against_the_oracle():
    lens = np.concatenate([RAGGED, synth.lognormal_lengths(1200, seed=9)])
    off = synth.offsets_from_lengths(lens)
    Q, Nq, B, T = 3, 32, len(lens), int(off[-1])
    q = synth.unit_tokens(Q * Nq, 128, torch.bfloat16, seed=41).view(Q, Nq, 128)
    C = synth.pq_codebooks(16, 256, 8, seed=42)
    codes = synth.pq_codes(T, 16, seed=43)
    ref = oracle.pq_maxsim(q, C, codes, off)
    for fn, need in ((tms.tms_pq_maxsim_host, tms.tms_pq_maxsim_host_workspace_min_bytes),
                     (tms.tms_pq_maxsim_decode_host, tms.tms_pq_maxsim_decode_host_workspace_min_bytes)):
        scores = torch.empty((Q, B), dtype=torch.float32).pin_memory()
        ws = torch.empty(need(Q, Nq, 128, torch.bfloat16, 16, 256, 1000) + (256 << 10), dtype=torch.uint8, device=DEV)
        fn(q, C, codes.pin_memory(), torch.from_numpy(off), scores, ws)
        assert_close(scores.numpy().astype(np.float64), ref, tol(torch.bfloat16, Nq))


# ---- top-k: -0.0 ties with +0.0 ----------------------------------------------------------------------------------------------

def test_topk_treats_negative_zero_as_zero():
    s = torch.tensor([[0.0, -0.0, -1.0, 0.0, -0.0, 2.0, float("-inf"), -0.0]], dtype=torch.float32, device=DEV)
    v, i = tms.tms_topk(s, 6)
    assert i.cpu().tolist() == [[5, 0, 1, 3, 4, 7]]
    ref_v, ref_i = oracle.topk(s.cpu().numpy(), 6)
    assert np.array_equal(ref_i, i.cpu().numpy()) and np.array_equal(ref_v, v.cpu().numpy())
