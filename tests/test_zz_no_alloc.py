"""GPU test of tms_topk_static, the library's one entry point that allocates nothing (include/tms.h).

Who needs it: callers that cannot get device memory for a workspace -- a process whose HBM already belongs, whole, to
another component's pool (so cudaMalloc fails), a hook inside a serving loop where the synchronising cudaMalloc /
cudaFree are off limits, a bare C caller without an allocator.  For them the top-k scratch sits in a fixed 4 MiB array
inside the library, shared by every call on the GPU and never cleared.

What is checked: the new entry point returns exactly what the existing tms_topk path returns (index work: the bar in
tests/test_gpu_topk.py is bit-exact, so it is here) on two calls IN A ROW -- the second, on a different shape, runs over
whatever the first left in the array -- and once more through raw ctypes with caller-owned outputs.  Shapes beyond the
array are refused with their own status instead of being served some other way.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide the parity tests)
and holds no state: it passes alone in a fresh process, where its first call performs the per-device address look-up,
and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_2606_26439_b200 import tms

pytestmark = pytest.mark.gpu
DEV = "cuda"


def scores_for(Q, B, seed, ties=False):
    rng = np.random.default_rng(seed)
    s = rng.integers(-3, 4, size=(Q, B)).astype(np.float32) if ties else rng.standard_normal((Q, B)).astype(np.float32)
    s[:, ::11] = -np.inf  # empty documents rank last
    return torch.from_numpy(s).to(DEV)


def same_as_existing_path(s, k):
    ref_v, ref_i = tms.tms_topk(s, k)  # existing path: caller-provided (here torch-allocated) workspace
    got_v, got_i = tms.tms_topk_static(s, k)
    torch.cuda.synchronize()
    assert torch.equal(got_i, ref_i)
    assert torch.equal(got_v.view(torch.int32), ref_v.view(torch.int32))  # bit for bit, not just ==


def test_two_calls_in_a_row_match_tms_topk_bit_for_bit():
    # first call: three selection levels, 3.1 MB of the 4 MiB array; thousands of ties decided by the index rule
    same_as_existing_path(scores_for(8, 1_000_000, seed=1, ties=True), 100)
    # second call right behind it, smaller and differently pitched: reads nothing the first call wrote
    same_as_existing_path(scores_for(3, 123_457, seed=2), 1024)
    # and a shape that needs no scratch at all (one chunk)
    same_as_existing_path(scores_for(5, 4096, seed=3), 7)


def test_raw_c_call_with_caller_owned_outputs_allocates_nothing():
    lib = tms.load()
    Q, B, k = 8, 500_000, 100
    s = scores_for(Q, B, seed=4)
    ref_v, ref_i = tms.tms_topk(s, k)
    vals = torch.full((Q, k), float("nan"), device=DEV)
    idx = torch.full((Q, k), -1, dtype=torch.int64, device=DEV)
    # the first call on a device looks the array's address up (and may load device code): do it before measuring
    tms.tms_topk_static(torch.zeros((1, 5000), device=DEV), 1)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    for _ in range(2):  # the same call twice: the second starts from the first one's leftovers
        st = lib.tms_topk_static(s.data_ptr(), Q, B, k, vals.data_ptr(), idx.data_ptr(),
                                 torch.cuda.current_stream().cuda_stream)
        assert st == 0, lib.tms_status_string(st)
        torch.cuda.synchronize()
        assert torch.equal(idx, ref_i) and torch.equal(vals.view(torch.int32), ref_v.view(torch.int32))
    # neither torch's allocator nor the device's free memory moved across the two calls
    assert (torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]) == before


def test_shapes_beyond_the_built_in_array_are_refused():
    lib = tms.load()
    cap = tms.tms_topk_static_scratch_bytes()
    assert cap == 4 << 20
    Q, B, k = 8, 1_000_000, 1024  # 32 MB of scratch through tms_topk
    assert tms.tms_topk_workspace_bytes(Q, B, k) > cap
    s = torch.zeros((Q, B), device=DEV)
    n0 = tms.tms_launch_count()
    with pytest.raises(RuntimeError, match="built-in static buffer"):
        tms.tms_topk_static(s, k)
    assert tms.tms_launch_count() == n0  # refused before any launch
    assert lib.tms_status_string(6).startswith(b"shape needs more scratch")
    # the largest shape that fits is served, one chunk more is not
    Q, k = 1, 1024
    fits = 256 * 4096
    assert tms.tms_topk_workspace_bytes(Q, fits, k) == cap
    same_as_existing_path(scores_for(Q, fits, seed=5), k)
    with pytest.raises(RuntimeError, match="status 6"):
        tms.tms_topk_static(torch.zeros((Q, fits + 1), device=DEV), k)
    # argument errors are tms_topk's
    with pytest.raises(RuntimeError, match="invalid"):
        tms.tms_topk_static(torch.zeros((2, 100), device=DEV), 101)
