"""C-ABI checks that need no GPU: libtms.so builds, loads and exports every symbol include/tms.h declares,
the binding covers the same set, and argument validation answers before any CUDA work."""
import ctypes
import os
import re

import pytest

from paper_2606_26439_b200 import build as tms_build
from paper_2606_26439_b200 import tms

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    tms_build.build()
    return tms.load()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "tms.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tms_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for required in ("tms_maxsim", "tms_pq_build_lut", "tms_pq_maxsim"):
        assert required in names


def test_library_exports_every_declared_symbol(lib):
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} declared in include/tms.h but not exported by libtms.so"


def test_binding_covers_every_declared_symbol():
    assert sorted(tms.SIGNATURES) == declared_functions()


def test_status_strings_and_version(lib):
    assert lib.tms_version() >= 100
    assert lib.tms_status_string(0) == b"ok"
    assert len({lib.tms_status_string(i) for i in range(7)}) == 7


def test_workspace_size_functions(lib):
    assert lib.tms_maxsim_workspace_bytes(8, 32, 128, 500000, tms.TMS_DTYPE_BF16) == 0
    assert lib.tms_pq_workspace_bytes(8, 32, 16, 256, 1000000) == 8 * 32 * 16 * 256 * 4 + 16  # table + header
    assert lib.tms_pq_workspace_bytes(8, 32, 8, 256, 1000) == 0
    assert lib.tms_maxsim_host_workspace_min_bytes(8, 32, 128, tms.TMS_DTYPE_BF16, 180) > 2 * 180 * 256


def test_pq_variant_used_is_a_pure_function_and_never_the_lossy_kernel(lib):
    assert lib.tms_pq_maxsim_variant_used(8, 32, 16, 256) == tms.TMS_VARIANT_PQ_SMEM   # configs[4]: fp32 entries
    assert lib.tms_pq_maxsim_variant_used(8, 24, 16, 256) == tms.TMS_VARIANT_PQ_SMEM
    assert lib.tms_pq_maxsim_variant_used(5, 7, 16, 256) == tms.TMS_VARIANT_SIMT
    assert lib.tms_pq_maxsim_variant_used(2, 12, 8, 64) == tms.TMS_VARIANT_SIMT
    assert lib.tms_pq_maxsim_variant_used(0, 32, 16, 256) == tms.TMS_VARIANT_AUTO
    assert tms.tms_pq_maxsim_variant_used(8, 32, 16, 256) == "pq_smem"


def test_topk_merge_rejects_a_shard_base_of_2_to_the_31(lib):
    buf = (ctypes.c_char * 4096)()
    p16 = (ctypes.addressof(buf) + 15) & ~15
    for bad in (1 << 31, -1):
        base = (ctypes.c_int64 * 2)(0, bad)
        assert lib.tms_topk_merge(p16, p16, ctypes.addressof(base), 2, 1, 4, 4, p16, p16, p16, 4096, None) == 1


def test_static_topk_limit_is_reported_without_a_device(lib):
    assert lib.tms_topk_static_scratch_bytes() == 4 << 20
    buf = (ctypes.c_char * 4096)()
    p16 = (ctypes.addressof(buf) + 15) & ~15
    assert lib.tms_topk_static(p16, 8, 1_000_000, 1024, p16, p16, None) == 6  # refused before any CUDA call
    assert b"static buffer" in lib.tms_status_string(6)


def test_argument_validation_happens_before_any_cuda_call(lib):
    buf = (ctypes.c_char * 4096)()
    p = ctypes.addressof(buf)
    p16 = (p + 15) & ~15
    ok = dict(Q=1, Nq=4, d=8)
    # non-positive sizes
    assert lib.tms_maxsim(p16, 0, 4, 8, p16, p16, 1, 4, 0, p16, None, 0, None) == 1
    assert lib.tms_maxsim(p16, 1, 4, 8, p16, p16, -1, 4, 0, p16, None, 0, None) == 1
    # NULL pointers
    assert lib.tms_maxsim(None, 1, 4, 8, p16, p16, 1, 4, 0, p16, None, 0, None) == 1
    assert lib.tms_maxsim(p16, 1, 4, 8, p16, None, 1, 4, 0, p16, None, 0, None) == 1
    # bad dtype enum
    assert lib.tms_maxsim(p16, 1, 4, 8, p16, p16, 1, 4, 7, p16, None, 0, None) == 1
    # row pitch not a multiple of 16 bytes: d=6 fp16 -> 12 bytes
    assert lib.tms_maxsim(p16, 1, 4, 6, p16, p16, 1, 4, 1, p16, None, 0, None) == 2
    # misaligned docs pointer
    assert lib.tms_maxsim(p16, 1, 4, 8, p16 + 4, p16, 1, 4, 0, p16, None, 0, None) == 3
    # PQ: d % M != 0, K > 256
    assert lib.tms_pq_build_lut(p16, 1, 4, 10, 0, p16, 4, 16, p16, None) == 2
    assert lib.tms_pq_build_lut(p16, 1, 4, 8, 0, p16, 4, 300, p16, None) == 2
    assert lib.tms_pq_maxsim(None, 1, 4, 4, 16, p16, p16, 1, 4, p16, None, 0, None) == 1
    assert ok


def test_no_cpu_fallback_without_a_device(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    buf = (ctypes.c_char * 4096)()
    p16 = (ctypes.addressof(buf) + 15) & ~15
    # valid arguments, no device: the call must fail with TMS_ERR_CUDA, never compute on the host
    assert lib.tms_maxsim(p16, 1, 4, 8, p16, p16, 1, 4, 0, p16, None, 0, None) == 5
