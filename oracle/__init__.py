"""fp64 CPU oracle for MaxSim scoring -- TEST INFRASTRUCTURE, not part of the product path.

Loads ``oracle/liboracle.so`` (plain C, built from ``oracle/oracle.c`` with gcc) through ctypes.
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It shares nothing with ``paper_2606_26439_b200`` and neither imports
the other.

Definitions implemented (PAPER.md line numbers, "P:L"):
  * dense MaxSim, Eq. 1: ``score(q,b) = sum_i max_{j in doc b} <q_i, d_j>``
  * PQ: explicit decompression followed by the dense definition; Eq. 8-9
    define the same value through a lookup table, which the tests check as an identity.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

# numeric values of the public dtype enum (include/tms.h), restated: they are part of the C-ABI contract
F32, F16, BF16 = 0, 1, 2
_DTYPE_CODE = {"f32": F32, "fp32": F32, "float32": F32, "f16": F16, "fp16": F16, "float16": F16,
               "bf16": BF16, "bfloat16": BF16}

_lib = None


def build(force: bool = False) -> str:
    """Compile oracle.c -> liboracle.so (no -march=native: the .so travels to other hosts)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-mavx2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64
        lib.oracle_bruteforce.argtypes = [vp, i32, i32, i32, vp, vp, i64, i32, vp]
        lib.oracle_bruteforce.restype = None
        lib.oracle_maxsim.argtypes = [vp, i32, i32, i32, vp, vp, i64, i32, vp, i32]
        lib.oracle_maxsim.restype = i32
        lib.oracle_pq_maxsim.argtypes = [vp, i32, i32, i32, i32, vp, i32, i32, vp, vp, i64, vp, i32]
        lib.oracle_pq_maxsim.restype = i32
        lib.oracle_max_threads.argtypes = []
        lib.oracle_max_threads.restype = i32
        _lib = lib
    return _lib


def dtype_code(name) -> int:
    return _DTYPE_CODE[str(name).replace("torch.", "")]


def raw(x):
    """(host ndarray of storage bytes, dtype code) from a numpy array or a CPU/GPU torch tensor.

    fp32 -> float32 array; fp16/bf16 -> uint16 array holding the exact storage bits.
    """
    if hasattr(x, "detach"):  # a torch tensor; torch is only needed when one is passed in
        import torch

        t = x.detach().cpu().contiguous()
        if t.dtype == torch.float32:
            return t.numpy(), F32
        if t.dtype == torch.float16:
            return t.view(torch.int16).numpy().view(np.uint16), F16
        if t.dtype == torch.bfloat16:
            return t.view(torch.int16).numpy().view(np.uint16), BF16
        raise TypeError(f"unsupported tensor dtype {t.dtype}")
    a = np.ascontiguousarray(x)
    if a.dtype == np.float32:
        return a, F32
    if a.dtype == np.float16:
        return a.view(np.uint16), F16
    raise TypeError("numpy input must be float32 or float16 (pass bf16 as a torch tensor or via raw bits + dtype)")


def _host_i64(offsets) -> np.ndarray:
    if hasattr(offsets, "detach"):
        offsets = offsets.detach().cpu().numpy()
    return np.ascontiguousarray(offsets, dtype=np.int64)


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _prep(queries, docs, offsets, dtype):
    if dtype is None:
        q, cq = raw(queries)
        D, cd = raw(docs)
        if cq != cd:
            raise TypeError("queries and docs must share a dtype")
        code = cq
    else:  # raw storage bits passed directly
        code = dtype_code(dtype)
        q, D = np.ascontiguousarray(queries), np.ascontiguousarray(docs)
    off = _host_i64(offsets)
    if q.ndim != 3 or D.ndim != 2 or q.shape[2] != D.shape[1]:
        raise ValueError("queries must be [Q,Nq,d] and docs [T,d]")
    B = off.shape[0] - 1
    if off[0] != 0 or off[B] != D.shape[0] or np.any(np.diff(off) < 0):
        raise ValueError("offsets must start at 0, be non-decreasing and end at total_tokens")
    return q, D, off, code, B


def bruteforce(queries, docs, offsets, dtype=None) -> np.ndarray:
    """Eq. 1 as literal nested loops (pin P1). Returns float64 [Q, B]."""
    q, D, off, code, B = _prep(queries, docs, offsets, dtype)
    out = np.empty((q.shape[0], B), dtype=np.float64)
    _load().oracle_bruteforce(_ptr(q), q.shape[0], q.shape[1], q.shape[2], _ptr(D), _ptr(off), B, code, _ptr(out))
    return out


def maxsim(queries, docs, offsets, dtype=None, threads: int = 0, return_threads: bool = False):
    """Eq. 1 in fp64 over the dtype-rounded inputs, parallel over documents. Returns float64 [Q, B]."""
    q, D, off, code, B = _prep(queries, docs, offsets, dtype)
    out = np.empty((q.shape[0], B), dtype=np.float64)
    used = _load().oracle_maxsim(_ptr(q), q.shape[0], q.shape[1], q.shape[2], _ptr(D), _ptr(off), B, code,
                                 _ptr(out), int(threads))
    return (out, used) if return_threads else out


def pq_maxsim(queries, codebooks, codes, offsets, threads: int = 0, return_threads: bool = False):
    """Decompress each document from its uint8 codes (fp32, exact), then Eq. 1 in fp64. float64 [Q, B]."""
    q, code = raw(queries)
    C = codebooks.detach().cpu().numpy() if hasattr(codebooks, "detach") else codebooks
    C = np.ascontiguousarray(C, dtype=np.float32)
    cd = codes.detach().cpu().numpy() if hasattr(codes, "detach") else codes
    cd = np.ascontiguousarray(cd, dtype=np.uint8)
    off = _host_i64(offsets)
    M, K, dsub = C.shape
    if q.ndim != 3 or q.shape[2] != M * dsub or cd.ndim != 2 or cd.shape[1] != M or K > 256:
        raise ValueError("shape mismatch between queries [Q,Nq,d], codebooks [M,K,d/M] and codes [T,M]")
    B = off.shape[0] - 1
    if off[0] != 0 or off[B] != cd.shape[0] or np.any(np.diff(off) < 0):
        raise ValueError("offsets must start at 0, be non-decreasing and end at total_tokens")
    if cd.size and int(cd.max()) >= K:
        raise ValueError("code value >= K")
    out = np.empty((q.shape[0], B), dtype=np.float64)
    used = _load().oracle_pq_maxsim(_ptr(q), q.shape[0], q.shape[1], q.shape[2], code, _ptr(C), M, K, _ptr(cd),
                                    _ptr(off), B, _ptr(out), int(threads))
    return (out, used) if return_threads else out


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def topk(scores, k: int):
    """Plain definition of per-query top-k (the step after scoring): documents ordered by score descending,
    ties by lower document index first; returns (values[Q,k] float64, indices[Q,k] int64).

    A stable sort of the negated scores keeps equal scores in index order, which is exactly the tie rule.
    Pins (tests/test_oracle_pins.py): brute-force selection on tiny inputs, ties, -inf, k = B.
    """
    s = np.asarray(scores, dtype=np.float64)
    order = np.argsort(-s, axis=1, kind="stable")[:, :k]
    return np.take_along_axis(s, order, axis=1), order.astype(np.int64)
