"""Algorithmic byte / FLOP accounting used by bench.py (the paper's IO model, section 2.3, 3.4, 4.4).

These are the bytes the method itself must move, not measured traffic.  tests/test_accounting.py pins
them to the totals the paper prints (tests/golden/paper_io_totals.txt).
"""
from __future__ import annotations


def flops_eq3(B: int, Nq: int, Nd: int, d: int) -> int:
    """Eq. 3: B*Nq*Nd*(2d+1) -- multiply+add per dimension plus one max compare."""
    return B * Nq * Nd * (2 * d + 1)


def io_naive_eq4(B: int, Nq: int, Nd: int, d: int, s: int = 2) -> int:
    """Eq. 4: read Q, read D, write + read the fp32 similarity matrix."""
    return Nq * d * s + B * Nd * d * s + 2 * B * Nq * Nd * 4


def io_fused_eq5(B: int, Nq: int, Nd: int, d: int, s: int = 2) -> int:
    """Eq. 5: fused, with B*Nq*4 output bytes (the paper's printed 328,968,192 uses this form)."""
    return Nq * d * s + B * Nd * d * s + B * Nq * 4


def io_optimal_eq7(B: int, Nq: int, Nd: int, d: int, s: int = 2) -> int:
    """Eq. 7: every embedding read once, one fp32 per document written."""
    return (Nq * d + B * Nd * d) * s + B * 4


def pq_io_decompress_then_score(B: int, Nq: int, Nd: int, d: int, M: int) -> int:
    """Section 4.4: B*Nd*(M + 2d) + 2*B*Nq*Nd*4."""
    return B * Nd * (M + d * 2) + 2 * B * Nq * Nd * 4


def pq_io_fused(B: int, Nq: int, Nd: int, M: int, K: int) -> int:
    """Section 4.4: Nq*M*K*4 + B*Nd*M + B*Nq*4."""
    return Nq * M * K * 4 + B * Nd * M + B * Nq * 4


# ---- generalised to Q queries per call and a packed store of T tokens (reading A3: Eq. 7 form) ---------------------

def dense_bytes(Q: int, Nq: int, d: int, T: int, B: int, elem_bytes: int) -> int:
    """Q*Nq*d*s (queries once) + T*d*s (every document token once) + Q*B*4 (scores)."""
    return Q * Nq * d * elem_bytes + T * d * elem_bytes + Q * B * 4


def dense_flops(Q: int, Nq: int, d: int, T: int) -> int:
    """2*Q*Nq*T*d (reading A4: the paper's reported TFLOP/s use 2d, not 2d+1)."""
    return 2 * Q * Nq * T * d


def pq_bytes(Q: int, Nq: int, M: int, K: int, T: int, B: int) -> int:
    """LUT once + codes once + scores."""
    return Q * Nq * M * K * 4 + T * M + Q * B * 4


def pq_lookups(Q: int, Nq: int, M: int, T: int) -> int:
    return Q * Nq * M * T
