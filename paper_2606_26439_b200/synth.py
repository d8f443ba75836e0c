"""Seeded synthetic inputs shaped like the paper's workloads.

This module only *generates inputs*: none of MaxSim's arithmetic lives here.  It is the one module
both the CUDA path's callers and the oracle's callers (tests, bench) use, so that the two sides see
the same bytes.  The paper's own large-scale rows use "synthetic (normalized random)" embeddings
(P:L595); its MS MARCO / BEIR embeddings are not available here and these inputs stand in for them
(DESIGN.md "Input recipe").

Recipe (reading A20): element ~ N(0,1) in fp32 -> L2-normalise each token in fp32 ->
round-to-nearest-even to the storage dtype; no re-normalisation.  Generation is chunked (2^20 tokens
per chunk, one generator seed per chunk) so 64M-token stores can be produced on the device without
a large fp32 temporary.  CPU and CUDA generators give different streams: generate once, copy the
bytes to whoever else needs them.
"""
from __future__ import annotations

import math

import numpy as np
import torch

CHUNK_TOKENS = 1 << 20


def _gen(device, seed: int, chunk: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed((int(seed) * 1000003 + chunk * 7919 + 12345) % (2**63 - 1))
    return g


def unit_tokens(n: int, d: int, dtype: torch.dtype, seed: int, device="cpu") -> torch.Tensor:
    """[n, d] L2-normalised Gaussian token vectors, rounded to `dtype`."""
    out = torch.empty((n, d), dtype=dtype, device=device)
    for c, lo in enumerate(range(0, n, CHUNK_TOKENS)):
        hi = min(n, lo + CHUNK_TOKENS)
        x = torch.randn((hi - lo, d), dtype=torch.float32, device=device, generator=_gen(device, seed, c))
        x /= x.norm(dim=1, keepdim=True).clamp_min(1e-20)
        out[lo:hi] = x.to(dtype)
    return out


def small_int_tokens(n: int, d: int, dtype: torch.dtype, seed: int, device="cpu", lo: int = -2, hi: int = 2):
    """[n, d] integers in [lo, hi]: exact in every dtype, every partial dot product exact in fp32."""
    out = torch.empty((n, d), dtype=dtype, device=device)
    for c, a in enumerate(range(0, n, CHUNK_TOKENS)):
        b = min(n, a + CHUNK_TOKENS)
        x = torch.randint(lo, hi + 1, (b - a, d), device=device, generator=_gen(device, seed, c))
        out[a:b] = x.to(dtype)
    return out


def onehot_queries(Q: int, Nq: int, d: int, dtype: torch.dtype, seed: int) -> tuple[torch.Tensor, np.ndarray]:
    """queries[q,i,:] = e_{pi[q,i]}; returns (queries, pi)."""
    rng = np.random.default_rng(seed)
    pi = rng.integers(0, d, size=(Q, Nq))
    q = torch.zeros((Q, Nq, d), dtype=torch.float32)
    q.view(-1, d)[torch.arange(Q * Nq), torch.from_numpy(pi.reshape(-1))] = 1.0
    return q.to(dtype), pi


def uniform_offsets(B: int, Nd: int) -> np.ndarray:
    return np.arange(B + 1, dtype=np.int64) * Nd


def lognormal_lengths(B: int, seed: int, median: float = 64.0, sigma: float = 0.5, lo: int = 8,
                      hi: int = 180) -> np.ndarray:
    """Nd ~ round(exp(N(ln median, sigma^2))) clipped to [lo, hi] (BASELINE.json configs[2])."""
    rng = np.random.default_rng(seed)
    x = np.exp(rng.normal(math.log(median), sigma, size=B))
    return np.clip(np.rint(x), lo, hi).astype(np.int64)


def offsets_from_lengths(lengths) -> np.ndarray:
    off = np.zeros(len(lengths) + 1, dtype=np.int64)
    np.cumsum(np.asarray(lengths, dtype=np.int64), out=off[1:])
    return off


def pq_codebooks(M: int, K: int, dsub: int, seed: int) -> torch.Tensor:
    """fp32 [M, K, dsub] ~ N(0, variance 1/8) (reading A12)."""
    g = _gen("cpu", seed, 0)
    return torch.randn((M, K, dsub), dtype=torch.float32, generator=g) * math.sqrt(1.0 / 8.0)


def pq_codes(T: int, M: int, seed: int, device="cpu", K: int = 256) -> torch.Tensor:
    """uint8 [T, M] uniform in [0, K)."""
    out = torch.empty((T, M), dtype=torch.uint8, device=device)
    step = CHUNK_TOKENS * 8
    for c, lo in enumerate(range(0, T, step)):
        hi = min(T, lo + step)
        out[lo:hi] = torch.randint(0, K, (hi - lo, M), device=device, generator=_gen(device, seed, c),
                                   dtype=torch.int32).to(torch.uint8)
    return out
