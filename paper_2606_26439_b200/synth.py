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


def plant_relevant(queries: torch.Tensor, docs: torch.Tensor, offsets: np.ndarray, seed: int, per_query: int = 128,
                   c_hi: float = 0.95, c_span: float = 0.5) -> np.ndarray:
    """Overwrite the first Nq tokens of `per_query` seeded documents per query with planted matches.

    Planted token = c_r * qhat_i + sqrt(1 - c_r^2) * u_i with u_i a unit vector orthogonal to qhat_i and
    c_r = c_hi - c_span * r / (per_query - 1), so planted document r of query q has cosine c_r with every
    token of q: scores are separated by ~Nq*c_span/(per_query-1), far above the bf16 tolerance
    (SURVEY.md 8(c) ranking rule).  Modifies `docs` in place; returns ids[Q, per_query] (rank order).
    """
    Q, Nq, d = queries.shape
    lengths = np.diff(offsets)
    eligible = np.nonzero(lengths >= Nq)[0]
    if eligible.size < Q * per_query:
        raise ValueError("not enough documents with Nd >= Nq to plant into")
    rng = np.random.default_rng(seed)
    ids = rng.choice(eligible, size=Q * per_query, replace=False).reshape(Q, per_query)
    g = _gen("cpu", seed, 1)
    qf = queries.detach().cpu().to(torch.float32)
    qhat = qf / qf.norm(dim=2, keepdim=True).clamp_min(1e-20)
    for q in range(Q):
        for r in range(per_query):
            c = c_hi - c_span * r / max(per_query - 1, 1)
            u = torch.randn((Nq, d), dtype=torch.float32, generator=g)
            u = u - (u * qhat[q]).sum(dim=1, keepdim=True) * qhat[q]
            u = u / u.norm(dim=1, keepdim=True)
            tok = c * qhat[q] + math.sqrt(1.0 - c * c) * u
            t0 = int(offsets[ids[q, r]])
            docs[t0:t0 + Nq] = tok.to(docs.dtype).to(docs.device)
    return ids


def plant_relevant_pq(queries: torch.Tensor, codebooks: torch.Tensor, codes: torch.Tensor, offsets: np.ndarray, seed: int,
                      per_query: int = 32) -> np.ndarray:
    """Planted PQ documents: document r of query q gets, as the codes of its first Nq - r tokens, the centroids closest (by
    inner product) to query tokens 0 .. Nq - r - 1 in every sub-quantiser; the other tokens keep their random codes.
    Each planted token lifts one query token's maximum far above what random codes reach, so the scores of a query's
    planted documents fall by a clear step from rank to rank (the test checks the steps on the oracle's scores).
    Modifies `codes` in place; returns ids[Q, per_query] in rank order.  per_query <= Nq."""
    Q, Nq, d = queries.shape
    M, K, dsub = codebooks.shape
    if per_query > Nq:
        raise ValueError("per_query <= Nq")
    lengths = np.diff(offsets)
    eligible = np.nonzero(lengths >= Nq)[0]
    rng = np.random.default_rng(seed)
    ids = rng.choice(eligible, size=Q * per_query, replace=False).reshape(Q, per_query)
    qf = queries.detach().cpu().to(torch.float32).reshape(Q, Nq, M, dsub)
    best = torch.einsum("qims,mks->qimk", qf, codebooks.detach().cpu().to(torch.float32)).argmax(dim=3)  # [Q, Nq, M]
    for q in range(Q):
        for r in range(per_query):
            n = Nq - r
            t0 = int(offsets[ids[q, r]])
            codes[t0:t0 + n] = best[q, :n].to(torch.uint8).to(codes.device)
    return ids
