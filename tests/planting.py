"""Planted relevant documents for the ranking tests (test-only helpers; they live here, not in the package's shared
input generator, because choosing WHAT to plant evaluates part of the method -- cosines, Eq. 8's table -- and the
module both sides share must hold none of the method's arithmetic).  The tests re-check the planted score steps on the
oracle's own scores, so nothing here is trusted."""
import math

import numpy as np
import torch

from paper_2606_26439_b200.synth import _gen


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
