"""Thin ctypes binding over libtms.so: same names as include/tms.h, argument marshalling only.

PyTorch is used for device memory and streams; every step of the hot path runs inside the library's
CUDA kernels.  There is no fallback: if libtms.so is missing or a call fails, a RuntimeError is raised.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtms.so")

TMS_OK = 0
TMS_DTYPE_F32, TMS_DTYPE_F16, TMS_DTYPE_BF16 = 0, 1, 2
TMS_VARIANT_AUTO, TMS_VARIANT_SIMT, TMS_VARIANT_TCGEN05, TMS_VARIANT_PQ_SMEM, TMS_VARIANT_PQ_SMEM_F16 = 0, 1, 2, 3, 4
VARIANTS = {"auto": 0, "simt": 1, "tcgen05": 2, "pq_smem": 3, "pq_smem_f16": 4}

_DTYPES = {torch.float32: TMS_DTYPE_F32, torch.float16: TMS_DTYPE_F16, torch.bfloat16: TMS_DTYPE_BF16}

# every symbol include/tms.h declares: (restype, argtypes)
_vp, _i, _i64, _sz, _u64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_size_t, ctypes.c_uint64
SIGNATURES = {
    "tms_maxsim": (_i, [_vp, _i, _i, _i, _vp, _vp, _i64, _i64, _i, _vp, _vp, _sz, _vp]),
    "tms_maxsim_variant": (_i, [_vp, _i, _i, _i, _vp, _vp, _i64, _i64, _i, _vp, _vp, _sz, _vp, _i]),
    "tms_maxsim_workspace_bytes": (_sz, [_i, _i, _i, _i64, _i]),
    "tms_maxsim_variant_used": (_i, [_i, _i, _i, _i64, _i64, _i]),
    "tms_pq_build_lut": (_i, [_vp, _i, _i, _i, _i, _vp, _i, _i, _vp, _vp]),
    "tms_pq_maxsim": (_i, [_vp, _i, _i, _i, _i, _vp, _vp, _i64, _i64, _vp, _vp, _sz, _vp]),
    "tms_pq_maxsim_variant": (_i, [_vp, _i, _i, _i, _i, _vp, _vp, _i64, _i64, _vp, _vp, _sz, _vp, _i]),
    "tms_pq_workspace_bytes": (_sz, [_i, _i, _i, _i, _i64]),
    "tms_pq_maxsim_variant_used": (_i, [_i, _i, _i, _i]),
    "tms_pq_maxsim_decode": (_i, [_vp, _i, _i, _i, _i, _vp, _i, _i, _vp, _vp, _i64, _i64, _vp, _vp, _sz, _vp]),
    "tms_pq_maxsim_decode_variant": (_i, [_vp, _i, _i, _i, _i, _vp, _i, _i, _vp, _vp, _i64, _i64, _vp, _vp, _sz, _vp, _i]),
    "tms_maxsim_host": (_i, [_vp, _i, _i, _i, _vp, _vp, _i64, _i64, _i, _vp, _vp, _sz, _vp]),
    "tms_pq_maxsim_host": (_i, [_vp, _i, _i, _i, _i, _vp, _i, _i, _vp, _vp, _i64, _i64, _vp, _vp, _sz, _vp]),
    "tms_pq_maxsim_decode_host": (_i, [_vp, _i, _i, _i, _i, _vp, _i, _i, _vp, _vp, _i64, _i64, _vp, _vp, _sz, _vp]),
    "tms_pq_maxsim_decode_host_workspace_min_bytes": (_sz, [_i, _i, _i, _i, _i, _i, _i64]),
    "tms_maxsim_host_workspace_min_bytes": (_sz, [_i, _i, _i, _i, _i64]),
    "tms_pq_maxsim_host_workspace_min_bytes": (_sz, [_i, _i, _i, _i, _i, _i, _i64]),
    "tms_topk": (_i, [_vp, _i, _i64, _i, _vp, _vp, _vp, _sz, _vp]),
    "tms_topk_workspace_bytes": (_sz, [_i, _i64, _i]),
    "tms_topk_static": (_i, [_vp, _i, _i64, _i, _vp, _vp, _vp]),
    "tms_topk_static_scratch_bytes": (_sz, []),
    "tms_topk_merge": (_i, [_vp, _vp, _vp, _i, _i, _i, _i, _vp, _vp, _vp, _sz, _vp]),
    "tms_topk_merge_workspace_bytes": (_sz, [_i, _i, _i, _i]),
    "tms_launch_count": (_u64, []),
    "tms_status_string": (ctypes.c_char_p, [_i]),
    "tms_version": (_i, []),
}

_lib = None


def load() -> ctypes.CDLL:
    """Load libtms.so (built by `python -m paper_2606_26439_b200.build`); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_2606_26439_b200.build` "
                               "(there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def _check(status: int, what: str) -> None:
    if status != TMS_OK:
        raise RuntimeError(f"{what} failed: {load().tms_status_string(status).decode()} (status {status})")


def _stream(stream) -> int:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def _dev(t: torch.Tensor, name: str) -> int:
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError(f"{name} must be a contiguous CUDA tensor")
    return t.data_ptr()


def tms_launch_count() -> int:
    return int(load().tms_launch_count())


def tms_version() -> int:
    return int(load().tms_version())


def tms_maxsim_workspace_bytes(Q, Nq, d, B, dtype) -> int:
    return int(load().tms_maxsim_workspace_bytes(Q, Nq, d, B, _DTYPES[dtype]))


def tms_maxsim_variant_used(Q, Nq, d, B, total_tokens, dtype) -> str:
    """Name of the kernel tms_maxsim picks for this shape ("tcgen05" / "simt"; "auto" when nothing is scored)."""
    v = int(load().tms_maxsim_variant_used(Q, Nq, d, B, total_tokens, _DTYPES[dtype]))
    return {val: name for name, val in VARIANTS.items()}[v]


def tms_pq_maxsim_variant_used(Q, Nq, M, K) -> str:
    """Name of the kernel tms_pq_maxsim picks for this shape ("pq_smem" = fp32 entries in shared memory, or "simt")."""
    v = int(load().tms_pq_maxsim_variant_used(Q, Nq, M, K))
    return {val: name for name, val in VARIANTS.items()}[v]


def tms_topk_workspace_bytes(Q, B, k) -> int:
    return int(load().tms_topk_workspace_bytes(Q, B, k))


def tms_pq_workspace_bytes(Q, Nq, M, K, B) -> int:
    return int(load().tms_pq_workspace_bytes(Q, Nq, M, K, B))


def tms_maxsim(queries: torch.Tensor, docs: torch.Tensor, offsets: torch.Tensor, scores: torch.Tensor | None = None,
               stream=None, variant: str = "auto", workspace: torch.Tensor | None = None) -> torch.Tensor:
    """scores[q,b] = sum_i max_{t in doc b} <queries[q,i], docs[t]>  (include/tms.h: tms_maxsim)."""
    Q, Nq, d = queries.shape
    T = docs.shape[0]
    B = offsets.numel() - 1
    if docs.dim() != 2 or docs.shape[1] != d or docs.dtype != queries.dtype or offsets.dtype != torch.int64:
        raise ValueError("docs must be [T,d] in the queries' dtype and offsets int64 [B+1]")
    if scores is None:
        scores = torch.empty((Q, B), dtype=torch.float32, device=queries.device)
    elif scores.shape != (Q, B) or scores.dtype != torch.float32:
        raise ValueError("scores must be fp32 [Q,B]")
    lib = load()
    need = int(lib.tms_maxsim_workspace_bytes(Q, Nq, d, B, _DTYPES[queries.dtype]))
    if workspace is None and need:
        workspace = torch.empty(need, dtype=torch.uint8, device=queries.device)
    ws_ptr = _dev(workspace, "workspace") if workspace is not None else None
    ws_len = workspace.numel() * workspace.element_size() if workspace is not None else 0
    st = lib.tms_maxsim_variant(_dev(queries, "queries"), Q, Nq, d, _dev(docs, "docs") if T else None,
                                _dev(offsets, "offsets"), B, T, _DTYPES[queries.dtype],
                                _dev(scores, "scores") if B else None, ws_ptr, ws_len, _stream(stream),
                                VARIANTS[variant])
    _check(st, "tms_maxsim")
    return scores


def tms_pq_build_lut(queries: torch.Tensor, codebooks: torch.Tensor, lut: torch.Tensor | None = None,
                     stream=None) -> torch.Tensor:
    """lut[q,i,m,k] = <queries[q,i,m-th slice], codebooks[m,k]>  (Eq. 8)."""
    Q, Nq, d = queries.shape
    M, K, dsub = codebooks.shape
    if codebooks.dtype != torch.float32 or M * dsub != d:
        raise ValueError("codebooks must be fp32 [M,K,d/M]")
    if lut is None:
        lut = torch.empty((Q, Nq, M, K), dtype=torch.float32, device=queries.device)
    st = load().tms_pq_build_lut(_dev(queries, "queries"), Q, Nq, d, _DTYPES[queries.dtype],
                                 _dev(codebooks, "codebooks"), M, K, _dev(lut, "lut"), _stream(stream))
    _check(st, "tms_pq_build_lut")
    return lut


def tms_pq_maxsim(lut: torch.Tensor, codes: torch.Tensor, offsets: torch.Tensor, scores: torch.Tensor | None = None,
                  workspace: torch.Tensor | None = None, stream=None, variant: str = "auto") -> torch.Tensor:
    """scores[q,b] = sum_i max_{t in doc b} sum_m lut[q,i,m,codes[t,m]]  (Eq. 9)."""
    Q, Nq, M, K = lut.shape
    T = codes.shape[0]
    B = offsets.numel() - 1
    if codes.dtype != torch.uint8 or codes.dim() != 2 or codes.shape[1] != M or lut.dtype != torch.float32:
        raise ValueError("codes must be uint8 [T,M] and lut fp32 [Q,Nq,M,K]")
    if scores is None:
        scores = torch.empty((Q, B), dtype=torch.float32, device=lut.device)
    lib = load()
    need = int(lib.tms_pq_workspace_bytes(Q, Nq, M, K, B))
    if workspace is None and need:
        workspace = torch.empty(need, dtype=torch.uint8, device=lut.device)
    ws_ptr = _dev(workspace, "workspace") if workspace is not None else None
    ws_len = workspace.numel() * workspace.element_size() if workspace is not None else 0
    st = lib.tms_pq_maxsim_variant(_dev(lut, "lut"), Q, Nq, M, K, _dev(codes, "codes") if T else None,
                                   _dev(offsets, "offsets"), B, T, _dev(scores, "scores") if B else None, ws_ptr,
                                   ws_len, _stream(stream), VARIANTS[variant])
    _check(st, "tms_pq_maxsim")
    return scores


PQ_PRECISIONS = {"split_bf16": 0, "fp16": 1}


def tms_pq_maxsim_decode(queries: torch.Tensor, codebooks: torch.Tensor, codes: torch.Tensor, offsets: torch.Tensor,
                         scores: torch.Tensor | None = None, workspace: torch.Tensor | None = None,
                         stream=None, precision: str = "split_bf16") -> torch.Tensor:
    """Same value as tms_pq_build_lut + tms_pq_maxsim, decoded tile by tile in shared memory and contracted on the
    tensor cores (include/tms.h: tms_pq_maxsim_decode)."""
    Q, Nq, d = queries.shape
    M, K, dsub = codebooks.shape
    T, B = codes.shape[0], offsets.numel() - 1
    if codes.dtype != torch.uint8 or codes.dim() != 2 or codes.shape[1] != M or codebooks.dtype != torch.float32:
        raise ValueError("codes must be uint8 [T,M] and codebooks fp32 [M,K,d/M]")
    if scores is None:
        scores = torch.empty((Q, B), dtype=torch.float32, device=queries.device)
    lib = load()
    need = int(lib.tms_maxsim_workspace_bytes(Q, Nq, d, B, _DTYPES[queries.dtype]))
    if workspace is None and need:
        workspace = torch.empty(need, dtype=torch.uint8, device=queries.device)
    ws_ptr = _dev(workspace, "workspace") if workspace is not None else None
    ws_len = workspace.numel() * workspace.element_size() if workspace is not None else 0
    st = lib.tms_pq_maxsim_decode_variant(_dev(queries, "queries"), Q, Nq, d, _DTYPES[queries.dtype],
                                          _dev(codebooks, "codebooks"), M, K, _dev(codes, "codes") if T else None,
                                          _dev(offsets, "offsets"), B, T, _dev(scores, "scores") if B else None, ws_ptr,
                                          ws_len, _stream(stream), PQ_PRECISIONS[precision])
    _check(st, "tms_pq_maxsim_decode")
    return scores


def tms_topk(scores: torch.Tensor, k: int, values: torch.Tensor | None = None, indices: torch.Tensor | None = None,
             workspace: torch.Tensor | None = None, stream=None):
    """(values[Q,k], indices[Q,k]): per query the k best documents, score descending, ties by lower index first."""
    Q, B = scores.shape
    if scores.dtype != torch.float32:
        raise ValueError("scores must be fp32 [Q,B]")
    if values is None:
        values = torch.empty((Q, k), dtype=torch.float32, device=scores.device)
    if indices is None:
        indices = torch.empty((Q, k), dtype=torch.int64, device=scores.device)
    lib = load()
    need = int(lib.tms_topk_workspace_bytes(Q, B, k))
    if workspace is None and need:
        workspace = torch.empty(need, dtype=torch.uint8, device=scores.device)
    ws_ptr = _dev(workspace, "workspace") if workspace is not None else None
    ws_len = workspace.numel() * workspace.element_size() if workspace is not None else 0
    st = lib.tms_topk(_dev(scores, "scores"), Q, B, k, _dev(values, "values"), _dev(indices, "indices"), ws_ptr, ws_len,
                      _stream(stream))
    _check(st, "tms_topk")
    return values, indices


def tms_topk_static_scratch_bytes() -> int:
    """Size of the library's built-in top-k scratch array (TMS_TOPK_STATIC_SCRATCH_BYTES)."""
    return int(load().tms_topk_static_scratch_bytes())


def tms_topk_static(scores: torch.Tensor, k: int, values: torch.Tensor | None = None,
                    indices: torch.Tensor | None = None, stream=None):
    """tms_topk for callers that cannot allocate device memory (include/tms.h: tms_topk_static): same result, bit for
    bit, but the scratch is a fixed 4 MiB array inside the library instead of a workspace, and the library allocates
    nothing.  Pass `values` (fp32 [Q,k]) and `indices` (int64 [Q,k]) to keep this wrapper from allocating them too.
    Shapes whose scratch exceeds the array raise (status 6) -- use tms_topk with a workspace for those.  All calls on
    one GPU share the array: keep them on one stream, and make the first call on a device outside stream capture."""
    Q, B = scores.shape
    if scores.dtype != torch.float32:
        raise ValueError("scores must be fp32 [Q,B]")
    if values is None:
        values = torch.empty((Q, k), dtype=torch.float32, device=scores.device)
    if indices is None:
        indices = torch.empty((Q, k), dtype=torch.int64, device=scores.device)
    if values.shape != (Q, k) or values.dtype != torch.float32 or indices.shape != (Q, k) or indices.dtype != torch.int64:
        raise ValueError("values must be fp32 [Q,k] and indices int64 [Q,k]")
    st = load().tms_topk_static(_dev(scores, "scores"), Q, B, k, _dev(values, "values"), _dev(indices, "indices"),
                                _stream(stream))
    _check(st, "tms_topk_static")
    return values, indices


def _host(t: torch.Tensor, name: str) -> int:
    if t.is_cuda or not t.is_contiguous():
        raise ValueError(f"{name} must be a contiguous host tensor")
    return t.data_ptr()


def tms_maxsim_host_workspace_min_bytes(Q, Nq, d, dtype, max_doc_tokens) -> int:
    return int(load().tms_maxsim_host_workspace_min_bytes(Q, Nq, d, _DTYPES[dtype], max_doc_tokens))


def tms_pq_maxsim_host_workspace_min_bytes(Q, Nq, d, q_dtype, M, K, max_doc_tokens) -> int:
    return int(load().tms_pq_maxsim_host_workspace_min_bytes(Q, Nq, d, _DTYPES[q_dtype], M, K, max_doc_tokens))


def tms_maxsim_host(queries: torch.Tensor, docs: torch.Tensor, offsets: torch.Tensor, scores: torch.Tensor,
                    dev_workspace: torch.Tensor, stream=None) -> torch.Tensor:
    """Same result with HOST tensors (pinned recommended); the store is streamed through dev_workspace."""
    Q, Nq, d = queries.shape
    T, B = docs.shape[0], offsets.numel() - 1
    st = load().tms_maxsim_host(_host(queries, "queries"), Q, Nq, d, _host(docs, "docs"), _host(offsets, "offsets"),
                                B, T, _DTYPES[queries.dtype], _host(scores, "scores"),
                                _dev(dev_workspace, "dev_workspace"),
                                dev_workspace.numel() * dev_workspace.element_size(), _stream(stream))
    _check(st, "tms_maxsim_host")
    return scores


def tms_pq_maxsim_host(queries: torch.Tensor, codebooks: torch.Tensor, codes: torch.Tensor, offsets: torch.Tensor,
                       scores: torch.Tensor, dev_workspace: torch.Tensor, stream=None) -> torch.Tensor:
    Q, Nq, d = queries.shape
    M, K, _ = codebooks.shape
    T, B = codes.shape[0], offsets.numel() - 1
    st = load().tms_pq_maxsim_host(_host(queries, "queries"), Q, Nq, d, _DTYPES[queries.dtype],
                                   _host(codebooks, "codebooks"), M, K, _host(codes, "codes"),
                                   _host(offsets, "offsets"), B, T, _host(scores, "scores"),
                                   _dev(dev_workspace, "dev_workspace"),
                                   dev_workspace.numel() * dev_workspace.element_size(), _stream(stream))
    _check(st, "tms_pq_maxsim_host")
    return scores


def tms_pq_maxsim_decode_host_workspace_min_bytes(Q, Nq, d, q_dtype, M, K, max_doc_tokens) -> int:
    return int(load().tms_pq_maxsim_decode_host_workspace_min_bytes(Q, Nq, d, _DTYPES[q_dtype], M, K, max_doc_tokens))


def tms_pq_maxsim_decode_host(queries: torch.Tensor, codebooks: torch.Tensor, codes: torch.Tensor,
                              offsets: torch.Tensor, scores: torch.Tensor, dev_workspace: torch.Tensor,
                              stream=None) -> torch.Tensor:
    Q, Nq, d = queries.shape
    M, K, _ = codebooks.shape
    T, B = codes.shape[0], offsets.numel() - 1
    st = load().tms_pq_maxsim_decode_host(_host(queries, "queries"), Q, Nq, d, _DTYPES[queries.dtype],
                                          _host(codebooks, "codebooks"), M, K, _host(codes, "codes"),
                                          _host(offsets, "offsets"), B, T, _host(scores, "scores"),
                                          _dev(dev_workspace, "dev_workspace"),
                                          dev_workspace.numel() * dev_workspace.element_size(), _stream(stream))
    _check(st, "tms_pq_maxsim_decode_host")
    return scores


def tms_topk_merge(values: torch.Tensor, indices: torch.Tensor, shard_base, k: int, stream=None):
    """k best of G per-shard top-k lists: values / indices [G,Q,k_in] (shard-local indices), shard_base[g] = first
    global document of shard g.  Returns (values[Q,k], indices[Q,k]) with GLOBAL document indices."""
    G, Q, k_in = values.shape
    if values.dtype != torch.float32 or indices.dtype != torch.int64 or indices.shape != values.shape:
        raise ValueError("values fp32 [G,Q,k_in] and indices int64 [G,Q,k_in] expected")
    base = (ctypes.c_int64 * G)(*[int(b) for b in shard_base])
    out_v = torch.empty((Q, k), dtype=torch.float32, device=values.device)
    out_i = torch.empty((Q, k), dtype=torch.int64, device=values.device)
    lib = load()
    need = int(lib.tms_topk_merge_workspace_bytes(G, Q, k_in, k))
    ws = torch.empty(max(need, 8), dtype=torch.uint8, device=values.device)
    st = lib.tms_topk_merge(_dev(values, "values"), _dev(indices, "indices"), ctypes.addressof(base), G, Q, k_in, k,
                            _dev(out_v, "out_values"), _dev(out_i, "out_indices"), _dev(ws, "workspace"), ws.numel(),
                            _stream(stream))
    _check(st, "tms_topk_merge")
    return out_v, out_i
