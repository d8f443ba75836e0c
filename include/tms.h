/*
 * tms.h -- C ABI of the B200-native MaxSim scoring library (libtms.so).
 *
 * Implements the data-parallel hot path of "TileMaxSim" (arXiv 2606.26439; the paper text is cited
 * below as P:L<line> of PAPER.md):
 *   - tms_maxsim        : fused multi-query MaxSim over a packed token-major document store,
 *                         including the dimension-tiled form for d > 128 (Eq. 1;
 *                         P:L182-204 Alg. 3).
 *   - tms_pq_build_lut  : product-quantisation distance table, Eq. 8.
 *   - tms_pq_maxsim     : fused lookup + max + sum over uint8 PQ codes, Eq. 9.
 *   - tms_pq_maxsim_decode : the same PQ scores from codes + codebooks, decoded in shared memory and
 *                         contracted on the tensor cores (no lookup table).
 *   - tms_topk          : per-query top-k over the scores, the step that follows scoring.
 *   - tms_maxsim_host / tms_pq_maxsim_host : the same scoring from HOST buffers, the document store
 *                         streamed through a caller-provided device workspace.
 *
 * Conventions, unless a function says otherwise:
 *   - "device" pointers are CUDA device memory on the current device, owned by the caller.  The
 *     library never allocates or frees device memory; scratch comes through `workspace`.
 *   - Calls enqueue work on `stream` (a cudaStream_t passed as void*; NULL = the legacy default
 *     stream) and return without synchronising the host.
 *   - The return value is a tms_status describing host-side argument / launch errors.  There are no
 *     exceptions, no errno, no logging.  Data errors the host cannot see without a sync (for
 *     instance non-monotone `offsets`) are undefined behaviour.
 *   - `scores` is fully overwritten for all Q*B entries; it is never accumulated into and needs no
 *     initialisation.
 *   - Inputs must be finite.  An empty document (offsets[b+1] == offsets[b]) scores -INFINITY, the
 *     literal outcome of "m <- -inf" in Alg. 3 line 4.
 *   - Similarity is the raw dot product of Eq. 1; normalisation is the caller's business.
 *   - There is no CPU fallback: on a machine without a usable sm_100 device the compute entry points
 *     return TMS_ERR_UNSUPPORTED or TMS_ERR_CUDA.
 */
#ifndef TMS_H_
#define TMS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TMS_OK = 0,
    TMS_ERR_INVALID_ARG = 1, /* NULL pointer, non-positive size, inconsistent sizes            */
    TMS_ERR_UNSUPPORTED = 2, /* shape / dtype / device outside what this build implements      */
    TMS_ERR_ALIGNMENT = 3,   /* a pointer or row pitch is not 16-byte aligned                  */
    TMS_ERR_WORKSPACE = 4,   /* workspace is NULL or smaller than the *_workspace_bytes() size  */
    TMS_ERR_CUDA = 5,        /* a CUDA runtime / driver call failed (launch, copy, attribute)  */
    TMS_ERR_STATIC_SCRATCH = 6 /* tms_topk_static: the shape needs more scratch than the built-in buffer holds */
} tms_status;

/* Storage dtype of query and document embeddings.  Arithmetic: products of the stored values,
 * accumulated in fp32 ("FP16 embeddings with FP32 accumulation"). */
typedef enum { TMS_DTYPE_F32 = 0, TMS_DTYPE_F16 = 1, TMS_DTYPE_BF16 = 2 } tms_dtype;

/* Kernel selection for tms_maxsim_variant / tms_pq_maxsim_variant (tests, benches, ablations). */
typedef enum {
    TMS_VARIANT_AUTO = 0,     /* what tms_maxsim / tms_pq_maxsim pick                                  */
    TMS_VARIANT_SIMT = 1,     /* CUDA-core tiled kernel: any dtype, any d, any Nq (the general path)   */
    TMS_VARIANT_TCGEN05 = 2,  /* TMA + tcgen05 tensor-core kernel (sm_100a), dimension-tiled for d>128 */
    TMS_VARIANT_PQ_SMEM = 3,  /* PQ: LUT slices resident in shared memory, fp32 entries (AUTO's choice)    */
    TMS_VARIANT_PQ_SMEM_F16 = 4 /* PQ, opt-in only: the same with table entries held as (block-scaled) fp16 in
                                 shared memory: half the gather bytes, lossy; see tms_pq_maxsim          */
} tms_variant;

/*
 * Dense MaxSim (Eq. 1):
 *     scores[q*B + b] = sum_{i<Nq}  max_{t in [offsets[b], offsets[b+1])}  <queries[q,i,:], docs[t,:]>
 *
 * queries       device, [Q, Nq, d] row-major, `dtype`, 16-byte aligned.
 * docs          device, packed token-major store [total_tokens, d] row-major, `dtype`, 16-byte
 *               aligned base; the row pitch d*sizeof(dtype) must be a multiple of 16 bytes.
 * offsets       device, int64 [B+1]; offsets[0] = 0, non-decreasing, offsets[B] = total_tokens.
 * total_tokens  = offsets[B]; passed by value so the host never reads device memory.
 * scores        device, fp32 [Q, B] row-major, overwritten.
 * workspace     device scratch of at least tms_maxsim_workspace_bytes(...) bytes, 16-byte aligned; may be
 *               NULL when that size is 0 (it is 0 for Nq <= 32).  Longer queries are scored as n equal parts
 *               of Nq/n <= 32 tokens (n = Nq/32 for multiples of 32) whose partial scores (fp32 [Q*n, B])
 *               live in the workspace and are added by a second kernel.  A workspace that is missing or too
 *               small for such a shape is TMS_ERR_WORKSPACE, a mis-aligned one TMS_ERR_ALIGNMENT -- the call
 *               never switches to a slower kernel because of its scratch.
 * Every document embedding is read from HBM once per group of up to 256 query rows (Q*Nq, Nq rounded up to a power of
 * two): for d*sizeof(dtype) <= 512 bytes both 128-row blocks sit in one SM's tensor memory next to their accumulators;
 * for 16-bit d in (256, 768] only one block fits, and 256 rows run as clusters of two CTAs -- one block each -- that
 * share every document tile by TMA multicast, so the store still crosses the HBM interface once.  fp32 inputs with
 * d > 128 keep one block per launch (128 rows).  A call with more rows runs ceil(rows / group) launches, each
 * streaming the store once -- the ceil(Nq/BQ) factor of Thm 1.  No similarity matrix is written to memory
 * (Eq. 7).
 * d > 128 accumulates partial dot products over dimension chunks before the max is taken.
 * Stores of 2^31 - 128 tokens or more (TMA tile coordinates are 32-bit) are scored in segments of 2^30 tokens, one
 * launch per segment; a single document must then be no longer than 2^30 - 128 tokens (it may start on a segment's
 * last token and must end inside the next segment's tensor map; a longer one is scored wrongly, without an error --
 * lengths live in device memory).  The same holds for tms_pq_maxsim_decode.
 */
int tms_maxsim(const void* queries, int Q, int Nq, int d, const void* docs, const int64_t* offsets, int64_t B,
               int64_t total_tokens, tms_dtype dtype, float* scores, void* workspace, size_t workspace_bytes,
               void* stream);

/* Same as tms_maxsim with an explicit kernel choice.  A variant that cannot run the given shape
 * returns TMS_ERR_UNSUPPORTED instead of silently switching. */
int tms_maxsim_variant(const void* queries, int Q, int Nq, int d, const void* docs, const int64_t* offsets,
                       int64_t B, int64_t total_tokens, tms_dtype dtype, float* scores, void* workspace,
                       size_t workspace_bytes, void* stream, tms_variant variant);

size_t tms_maxsim_workspace_bytes(int Q, int Nq, int d, int64_t B, tms_dtype dtype);

/* Which kernel tms_maxsim (TMS_VARIANT_AUTO) runs for this shape on an sm_100 device, given an adequate workspace:
 * TMS_VARIANT_TCGEN05 or TMS_VARIANT_SIMT (the general CUDA-core kernel, far below the HBM roofline: d*sizeof(dtype)
 * beyond tensor-memory residency, fp32 with d % 64 != 0).  TMS_VARIANT_AUTO when nothing
 * is scored (B == 0 or total_tokens == 0).  A pure function of its arguments: no device is touched. */
int tms_maxsim_variant_used(int Q, int Nq, int d, int64_t B, int64_t total_tokens, tms_dtype dtype);

/*
 * PQ distance table (Eq. 8):
 *     lut[q,i,m,k] = sum_{s<d/M} queries[q,i,m*(d/M)+s] * codebooks[m,k,s]      (fp32 FMA, s ascending)
 * queries    device, [Q, Nq, d], `q_dtype`.      codebooks  device, fp32 [M, K, d/M].
 * lut        device, fp32 [Q, Nq, M, K], overwritten.     Requires d % M == 0 and 1 <= K <= 256.
 */
int tms_pq_build_lut(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks, int M,
                     int K, float* lut, void* stream);

/*
 * Fused PQ scoring (Eq. 9; phase 2 of P:L270):
 *     scores[q*B + b] = sum_{i<Nq}  max_{t in doc b}  sum_{m<M} lut[q,i,m,codes[t,m]]
 * lut      device, fp32 [Q, Nq, M, K] as written by tms_pq_build_lut.
 * codes    device, uint8 [total_tokens, M] row-major, 16-byte aligned base; values < K.
 * The decompressed vectors are never materialised.  The sum over m is fp32 in a fixed, kernel-defined
 * order (run-to-run reproducible).
 * workspace  device scratch of at least tms_pq_workspace_bytes(...) bytes (the re-laid-out table).
 * Precision contract: tms_pq_maxsim (TMS_VARIANT_AUTO) adds the fp32 table entries as they are (the paper's table is
 * fp32) -- the only rounding is the fp32 sum over m and, before it, the fp32 FMA chain of tms_pq_build_lut.
 * Whatever the queries' dtype was, the scores are within 1e-5 * Nq * max|dhat| of Eq. 9 evaluated on the stored query
 * values (so within the 1e-5*Nq bound of fp32 inputs and, a fortiori, the 2e-3*Nq bound of 16-bit ones).  The call
 * cannot know what `lut` was built from and therefore never narrows it on its own.
 * Kernels: for M = 16, K = 256, Nq % 8 == 0 the table is re-laid-out into the workspace and served from shared memory
 * in 8-row slices (P:L268 keeps it in L2; here the gathers are the bound): TMS_VARIANT_PQ_SMEM, what AUTO picks for
 * that shape; any other shape (any M, K <= 256, Nq) runs the general kernel, TMS_VARIANT_SIMT, with the table read
 * through L1/L2.
 * OPT-IN, through tms_pq_maxsim_variant only: TMS_VARIANT_PQ_SMEM_F16 (Nq % 16 == 0) holds the re-laid-out copy as fp16
 * after one power-of-two scale of the whole table (max|entry| -> [2^14, 2^15): no overflow or subnormals for any
 * finite table); entries are widened back inside the fp32 additions and the scale is undone exactly.  Half the gather
 * bytes (1.9x faster on config 5) for one rounding of relative 2^-11 per entry: |dscore| <= Nq * M * max|entry| * 2^-12
 * in the worst case, ~2e-3 measured on config 5's data -- inside the 2e-3*Nq tolerance of 16-bit
 * queries, NOT inside the 1e-5*Nq one of fp32 queries, and near-ties in a ranking can swap.  Choose it only for tables
 * built from 16-bit queries.  `lut` itself is never modified.
 */
int tms_pq_maxsim(const float* lut, int Q, int Nq, int M, int K, const uint8_t* codes, const int64_t* offsets,
                  int64_t B, int64_t total_tokens, float* scores, void* workspace, size_t workspace_bytes,
                  void* stream);

int tms_pq_maxsim_variant(const float* lut, int Q, int Nq, int M, int K, const uint8_t* codes,
                          const int64_t* offsets, int64_t B, int64_t total_tokens, float* scores, void* workspace,
                          size_t workspace_bytes, void* stream, tms_variant variant);

size_t tms_pq_workspace_bytes(int Q, int Nq, int M, int K, int64_t B);

/* Which kernel tms_pq_maxsim (TMS_VARIANT_AUTO) runs for this shape: TMS_VARIANT_PQ_SMEM (fp32 entries in shared
 * memory) or TMS_VARIANT_SIMT (the general kernel); never TMS_VARIANT_PQ_SMEM_F16.  TMS_VARIANT_AUTO for non-positive
 * sizes.  A pure function of its arguments: no device is touched. */
int tms_pq_maxsim_variant_used(int Q, int Nq, int M, int K);

/*
 * Decode-and-contract PQ scoring: the same value as tms_pq_build_lut + tms_pq_maxsim,
 *     scores[q*B + b] = sum_{i<Nq}  max_{t in doc b}  <queries[q,i,:], dhat_t>,   dhat_t = concat_m codebooks[m, codes[t,m], :]
 * (Eq. 9), computed without a lookup table: every tile of 128 tokens is decompressed inside
 * shared memory from the resident codebook and contracted on the tensor cores; the decompressed vectors never reach
 * HBM.  Arithmetic: queries and centroids are split into bf16 hi + lo parts (hi*hi + hi*lo + lo*hi, fp32
 * accumulate), i.e. about 16 mantissa bits per factor -- the result agrees with tms_pq_maxsim to ~1e-5.
 * Supported: d = 128, M = 16, K = 256 (8-dimensional sub-vectors); any Q; Nq <= 32 or a multiple of 32 (then
 * `workspace` as for tms_maxsim: tms_maxsim_workspace_bytes(Q, Nq, d, B, q_dtype)); otherwise TMS_ERR_UNSUPPORTED.
 * queries device [Q, Nq, d] `q_dtype`;  codebooks device fp32 [M, K, d/M];  codes device uint8 [total_tokens, M].
 */
int tms_pq_maxsim_decode(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks, int M,
                         int K, const uint8_t* codes, const int64_t* offsets, int64_t B, int64_t total_tokens,
                         float* scores, void* workspace, size_t workspace_bytes, void* stream);

/* Operand precision of tms_pq_maxsim_decode_variant. */
typedef enum {
    TMS_PQ_SPLIT_BF16 = 0, /* the default: bf16 hi + lo parts, two MMAs per product, ~1e-5 from the fp32 table form  */
    TMS_PQ_FP16 = 1        /* queries and centroids rounded to fp16 (11-bit mantissa), ONE MMA per product: half the
                              tensor work; per-element rounding 2^-12 relative, measured |dscore| <= 1e-3*Nq on config
                              5's data (inside the 2e-3*Nq tolerance of 16-bit inputs); inputs must fit fp16's range  */
} tms_pq_precision;

/* tms_pq_maxsim_decode with an explicit operand precision (tms_pq_maxsim_decode = TMS_PQ_SPLIT_BF16). */
int tms_pq_maxsim_decode_variant(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks,
                                 int M, int K, const uint8_t* codes, const int64_t* offsets, int64_t B,
                                 int64_t total_tokens, float* scores, void* workspace, size_t workspace_bytes,
                                 void* stream, tms_pq_precision precision);

/*
 * Host-buffer entry points: identical results, but `queries`, `docs` / `codes`, `offsets`, `codebooks` and
 * `scores` are HOST pointers (pinned memory makes the copies asynchronous and fast).  The document store
 * is streamed through `dev_workspace` in document-aligned chunks; the host->device copy of chunk n+1 runs
 * on an internal copy stream while chunk n is scored on `stream`; each chunk's scores return with one
 * strided device->host copy.  Unlike the device entry points these calls validate `offsets` (host memory)
 * and return only after the scores have landed in `scores` (they synchronise `stream`).
 *
 * dev_workspace   device memory, at least *_host_workspace_min_bytes(..., max_doc_tokens) bytes where
 *                 max_doc_tokens is the longest document; a larger workspace means fewer, larger chunks.  The
 *                 scratch of queries longer than 32 tokens is carved out of it (per chunk), so every shape runs the
 *                 same kernel as through the device entry point.
 *                 TMS_ERR_WORKSPACE if a single document does not fit in half of what remains after the
 *                 query (and, for PQ, table) staging area.
 * tms_pq_maxsim_host builds the distance table on the device from host `queries` and `codebooks` first.
 */
int tms_maxsim_host(const void* queries, int Q, int Nq, int d, const void* docs, const int64_t* offsets, int64_t B,
                    int64_t total_tokens, tms_dtype dtype, float* scores, void* dev_workspace,
                    size_t dev_workspace_bytes, void* stream);

int tms_pq_maxsim_host(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks, int M,
                       int K, const uint8_t* codes, const int64_t* offsets, int64_t B, int64_t total_tokens,
                       float* scores, void* dev_workspace, size_t dev_workspace_bytes, void* stream);

/* tms_pq_maxsim_decode from host buffers (same shapes as tms_pq_maxsim_decode; no table is built). */
int tms_pq_maxsim_decode_host(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks,
                              int M, int K, const uint8_t* codes, const int64_t* offsets, int64_t B,
                              int64_t total_tokens, float* scores, void* dev_workspace, size_t dev_workspace_bytes,
                              void* stream);

size_t tms_maxsim_host_workspace_min_bytes(int Q, int Nq, int d, tms_dtype dtype, int64_t max_doc_tokens);
size_t tms_pq_maxsim_host_workspace_min_bytes(int Q, int Nq, int d, tms_dtype q_dtype, int M, int K,
                                              int64_t max_doc_tokens);
size_t tms_pq_maxsim_decode_host_workspace_min_bytes(int Q, int Nq, int d, tms_dtype q_dtype, int M, int K,
                                                     int64_t max_doc_tokens);

/*
 * Per-query top-k over a score matrix -- the step right after scoring ("followed by torch.topk"):
 *     for every q: (values[q, r], indices[q, r]), r < k = the k best documents of scores[q, 0..B), ordered by score
 *     descending, ties by lower document index first; -INFINITY (empty documents) ranks last.
 * scores   device, fp32 [Q, B] row-major (as written by tms_maxsim / tms_pq_maxsim); not modified; no NaN.
 * values   device, fp32 [Q, k];   indices  device, int64 [Q, k];   1 <= k <= min(B, 1024);  B <= 2^31.
 * workspace  device scratch of at least tms_topk_workspace_bytes(Q, B, k) bytes, 8-byte aligned (0 for B <= 4096).
 * Values are copies of the scores (a score of -0.0 ties with and is reported as +0.0); the result is unique and
 * bit-reproducible.
 */
int tms_topk(const float* scores, int Q, int64_t B, int k, float* values, int64_t* indices, void* workspace,
             size_t workspace_bytes, void* stream);

size_t tms_topk_workspace_bytes(int Q, int64_t B, int k);

/*
 * tms_topk without a workspace argument and without any allocation -- the one entry point of this library for callers
 * that have no device memory to give and no way to get some:
 *   - a process whose HBM was handed, whole, to another component's pool at start-up (an inference server's KV-cache
 *     arena, a framework's caching allocator run at its memory limit), so cudaMalloc would return out-of-memory;
 *   - a plug-in or callback that runs where the host forbids calls that synchronise the device or take the driver's
 *     allocation lock (cudaMalloc and cudaFree do both), e.g. a scoring hook inside a latency-bound serving loop;
 *   - a plain C caller with no allocator of its own that wants one call and no buffer whose lifetime it must manage.
 * Everything else in the library takes its scratch through `workspace`; this call takes none.  The selection levels'
 * two key buffers live instead in a fixed array inside the library's device image:
 *
 *     TMS_TOPK_STATIC_SCRATCH_BYTES = 4 MiB, held by EVERY GPU that loads libtms.so from load until process exit,
 *     whether or not this function is ever called.
 *
 * Result, order, tie rule and argument meaning are exactly tms_topk's (same kernels, same launch sequence: the outputs
 * are bit-identical).  The caller still owns and passes `scores`, `values` and `indices`.
 * Limit: shapes with tms_topk_workspace_bytes(Q, B, k) > TMS_TOPK_STATIC_SCRATCH_BYTES are rejected with
 * TMS_ERR_STATIC_SCRATCH before anything is launched (the need is 16 * Q * ceil(B/4096) * k bytes for B > 4096, else
 * 0: Q=8, k=100 fits up to B = 1.3M documents; Q=1, k=1024 up to B = 1.0M; Q=8, k=1024 up to B = 131K).  Such shapes
 * need tms_topk with a caller-provided workspace; nothing falls back silently.
 * First call on each device: the library asks the CUDA runtime for the array's address on the current device (once
 * per device, cached; the device current at the time of the call is the one used).  That look-up can make the runtime
 * load the library's device code onto that GPU, so make the first call on a device during start-up, outside any stream
 * capture.  Later calls do no set-up.
 * Sharing: there is ONE array per GPU and every call on that GPU uses it.  It keeps whatever the last call left there;
 * no call depends on its contents (every key a level reads was written by the level before it, in the same call), so
 * nothing needs clearing between calls.  Two calls whose kernels can overlap on the GPU -- different streams without
 * an event between them, or two host threads -- race on the array and both results are garbage: keep all
 * tms_topk_static calls of a device on one stream or order them with events.
 * Makes no CUDA allocation and calls no allocating library routine.  Errors: as tms_topk, plus TMS_ERR_STATIC_SCRATCH;
 * TMS_ERR_CUDA if the address look-up fails.
 */
#define TMS_TOPK_STATIC_SCRATCH_BYTES (4u << 20)
int tms_topk_static(const float* scores, int Q, int64_t B, int k, float* values, int64_t* indices, void* stream);

/* = TMS_TOPK_STATIC_SCRATCH_BYTES of the loaded library (for callers that cannot see this header). */
size_t tms_topk_static_scratch_bytes(void);

/*
 * k-way merge of per-shard top-k lists -- the step after data-parallel scoring ("only a final concatenation of
 * per-shard scores"; with per-shard tms_topk only G*k candidates per query cross GPUs instead of B scores):
 *     (out_values[q, :], out_indices[q, :]) = the k best of the G*k_in candidates
 *         (values[g, q, r], shard_base[g] + indices[g, q, r]),  same order as tms_topk (score descending, lower GLOBAL
 *         document index first, -INFINITY last).  With k_in >= k this equals tms_topk over the concatenated scores.
 * values / indices   device, fp32 / int64 [G, Q, k_in] (shard-local document indices, as tms_topk wrote them).
 * shard_base         HOST, int64 [G]: first global document index of every shard; 0 <= base < 2^31 (else
 *                    TMS_ERR_INVALID_ARG).  base + index < 2^31 for every candidate is the caller's contract: the
 *                    indices live in device memory, the host cannot check them, and a larger sum wraps silently.
 * G <= 64; k, k_in <= 1024; k <= G*k_in.  workspace: device, >= tms_topk_merge_workspace_bytes(...), 8-byte aligned.
 */
int tms_topk_merge(const float* values, const int64_t* indices, const int64_t* shard_base, int G, int Q, int k_in, int k,
                   float* out_values, int64_t* out_indices, void* workspace, size_t workspace_bytes, void* stream);

size_t tms_topk_merge_workspace_bytes(int G, int Q, int k_in, int k);

/* Number of kernels this library has launched in this process since load (all entry points). */
uint64_t tms_launch_count(void);

const char* tms_status_string(int status);
int tms_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TMS_H_ */
