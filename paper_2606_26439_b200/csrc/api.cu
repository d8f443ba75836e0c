// api.cu -- the C ABI of libtms.so (include/tms.h): argument validation and kernel dispatch only.
#include <atomic>
#include <mutex>

#include "tms_internal.h"

namespace tms {

static std::atomic<uint64_t> g_launches{0};
void count_launch(int n) { g_launches.fetch_add((uint64_t)n, std::memory_order_relaxed); }

const DeviceInfo* device_info() {
    static std::mutex mu;
    static DeviceInfo cache[64];
    static bool have[64] = {};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) {
        cudaGetLastError();
        return nullptr;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (!have[dev]) {
        DeviceInfo di;
        di.device = dev;
        if (cudaDeviceGetAttribute(&di.cc_major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&di.cc_minor, cudaDevAttrComputeCapabilityMinor, dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&di.num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&di.max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) {
            cudaGetLastError();
            return nullptr;
        }
        cache[dev] = di;
        have[dev] = true;
    }
    return &cache[dev];
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

__global__ void fill_neg_inf_kernel(float* __restrict__ x, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) x[i] = -INFINITY;
}
// every document is empty: all scores are -inf (Alg. 3 line 4 summed Nq times; reading A2)
static int fill_empty(float* scores, int64_t n, cudaStream_t stream) {
    fill_neg_inf_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(scores, n);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? TMS_OK : TMS_ERR_CUDA;
}

static int check_dense(const void* queries, int Q, int Nq, int d, const void* docs, const int64_t* offsets, int64_t B,
                       int64_t T, tms_dtype dtype, float* scores) {
    if (Q <= 0 || Nq <= 0 || d <= 0 || B < 0 || T < 0) return TMS_ERR_INVALID_ARG;
    if (dtype != TMS_DTYPE_F32 && dtype != TMS_DTYPE_F16 && dtype != TMS_DTYPE_BF16) return TMS_ERR_INVALID_ARG;
    if (!queries || !offsets || (B > 0 && !scores) || (T > 0 && !docs)) return TMS_ERR_INVALID_ARG;
    if ((int64_t)Q * Nq > (1 << 20) || (int64_t)Q * B < 0) return TMS_ERR_UNSUPPORTED;
    if (((size_t)d * dtype_size(dtype)) % 16 != 0) return TMS_ERR_UNSUPPORTED;  // row pitch (a1)
    if (!aligned16(queries) || !aligned16(docs) || (reinterpret_cast<uintptr_t>(offsets) & 7u) ||
        (reinterpret_cast<uintptr_t>(scores) & 3u))
        return TMS_ERR_ALIGNMENT;
    return TMS_OK;
}

static int dense_dispatch(const void* queries, int Q, int Nq, int d, const void* docs, const int64_t* offsets,
                          int64_t B, int64_t T, tms_dtype dtype, float* scores, void* workspace,
                          size_t workspace_bytes, void* stream, tms_variant variant) {
    int st = check_dense(queries, Q, Nq, d, docs, offsets, B, T, dtype, scores);
    if (st != TMS_OK) return st;
    if (variant != TMS_VARIANT_AUTO && variant != TMS_VARIANT_SIMT && variant != TMS_VARIANT_TCGEN05)
        return TMS_ERR_INVALID_ARG;
    if (!device_info()) return TMS_ERR_CUDA;
    if (B == 0) return TMS_OK;
    if (T == 0) return fill_empty(scores, (int64_t)Q * B, static_cast<cudaStream_t>(stream));  // every document empty (A2)
    // The long-query scratch is never optional: a missing, short or mis-aligned workspace is an error, not a reason
    // to run a slower kernel behind the caller's back.
    const size_t need = dense_tc_workspace_bytes(Q, Nq, B);
    DenseArgs a{queries, Q, Nq, d, docs, offsets, B, T, dtype, scores, static_cast<cudaStream_t>(stream), workspace,
                workspace_bytes};
    if (variant != TMS_VARIANT_SIMT && need != 0) {
        a.workspace = reinterpret_cast<void*>(static_cast<uintptr_t>(16));  // "present" for the shape test below
        a.workspace_bytes = need;
        const bool tc = dense_tc_supports(a);
        a.workspace = workspace;
        a.workspace_bytes = workspace_bytes;
        if (tc) {
            if (!workspace || workspace_bytes < need) return TMS_ERR_WORKSPACE;
            if (!aligned16(workspace)) return TMS_ERR_ALIGNMENT;
        }
    }
    switch (variant) {
        case TMS_VARIANT_AUTO: return dense_tc_supports(a) ? launch_dense_tc(a) : launch_dense_simt(a);
        case TMS_VARIANT_SIMT: return launch_dense_simt(a);
        default: return dense_tc_supports(a) ? launch_dense_tc(a) : TMS_ERR_UNSUPPORTED;
    }
}

static int check_pq(const float* lut, int Q, int Nq, int M, int K, const uint8_t* codes, const int64_t* offsets,
                    int64_t B, int64_t T, float* scores) {
    if (Q <= 0 || Nq <= 0 || M <= 0 || K <= 0 || B < 0 || T < 0) return TMS_ERR_INVALID_ARG;
    if (!lut || !offsets || (B > 0 && !scores) || (T > 0 && !codes)) return TMS_ERR_INVALID_ARG;
    if (K > 256 || M > 256 || (int64_t)Q * Nq > (1 << 20)) return TMS_ERR_UNSUPPORTED;
    if (!aligned16(lut) || !aligned16(codes) || (reinterpret_cast<uintptr_t>(offsets) & 7u) ||
        (reinterpret_cast<uintptr_t>(scores) & 3u))
        return TMS_ERR_ALIGNMENT;
    return TMS_OK;
}

static int pq_dispatch(const float* lut, int Q, int Nq, int M, int K, const uint8_t* codes, const int64_t* offsets,
                       int64_t B, int64_t T, float* scores, void* workspace, size_t workspace_bytes, void* stream,
                       tms_variant variant) {
    int st = check_pq(lut, Q, Nq, M, K, codes, offsets, B, T, scores);
    if (st != TMS_OK) return st;
    if (!device_info()) return TMS_ERR_CUDA;
    if (B == 0) return TMS_OK;
    if (variant != TMS_VARIANT_AUTO && variant != TMS_VARIANT_SIMT && variant != TMS_VARIANT_PQ_SMEM &&
        variant != TMS_VARIANT_PQ_SMEM_F16)
        return TMS_ERR_INVALID_ARG;
    // AUTO never narrows the table: the call sees only `lut`, not what it was built from, and a table built from fp32
    // queries is held to 1e-5*Nq (the paper's table is fp32).  AUTO = the shared-memory kernel over fp32 entries
    // when the shape has whole 8-row slices, else the general kernel.  fp16 entries (half the gather bytes, 1.9x faster
    // on config 5, one 2^-11 rounding per entry: DESIGN.md 5.4) are the caller's explicit choice: TMS_VARIANT_PQ_SMEM_F16.
    PqArgs a{lut, Q, Nq, M, K, codes, offsets, B, T, scores, static_cast<cudaStream_t>(stream)};
    const bool f16 = variant == TMS_VARIANT_PQ_SMEM_F16;
    const bool smem_ok = pq_smem_supports(a, f16);
    if (variant == TMS_VARIANT_SIMT || (variant == TMS_VARIANT_AUTO && !smem_ok)) return launch_pq_simt(a);
    if (!smem_ok) return TMS_ERR_UNSUPPORTED;
    if (!workspace || workspace_bytes < pq_smem_workspace_bytes(Q, Nq) || !aligned16(workspace))
        return TMS_ERR_WORKSPACE;
    return launch_pq_smem(a, workspace, f16);
}

}  // namespace tms

using namespace tms;

extern "C" {

int tms_maxsim(const void* queries, int Q, int Nq, int d, const void* docs, const int64_t* offsets, int64_t B,
               int64_t total_tokens, tms_dtype dtype, float* scores, void* workspace, size_t workspace_bytes,
               void* stream) {
    return dense_dispatch(queries, Q, Nq, d, docs, offsets, B, total_tokens, dtype, scores, workspace, workspace_bytes,
                          stream, TMS_VARIANT_AUTO);
}

int tms_maxsim_variant(const void* queries, int Q, int Nq, int d, const void* docs, const int64_t* offsets,
                       int64_t B, int64_t total_tokens, tms_dtype dtype, float* scores, void* workspace,
                       size_t workspace_bytes, void* stream, tms_variant variant) {
    return dense_dispatch(queries, Q, Nq, d, docs, offsets, B, total_tokens, dtype, scores, workspace, workspace_bytes,
                          stream, variant);
}

int tms_maxsim_variant_used(int Q, int Nq, int d, int64_t B, int64_t total_tokens, tms_dtype dtype) {
    if (Q <= 0 || Nq <= 0 || d <= 0 || B <= 0 || total_tokens <= 0) return TMS_VARIANT_AUTO;  // nothing is scored
    DenseArgs a{reinterpret_cast<const void*>(static_cast<uintptr_t>(16)), Q, Nq, d,
                reinterpret_cast<const void*>(static_cast<uintptr_t>(16)), nullptr, B, total_tokens, dtype, nullptr,
                nullptr, reinterpret_cast<void*>(static_cast<uintptr_t>(16)), dense_tc_workspace_bytes(Q, Nq, B)};
    return dense_tc_shape_ok(a) ? TMS_VARIANT_TCGEN05 : TMS_VARIANT_SIMT;
}

size_t tms_maxsim_workspace_bytes(int Q, int Nq, int d, int64_t B, tms_dtype dtype) {
    (void)d; (void)dtype;
    // Nq <= 32: no scratch, no partial result ever leaves the SM.  Longer queries are scored as 32-token parts whose
    // partial scores are added by a second small kernel.
    if (Q <= 0 || Nq <= 0 || B <= 0) return 0;
    return dense_tc_workspace_bytes(Q, Nq, B);
}

int tms_pq_build_lut(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks, int M,
                     int K, float* lut, void* stream) {
    if (Q <= 0 || Nq <= 0 || d <= 0 || M <= 0 || K <= 0) return TMS_ERR_INVALID_ARG;
    if (!queries || !codebooks || !lut) return TMS_ERR_INVALID_ARG;
    if (q_dtype != TMS_DTYPE_F32 && q_dtype != TMS_DTYPE_F16 && q_dtype != TMS_DTYPE_BF16) return TMS_ERR_INVALID_ARG;
    if (d % M != 0 || K > 256 || M > 65535) return TMS_ERR_UNSUPPORTED;
    if (!device_info()) return TMS_ERR_CUDA;
    return launch_pq_build_lut(queries, Q, Nq, d, q_dtype, codebooks, M, K, lut, static_cast<cudaStream_t>(stream));
}

int tms_pq_maxsim(const float* lut, int Q, int Nq, int M, int K, const uint8_t* codes, const int64_t* offsets,
                  int64_t B, int64_t total_tokens, float* scores, void* workspace, size_t workspace_bytes,
                  void* stream) {
    return pq_dispatch(lut, Q, Nq, M, K, codes, offsets, B, total_tokens, scores, workspace, workspace_bytes, stream,
                       TMS_VARIANT_AUTO);
}

int tms_pq_maxsim_variant(const float* lut, int Q, int Nq, int M, int K, const uint8_t* codes,
                          const int64_t* offsets, int64_t B, int64_t total_tokens, float* scores, void* workspace,
                          size_t workspace_bytes, void* stream, tms_variant variant) {
    return pq_dispatch(lut, Q, Nq, M, K, codes, offsets, B, total_tokens, scores, workspace, workspace_bytes, stream,
                       variant);
}

int tms_pq_maxsim_variant_used(int Q, int Nq, int M, int K) {
    if (Q <= 0 || Nq <= 0 || M <= 0 || K <= 0) return TMS_VARIANT_AUTO;  // nothing is scored
    PqArgs a{nullptr, Q, Nq, M, K, nullptr, nullptr, 0, 0, nullptr, nullptr};
    return pq_smem_supports(a, false) ? TMS_VARIANT_PQ_SMEM : TMS_VARIANT_SIMT;
}

size_t tms_pq_workspace_bytes(int Q, int Nq, int M, int K, int64_t B) {
    (void)B;
    if (Q <= 0 || Nq <= 0 || M != 16 || K != 256 || Nq % 8 != 0) return 0;  // general kernel: no scratch
    return pq_smem_workspace_bytes(Q, Nq);
}

int tms_pq_maxsim_decode_variant(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks,
                                 int M, int K, const uint8_t* codes, const int64_t* offsets, int64_t B,
                                 int64_t total_tokens, float* scores, void* workspace, size_t workspace_bytes,
                                 void* stream, tms_pq_precision precision) {
    if (precision != TMS_PQ_SPLIT_BF16 && precision != TMS_PQ_FP16) return TMS_ERR_INVALID_ARG;
    if (Q <= 0 || Nq <= 0 || d <= 0 || M <= 0 || K <= 0 || B < 0 || total_tokens < 0) return TMS_ERR_INVALID_ARG;
    if (q_dtype != TMS_DTYPE_F32 && q_dtype != TMS_DTYPE_F16 && q_dtype != TMS_DTYPE_BF16) return TMS_ERR_INVALID_ARG;
    if (!queries || !codebooks || !offsets || (B > 0 && !scores) || (total_tokens > 0 && !codes))
        return TMS_ERR_INVALID_ARG;
    if (d != 128 || M != 16 || K != 256) return TMS_ERR_UNSUPPORTED;  // the shape of BASELINE.json configs[4]
    if (!aligned16(queries) || !aligned16(codebooks) || !aligned16(codes) || (reinterpret_cast<uintptr_t>(offsets) & 7u) ||
        (reinterpret_cast<uintptr_t>(scores) & 3u))
        return TMS_ERR_ALIGNMENT;
    if (!device_info()) return TMS_ERR_CUDA;
    if (B == 0) return TMS_OK;
    if (total_tokens == 0) return fill_empty(scores, (int64_t)Q * B, static_cast<cudaStream_t>(stream));
    const size_t need = dense_tc_workspace_bytes(Q, Nq, B);
    if (need != 0) {
        if (!workspace || workspace_bytes < need) return TMS_ERR_WORKSPACE;
        if (!aligned16(workspace)) return TMS_ERR_ALIGNMENT;
    }
    DenseArgs a{queries, Q, Nq, d, nullptr, offsets, B, total_tokens, q_dtype, scores, static_cast<cudaStream_t>(stream),
                workspace, workspace_bytes};
    a.codes = codes;
    a.codebooks = codebooks;
    a.pq_half = precision == TMS_PQ_FP16;
    return dense_tc_supports(a) ? launch_dense_tc(a) : TMS_ERR_UNSUPPORTED;
}

int tms_pq_maxsim_decode(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks, int M,
                         int K, const uint8_t* codes, const int64_t* offsets, int64_t B, int64_t total_tokens,
                         float* scores, void* workspace, size_t workspace_bytes, void* stream) {
    return tms_pq_maxsim_decode_variant(queries, Q, Nq, d, q_dtype, codebooks, M, K, codes, offsets, B, total_tokens,
                                        scores, workspace, workspace_bytes, stream, TMS_PQ_SPLIT_BF16);
}

int tms_topk(const float* scores, int Q, int64_t B, int k, float* values, int64_t* indices, void* workspace,
             size_t workspace_bytes, void* stream) {
    if (Q <= 0 || B <= 0 || k <= 0 || !scores || !values || !indices) return TMS_ERR_INVALID_ARG;
    if (k > B) return TMS_ERR_INVALID_ARG;
    if (k > 1024 || B > (1ll << 31) || Q > 65535) return TMS_ERR_UNSUPPORTED;
    if ((reinterpret_cast<uintptr_t>(scores) & 3u) || (reinterpret_cast<uintptr_t>(values) & 3u) ||
        (reinterpret_cast<uintptr_t>(indices) & 7u))
        return TMS_ERR_ALIGNMENT;
    const size_t need = topk_workspace_bytes(Q, B, k);
    if (need && (!workspace || workspace_bytes < need || (reinterpret_cast<uintptr_t>(workspace) & 7u)))
        return TMS_ERR_WORKSPACE;
    if (!device_info()) return TMS_ERR_CUDA;
    return launch_topk(scores, Q, B, k, values, indices, workspace, static_cast<cudaStream_t>(stream));
}

size_t tms_topk_workspace_bytes(int Q, int64_t B, int k) {
    if (Q <= 0 || B <= 0 || k <= 0) return 0;
    return topk_workspace_bytes(Q, B, k);
}

// tms_topk for callers that cannot provide a workspace: same checks, scratch in the library's built-in device array.
// No cudaMalloc / cudaFree / allocating library routine anywhere below this call.
int tms_topk_static(const float* scores, int Q, int64_t B, int k, float* values, int64_t* indices, void* stream) {
    if (Q <= 0 || B <= 0 || k <= 0 || !scores || !values || !indices) return TMS_ERR_INVALID_ARG;
    if (k > B) return TMS_ERR_INVALID_ARG;
    if (k > 1024 || B > (1ll << 31) || Q > 65535) return TMS_ERR_UNSUPPORTED;
    if ((reinterpret_cast<uintptr_t>(scores) & 3u) || (reinterpret_cast<uintptr_t>(values) & 3u) ||
        (reinterpret_cast<uintptr_t>(indices) & 7u))
        return TMS_ERR_ALIGNMENT;
    if (topk_workspace_bytes(Q, B, k) > (size_t)TMS_TOPK_STATIC_SCRATCH_BYTES) return TMS_ERR_STATIC_SCRATCH;
    if (!device_info()) return TMS_ERR_CUDA;
    return launch_topk_static(scores, Q, B, k, values, indices, static_cast<cudaStream_t>(stream));
}

size_t tms_topk_static_scratch_bytes(void) { return (size_t)TMS_TOPK_STATIC_SCRATCH_BYTES; }

int tms_topk_merge(const float* values, const int64_t* indices, const int64_t* shard_base, int G, int Q, int k_in, int k,
                   float* out_values, int64_t* out_indices, void* workspace, size_t workspace_bytes, void* stream) {
    if (G <= 0 || Q <= 0 || k_in <= 0 || k <= 0 || !values || !indices || !shard_base || !out_values || !out_indices)
        return TMS_ERR_INVALID_ARG;
    if ((int64_t)k > (int64_t)G * k_in) return TMS_ERR_INVALID_ARG;
    if (G > 64 || k > 1024 || k_in > 1024 || Q > 65535) return TMS_ERR_UNSUPPORTED;
    for (int g = 0; g < G; ++g)
        if (shard_base[g] < 0 || shard_base[g] >= (1ll << 31)) return TMS_ERR_INVALID_ARG;  // base + index < 2^31
    if ((reinterpret_cast<uintptr_t>(values) & 3u) || (reinterpret_cast<uintptr_t>(out_values) & 3u) ||
        (reinterpret_cast<uintptr_t>(indices) & 7u) || (reinterpret_cast<uintptr_t>(out_indices) & 7u))
        return TMS_ERR_ALIGNMENT;
    if (!workspace || workspace_bytes < topk_merge_workspace_bytes(G, Q, k_in, k) ||
        (reinterpret_cast<uintptr_t>(workspace) & 7u))
        return TMS_ERR_WORKSPACE;
    if (!device_info()) return TMS_ERR_CUDA;
    return launch_topk_merge(values, indices, shard_base, G, Q, k_in, k, out_values, out_indices, workspace,
                             static_cast<cudaStream_t>(stream));
}

size_t tms_topk_merge_workspace_bytes(int G, int Q, int k_in, int k) {
    if (G <= 0 || Q <= 0 || k_in <= 0 || k <= 0) return 0;
    return topk_merge_workspace_bytes(G, Q, k_in, k);
}

uint64_t tms_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char* tms_status_string(int status) {
    switch (status) {
        case TMS_OK: return "ok";
        case TMS_ERR_INVALID_ARG: return "invalid argument";
        case TMS_ERR_UNSUPPORTED: return "unsupported shape, dtype or device";
        case TMS_ERR_ALIGNMENT: return "pointer or row pitch not 16-byte aligned";
        case TMS_ERR_WORKSPACE: return "workspace missing or too small";
        case TMS_ERR_CUDA: return "CUDA error";
        case TMS_ERR_STATIC_SCRATCH:
            return "shape needs more scratch than the library's built-in static buffer holds "
                   "(tms_topk_workspace_bytes > TMS_TOPK_STATIC_SCRATCH_BYTES): use tms_topk with a workspace";
        default: return "unknown status";
    }
}

int tms_version(void) { return 100; }

}  // extern "C"
