// host_api.cu -- the HOST-buffer entry points of include/tms.h (tms_maxsim_host, tms_pq_maxsim_host).
//
// The document store lives in host memory and is streamed through a caller-provided device workspace in
// document-aligned chunks.  Two chunk buffers alternate: the host->device copy of chunk n+1 runs on an
// internal copy stream while the scoring kernels of chunk n run on the caller's stream; scores of each
// chunk go back with one strided device->host copy.  Scoring itself is the same kernels as the device
// entry points (dispatch through tms_maxsim / tms_pq_maxsim).
#include <mutex>

#include "tms_internal.h"

namespace tms {
namespace {

constexpr size_t ALIGN = 256;
size_t up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

__global__ void rebase_offsets_kernel(int64_t* off, int64_t n, int64_t base) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) off[i] -= base;
}

cudaStream_t copy_stream() {
    static std::mutex mu;
    static cudaStream_t streams[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lock(mu);
    if (!streams[dev] && cudaStreamCreateWithFlags(&streams[dev], cudaStreamNonBlocking) != cudaSuccess)
        return nullptr;
    return streams[dev];
}

// bytes of one chunk buffer: rows of the store, rebased offsets, scores, and `ws_per_doc` bytes of kernel scratch per
// document (the partial scores of queries longer than 32 tokens; 0 otherwise)
size_t chunk_bytes(int64_t nt, int64_t nb, size_t row_bytes, int Q, size_t ws_per_doc) {
    return up((size_t)nt * row_bytes) + up((size_t)(nb + 1) * 8) + up((size_t)Q * nb * 4) + up(ws_per_doc * (size_t)nb);
}

struct Chunk {
    uint8_t* store;    // device: this chunk's rows of the document store (embeddings or codes)
    int64_t* offsets;  // device: rebased offsets [nb+1]
    float* scores;     // device: [Q, nb]
    void* ws;          // device: kernel scratch (ws_bytes; NULL when none is needed)
    size_t ws_bytes;
    int64_t nb, nt;
};

struct Events {  // destroyed on every exit path
    cudaEvent_t copied[2] = {nullptr, nullptr}, consumed[2] = {nullptr, nullptr}, entry = nullptr;
    bool create() {
        for (int i = 0; i < 2; ++i)
            if (cudaEventCreateWithFlags(&copied[i], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&consumed[i], cudaEventDisableTiming) != cudaSuccess)
                return false;
        return cudaEventCreateWithFlags(&entry, cudaEventDisableTiming) == cudaSuccess;
    }
    ~Events() {
        for (int i = 0; i < 2; ++i) {
            if (copied[i]) cudaEventDestroy(copied[i]);
            if (consumed[i]) cudaEventDestroy(consumed[i]);
        }
        if (entry) cudaEventDestroy(entry);
    }
};

#define TMS_CUDA_OK(call) ((call) == cudaSuccess)

// Streams the store through two buffers; `score` enqueues the scoring of one chunk on `stream`.
template <typename ScoreFn>
int stream_chunks(const uint8_t* store_h, size_t row_bytes, const int64_t* offsets_h, int64_t B, int64_t T, int Q,
                  size_t ws_per_doc, float* scores_h, uint8_t* bufs, size_t per_buf, cudaStream_t stream,
                  ScoreFn score) {
    if (offsets_h[0] != 0 || offsets_h[B] != T) return TMS_ERR_INVALID_ARG;
    cudaStream_t cs = copy_stream();
    if (!cs) return TMS_ERR_CUDA;
    Events ev;
    if (!ev.create()) { cudaGetLastError(); return TMS_ERR_CUDA; }
    int status = TMS_OK;
    // the copy stream must not touch the workspace before earlier work on `stream` is done with it
    if (!TMS_CUDA_OK(cudaEventRecord(ev.entry, stream)) || !TMS_CUDA_OK(cudaStreamWaitEvent(cs, ev.entry, 0)))
        status = TMS_ERR_CUDA;

    int64_t b0 = 0;
    for (int n = 0; b0 < B && status == TMS_OK; ++n) {
        const int buf = n & 1;
        const int64_t t0 = offsets_h[b0];
        int64_t b1 = b0;
        while (b1 < B) {  // grow the chunk document by document while it fits
            if (offsets_h[b1 + 1] < offsets_h[b1]) { status = TMS_ERR_INVALID_ARG; break; }
            if (chunk_bytes(offsets_h[b1 + 1] - t0, b1 + 1 - b0, row_bytes, Q, ws_per_doc) > per_buf) break;
            ++b1;
        }
        if (status != TMS_OK) break;
        if (b1 == b0) { status = TMS_ERR_WORKSPACE; break; }  // a single document does not fit
        Chunk c;
        c.nb = b1 - b0;
        c.nt = offsets_h[b1] - t0;
        uint8_t* base = bufs + (size_t)buf * per_buf;
        c.store = base;
        c.offsets = reinterpret_cast<int64_t*>(base + up((size_t)c.nt * row_bytes));
        c.scores = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(c.offsets) + up((size_t)(c.nb + 1) * 8));
        c.ws_bytes = ws_per_doc * (size_t)c.nb;
        c.ws = c.ws_bytes ? reinterpret_cast<uint8_t*>(c.scores) + up((size_t)Q * c.nb * 4) : nullptr;

        bool ok = true;
        if (n >= 2) ok = ok && TMS_CUDA_OK(cudaStreamWaitEvent(cs, ev.consumed[buf], 0));
        if (c.nt > 0)
            ok = ok && TMS_CUDA_OK(cudaMemcpyAsync(c.store, store_h + (size_t)t0 * row_bytes, (size_t)c.nt * row_bytes,
                                                   cudaMemcpyHostToDevice, cs));
        ok = ok && TMS_CUDA_OK(cudaMemcpyAsync(c.offsets, offsets_h + b0, (size_t)(c.nb + 1) * 8, cudaMemcpyHostToDevice, cs));
        if (ok) {
            rebase_offsets_kernel<<<(unsigned)((c.nb + 1 + 255) / 256), 256, 0, cs>>>(c.offsets, c.nb + 1, t0);
            count_launch();
            ok = TMS_CUDA_OK(cudaGetLastError());
        }
        ok = ok && TMS_CUDA_OK(cudaEventRecord(ev.copied[buf], cs)) && TMS_CUDA_OK(cudaStreamWaitEvent(stream, ev.copied[buf], 0));
        if (!ok) { status = TMS_ERR_CUDA; break; }
        status = score(c);
        if (status != TMS_OK) break;
        if (!TMS_CUDA_OK(cudaMemcpy2DAsync(scores_h + b0, (size_t)B * 4, c.scores, (size_t)c.nb * 4, (size_t)c.nb * 4,
                                           (size_t)Q, cudaMemcpyDeviceToHost, stream)) ||
            !TMS_CUDA_OK(cudaEventRecord(ev.consumed[buf], stream))) {
            status = TMS_ERR_CUDA;
            break;
        }
        b0 = b1;
    }
    // both streams are drained before the workspace (and the events) can be reused, whatever happened above
    if (cudaStreamSynchronize(stream) != cudaSuccess && status == TMS_OK) status = TMS_ERR_CUDA;
    if (cudaStreamSynchronize(cs) != cudaSuccess && status == TMS_OK) status = TMS_ERR_CUDA;
    if (cudaGetLastError() != cudaSuccess && status == TMS_OK) status = TMS_ERR_CUDA;
    return status;
}

}  // namespace
}  // namespace tms

using namespace tms;

extern "C" {

size_t tms_maxsim_host_workspace_min_bytes(int Q, int Nq, int d, tms_dtype dtype, int64_t max_doc_tokens) {
    if (Q <= 0 || Nq <= 0 || d <= 0 || max_doc_tokens < 0) return 0;
    const size_t row = (size_t)d * dtype_size(dtype);
    return up((size_t)Q * Nq * row) + 2 * chunk_bytes(max_doc_tokens, 1, row, Q, dense_tc_workspace_bytes(Q, Nq, 1)) +
           2 * ALIGN;
}

int tms_maxsim_host(const void* queries, int Q, int Nq, int d, const void* docs, const int64_t* offsets, int64_t B,
                    int64_t total_tokens, tms_dtype dtype, float* scores, void* dev_workspace,
                    size_t dev_workspace_bytes, void* stream_) {
    if (Q <= 0 || Nq <= 0 || d <= 0 || B < 0 || total_tokens < 0) return TMS_ERR_INVALID_ARG;
    if (dtype != TMS_DTYPE_F32 && dtype != TMS_DTYPE_F16 && dtype != TMS_DTYPE_BF16) return TMS_ERR_INVALID_ARG;
    if (!queries || !offsets || (B > 0 && !scores) || (total_tokens > 0 && !docs)) return TMS_ERR_INVALID_ARG;
    const size_t row = (size_t)d * dtype_size(dtype);
    if (row % 16 != 0) return TMS_ERR_UNSUPPORTED;
    if (!device_info()) return TMS_ERR_CUDA;
    if (B == 0) return TMS_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    uint8_t* ws = static_cast<uint8_t*>(dev_workspace);
    if (!ws) return TMS_ERR_WORKSPACE;
    const size_t skew = (ALIGN - (reinterpret_cast<uintptr_t>(ws) % ALIGN)) % ALIGN;
    const size_t qbytes = up((size_t)Q * Nq * row);
    if (dev_workspace_bytes < skew + qbytes + 4 * ALIGN) return TMS_ERR_WORKSPACE;
    uint8_t* q_dev = ws + skew;
    uint8_t* bufs = q_dev + qbytes;
    const size_t per_buf = ((dev_workspace_bytes - skew - qbytes) / 2) / ALIGN * ALIGN;
    if (cudaMemcpyAsync(q_dev, queries, (size_t)Q * Nq * row, cudaMemcpyHostToDevice, stream) != cudaSuccess)
        return TMS_ERR_CUDA;
    // queries longer than 32 tokens: every chunk buffer carries the kernel's scratch for its own documents
    return stream_chunks(static_cast<const uint8_t*>(docs), row, offsets, B, total_tokens, Q,
                         dense_tc_workspace_bytes(Q, Nq, 1), scores, bufs, per_buf, stream, [&](const Chunk& c) {
                             return tms_maxsim(q_dev, Q, Nq, d, c.store, c.offsets, c.nb, c.nt, dtype, c.scores, c.ws,
                                               c.ws_bytes, stream);
                         });
}

size_t tms_pq_maxsim_host_workspace_min_bytes(int Q, int Nq, int d, tms_dtype q_dtype, int M, int K,
                                              int64_t max_doc_tokens) {
    if (Q <= 0 || Nq <= 0 || d <= 0 || M <= 0 || K <= 0 || max_doc_tokens < 0) return 0;
    const size_t lut = up((size_t)Q * Nq * M * K * 4 + 16);  // the table, and the re-laid-out table + its header
    return up((size_t)Q * Nq * d * dtype_size(q_dtype)) + up((size_t)M * K * (d / M) * 4) + 2 * lut +
           2 * chunk_bytes(max_doc_tokens, 1, (size_t)M, Q, 0) + 2 * ALIGN;
}

int tms_pq_maxsim_host(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks, int M,
                       int K, const uint8_t* codes, const int64_t* offsets, int64_t B, int64_t total_tokens,
                       float* scores, void* dev_workspace, size_t dev_workspace_bytes, void* stream_) {
    if (Q <= 0 || Nq <= 0 || d <= 0 || M <= 0 || K <= 0 || B < 0 || total_tokens < 0) return TMS_ERR_INVALID_ARG;
    if (q_dtype != TMS_DTYPE_F32 && q_dtype != TMS_DTYPE_F16 && q_dtype != TMS_DTYPE_BF16) return TMS_ERR_INVALID_ARG;
    if (!queries || !codebooks || !offsets || (B > 0 && !scores) || (total_tokens > 0 && !codes))
        return TMS_ERR_INVALID_ARG;
    if (d % M != 0 || K > 256) return TMS_ERR_UNSUPPORTED;
    if (!device_info()) return TMS_ERR_CUDA;
    if (B == 0) return TMS_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    uint8_t* ws = static_cast<uint8_t*>(dev_workspace);
    if (!ws) return TMS_ERR_WORKSPACE;
    const size_t skew = (ALIGN - (reinterpret_cast<uintptr_t>(ws) % ALIGN)) % ALIGN;
    const size_t qbytes = up((size_t)Q * Nq * d * dtype_size(q_dtype));
    const size_t cbytes = up((size_t)M * K * (d / M) * 4);
    const size_t lbytes = up((size_t)Q * Nq * M * K * 4 + 16);  // the table, and the re-laid-out table + its header
    const size_t fixed = skew + qbytes + cbytes + 2 * lbytes;
    if (dev_workspace_bytes < fixed + 4 * ALIGN) return TMS_ERR_WORKSPACE;
    uint8_t* q_dev = ws + skew;
    float* cb_dev = reinterpret_cast<float*>(q_dev + qbytes);
    float* lut_dev = reinterpret_cast<float*>(q_dev + qbytes + cbytes);
    uint8_t* pq_ws = q_dev + qbytes + cbytes + lbytes;
    uint8_t* bufs = pq_ws + lbytes;
    const size_t per_buf = ((dev_workspace_bytes - fixed) / 2) / ALIGN * ALIGN;
    if (cudaMemcpyAsync(q_dev, queries, (size_t)Q * Nq * d * dtype_size(q_dtype), cudaMemcpyHostToDevice, stream) !=
            cudaSuccess ||
        cudaMemcpyAsync(cb_dev, codebooks, (size_t)M * K * (d / M) * 4, cudaMemcpyHostToDevice, stream) != cudaSuccess)
        return TMS_ERR_CUDA;
    int st = tms_pq_build_lut(q_dev, Q, Nq, d, q_dtype, cb_dev, M, K, lut_dev, stream);
    if (st != TMS_OK) return st;
    return stream_chunks(codes, (size_t)M, offsets, B, total_tokens, Q, 0, scores, bufs, per_buf, stream,
                         [&](const Chunk& c) {
                             return tms_pq_maxsim(lut_dev, Q, Nq, M, K, c.store, c.offsets, c.nb, c.nt, c.scores, pq_ws,
                                                  lbytes, stream);
                         });
}

size_t tms_pq_maxsim_decode_host_workspace_min_bytes(int Q, int Nq, int d, tms_dtype q_dtype, int M, int K,
                                                     int64_t max_doc_tokens) {
    if (Q <= 0 || Nq <= 0 || d <= 0 || M <= 0 || K <= 0 || max_doc_tokens < 0) return 0;
    return up((size_t)Q * Nq * d * dtype_size(q_dtype)) + up((size_t)M * K * (d / M) * 4) +
           2 * chunk_bytes(max_doc_tokens, 1, (size_t)M, Q, dense_tc_workspace_bytes(Q, Nq, 1)) + 2 * ALIGN;
}

int tms_pq_maxsim_decode_host(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks,
                              int M, int K, const uint8_t* codes, const int64_t* offsets, int64_t B,
                              int64_t total_tokens, float* scores, void* dev_workspace, size_t dev_workspace_bytes,
                              void* stream_) {
    if (Q <= 0 || Nq <= 0 || d <= 0 || M <= 0 || K <= 0 || B < 0 || total_tokens < 0) return TMS_ERR_INVALID_ARG;
    if (q_dtype != TMS_DTYPE_F32 && q_dtype != TMS_DTYPE_F16 && q_dtype != TMS_DTYPE_BF16) return TMS_ERR_INVALID_ARG;
    if (!queries || !codebooks || !offsets || (B > 0 && !scores) || (total_tokens > 0 && !codes))
        return TMS_ERR_INVALID_ARG;
    if (d != 128 || M != 16 || K != 256) return TMS_ERR_UNSUPPORTED;
    if (!device_info()) return TMS_ERR_CUDA;
    if (B == 0) return TMS_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    uint8_t* ws = static_cast<uint8_t*>(dev_workspace);
    if (!ws) return TMS_ERR_WORKSPACE;
    const size_t skew = (ALIGN - (reinterpret_cast<uintptr_t>(ws) % ALIGN)) % ALIGN;
    const size_t qbytes = up((size_t)Q * Nq * d * dtype_size(q_dtype));
    const size_t cbytes = up((size_t)M * K * (d / M) * 4);
    const size_t fixed = skew + qbytes + cbytes;
    if (dev_workspace_bytes < fixed + 4 * ALIGN) return TMS_ERR_WORKSPACE;
    uint8_t* q_dev = ws + skew;
    float* cb_dev = reinterpret_cast<float*>(q_dev + qbytes);
    uint8_t* bufs = q_dev + qbytes + cbytes;
    const size_t per_buf = ((dev_workspace_bytes - fixed) / 2) / ALIGN * ALIGN;
    if (cudaMemcpyAsync(q_dev, queries, (size_t)Q * Nq * d * dtype_size(q_dtype), cudaMemcpyHostToDevice, stream) !=
            cudaSuccess ||
        cudaMemcpyAsync(cb_dev, codebooks, (size_t)M * K * (d / M) * 4, cudaMemcpyHostToDevice, stream) != cudaSuccess)
        return TMS_ERR_CUDA;
    return stream_chunks(codes, (size_t)M, offsets, B, total_tokens, Q, dense_tc_workspace_bytes(Q, Nq, 1), scores, bufs,
                         per_buf, stream, [&](const Chunk& c) {
                             return tms_pq_maxsim_decode(q_dev, Q, Nq, d, q_dtype, cb_dev, M, K, c.store, c.offsets, c.nb,
                                                         c.nt, c.scores, c.ws, c.ws_bytes, stream);
                         });
}

}  // extern "C"
