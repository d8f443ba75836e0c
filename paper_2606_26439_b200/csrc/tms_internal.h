// Internal declarations shared by the translation units of libtms.so (never installed).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/tms.h"

namespace tms {

inline size_t dtype_size(tms_dtype t) { return t == TMS_DTYPE_F32 ? 4 : 2; }

// Every kernel launch in the library goes through this counter (tms_launch_count()).
void count_launch(int n = 1);

struct DeviceInfo {
    int device = -1;
    int cc_major = 0, cc_minor = 0;
    int num_sms = 0;
    int max_smem_optin = 0;
};
// Cached per device; returns nullptr when no CUDA device is usable.
const DeviceInfo* device_info();

// ---- dense -----------------------------------------------------------------------------------------------------
struct DenseArgs {
    const void* queries;
    int Q, Nq, d;
    const void* docs;
    const int64_t* offsets;
    int64_t B, T;
    tms_dtype dtype;
    float* scores;
    cudaStream_t stream;
    void* workspace = nullptr;  // device scratch (tms_maxsim_workspace_bytes)
    size_t workspace_bytes = 0;
    // decode-and-contract PQ variant: `docs` is unused, the store is codes[T,16] + codebooks[16,256,8]; `dtype` is the
    // queries' dtype and d = 128
    const uint8_t* codes = nullptr;
    const float* codebooks = nullptr;
    bool pq_half = false;  // TMS_PQ_FP16: queries and centroids rounded to fp16, one MMA per product
};

// CUDA-core tiled kernel: any dtype / d / Nq / Q (csrc/dense_simt.cu).
int launch_dense_simt(const DenseArgs& a);
// TMA + tcgen05 kernel (csrc/dense_tc.cu). supports() says whether the shape is covered.
bool dense_tc_supports(const DenseArgs& a);
// the shape test alone (no device query): what an sm_100 device with 227 KB of shared memory would run
bool dense_tc_shape_ok(const DenseArgs& a);
int launch_dense_tc(const DenseArgs& a);
// Scratch the tcgen05 path needs for this shape (0 for Nq <= 32).
size_t dense_tc_workspace_bytes(int Q, int Nq, int64_t B);

// ---- PQ --------------------------------------------------------------------------------------------------------
struct PqArgs {
    const float* lut;
    int Q, Nq, M, K;
    const uint8_t* codes;
    const int64_t* offsets;
    int64_t B, T;
    float* scores;
    cudaStream_t stream;
};
int launch_pq_build_lut(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks, int M,
                        int K, float* lut, cudaStream_t stream);
int launch_pq_simt(const PqArgs& a);
// f16: table entries stored as scaled fp16 (16 query rows per shared-memory slice, Nq % 16 == 0)
bool pq_smem_supports(const PqArgs& a, bool f16);
size_t pq_smem_workspace_bytes(int Q, int Nq);
int launch_pq_smem(const PqArgs& a, void* workspace, bool f16);

// ---- top-k (csrc/topk.cu) ---------------------------------------------------------------------------------------
size_t topk_workspace_bytes(int Q, int64_t B, int k);
int launch_topk(const float* scores, int Q, int64_t B, int k, float* values, int64_t* indices, void* workspace,
                cudaStream_t stream);

// the same with the key buffers in the library's built-in device array (tms_topk_static)
int launch_topk_static(const float* scores, int Q, int64_t B, int k, float* values, int64_t* indices,
                       cudaStream_t stream);

size_t topk_merge_workspace_bytes(int G, int Q, int k_in, int k);
int launch_topk_merge(const float* values, const int64_t* indices, const int64_t* shard_base, int G, int Q, int k_in,
                      int k, float* out_values, int64_t* out_indices, void* workspace, cudaStream_t stream);

}  // namespace tms
