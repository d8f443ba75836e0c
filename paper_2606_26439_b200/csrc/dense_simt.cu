// dense_simt.cu -- general CUDA-core MaxSim kernel (TMS_VARIANT_SIMT).
//
// Covers every shape the C ABI admits (any dtype, any d with a 16-byte row pitch, any Nq, any Q): it is
// the path for shapes the tcgen05 kernel does not take, and the on-GPU cross-check for it.
//
// One CTA scores one document at a time (grid-stride over documents).  For each 64-row x 64-token tile it
// accumulates partial dot products over 32-wide dimension chunks in fp32 registers -- the paper's
// dimension tiling, "accumulating partial dot products before computing the max" -- then folds
// the tile into per-row running maxima (Alg. 3 lines 7-8) and finally sums the Nq maxima of
// each query in ascending i (Eq. 1).  Nothing but scores[Q,B] is written to global memory.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "tms_internal.h"

namespace tms {
namespace {

constexpr int TR = 64;   // query rows per tile
constexpr int TT = 64;   // document tokens per tile
constexpr int TK = 32;   // dimension chunk
constexpr int NTHREADS = 256;

__device__ __forceinline__ float to_f32(float v) { return v; }
__device__ __forceinline__ float to_f32(__half v) { return __half2float(v); }
__device__ __forceinline__ float to_f32(__nv_bfloat16 v) { return __bfloat162float(v); }

template <typename T>
__global__ void __launch_bounds__(NTHREADS)
dense_simt_kernel(const T* __restrict__ queries, int Q, int Nq, int d, const T* __restrict__ docs,
                  const int64_t* __restrict__ offsets, int64_t B, float* __restrict__ scores) {
    __shared__ float Qs[TR][TK + 1];
    __shared__ float Ds[TT][TK + 1];
    extern __shared__ float rowmax[];  // [Q*Nq]

    const int R = Q * Nq;
    const int tid = threadIdx.x;
    const int tx = tid & 15;  // token direction
    const int ty = tid >> 4;  // row direction

    for (int64_t b = blockIdx.x; b < B; b += gridDim.x) {
        const int64_t t0 = offsets[b];
        const int64_t nd = offsets[b + 1] - t0;
        for (int r = tid; r < R; r += NTHREADS) rowmax[r] = -INFINITY;  // Alg. 3 line 4: m <- -inf
        __syncthreads();

        for (int r0 = 0; r0 < R; r0 += TR) {
            for (int64_t j0 = 0; j0 < nd; j0 += TT) {
                float acc[4][4];
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

                for (int k0 = 0; k0 < d; k0 += TK) {
#pragma unroll
                    for (int e = 0; e < (TR * TK) / NTHREADS; ++e) {
                        const int idx = tid + e * NTHREADS;
                        const int row = idx / TK, kk = idx % TK;
                        const int r = r0 + row, k = k0 + kk;
                        Qs[row][kk] = (r < R && k < d) ? to_f32(queries[(int64_t)r * d + k]) : 0.f;
                        const int64_t j = j0 + row;
                        Ds[row][kk] = (j < nd && k < d) ? to_f32(docs[(t0 + j) * d + k]) : 0.f;
                    }
                    __syncthreads();
#pragma unroll
                    for (int kk = 0; kk < TK; ++kk) {
                        float a[4], c[4];
#pragma unroll
                        for (int i = 0; i < 4; ++i) a[i] = Qs[ty * 4 + i][kk];
#pragma unroll
                        for (int j = 0; j < 4; ++j) c[j] = Ds[tx + 16 * j][kk];
#pragma unroll
                        for (int i = 0; i < 4; ++i)
#pragma unroll
                            for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], c[j], acc[i][j]);
                    }
                    __syncthreads();
                }

                // rowmax over this tile's valid tokens, then across the 16 lanes that share a row
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    float m = -INFINITY;
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        if (j0 + tx + 16 * j < nd) m = fmaxf(m, acc[i][j]);
#pragma unroll
                    for (int o = 8; o >= 1; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
                    const int r = r0 + ty * 4 + i;
                    if (tx == 0 && r < R) rowmax[r] = fmaxf(rowmax[r], m);
                }
            }
        }
        __syncthreads();
        for (int q = tid; q < Q; q += NTHREADS) {
            float s = 0.f;
            for (int i = 0; i < Nq; ++i) s += rowmax[q * Nq + i];
            scores[(int64_t)q * B + b] = s;
        }
        __syncthreads();
    }
}

template <typename T>
int launch(const DenseArgs& a, int num_sms) {
    const size_t smem = sizeof(float) * (size_t)a.Q * a.Nq;
    if (smem > 160 * 1024) return TMS_ERR_UNSUPPORTED;
    if (smem > 30 * 1024 &&
        cudaFuncSetAttribute(dense_simt_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
            cudaSuccess)
        return TMS_ERR_CUDA;
    const int64_t grid = a.B < (int64_t)num_sms * 8 ? a.B : (int64_t)num_sms * 8;
    dense_simt_kernel<T><<<(unsigned)grid, NTHREADS, smem, a.stream>>>(
        static_cast<const T*>(a.queries), a.Q, a.Nq, a.d, static_cast<const T*>(a.docs), a.offsets, a.B, a.scores);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? TMS_OK : TMS_ERR_CUDA;
}

}  // namespace

int launch_dense_simt(const DenseArgs& a) {
    const DeviceInfo* di = device_info();
    if (!di) return TMS_ERR_CUDA;
    if (a.B == 0) return TMS_OK;
    switch (a.dtype) {
        case TMS_DTYPE_F32: return launch<float>(a, di->num_sms);
        case TMS_DTYPE_F16: return launch<__half>(a, di->num_sms);
        case TMS_DTYPE_BF16: return launch<__nv_bfloat16>(a, di->num_sms);
    }
    return TMS_ERR_INVALID_ARG;
}

}  // namespace tms
