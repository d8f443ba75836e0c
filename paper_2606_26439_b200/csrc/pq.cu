// pq.cu -- product-quantisation path: LUT build (Eq. 8), general fused lookup kernel, and the
// shared-memory-resident LUT kernel (Eq. 9).
//
// The paper's phase 2 runs one program per (document, query token) with the table served from L2
// (P:L268-270).  On B200 the lookups, not HBM, bound this path: Q*Nq*T*M 4-byte gathers against 2 GB of
// codes.  The main kernel therefore keeps a 128 KB slice of the table -- 8 query
// rows x M=16 x K=256 -- resident in shared memory, laid out so that every LDS.128 of a quarter-warp hits
// eight different 16-byte bank groups whatever the codes are, and walks all slices over a document chunk
// while the chunk's codes stay in L2, so codes come from HBM once.  No decompressed vector ever exists.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "tms_internal.h"

namespace tms {
namespace {

__device__ __forceinline__ float to_f32(float v) { return v; }
__device__ __forceinline__ float to_f32(__half v) { return __half2float(v); }
__device__ __forceinline__ float to_f32(__nv_bfloat16 v) { return __bfloat162float(v); }

// ---------------------------------------------------------------------------------------------------------------
// Eq. 8: lut[q,i,m,k] = sum_s queries[q,i,m*dsub+s] * C[m,k,s]   (fp32 FMA, s ascending)
// grid (Q*Nq, M), one thread per centroid k.
// ---------------------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
pq_build_lut_kernel(const T* __restrict__ queries, int d, const float* __restrict__ codebooks, int M, int K,
                    float* __restrict__ lut) {
    const int row = blockIdx.x, m = blockIdx.y, dsub = d / M;
    const T* q = queries + (int64_t)row * d + m * dsub;
    for (int k = threadIdx.x; k < K; k += blockDim.x) {
        const float* c = codebooks + ((int64_t)m * K + k) * dsub;
        float acc = 0.f;
        for (int s = 0; s < dsub; ++s) acc = fmaf(to_f32(q[s]), c[s], acc);
        lut[((int64_t)row * M + m) * K + k] = acc;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// General fused lookup kernel (TMS_VARIANT_SIMT): any M, any K <= 256, any Nq.  One CTA per document
// (grid-stride), one thread per query row, table read through L1/L2 as in the paper.
// ---------------------------------------------------------------------------------------------------------------
constexpr int SIMT_THREADS = 256;
constexpr int SIMT_TOK = 128;  // tokens staged per pass

__global__ void __launch_bounds__(SIMT_THREADS)
pq_simt_kernel(const float* __restrict__ lut, int Q, int Nq, int M, int K, const uint8_t* __restrict__ codes,
               const int64_t* __restrict__ offsets, int64_t B, float* __restrict__ scores) {
    extern __shared__ unsigned char smem_raw[];
    const int R = Q * Nq;
    float* rowmax = reinterpret_cast<float*>(smem_raw);                    // [R]
    uint8_t* cs = smem_raw + sizeof(float) * (size_t)((R + 3) & ~3);       // [SIMT_TOK * M]
    const int tid = threadIdx.x;
    for (int64_t b = blockIdx.x; b < B; b += gridDim.x) {
        const int64_t t0 = offsets[b], nd = offsets[b + 1] - t0;
        for (int r = tid; r < R; r += SIMT_THREADS) rowmax[r] = -INFINITY;
        for (int64_t j0 = 0; j0 < nd; j0 += SIMT_TOK) {
            const int nt = (int)((nd - j0) < SIMT_TOK ? (nd - j0) : SIMT_TOK);
            __syncthreads();
            for (int e = tid; e < nt * M; e += SIMT_THREADS) cs[e] = codes[(t0 + j0) * M + e];
            __syncthreads();
            for (int r = tid; r < R; r += SIMT_THREADS) {
                const float* lr = lut + (int64_t)r * M * K;
                float mx = rowmax[r];
                for (int j = 0; j < nt; ++j) {
                    float s = 0.f;
                    for (int m = 0; m < M; ++m) s += lr[m * K + cs[j * M + m]];  // Eq. 9, m ascending
                    mx = fmaxf(mx, s);
                }
                rowmax[r] = mx;
            }
        }
        __syncthreads();
        for (int q = tid; q < Q; q += SIMT_THREADS) {
            float s = 0.f;
            for (int i = 0; i < Nq; ++i) s += rowmax[q * Nq + i];
            scores[(int64_t)q * B + b] = s;
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Shared-memory-resident LUT kernel (TMS_VARIANT_PQ_SMEM): M = 16, K = 256, Nq % 8 == 0.
//
// Slice sl holds query rows 8*sl .. 8*sl+7.  Slice layout (floats), one 128-byte line per (m/4, k):
//     line = (m >> 2) * 256 + k ;  within the line: [m & 3][row 0..7]
// A warp handles 16 document tokens per step: lane = 8*s4 + 2*u + h  ->  token slot 4*s4 + u, rows 4h..4h+3.
// At step (g, s) the lane looks up sub-quantiser m = 4g + ((s + u) & 3): the eight lanes of a quarter-warp
// then read 16-byte pieces 2*((s+u)&3) + h of their (code-dependent) lines -- eight distinct bank groups,
// conflict-free for any codes.  The per-lane order of the 16 additions is a fixed rotation of m.
// ---------------------------------------------------------------------------------------------------------------
//
// H16 (TMS_VARIANT_PQ_SMEM_F16): the same kernel over a table whose entries are stored as fp16 --
// a slice is then 16 query rows, every LDS.128 returns eight rows' entries and the gather bytes (the bound of this
// path) halve.  Entries are widened back to fp32 inside the addition (add.f32.f16: one FHADD per entry, as many ALU
// instructions as the fp32 table needs), so only the STORED entry is rounded: one relative 2^-11 error per entry,
// against the table's largest magnitude at worst, because the whole table is first scaled by a power of two that
// brings max|entry| into [2^14, 2^15) (no overflow, no subnormals for any finite table; the scale is undone exactly
// on the 16-row partial sums).
constexpr int PQS_M = 16, PQS_K = 256;
constexpr int PQS_SLICE_BYTES = 8 * PQS_M * PQS_K * 4;  // 128 KB: 8 rows of fp32 entries or 16 rows of fp16 entries
constexpr int PQS_WARPS = 24, PQS_THREADS = PQS_WARPS * 32;
constexpr int PQS_MAX_SC_FLOATS = 20480;  // 80 KB of per-chunk score accumulators

// lut [R, 16, 256] -> lutT [R/8 slices][4 g][256 k][4 sub][8 rows]
__global__ void pq_relayout_kernel(const float* __restrict__ lut, float* __restrict__ lutT, int64_t total) {
    const int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= total) return;
    const int row = (int)(o & 7), sub = (int)((o >> 3) & 3), k = (int)((o >> 5) & 255), g = (int)((o >> 13) & 3);
    const int64_t sl = o >> 15;
    lutT[o] = lut[((sl * 8 + row) * PQS_M + (4 * g + sub)) * PQS_K + k];
}

// max |lut| as float bits (non-negative floats order like unsigned integers); *out zeroed beforehand
__global__ void pq_absmax_kernel(const float* __restrict__ lut, int64_t total, uint32_t* __restrict__ out) {
    uint32_t m = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const uint32_t b = __float_as_uint(lut[i]) & 0x7fffffffu;
        m = b > m ? b : m;
    }
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0) atomicMax(out, m);
}

// lut [R, 16, 256] fp32 -> lutT [R/16 slices][4 g][256 k][4 sub][16 rows] fp16, scaled by the power of two that puts
// max|lut| into [2^14, 2^15); hdr[0] = max|lut| bits (input), hdr[1] = 1/scale as float bits (output).
__global__ void pq_relayout_f16_kernel(const float* __restrict__ lut, __half* __restrict__ lutT, int64_t total,
                                       uint32_t* __restrict__ hdr) {
    const float mx = __uint_as_float(hdr[0]);
    int e = 15;
    if (mx > 0.f && mx < INFINITY) frexpf(mx, &e);  // mx = f * 2^e, f in [0.5, 1)
    const float scale = ldexpf(1.f, 15 - e);        // 15 - e in [-113, 164]: clamp so that the scale stays finite
    const float sc = (15 - e > 126) ? ldexpf(1.f, 126) : scale;
    const int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o == 0) hdr[1] = __float_as_uint(1.f / sc);  // exact: a power of two
    if (o >= total) return;
    const int row = (int)(o & 15), sub = (int)((o >> 4) & 3), k = (int)((o >> 6) & 255), g = (int)((o >> 14) & 3);
    const int64_t sl = o >> 16;
    lutT[o] = __float2half_rn(lut[((sl * 16 + row) * PQS_M + (4 * g + sub)) * PQS_K + k] * sc);
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

// A chunk's codes are read once per table slice: every pass but the last asks L2 to keep the lines (evict_last), the last
// one marks them evict_first, so the chunk comes from HBM once even when 148 CTAs x 512 KB of live codes crowd L2.
__device__ __forceinline__ uint4 ldg_codes(const uint8_t* p, uint64_t policy) {
    uint4 r;
    asm volatile("ld.global.nc.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p), "l"(policy));
    return r;
}

__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds128u(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
// a += lo half of w, b += hi half of w, both widened exactly to fp32 inside the addition (one FHADD each)
__device__ __forceinline__ void add_h2(float& a, float& b, uint32_t w) {
    asm("add.rn.f32.f16 %0, %1, %0;" : "+f"(a) : "h"((unsigned short)(w & 0xffffu)));
    asm("add.rn.f32.f16 %0, %1, %0;" : "+f"(b) : "h"((unsigned short)(w >> 16)));
}

template <bool H16>
__global__ void __launch_bounds__(PQS_THREADS, 1)
pq_smem_kernel(const void* __restrict__ lutT, int Q, int Nq, const uint8_t* __restrict__ codes,
               const int64_t* __restrict__ offsets, int64_t B, int dpc /* docs per chunk */, int64_t nchunks,
               float* __restrict__ scores, const float* __restrict__ inv_scale) {
    constexpr int PQS_ROWS = H16 ? 16 : 8;  // query rows per 128 KB slice
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* lut_s = reinterpret_cast<float*>(smem_raw);                          // 128 KB slice
    float* sc = reinterpret_cast<float*>(smem_raw + PQS_SLICE_BYTES);           // [Q][dpc]
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + PQS_SLICE_BYTES + sizeof(float) * PQS_MAX_SC_FLOATS);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int s4 = lane >> 3, u = (lane >> 1) & 3, h = lane & 1;
    const int slot = s4 * 4 + u;
    const int nslices = (Q * Nq) / PQS_ROWS;
    const uint32_t bar_a = smem_u32(bar);
    const uint32_t lut_a = smem_u32(lut_s);

    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_a));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // per-lane constants: byte selector and 16-byte piece for each rotation step s
    uint32_t sel[4], base[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) {
        const uint32_t sub = (uint32_t)((s + u) & 3);
        sel[s] = 0x4440u | sub;  // PRMT: byte `sub` of the code word into bits 0..7, zeros above
        base[s] = lut_a + sub * 32u + (uint32_t)h * 16u;
    }
    uint32_t phase = 0;
    const float unscale = H16 ? *inv_scale : 1.f;
    uint64_t pol_keep, pol_drop;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_drop));
    __syncthreads();

    for (int64_t chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
        const int64_t d0 = chunk * dpc;
        const int nd = (int)((B - d0) < dpc ? (B - d0) : dpc);
        for (int sl = 0; sl < nslices; ++sl) {
            __syncthreads();  // every warp is done reading the previous slice (and, at sl == 0, done with sc)
            if (tid == 0) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a),
                             "r"((uint32_t)PQS_SLICE_BYTES)
                             : "memory");
                const uint8_t* src = static_cast<const uint8_t*>(lutT) + (int64_t)sl * PQS_SLICE_BYTES;
#pragma unroll
                for (int p = 0; p < 4; ++p)
                    asm volatile(
                        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                            lut_a + p * (PQS_SLICE_BYTES / 4)),
                        "l"(src + p * (PQS_SLICE_BYTES / 4)), "r"((uint32_t)(PQS_SLICE_BYTES / 4)), "r"(bar_a)
                        : "memory");
            }
            mbar_wait(bar_a, phase);
            phase ^= 1;

            const uint64_t pol = sl + 1 < nslices ? pol_keep : pol_drop;
            const int q = (sl * PQS_ROWS) / Nq;
            const bool first = (sl * PQS_ROWS) % Nq == 0;
            for (int dd = warp; dd < nd; dd += PQS_WARPS) {
                const int64_t t0 = offsets[d0 + dd];
                const int n = (int)(offsets[d0 + dd + 1] - t0);
                const uint8_t* cp = codes + (t0 + slot) * PQS_M;
                float part;
                uint4 c = make_uint4(0, 0, 0, 0);
                if (slot < n) c = ldg_codes(cp, pol);
                if constexpr (H16) {
                    float r[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) r[j] = -INFINITY;
                    for (int tb = 0; tb < n; tb += 16) {
                        uint4 cn = make_uint4(0, 0, 0, 0);
                        if (tb + 16 + slot < n) cn = ldg_codes(cp + (int64_t)(tb + 16) * PQS_M, pol);  // prefetch next step
                        float a[8];
#pragma unroll
                        for (int j = 0; j < 8; ++j) a[j] = 0.f;
                        const uint32_t w[4] = {c.x, c.y, c.z, c.w};
#pragma unroll
                        for (int g = 0; g < 4; ++g) {
#pragma unroll
                            for (int s = 0; s < 4; ++s) {
                                const uint32_t code = __byte_perm(w[g], 0u, sel[s]);
                                const uint4 v = lds128u(base[s] + code * 128u + (uint32_t)g * (PQS_K * 128u));
                                add_h2(a[0], a[1], v.x); add_h2(a[2], a[3], v.y);
                                add_h2(a[4], a[5], v.z); add_h2(a[6], a[7], v.w);
                            }
                        }
                        if (tb + slot < n) {
#pragma unroll
                            for (int j = 0; j < 8; ++j) r[j] = fmaxf(r[j], a[j]);
                        }
                        c = cn;
                    }
                    // max over the 16 token slots (lane bits 1..4), then sum of the 16 rows (8 here, 8 in lane ^ 1)
#pragma unroll
                    for (int o = 2; o <= 16; o <<= 1) {
#pragma unroll
                        for (int j = 0; j < 8; ++j) r[j] = fmaxf(r[j], __shfl_xor_sync(0xffffffffu, r[j], o));
                    }
                    part = ((r[0] + r[1]) + (r[2] + r[3])) + ((r[4] + r[5]) + (r[6] + r[7]));
                    part += __shfl_xor_sync(0xffffffffu, part, 1);
                    part *= unscale;  // exact: a power of two
                } else {
                float r0 = -INFINITY, r1 = -INFINITY, r2 = -INFINITY, r3 = -INFINITY;
                for (int tb = 0; tb < n; tb += 16) {
                    uint4 cn = make_uint4(0, 0, 0, 0);
                    if (tb + 16 + slot < n) cn = ldg_codes(cp + (int64_t)(tb + 16) * PQS_M, pol);  // prefetch next step
                    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
                    const uint32_t w[4] = {c.x, c.y, c.z, c.w};
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
#pragma unroll
                        for (int s = 0; s < 4; ++s) {
                            const uint32_t code = __byte_perm(w[g], 0u, sel[s]);
                            const float4 v = lds128(base[s] + code * 128u + (uint32_t)g * (PQS_K * 128u));
                            a0 += v.x; a1 += v.y; a2 += v.z; a3 += v.w;
                        }
                    }
                    if (tb + slot < n) {
                        r0 = fmaxf(r0, a0); r1 = fmaxf(r1, a1); r2 = fmaxf(r2, a2); r3 = fmaxf(r3, a3);
                    }
                    c = cn;
                }
                // max over the 16 token slots (lane bits 1..4), then sum of the 8 rows (4 here, 4 in lane ^ 1)
#pragma unroll
                for (int o = 2; o <= 16; o <<= 1) {
                    r0 = fmaxf(r0, __shfl_xor_sync(0xffffffffu, r0, o));
                    r1 = fmaxf(r1, __shfl_xor_sync(0xffffffffu, r1, o));
                    r2 = fmaxf(r2, __shfl_xor_sync(0xffffffffu, r2, o));
                    r3 = fmaxf(r3, __shfl_xor_sync(0xffffffffu, r3, o));
                }
                part = (r0 + r1) + (r2 + r3);
                part += __shfl_xor_sync(0xffffffffu, part, 1);
                }
                if (lane == 0) {
                    float* dst = sc + q * dpc + dd;
                    *dst = first ? part : (*dst + part);
                }
            }
        }
        __syncthreads();
        for (int idx = tid; idx < Q * nd; idx += PQS_THREADS) {
            const int q = idx / nd, dd = idx - q * nd;
            scores[(int64_t)q * B + d0 + dd] = sc[q * dpc + dd];
        }
    }
}

}  // namespace

int launch_pq_build_lut(const void* queries, int Q, int Nq, int d, tms_dtype q_dtype, const float* codebooks, int M,
                        int K, float* lut, cudaStream_t stream) {
    dim3 grid((unsigned)(Q * Nq), (unsigned)M);
    switch (q_dtype) {
        case TMS_DTYPE_F32:
            pq_build_lut_kernel<float><<<grid, 256, 0, stream>>>(static_cast<const float*>(queries), d, codebooks,
                                                                  M, K, lut);
            break;
        case TMS_DTYPE_F16:
            pq_build_lut_kernel<__half><<<grid, 256, 0, stream>>>(static_cast<const __half*>(queries), d,
                                                                   codebooks, M, K, lut);
            break;
        case TMS_DTYPE_BF16:
            pq_build_lut_kernel<__nv_bfloat16><<<grid, 256, 0, stream>>>(
                static_cast<const __nv_bfloat16*>(queries), d, codebooks, M, K, lut);
            break;
        default: return TMS_ERR_INVALID_ARG;
    }
    count_launch();
    return cudaGetLastError() == cudaSuccess ? TMS_OK : TMS_ERR_CUDA;
}

int launch_pq_simt(const PqArgs& a) {
    const DeviceInfo* di = device_info();
    if (!di) return TMS_ERR_CUDA;
    if (a.B == 0) return TMS_OK;
    const int R = a.Q * a.Nq;
    const size_t smem = sizeof(float) * (size_t)((R + 3) & ~3) + (size_t)SIMT_TOK * a.M;
    if (smem > 200 * 1024) return TMS_ERR_UNSUPPORTED;
    if (smem > 40 * 1024 &&
        cudaFuncSetAttribute(pq_simt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return TMS_ERR_CUDA;
    const int64_t grid = a.B < (int64_t)di->num_sms * 8 ? a.B : (int64_t)di->num_sms * 8;
    pq_simt_kernel<<<(unsigned)grid, SIMT_THREADS, smem, a.stream>>>(a.lut, a.Q, a.Nq, a.M, a.K, a.codes, a.offsets,
                                                                     a.B, a.scores);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? TMS_OK : TMS_ERR_CUDA;
}

bool pq_smem_supports(const PqArgs& a, bool f16) {
    return a.M == PQS_M && a.K == PQS_K && a.Nq % (f16 ? 16 : 8) == 0 && a.Q >= 1 && a.Q <= PQS_MAX_SC_FLOATS / 16;
}

// the re-laid-out table (fp32 entries: as large as lut; fp16 entries: half of it) + a 16-byte header (fp16: max, 1/scale)
size_t pq_smem_workspace_bytes(int Q, int Nq) { return sizeof(float) * (size_t)Q * Nq * PQS_M * PQS_K + 16; }

template <bool H16>
static int launch_pq_smem_t(const PqArgs& a, const void* lutT, const float* inv_scale, const DeviceInfo* di) {
    // docs per chunk: as large as the smem score accumulators allow (amortises the 128 KB slice reloads),
    // but no larger than one CTA's share of a small batch
    int dpc_max = PQS_MAX_SC_FLOATS / a.Q;
    if (dpc_max > 256) dpc_max = 256;
    int64_t dpc = (a.B + di->num_sms - 1) / di->num_sms;
    if (dpc < 16) dpc = 16;
    if (dpc > dpc_max) dpc = dpc_max;
    const int64_t nchunks = (a.B + dpc - 1) / dpc;
    const size_t smem = (size_t)PQS_SLICE_BYTES + sizeof(float) * PQS_MAX_SC_FLOATS + 16;
    if (cudaFuncSetAttribute(pq_smem_kernel<H16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return TMS_ERR_CUDA;
    const int64_t grid = nchunks < di->num_sms ? nchunks : di->num_sms;
    pq_smem_kernel<H16><<<(unsigned)grid, PQS_THREADS, smem, a.stream>>>(lutT, a.Q, a.Nq, a.codes, a.offsets, a.B,
                                                                         (int)dpc, nchunks, a.scores, inv_scale);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? TMS_OK : TMS_ERR_CUDA;
}

// workspace: [16-byte header][the re-laid-out table lutT]
int launch_pq_smem(const PqArgs& a, void* workspace, bool f16) {
    const DeviceInfo* di = device_info();
    if (!di) return TMS_ERR_CUDA;
    if (a.B == 0) return TMS_OK;
    uint32_t* hdr = static_cast<uint32_t*>(workspace);
    void* lutT = static_cast<uint8_t*>(workspace) + 16;
    const int64_t total = (int64_t)a.Q * a.Nq * PQS_M * PQS_K;
    if (f16) {
        if (cudaMemsetAsync(hdr, 0, 16, a.stream) != cudaSuccess) return TMS_ERR_CUDA;
        int64_t nb = (total + 1023) / 1024;
        if (nb > 4 * di->num_sms) nb = 4 * di->num_sms;
        pq_absmax_kernel<<<(unsigned)nb, 256, 0, a.stream>>>(a.lut, total, hdr);
        pq_relayout_f16_kernel<<<(unsigned)((total + 255) / 256), 256, 0, a.stream>>>(a.lut, static_cast<__half*>(lutT),
                                                                                     total, hdr);
        count_launch(2);
        if (cudaGetLastError() != cudaSuccess) return TMS_ERR_CUDA;
        return launch_pq_smem_t<true>(a, lutT, reinterpret_cast<const float*>(hdr + 1), di);
    }
    pq_relayout_kernel<<<(unsigned)((total + 255) / 256), 256, 0, a.stream>>>(a.lut, static_cast<float*>(lutT), total);
    count_launch();
    if (cudaGetLastError() != cudaSuccess) return TMS_ERR_CUDA;
    return launch_pq_smem_t<false>(a, lutT, nullptr, di);
}

}  // namespace tms
