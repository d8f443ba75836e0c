// dense_tc.cu -- fused multi-query MaxSim on sm_100a: TMA-fed, tcgen05 tensor cores, TMEM accumulators
// (TMS_VARIANT_TCGEN05).  Rebuilds the paper's V2-MQ kernel (Alg. 3) and its dimension-tiled
// form for Blackwell; the Triton/H100 tiling of the paper is prior art, not the blueprint.
//
// Persistent kernel, one CTA per SM.  Each CTA owns a contiguous, token-balanced range of documents cut at
// document boundaries (no cross-CTA merge, no atomics: the paper's atomic_add of Alg. 3 line 10 is gone).
//
//   A operand  Qmat[rows, d]: all Q queries x Nq tokens (Nq padded to a power of two), resident in shared
//              memory for the whole kernel, K-major, 128-byte swizzle       ("Load Q_tile once", Alg. 3 line 3)
//   B operand  128 packed document tokens x (1 or 2) 128-byte dimension blocks per pipeline stage, brought by
//              TMA exactly once from HBM                                                   (Alg. 3 line 6; Eq. 7)
//   D          S = Qmat . D_tile^T in TMEM, fp32, one 128-lane x 128-column block per 128 query rows; for
//              d*sizeof > one stage the MMAs of successive dimension chunks accumulate into the same TMEM
//              block and the max is taken once after the last chunk
//   epilogue   tcgen05.ld -> registers; running max per query row, segmented by document with a carry across
//              tiles (Alg. 3 line 8); at a document's last token the Nq maxima are summed with warp shuffles
//              and ONE fp32 is stored to scores[q, b]                                        (Eq. 1)
//
// Warp roles (blockDim = 128 + 128*MB): warp 0 TMA producer, warp 1 MMA issuer + TMEM owner, warp 2 document
// segmenter (turns `offsets` into per-tile boundary masks, writes -inf for empty documents), warp 3 idle,
// warps 4.. epilogue (warp w reads TMEM lanes 32*(w%4)..+31 of M-block (w-4)/4).
#include <cuda.h>
#include <cstdlib>
#include <cuda_runtime.h>

#include "tms_internal.h"

namespace tms {
namespace {

constexpr int BN = 128;            // document tokens per tile (= UMMA N)
constexpr int KB_BYTES = 128;      // one dimension block: 128 bytes of a row (64 x 16-bit or 32 x fp32)
constexpr int KB_TILE_BYTES = BN * KB_BYTES;  // 16 KB: one dimension block of one document tile
constexpr int A_BLOCK_BYTES = 128 * KB_BYTES; // 16 KB: one dimension block of one 128-row query block
constexpr int NSEG = 4;            // depth of the segment-info ring
constexpr int MAX_STAGES = 12;
constexpr int TMEM_COLS = 512;
constexpr uint32_t SMEM_LIMIT = 232448;  // 227 KB

struct Params {
    const int64_t* offsets;
    float* scores;
    int64_t B, T;
    int Q, Nq, Nq_pad;
    int MB;        // 128-row query blocks (1 or 2)
    int NKB;       // dimension blocks per row = d*sizeof/128
    int KBS;       // dimension blocks per pipeline stage
    int NS;        // pipeline stages
    int NT;        // TMEM accumulator stages = 512 / (MB*128)
    uint32_t idesc;
    int kb_elems;  // elements per dimension block (64 or 32)
    int debug;     // TMS_DEBUG bits (measurement probes only): 1 skip epilogue math, 2 skip MMAs
};

// ---- PTX wrappers ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
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
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1,
                                            uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4}], [%2], %5;" ::"r"(dst),
        "l"(map), "r"(bar), "r"(c0), "r"(c1), "l"(policy)
        : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] . B[smem]^T, kind::f16 (fp16/bf16 in, fp32 accumulate) or kind::tf32
template <bool TF32>
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                       uint32_t accumulate) {
    if constexpr (TF32) {
        asm volatile(
            "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
            "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}\n" ::"r"(d_tmem),
            "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
            : "memory");
    } else {
        asm volatile(
            "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}\n" ::"r"(d_tmem),
            "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
            : "memory");
    }
}
// 32 lanes x 32 consecutive fp32 columns -> 32 registers per thread (lane l of the warp gets TMEM lane base+l)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float* v) {
    uint32_t* r = reinterpret_cast<uint32_t*>(v);
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// K-major, 128-byte-swizzled operand tile: rows of 128 bytes, 8-row groups 1024 bytes apart (SBO),
// descriptor version 1 (sm_100), layout type 2 (SWIZZLE_128B).  LBO is unused for this layout.
__device__ __forceinline__ uint64_t umma_desc(uint32_t smem_addr) {
    return (uint64_t)((smem_addr & 0x3FFFFu) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) |
           (2ull << 61);
}

// smallest b in [0, B] with offsets[b] >= target; whole warp, 32 probes per round
__device__ int64_t warp_lower_bound(const int64_t* __restrict__ offsets, int64_t B, int64_t target, int lane) {
    int64_t lo = 0, hi = B;  // the answer lies in [lo, hi]; offsets[B] = T >= target always holds
    while (hi - lo > 32) {
        const int64_t n = hi - lo;
        const int64_t p = lo + (n * (lane + 1)) / 33;  // lo <= p < hi, increasing in lane
        const bool ge = offsets[p] >= target;
        const unsigned ball = __ballot_sync(0xffffffffu, ge);
        const int f = ball ? __ffs(ball) - 1 : 32;
        const int64_t p_f = __shfl_sync(0xffffffffu, p, f & 31);
        const int64_t p_fm1 = __shfl_sync(0xffffffffu, p, (f - 1) & 31);
        if (f < 32) hi = p_f;
        if (f > 0) lo = p_fm1 + 1;
    }
    const int64_t p = lo + lane;
    const bool ge = (p < hi) && (offsets[p] >= target);
    const unsigned ball = __ballot_sync(0xffffffffu, ge);
    return ball ? lo + (__ffs(ball) - 1) : hi;
}

struct SegInfo {
    uint32_t mask[4];     // bit c set: column c of the tile is the last token of a (non-empty) document
    uint32_t pad[4];
    uint32_t doc[BN];     // k-th set bit  ->  document index relative to the CTA's first document
};

// ---- epilogue helpers ------------------------------------------------------------------------------------------
// flags: bits 0-7 Nq_pad (a power of two <= 32), bit 8 row holds a real query token, bit 9 row writes the score.

// max -> sum (Eq. 1): the Nq running maxima of one query sit in Nq adjacent lanes; they are summed in a fixed
// xor-shuffle order and the lane of query token 0 stores the score of the k-th document that ends in this tile.
__device__ __forceinline__ void flush_inline(float m, uint32_t k, uint32_t flags, const uint32_t* doc, float* out) {
    const uint32_t nqp = flags & 0xffu;
    float v = (flags & 0x100u) ? m : 0.f;
    if (nqp > 16) v += __shfl_xor_sync(0xffffffffu, v, 16);
    if (nqp > 8) v += __shfl_xor_sync(0xffffffffu, v, 8);
    if (nqp > 4) v += __shfl_xor_sync(0xffffffffu, v, 4);
    if (nqp > 2) v += __shfl_xor_sync(0xffffffffu, v, 2);
    if (nqp > 1) v += __shfl_xor_sync(0xffffffffu, v, 1);
    if (flags & 0x200u) out[doc[k]] = v;
}
__device__ __noinline__ void epi_flush(float m, uint32_t k, uint32_t flags, const uint32_t* doc, float* out) {
    flush_inline(m, k, flags, doc, out);
}

// max of 32 accumulator columns and the running max, three inputs per FMNMX3
__device__ __forceinline__ float max_tree32(float m, const float* x) {
    float a[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = fmaxf(fmaxf(x[4 * j], x[4 * j + 1]), fmaxf(x[4 * j + 2], x[4 * j + 3]));
    const float b0 = fmaxf(fmaxf(a[0], a[1]), a[2]), b1 = fmaxf(fmaxf(a[3], a[4]), a[5]);
    return fmaxf(fmaxf(m, b0), fmaxf(fmaxf(b1, a[6]), a[7]));
}

// 32 accumulator columns in which at least one document ends (bit c of `bits`: column c is a document's last token).
// Out of line and re-reading its columns from TMEM on purpose: boundary words are the minority, and one compact copy
// of this code keeps the epilogue's hot loop inside the instruction cache.  One iteration per document end: the
// segment's columns are selected by predicate, folded into the running max, and the document is flushed.
__device__ __noinline__ uint2 epi_boundary_word(uint32_t taddr, uint32_t bits, float m, uint32_t k, uint32_t flags,
                                                const uint32_t* doc, float* out) {
    float x[32];
    tmem_ld32(taddr, x);
    tmem_ld_wait();
    uint32_t done = 0;  // columns that belong to documents already flushed
    while (bits) {
        const uint32_t low = bits & (0u - bits);
        const uint32_t seg = ((low << 1) - 1u) & ~done;
        float a0 = m, a1 = -INFINITY;
#pragma unroll
        for (int c = 0; c < 32; c += 2) {
            a0 = fmaxf(a0, (seg >> c) & 1u ? x[c] : -INFINITY);
            a1 = fmaxf(a1, (seg >> (c + 1)) & 1u ? x[c + 1] : -INFINITY);
        }
        flush_inline(fmaxf(a0, a1), k, flags, doc, out);
        ++k;
        m = -INFINITY;
        done |= seg;
        bits ^= low;
    }
    float a0 = m, a1 = -INFINITY;
#pragma unroll
    for (int c = 0; c < 32; c += 2) {
        a0 = fmaxf(a0, (done >> c) & 1u ? -INFINITY : x[c]);
        a1 = fmaxf(a1, (done >> (c + 1)) & 1u ? -INFINITY : x[c + 1]);
    }
    return make_uint2(__float_as_uint(fmaxf(a0, a1)), k);
}

template <bool TF32, int MB, int KBS>
__global__ void __launch_bounds__(128 + 128 * MB, 1)
dense_tc_kernel(const __grid_constant__ CUtensorMap map_docs, const __grid_constant__ CUtensorMap map_q,
                const Params p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    // 128-byte-swizzled operand tiles need 1024-byte alignment in the shared window
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    // layout: [A: MB*NKB*16 KB] [stages: NS * KBS*16 KB] [SegInfo x NSEG] [barriers] [misc]
    const uint32_t a_bytes = (uint32_t)MB * p.NKB * A_BLOCK_BYTES;
    const uint32_t stage_bytes = (uint32_t)KBS * KB_TILE_BYTES;
    uint8_t* a_ptr = smem;
    uint8_t* st_ptr = smem + a_bytes;
    SegInfo* seg = reinterpret_cast<SegInfo*>(st_ptr + (size_t)p.NS * stage_bytes);
    uint64_t* bars = reinterpret_cast<uint64_t*>(seg + NSEG);
    // barrier indices
    uint64_t* full = bars;                       // [NS]
    uint64_t* empty = full + MAX_STAGES;         // [NS]
    uint64_t* tfull = empty + MAX_STAGES;        // [4]
    uint64_t* tempty = tfull + 4;                // [4]
    uint64_t* sfull = tempty + 4;                // [NSEG]
    uint64_t* sempty = sfull + NSEG;             // [NSEG]
    uint64_t* qfull = sempty + NSEG;             // [1]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(qfull + 1);
    int64_t* range = reinterpret_cast<int64_t*>(qfull + 2);  // b_lo, b_hi, t_lo, t_hi

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_epi_warps = 4 * MB;

    // ---- one-time setup ------------------------------------------------------------------------------------
    if (warp == 0) {
        if (lane == 0) {
            for (int s = 0; s < p.NS; ++s) { mbar_init(smem_u32(full + s), 1); mbar_init(smem_u32(empty + s), 1); }
            for (int s = 0; s < 4; ++s) { mbar_init(smem_u32(tfull + s), 1); mbar_init(smem_u32(tempty + s), n_epi_warps); }
            for (int s = 0; s < NSEG; ++s) { mbar_init(smem_u32(sfull + s), 1); mbar_init(smem_u32(sempty + s), n_epi_warps); }
            mbar_init(smem_u32(qfull), 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(&map_docs) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(&map_q) : "memory");
        }
        // work partition (a3): documents [b_lo, b_hi) whose first tokens lie in [c*T/G, (c+1)*T/G)
        const int64_t G = gridDim.x, c = blockIdx.x;
        const int64_t tgt_lo = (c * p.T) / G, tgt_hi = ((c + 1) * p.T) / G;
        const int64_t b_lo = (c == 0) ? 0 : warp_lower_bound(p.offsets, p.B, tgt_lo, lane);
        const int64_t b_hi = (c == G - 1) ? p.B : warp_lower_bound(p.offsets, p.B, tgt_hi, lane);
        if (lane == 0) {
            range[0] = b_lo;
            range[1] = b_hi;
            range[2] = p.offsets[b_lo];
            range[3] = p.offsets[b_hi];
        }
    } else if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                     "r"((uint32_t)TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    } else {
        // zero the A operand so rows that no query owns are finite (they never reach a score)
        const int nthr = blockDim.x - 64;
        uint4* a4 = reinterpret_cast<uint4*>(a_ptr);
        for (uint32_t i = threadIdx.x - 64; i < a_bytes / 16; i += nthr) a4[i] = make_uint4(0, 0, 0, 0);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy zeros before TMA writes
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    const uint32_t tmem_base = *tmem_slot;
    const int64_t b_lo = range[0], b_hi = range[1], t_lo = range[2], t_hi = range[3];
    const int64_t ntiles = (t_hi - t_lo + BN - 1) / BN;
    const int nchunks = p.NKB / KBS;  // pipeline stages consumed per tile

    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            const uint64_t pol_docs = policy_evict_first();  // streamed once
            const uint64_t pol_q = policy_evict_last();      // every CTA reads the same queries
            // queries: one box of Nq rows x 128 bytes per (query, dimension block)
            mbar_expect_tx(smem_u32(qfull), (uint32_t)p.Q * p.Nq * KB_BYTES * p.NKB);
            for (int q = 0; q < p.Q; ++q) {
                const int row0 = q * p.Nq_pad;
                const int mb = row0 >> 7, r = row0 & 127;
                for (int kb = 0; kb < p.NKB; ++kb)
                    tma_load_2d(smem_u32(a_ptr + (size_t)(mb * p.NKB + kb) * A_BLOCK_BYTES + r * KB_BYTES), &map_q,
                                smem_u32(qfull), kb * p.kb_elems, q * p.Nq, pol_q);
            }
            uint32_t s = 0, ph = 0;  // ring slot and its phase bit
            for (int64_t t = 0; t < ntiles; ++t) {
                const int tok = (int)(t_lo + t * BN);
                for (int ch = 0; ch < nchunks; ++ch) {
                    mbar_wait(smem_u32(empty + s), ph ^ 1);
                    mbar_expect_tx(smem_u32(full + s), stage_bytes);
                    for (int k = 0; k < KBS; ++k)
                        tma_load_2d(smem_u32(st_ptr + (size_t)s * stage_bytes + k * KB_TILE_BYTES), &map_docs,
                                    smem_u32(full + s), (ch * KBS + k) * p.kb_elems, tok, pol_docs);
                    if (++s == (uint32_t)p.NS) { s = 0; ph ^= 1; }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        // ===== MMA issuer =====
        // One thread issues every tcgen05.mma of the CTA, so its instruction stream must stay short: the loops
        // over K steps and query blocks are compile-time, and a descriptor is the previous one plus a constant.
        if (lane == 0) {
            mbar_wait(smem_u32(qfull), 0);
            tc_fence_after();
            constexpr uint32_t DESC_HI = (1024u >> 4) | (1u << 14) | (2u << 29);  // SBO 1024 B, version 1, SWIZZLE_128B
            constexpr uint32_t DESC_LO = 1u << 16;                                // LBO field (unused for this layout)
            const uint32_t a_lo0 = ((smem_u32(a_ptr) & 0x3FFFFu) >> 4) | DESC_LO;
            const uint32_t a_mb_step = (uint32_t)p.NKB * (A_BLOCK_BYTES >> 4);    // next 128-row query block
            const uint32_t b_lo0 = ((smem_u32(st_ptr) & 0x3FFFFu) >> 4) | DESC_LO;
            const uint32_t stage_step = stage_bytes >> 4;
            const uint32_t idesc = p.idesc;
            const bool skip = (p.debug & 2) != 0;
            uint32_t s = 0, ph = 0, ts = 0, tph = 0;
            for (int64_t t = 0; t < ntiles; ++t) {
                mbar_wait(smem_u32(tempty + ts), tph ^ 1);  // epilogue has drained this accumulator stage
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + ts * (uint32_t)(MB * BN);
                uint32_t a_lo = a_lo0;
                for (int ch = 0; ch < nchunks; ++ch) {
                    mbar_wait(smem_u32(full + s), ph);
                    tc_fence_after();
                    const uint32_t b_lo = b_lo0 + s * stage_step;
                    if (!skip) {
#pragma unroll
                        for (int k = 0; k < KBS; ++k) {
#pragma unroll
                            for (int kk = 0; kk < 4; ++kk) {  // four 32-byte K steps per 128-byte dimension block
                                const uint64_t bd = ((uint64_t)DESC_HI << 32) | (b_lo + k * (KB_TILE_BYTES >> 4) + kk * 2);
#pragma unroll
                                for (int mb = 0; mb < MB; ++mb) {
                                    const uint64_t ad = ((uint64_t)DESC_HI << 32) |
                                                        (a_lo + mb * a_mb_step + k * (A_BLOCK_BYTES >> 4) + kk * 2);
                                    if (k == 0 && kk == 0)
                                        tc_mma<TF32>(d_tmem + mb * BN, ad, bd, idesc, ch != 0);
                                    else
                                        tc_mma<TF32>(d_tmem + mb * BN, ad, bd, idesc, 1u);
                                }
                            }
                        }
                    }
                    a_lo += KBS * (A_BLOCK_BYTES >> 4);
                    tc_commit(smem_u32(empty + s));  // frees the smem stage once these MMAs have read it
                    if (++s == (uint32_t)p.NS) { s = 0; ph ^= 1; }
                }
                tc_commit(smem_u32(tfull + ts));     // accumulator stage complete -> epilogue
                if (++ts == (uint32_t)p.NT) { ts = 0; tph ^= 1; }
            }
        }
        __syncwarp();
    } else if (warp == 2) {
        // ===== document segmenter =====
        // Lane l holds the end offset of document wb + l (a 32-document window in registers); the next window is
        // loaded one window ahead, so no tile waits on a global load.  A document's start is its predecessor's end.
        const uint32_t lt_mask = (1u << lane) - 1u;
        const float ninf = -INFINITY;
        const int64_t never = INT64_MAX;
        auto load_ends = [&](int64_t base) -> int64_t {
            const int64_t idx = base + lane;
            return idx < b_hi ? p.offsets[idx + 1] : never;
        };
        int64_t wb = b_lo;
        int64_t e_cur = load_ends(wb), e_nxt = load_ends(wb + 32);
        int64_t s_first = t_lo;  // start of document wb
        int consumed = 0;        // documents of the current window already assigned to a tile
        for (int64_t t = 0; t < ntiles; ++t) {
            const uint32_t g = (uint32_t)(t % NSEG), gph = (uint32_t)((t / NSEG) & 1);
            const int64_t tile_start = t_lo + t * BN, tile_end = tile_start + BN;
            mbar_wait(smem_u32(sempty + g), gph ^ 1);
            uint32_t m0 = 0, m1 = 0, m2 = 0, m3 = 0, nseg = 0;
            while (true) {
                const int64_t idx = wb + lane;
                const int64_t e = e_cur;
                const int64_t e_prev = __shfl_up_sync(0xffffffffu, e_cur, 1);
                const int64_t s = lane == 0 ? s_first : e_prev;
                const bool in_tile = lane >= consumed && e <= tile_end;  // ends are monotone: a run of lanes
                const unsigned ball = __ballot_sync(0xffffffffu, in_tile);
                const bool nonempty = in_tile && e > s;
                const unsigned nb = __ballot_sync(0xffffffffu, nonempty);
                uint32_t w0 = 0, w1 = 0, w2 = 0, w3 = 0;
                if (nonempty) {
                    const uint32_t col = (uint32_t)(e - 1 - tile_start);
                    seg[g].doc[nseg + __popc(nb & lt_mask)] = (uint32_t)(idx - b_lo);
                    const uint32_t bit = 1u << (col & 31);
                    w0 = (col >> 5) == 0 ? bit : 0; w1 = (col >> 5) == 1 ? bit : 0;
                    w2 = (col >> 5) == 2 ? bit : 0; w3 = (col >> 5) == 3 ? bit : 0;
                } else if (in_tile) {
                    for (int q = 0; q < p.Q; ++q) p.scores[(int64_t)q * p.B + idx] = ninf;  // empty document (A2)
                }
                if (nb) {
                    m0 |= __reduce_or_sync(0xffffffffu, w0); m1 |= __reduce_or_sync(0xffffffffu, w1);
                    m2 |= __reduce_or_sync(0xffffffffu, w2); m3 |= __reduce_or_sync(0xffffffffu, w3);
                }
                nseg += __popc(nb);
                consumed += __popc(ball);
                if (consumed < 32) break;
                s_first = __shfl_sync(0xffffffffu, e_cur, 31);  // window exhausted: slide to the prefetched one
                wb += 32;
                e_cur = e_nxt;
                e_nxt = load_ends(wb + 32);
                consumed = 0;
            }
            if (lane == 0) { seg[g].mask[0] = m0; seg[g].mask[1] = m1; seg[g].mask[2] = m2; seg[g].mask[3] = m3; }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(sfull + g));
        }
        // documents after the last token of the range can only be empty
        for (int64_t idx = wb + consumed + lane; idx < b_hi; idx += 32)
            for (int q = 0; q < p.Q; ++q) p.scores[(int64_t)q * p.B + idx] = ninf;
    } else if (warp >= 4) {
        // ===== epilogue: running rowmax, segmented by document; max -> sum =====
        const int ew = warp - 4, mb = ew >> 2, quad = warp & 3;
        const int row = mb * 128 + quad * 32 + lane;
        const int q = row / p.Nq_pad, i = row - q * p.Nq_pad;
        const bool row_valid = (q < p.Q) && (i < p.Nq);
        const bool writer = row_valid && (i == 0);
        float* out = p.scores + (int64_t)(q < p.Q ? q : 0) * p.B + b_lo;
        const uint32_t flags = (uint32_t)p.Nq_pad | (row_valid ? 0x100u : 0u) | (writer ? 0x200u : 0u);
        float m = -INFINITY;  // Alg. 3 line 4

        const uint32_t nt = (uint32_t)p.NT, tstride = (uint32_t)(MB * BN);
        const uint32_t taddr0 = tmem_base + ((uint32_t)(quad * 32) << 16) + mb * BN;
        uint32_t ts = 0, tph = 0, g = 0, gph = 0;
        for (int64_t t = 0; t < ntiles; ++t) {
            mbar_wait(smem_u32(tfull + ts), tph);
            tc_fence_after();
            const uint32_t taddr = taddr0 + ts * tstride;
            float v[BN];
            tmem_ld32(taddr + 0, v + 0);
            tmem_ld32(taddr + 32, v + 32);
            tmem_ld32(taddr + 64, v + 64);
            tmem_ld32(taddr + 96, v + 96);
            mbar_wait(smem_u32(sfull + g), gph);
            const uint4 mask = *reinterpret_cast<const uint4*>(seg[g].mask);
            tmem_ld_wait();
            uint32_t k = 0;
            const uint32_t mw[4] = {mask.x, mask.y, mask.z, mask.w};
#pragma unroll
            for (int c4 = 0; c4 < 4; ++c4) {
                const uint32_t bits = (p.debug & 1) ? 0u : mw[c4];
                if (p.debug & 1) {
                    m = fmaxf(m, v[c4 * 32]);
                } else if (bits == 0) {  // no document ends inside these 32 columns
                    m = max_tree32(m, v + c4 * 32);
                } else if (bits == 0x80000000u) {  // exactly one document ends, at the last of the 32 columns
                    epi_flush(max_tree32(m, v + c4 * 32), k, flags, seg[g].doc, out);
                    ++k;
                    m = -INFINITY;
                } else {
                    const uint2 r = epi_boundary_word(taddr + c4 * 32, bits, m, k, flags, seg[g].doc, out);
                    m = __uint_as_float(r.x);
                    k = r.y;
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(tempty + ts));  // accumulator stage is free again
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(sempty + g));
            if (++ts == nt) { ts = 0; tph ^= 1; }
            if (++g == NSEG) { g = 0; gph ^= 1; }
        }
    }

    // ---- teardown --------------------------------------------------------------------------------------------
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"((uint32_t)TMEM_COLS)
                     : "memory");
    }
}

// ---- host side -----------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* ptr = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(ptr);
    }
    return fn;
}

bool make_map_2d(CUtensorMap* map, tms_dtype dtype, const void* base, uint64_t rows, uint64_t cols, uint32_t box_cols,
                 uint32_t box_rows) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return false;
    const CUtensorMapDataType dt = dtype == TMS_DTYPE_F32   ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                                   : dtype == TMS_DTYPE_F16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16
                                                            : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
    const cuuint64_t dims[2] = {cols, rows};
    const cuuint64_t strides[1] = {cols * dtype_size(dtype)};
    const cuuint32_t box[2] = {box_cols, box_rows};
    const cuuint32_t estr[2] = {1, 1};
    return fn(map, dt, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int next_pow2(int v) {
    int p = 1;
    while (p < v) p <<= 1;
    return p;
}

// Shape -> kernel parameters; false when the tcgen05 path does not cover it.
bool plan(const DenseArgs& a, Params& p, uint32_t& smem_bytes) {
    if (a.B <= 0 || a.T <= 0 || a.T >= (1ll << 31) - BN) return false;
    if (a.dtype == TMS_DTYPE_F32) return false;  // fp32 inputs: plain TF32 would break the 1e-5*Nq tolerance
    const int esize = (int)dtype_size(a.dtype);
    if ((a.d * esize) % KB_BYTES != 0) return false;
    const int nqp = next_pow2(a.Nq);
    if (nqp > 32) return false;
    const int nqp8 = nqp < 8 ? 8 : nqp;  // query blocks start on 8-row (1024-byte) swizzle-atom boundaries
    const int rows = a.Q * nqp8;
    if (rows > 256) return false;
    p.offsets = a.offsets;
    p.scores = a.scores;
    p.B = a.B;
    p.T = a.T;
    p.Q = a.Q;
    p.Nq = a.Nq;
    p.Nq_pad = nqp8;
    p.MB = (rows + 127) / 128;
    p.NKB = a.d * esize / KB_BYTES;
    p.kb_elems = KB_BYTES / esize;
    p.NT = TMEM_COLS / (p.MB * BN);
    {
        const char* dbg = getenv("TMS_DEBUG");
        p.debug = dbg ? atoi(dbg) : 0;
    }
    p.KBS = (p.NKB % 2 == 0) ? 2 : 1;
    const uint32_t fmt = a.dtype == TMS_DTYPE_BF16 ? 1u : (a.dtype == TMS_DTYPE_F16 ? 0u : 2u);
    // instruction descriptor: fp32 accumulate, A/B format, both K-major, N = 128, M = 128
    p.idesc = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    const uint32_t a_bytes = (uint32_t)p.MB * p.NKB * A_BLOCK_BYTES;
    const uint32_t fixed = sizeof(SegInfo) * NSEG + 8 * (2 * MAX_STAGES + 8 + 2 * NSEG + 2) + 4 * 8 + 1024;
    if (a_bytes + fixed + 2u * KB_TILE_BYTES > SMEM_LIMIT) return false;
    uint32_t stage_bytes = (uint32_t)p.KBS * KB_TILE_BYTES;
    int ns = (int)((SMEM_LIMIT - a_bytes - fixed) / stage_bytes);
    if (ns < 3 && p.KBS == 2) {  // fall back to 16 KB stages when the resident queries leave little room
        p.KBS = 1;
        stage_bytes = KB_TILE_BYTES;
        ns = (int)((SMEM_LIMIT - a_bytes - fixed) / stage_bytes);
    }
    if (ns < 2) return false;
    p.NS = ns > MAX_STAGES ? MAX_STAGES : ns;
    smem_bytes = a_bytes + (uint32_t)p.NS * stage_bytes + fixed;
    return true;
}

}  // namespace

bool dense_tc_supports(const DenseArgs& a) {
    const DeviceInfo* di = device_info();
    if (!di || di->cc_major != 10) return false;
    Params p;
    uint32_t smem;
    return plan(a, p, smem) && smem <= (uint32_t)di->max_smem_optin;
}

int launch_dense_tc(const DenseArgs& a) {
    const DeviceInfo* di = device_info();
    if (!di) return TMS_ERR_CUDA;
    Params p;
    uint32_t smem = 0;
    if (di->cc_major != 10 || !plan(a, p, smem) || smem > (uint32_t)di->max_smem_optin) return TMS_ERR_UNSUPPORTED;

    CUtensorMap map_docs, map_q;
    if (!make_map_2d(&map_docs, a.dtype, a.docs, (uint64_t)a.T, (uint64_t)a.d, (uint32_t)p.kb_elems, BN))
        return TMS_ERR_CUDA;
    if (!make_map_2d(&map_q, a.dtype, a.queries, (uint64_t)a.Q * a.Nq, (uint64_t)a.d, (uint32_t)p.kb_elems,
                     (uint32_t)a.Nq))
        return TMS_ERR_CUDA;

    void (*kern)(const CUtensorMap, const CUtensorMap, const Params) = nullptr;
    if (p.MB == 1) kern = p.KBS == 1 ? dense_tc_kernel<false, 1, 1> : dense_tc_kernel<false, 1, 2>;
    else kern = p.KBS == 1 ? dense_tc_kernel<false, 2, 1> : dense_tc_kernel<false, 2, 2>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return TMS_ERR_CUDA;
    // no more CTAs than 128-token tiles; one CTA per SM
    int64_t grid = (a.T + BN - 1) / BN;
    if (grid > di->num_sms) grid = di->num_sms;
    kern<<<(unsigned)grid, 128 + 128 * p.MB, smem, a.stream>>>(map_docs, map_q, p);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? TMS_OK : TMS_ERR_CUDA;
}

}  // namespace tms
