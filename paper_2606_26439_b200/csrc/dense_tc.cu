// dense_tc.cu -- fused multi-query MaxSim on sm_100a: TMA-fed, tcgen05 tensor cores, TMEM operands and
// accumulators (TMS_VARIANT_TCGEN05).  Rebuilds the paper's V2-MQ kernel (Alg. 3) and its
// dimension-tiled form for Blackwell; the Triton/H100 tiling of the paper is prior art, not the blueprint.
//
// Persistent kernel, one CTA per SM.  Each CTA owns a contiguous, token-balanced range of documents cut at
// document boundaries (no cross-CTA merge, no atomics: the paper's atomic_add of Alg. 3 line 10 is gone).
//
//   A operand  Qmat[rows, d]: up to 256 query rows (Q queries x Nq tokens, Nq padded to a power of two) resident
//              in TENSOR MEMORY for the whole kernel ("Load Q_tile once", Alg. 3 line 3).  Each epilogue thread
//              owns one row and writes it with tcgen05.st; shared memory then only carries document tiles, so
//              the tensor pipe reads half the shared-memory bytes an SS-mode MMA would.
//   B operand  128 packed document tokens x (1 or 2) 128-byte dimension blocks per pipeline stage, brought by
//              TMA exactly once from HBM, 128-byte swizzle                              (Alg. 3 line 6; Eq. 7)
//   D          S = Qmat . D_tile^T in TMEM, fp32, one 128-lane x 128-column accumulator per 128 query rows, in
//              a ring of accumulators.  For d*sizeof > one stage the MMAs of successive dimension chunks
//              accumulate into the same accumulator; the max is taken once after the last chunk
//   epilogue   tcgen05.ld of 32 accumulator columns per thread at a time (pipelined against the reduction when two
//              epilogue warps share a scheduler) -> running max per query row, segmented by document with a carry
//              across tiles (Alg. 3 line 8).  At a document's last token each row parks its maximum in a small
//              per-warp shared-memory buffer; when 16 documents are parked the warp adds the Nq maxima of each
//              query in a fixed order and stores 16 scores                                           (Eq. 1)
//
// Warp roles (blockDim = 128 + 128*MB, + 128 for the split paths): warp 0 TMA producer, warp 1 MMA issuer + TMEM
// owner, warp 2 document segmenter (turns `offsets` into per-tile boundary masks, writes -inf for empty documents),
// warp 3 idle, warps 4.. epilogue (warp w reads TMEM lanes 32*(w%4)..+31 of query block (w-4)/4), and for fp32 inputs
// / PQ codes four more warps that turn what TMA lands into bf16 hi/lo operand stages (see the kernel's comment).
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <cuda_runtime.h>

#include "tms_internal.h"

namespace tms {
namespace {

constexpr int BN = 128;            // document tokens per tile (= UMMA N) = columns of one accumulator
constexpr int KB_BYTES = 128;      // one dimension block: 128 bytes of a row (64 x 16-bit)
constexpr int KB_WORDS = 32;       // ... = 32 TMEM columns of the A operand
constexpr int KB_TILE_BYTES = BN * KB_BYTES;  // 16 KB: one dimension block of one document tile
constexpr int NSEG = 4;            // depth of the segment-info ring
constexpr int MAX_STAGES = 14;
constexpr int MAX_ACC = 4;
constexpr int MAX_RAW = 4;
constexpr int TMEM_COLS = 512;
constexpr int PEND = 16;           // documents parked per epilogue warp before their scores are summed and stored
constexpr int PEND_PITCH = 36;     // floats per parked document: 32 rows, padded so that 16-byte row reads of 8
                                   // consecutive documents fall into different banks
constexpr uint32_t SMEM_LIMIT = 232448;  // 227 KB

struct Params {
    const void* queries;   // this launch's first query
    const int64_t* offsets;
    float* scores;         // this launch's first score row
    int64_t B, T;
    // Stores of 2^31 tokens or more (TMA coordinates are 32-bit) are scored in token segments, one launch each: this
    // launch takes the documents whose FIRST token lies in [tok0, tok0 + Tseg); its tensor map starts at token tok0.
    int64_t tok0, Tseg;
    int seg_first, seg_last;  // the first segment owns leading empty documents, the last one trailing ones
    int Q, Nq, Nq_pad;     // queries in this launch
    int row_bytes;         // d * sizeof(element)
    int NKB;               // dimension blocks per row = row_bytes / 128
    int NS;                // pipeline (operand) stages
    int NR;                // fp32 inputs: raw fp32 stages that TMA fills and the splitter warps drain
    int NACC;              // accumulators in the TMEM ring
    int acc_col0;          // first TMEM column of the ring (the A operand sits in columns [0, MB*NKB*32))
    uint32_t idesc;
    int kb_elems;          // elements per dimension block (64)
    // PQD (decode-and-contract PQ variant): the store is uint8 codes[T,16] + fp32 codebooks[16,256,8]
    const uint8_t* codes;
    const float* codebooks;
    int q_fmt;             // element type of the query rows: 0 fp32, 1 fp16, 2 bf16 (fp32-split paths only)
    int skip_alo;          // the queries' lo halves are all zero (bf16 queries): leave out the a_lo * b_hi MMAs
    int half_mode;         // PQD, TMS_PQ_FP16: queries and centroids rounded to fp16, one MMA per product (no lo parts)
#ifdef TMS_PROBES
    const void* docs_raw;
    int debug;             // probe builds only (-DTMS_PROBES, never set by build.py): TMS_DEBUG bits 1 skip epilogue
                           // math, 2 skip MMAs, 4 skip TMEM reads.  The product library has none of this.
#endif
};

// Measurement probes exist only in builds made with -DTMS_PROBES (a separate library for experiments; build.py never
// sets it): skip switches read from the environment, and a per-role clock trace of one CTA.
#ifdef TMS_PROBES
#define PROBE(p, bit) (((p).debug & (bit)) != 0)
constexpr int TRACE_NT = 64, TRACE_T0 = 200, TRACE_CTA = 5, TRACE_EV = 8, TRACE_ROLES = 4;
__device__ long long g_trace[TRACE_ROLES * TRACE_NT * TRACE_EV];
#define TRACE(role, t, ev)                                                                                    \
    do {                                                                                                      \
        if (blockIdx.x == TRACE_CTA && lane == 0 && (t) >= TRACE_T0 && (t) < TRACE_T0 + TRACE_NT)             \
            g_trace[((role) * TRACE_NT + (int)((t) - TRACE_T0)) * TRACE_EV + (ev)] = clock64();               \
    } while (0)
// same from a region only one thread executes
#define TRACE1(role, t, ev)                                                                                   \
    do {                                                                                                      \
        if (blockIdx.x == TRACE_CTA && (t) >= TRACE_T0 && (t) < TRACE_T0 + TRACE_NT)                          \
            g_trace[((role) * TRACE_NT + (int)((t) - TRACE_T0)) * TRACE_EV + (ev)] = clock64();               \
    } while (0)
#ifdef TMS_TRACE_DETAIL
#define TRACED(role, t, ev) TRACE(role, t, ev)
#else
#define TRACED(role, t, ev) do { } while (0)
#endif
#else
#define PROBE(p, bit) false
#define TRACE(role, t, ev) do { } while (0)
#define TRACE1(role, t, ev) do { } while (0)
#define TRACED(role, t, ev) do { } while (0)
#endif

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
// try_wait (unlike test_wait) lets the hardware suspend the warp until the phase completes or an implementation time
// limit expires, instead of returning at once: a warp that spins takes issue slots from the working warps of its
// sub-partition.
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
// non-blocking: has the phase with this parity completed?
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n.reg .pred p;\nmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.b32 %0, 1, 0, p;\n}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1,
                                            uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4}], [%2], %5;" ::"r"(dst),
        "l"(map), "r"(bar), "r"(c0), "r"(c1), "l"(policy)
        : "memory");
}
// The same copy delivered to the same shared-memory offset of every CTA of the cluster named in cta_mask; each
// destination CTA's mbarrier (same offset) receives the bytes that landed in it.
__device__ __forceinline__ void tma_load_2d_multicast(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1,
                                                      uint16_t cta_mask, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster.L2::cache_hint"
        " [%0], [%1, {%4, %5}], [%2], %3, %6;" ::"r"(dst),
        "l"(map), "r"(bar), "h"(cta_mask), "r"(c0), "r"(c1), "l"(policy)
        : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// every thread of every CTA of the cluster
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier (size and addresses multiples of 16)
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// true in exactly one lane of the (converged) warp
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n.reg .pred P;\nelect.sync _|P, 0xffffffff;\nselp.b32 %0, 1, 0, P;\n}\n" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// the same arrive on the mbarrier at this shared-memory offset in every CTA of cta_mask (a CTA pair shares stages)
__device__ __forceinline__ void tc_commit_multicast(uint32_t bar, uint16_t cta_mask) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
                 "h"(cta_mask)
                 : "memory");
}
// D[tmem] (+)= A[tmem] . B[smem]^T, kind::f16 (fp16/bf16 in, fp32 accumulate)
__device__ __forceinline__ void tc_mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc,
                                          uint32_t accumulate) {
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n}\n" ::"r"(d_tmem),
        "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// 32 lanes x 32 consecutive 32-bit columns <-> 32 registers per thread (lane l of the warp owns TMEM lane base+l)
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
// Waits for every tcgen05.ld of this thread.  The 32 registers of the load being waited for pass through the
// statement as in/out operands so that no use of them can be scheduled above the wait.
__device__ __forceinline__ void tmem_ld_wait32(float* v) {
    uint32_t* r = reinterpret_cast<uint32_t*>(v);
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]),
                   "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]),
                   "+r"(r[15]), "+r"(r[16]), "+r"(r[17]), "+r"(r[18]), "+r"(r[19]), "+r"(r[20]), "+r"(r[21]),
                   "+r"(r[22]), "+r"(r[23]), "+r"(r[24]), "+r"(r[25]), "+r"(r[26]), "+r"(r[27]), "+r"(r[28]),
                   "+r"(r[29]), "+r"(r[30]), "+r"(r[31])
                 :
                 : "memory");
}
// No instruction: makes later uses of these 32 registers depend on a statement that follows the wait above.
__device__ __forceinline__ void tmem_ld_pin32(float* v) {
    uint32_t* r = reinterpret_cast<uint32_t*>(v);
    asm volatile(""
                 : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]),
                   "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]),
                   "+r"(r[15]), "+r"(r[16]), "+r"(r[17]), "+r"(r[18]), "+r"(r[19]), "+r"(r[20]), "+r"(r[21]),
                   "+r"(r[22]), "+r"(r[23]), "+r"(r[24]), "+r"(r[25]), "+r"(r[26]), "+r"(r[27]), "+r"(r[28]),
                   "+r"(r[29]), "+r"(r[30]), "+r"(r[31])
                 :
                 : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t* r) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
        "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]),
        "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]),
        "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
        : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
// Two fp32 values -> packed bf16 pairs (first value in the low half): hi = bf16(x) rounded to nearest even,
// lo = bf16(x - hi); x - hi is exact in fp32, and hi + lo carries 16 to 18 of x's 24 mantissa bits.
__device__ __forceinline__ void split_pair(float x0, float x1, uint32_t& hi, uint32_t& lo) {
    const __nv_bfloat162 h = __floats2bfloat162_rn(x0, x1);
    const float2 hf = __bfloat1622float2(h);
    const __nv_bfloat162 l = __floats2bfloat162_rn(x0 - hf.x, x1 - hf.y);
    hi = *reinterpret_cast<const uint32_t*>(&h);
    lo = *reinterpret_cast<const uint32_t*>(&l);
}
// operand encoding of the split paths: bf16 hi/lo pair, or (half_mode) one fp16 value rounded to nearest even, lo = 0
__device__ __forceinline__ void encode_pair(float x0, float x1, uint32_t& hi, uint32_t& lo, bool half_mode) {
    if (half_mode) {
        const __half2 h = __floats2half2_rn(x0, x1);
        hi = *reinterpret_cast<const uint32_t*>(&h);
        lo = 0u;
    } else {
        split_pair(x0, x1, hi, lo);
    }
}
__device__ __forceinline__ uint4 ldg_nc16(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

// K-major, 128-byte-swizzled operand tile: rows of 128 bytes, 8-row groups 1024 bytes apart (SBO); descriptor
// version 1 (sm_100), layout type 2 (SWIZZLE_128B).  LBO is unused for this layout.  High word / constant low bits:
constexpr uint32_t DESC_HI = (1024u >> 4) | (1u << 14) | (2u << 29);
constexpr uint32_t DESC_LO = 1u << 16;

// One 33-ary search state: the answer (smallest b in [0, B] with offsets[b] >= target) lies in [lo, hi]; val = offsets[hi].
struct Search {
    int64_t lo, hi, val, target;
};
// one round of 32 probes (n = hi - lo > 32): x is this lane's probe value at p = lo + n*(lane+1)/33
__device__ __forceinline__ int64_t search_probe(const Search& s, int lane) { return s.lo + ((s.hi - s.lo) * (lane + 1)) / 33; }
__device__ __forceinline__ void search_narrow(Search& s, int64_t p, int64_t x, int lane) {
    const unsigned ball = __ballot_sync(0xffffffffu, x >= s.target);
    const int f = ball ? __ffs(ball) - 1 : 32;
    const int64_t p_f = __shfl_sync(0xffffffffu, p, f & 31), x_f = __shfl_sync(0xffffffffu, x, f & 31);
    const int64_t p_fm1 = __shfl_sync(0xffffffffu, p, (f - 1) & 31);
    if (f < 32) { s.hi = p_f; s.val = x_f; }
    if (f > 0) s.lo = p_fm1 + 1;
}
// Both ends of a CTA's document range at once: the two searches run in lockstep so that their (dependent) global loads
// overlap, and each returns offsets[answer] with the index, so no further load follows -- the prologue of a small batch
// is a chain of ~3 load latencies instead of ~8.  offsets[B] = T is known without a load.
__device__ void warp_lower_bound2(const int64_t* __restrict__ offsets, int64_t B, int64_t T, int64_t target_a,
                                  int64_t target_b, int lane, int64_t& idx_a, int64_t& val_a, int64_t& idx_b,
                                  int64_t& val_b) {
    Search a{0, B, T, target_a}, b{0, B, T, target_b};
    while (a.hi - a.lo > 32 || b.hi - b.lo > 32) {
        const bool ra = a.hi - a.lo > 32, rb = b.hi - b.lo > 32;  // warp-uniform
        const int64_t pa = ra ? search_probe(a, lane) : 0, pb = rb ? search_probe(b, lane) : 0;
        const int64_t xa = ra ? offsets[pa] : 0, xb = rb ? offsets[pb] : 0;
        if (ra) search_narrow(a, pa, xa, lane);
        if (rb) search_narrow(b, pb, xb, lane);
    }
    const int64_t qa = a.lo + lane, qb = b.lo + lane;
    const int64_t xa = qa < a.hi ? offsets[qa] : INT64_MAX, xb = qb < b.hi ? offsets[qb] : INT64_MAX;
    const unsigned ba = __ballot_sync(0xffffffffu, qa < a.hi && xa >= a.target);
    const unsigned bb = __ballot_sync(0xffffffffu, qb < b.hi && xb >= b.target);
    const int64_t xa_f = __shfl_sync(0xffffffffu, xa, ba ? __ffs(ba) - 1 : 0), xb_f = __shfl_sync(0xffffffffu, xb, bb ? __ffs(bb) - 1 : 0);
    idx_a = ba ? a.lo + (__ffs(ba) - 1) : a.hi;
    val_a = ba ? xa_f : a.val;
    idx_b = bb ? b.lo + (__ffs(bb) - 1) : b.hi;
    val_b = bb ? xb_f : b.val;
}

struct __align__(16) SegInfo {
    uint32_t mask[4];     // bit c set: column c of the tile is the last token of a (non-empty) document
    uint32_t ord0;        // ordinal (see DOCRING) of the first document that ends in this tile
    uint32_t pad[3];
};
// The CTA's non-empty documents are numbered in order ("ordinals"); DOCRING maps ordinal -> document index relative to
// the CTA's first document.  An entry is read when its document is PARKED, i.e. while the epilogue warp still holds the
// tile the document ends in: the segmenter is at most NSEG tiles (<= 128 documents each) ahead of the slowest epilogue
// warp, so at most 128 + (NSEG - 1) * 128 = 512 < DOCRING ordinals separate the entry from the newest one written.
// (Reading it later, when the park buffer is drained, would not be safe: ordinals count ALL of the CTA's documents,
// while a warp of two epilogue sets parks only those that end in its own columns / tiles, so a parked document can
// wait while far more than DOCRING ordinals go by.)
constexpr uint32_t DOCRING = 1024;

// ---- epilogue helpers ------------------------------------------------------------------------------------------
__device__ __forceinline__ float max3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }  // one FMNMX3

// running max folded with 8 accumulator columns: four 3-input max instructions
__device__ __forceinline__ float max9(float m, const float* x) {
    return max3(max3(x[0], x[1], x[2]), max3(x[3], x[4], x[5]), max3(x[6], x[7], m));
}

// Per-warp constants of the max -> sum step, packed: bits 0-5 Nq, 6-11 Nq_pad, 12-17 queries of this warp that exist.
__device__ __forceinline__ uint32_t pack_cfg(int Nq, int Nq_pad, int nvalid) {
    return (uint32_t)Nq | ((uint32_t)Nq_pad << 6) | ((uint32_t)nvalid << 12);
}

__device__ __forceinline__ void sts_f32(uint32_t addr, float v) {
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ float4 lds_f32x4(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ float lds_f32(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
    return v;
}

// A document's last token has been folded in: row `lane` parks its maximum in slot np of the warp's buffer.
// pend: shared-window byte address of this warp's park buffer ([PEND][PEND_PITCH] floats, then PEND document indices,
// relative to the CTA's first document: the ordinal is resolved through DOCRING here, while its entry is live).
constexpr uint32_t PEND_IDS = PEND * PEND_PITCH * 4;  // byte offset of the ids inside a warp's park buffer
__device__ __forceinline__ void park(float m, uint32_t ord, uint32_t np, uint32_t pend, uint32_t ring, int lane) {
    sts_f32(pend + (np * PEND_PITCH + lane) * 4, m);
    if (lane == 0) sts_u32(pend + PEND_IDS + np * 4, lds_u32(ring + (ord & (DOCRING - 1)) * 4));
}

// max -> sum (Eq. 1) for the np parked documents.  Rows that no query token owns hold zero query vectors, so their
// maxima are exactly 0 and every one of the Nq_pad rows of a query can be added (A5).  Parked documents are
// consecutive in the usual case, so the stores of a warp coalesce.
//   Nq_pad = 32 (one query per warp): lanes j and j+16 add rows 0..15 / 16..31 of parked document j with four
//   16-byte loads each, in four interleaved partial sums, and lane j stores the score.
//   Nq_pad < 32: one lane per (document, query of this warp), rows added in ascending order.
__device__ __noinline__ void drain(uint32_t pend, uint32_t np, float* out, int64_t B, uint32_t cfg, int lane) {
    const uint32_t Nq_pad = (cfg >> 6) & 63u, nvalid = (cfg >> 12) & 63u;
    __syncwarp();
    if (Nq_pad == 32) {
        const uint32_t j = lane & 15u, h = (uint32_t)lane >> 4;
        const uint32_t p = pend + (j * PEND_PITCH + h * 16) * 4;
        const float4 x0 = lds_f32x4(p), x1 = lds_f32x4(p + 16), x2 = lds_f32x4(p + 32), x3 = lds_f32x4(p + 48);
        const float a0 = (x0.x + x1.x) + (x2.x + x3.x), a1 = (x0.y + x1.y) + (x2.y + x3.y);
        const float a2 = (x0.z + x1.z) + (x2.z + x3.z), a3 = (x0.w + x1.w) + (x2.w + x3.w);
        float acc = (a0 + a1) + (a2 + a3);
        acc += __shfl_xor_sync(0xffffffffu, acc, 16);
        if (h == 0 && j < np && nvalid) out[lds_u32(pend + PEND_IDS + j * 4)] = acc;
    } else {
        const uint32_t nsub = 32u / Nq_pad;
        for (uint32_t u = lane; u < np * nsub; u += 32) {
            const uint32_t slot = u / nsub, sub = u - slot * nsub;
            if (sub < nvalid) {
                const uint32_t p = pend + (slot * PEND_PITCH + sub * Nq_pad) * 4;
                float acc = lds_f32(p);
                for (uint32_t r = 1; r < Nq_pad; ++r) acc += lds_f32(p + r * 4);
                out[(int64_t)sub * B + lds_u32(pend + PEND_IDS + slot * 4)] = acc;
            }
        }
    }
    __syncwarp();
}

// running max folded with 32 accumulator columns: sixteen 3-input max instructions, four independent chains
__device__ __forceinline__ float max33(float m, const float* x) {
    const float a = max3(max3(x[0], x[1], x[2]), max3(x[3], x[4], x[5]), max3(x[6], x[7], x[8]));
    const float b = max3(max3(x[9], x[10], x[11]), max3(x[12], x[13], x[14]), max3(x[15], x[16], x[17]));
    const float c = max3(max3(x[18], x[19], x[20]), max3(x[21], x[22], x[23]), max3(x[24], x[25], x[26]));
    const float d = max3(max3(x[27], x[28], x[29]), max3(x[30], x[31], m), a);
    return max3(b, c, d);
}

constexpr uint32_t NONE = 0xffffffffu;
struct EpiState {
    float m;       // running max of this row over the current document's tokens seen so far
    uint32_t ord;  // ordinal of the next document to close (see DOCRING)
    uint32_t np;   // documents parked in the warp's buffer
    // Two epilogue warp sets on alternate tiles: a tile is reduced before the running max of the previous tile (the
    // other set's) is known.  Until that carry has been folded in (`unresolved`), the first document the tile closes is
    // parked without it: `first` is its slot in the park buffer (NONE: nothing closed yet), `head` the value parked.
    bool unresolved;
    uint32_t first;
    float head;
};
// a document closes with row maximum `value`
__device__ __forceinline__ void close_doc(float value, EpiState& s, uint32_t pend, uint32_t ring, int lane) {
    if (s.unresolved && s.first == NONE) {
        s.first = s.np;
        s.head = value;
    }
    park(value, s.ord, s.np, pend, ring, lane);
    ++s.ord;
    ++s.np;
}

// 8 accumulator columns in which documents end (bit c of `byte`: column c is a document's last token): columns
// are folded in order and every finished document is parked.  Out of line: boundary chunks are the minority, and
// one compact copy keeps the epilogue's hot loop short.  The caller has made sure the buffer has room.
__device__ __noinline__ float epi_chunk_slow(float x0, float x1, float x2, float x3, float x4, float x5, float x6,
                                             float x7, uint32_t byte, float m, uint32_t ord, uint32_t np, uint32_t pend,
                                             uint32_t ring, int lane) {
    const float x[8] = {x0, x1, x2, x3, x4, x5, x6, x7};
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        m = fmaxf(m, x[c]);
        if (byte & (1u << c)) {
            park(m, ord, np, pend, ring, lane);
            ++ord;
            ++np;
            m = -INFINITY;  // Alg. 3 line 4 for the next document
        }
    }
    return m;
}

// max of 8 columns
__device__ __forceinline__ float max8(const float* x) {
    return max3(max3(x[0], x[1], x[2]), max3(x[3], x[4], x[5]), fmaxf(x[6], x[7]));
}

// One document ends in this word, at column e of chunk J (8-column chunks; J compile-time): the columns up to e close the
// document (together with the running max m), the columns after e open the next one.  Whole chunks go to one side
// unconditionally; only chunk J is split, branch-free, with selects.
template <int J>
__device__ __forceinline__ void split_word(const float* v, int e8, float m, float& closed, float& open) {
    float l[8], r[8];
    const float* x = v + 8 * J;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const bool left = e8 >= c;
        l[c] = left ? x[c] : -INFINITY;
        r[c] = left ? -INFINITY : x[c];
    }
    float a = max3(max8(l), m, -INFINITY), b = max8(r);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        if (i < J) a = fmaxf(a, max8(v + 8 * i));
        if (i > J) b = fmaxf(b, max8(v + 8 * i));
    }
    closed = a;
    open = b;
}

// 32 accumulator columns (registers v) with boundary word w: bit c set = column c is a document's last token.
//   no boundary (the majority)              sixteen 3-input max instructions
//   one boundary                            dispatched ONCE on the boundary's 8-column chunk (a lone warp pays ~15 clk per
//                                           unpredicted branch, so no per-chunk tests), whole chunks folded to either side
//                                           and the boundary chunk split with selects
//   several boundaries (documents < 32 tokens)   walked in 8-column chunks
// `resolve` folds the previous range's carry in; it must have run before the park buffer is drained.
template <class Resolve>
__device__ __forceinline__ void process32(const float* v, uint32_t w, EpiState& s, uint32_t pend, uint32_t ring, float* out, int64_t B, uint32_t cfg, int lane,
                                          bool skip_math, Resolve resolve) {
    if (skip_math) {  // measurement probe: TMEM loads without the reduction
        s.m = fmaxf(s.m, v[0]);
        return;
    }
    if (w == 0) {
        s.m = max33(s.m, v);
        return;
    }
    if (w == 0x80000000u) {  // the word's last column (uniform 128-token documents)
        if (s.np == PEND) {
            if (s.unresolved) resolve();
            drain(pend, s.np, out, B, cfg, lane);
            s.np = 0;
        }
        close_doc(max33(s.m, v), s, pend, ring, lane);
        s.m = -INFINITY;  // Alg. 3 line 4 for the next document
        return;
    }
    if ((w & (w - 1)) == 0) {
        if (s.np == PEND) {
            if (s.unresolved) resolve();
            drain(pend, s.np, out, B, cfg, lane);
            s.np = 0;
        }
        float closed, open;
        const int e = 31 - __clz((int)w), e8 = e & 7;
        if (e < 16) {
            if (e < 8) split_word<0>(v, e8, s.m, closed, open);
            else split_word<1>(v, e8, s.m, closed, open);
        } else {
            if (e < 24) split_word<2>(v, e8, s.m, closed, open);
            else split_word<3>(v, e8, s.m, closed, open);
        }
        close_doc(closed, s, pend, ring, lane);
        s.m = open;
        return;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t byte = (w >> (8 * j)) & 0xffu;
        const float* x = v + 8 * j;
        if (byte == 0) {
            s.m = max9(s.m, x);
            continue;
        }
        if (s.np + __popc(byte) > PEND) {  // room for the documents that end in this chunk
            if (s.unresolved) resolve();
            drain(pend, s.np, out, B, cfg, lane);
            s.np = 0;
        }
        const bool rec = s.unresolved && s.first == NONE;
        s.m = epi_chunk_slow(x[0], x[1], x[2], x[3], x[4], x[5], x[6], x[7], byte, s.m, s.ord, s.np, pend, ring, lane);
        if (rec) {  // the first document this range closes was parked by the helper: pick its value up again
            s.first = s.np;
            s.head = lds_f32(pend + (s.np * PEND_PITCH + lane) * 4);
        }
        const uint32_t n = __popc(byte);
        s.ord += n;
        s.np += n;
    }
}

// KBS: dimension blocks per pipeline stage (2 = a whole 256-byte row block per stage).
// F32: fp32 inputs (a9).  The tensor pipe has no fp32 MMA, and TF32 alone would break the 1e-5*Nq tolerance, so
// every fp32 value x is split on the fly into two bf16 values, hi = bf16(x) and lo = bf16(x - hi) (16-18 mantissa
// bits together), and hi*hi + hi*lo + lo*hi is accumulated in fp32 -- three bf16 MMAs per K step.
// Four extra "splitter" warps turn each fp32 tile that TMA lands (a raw stage) into a bf16 hi block + lo block (an
// operand stage, KBS = 2 blocks); the query rows are split once by their epilogue threads.  p.NKB then counts
// 64-element units (64 fp32 = two 128-byte dimension blocks in, one bf16 hi block + one lo block out).
// PQD (with F32): the document tile is not loaded but DECODED: TMA brings 128 tokens x 16 code bytes, and the four
// splitter warps gather every token's 16 centroid slices (8 fp32 each) from the codebook, resident in shared memory,
// split them into bf16 hi/lo and write the same operand stages as the fp32 path.  The decompressed vectors exist only
// as MMA operands in shared memory, never in HBM (P:L244-249 names decompress-then-score as the costly baseline
// because of its HBM round trip; on-chip it costs 16 bytes of HBM per token and no lookup per query row).
// NSET: epilogue warp sets.  2 (16-bit inputs only): two warps per 32 TMEM lanes, one per half of a tile's columns --
// pays when documents are short (many boundaries per tile: the segmented reduction is the binding step); 1 otherwise.
// PAIR (16-bit inputs, MB = 1): "read once" for 256 query rows when d is too large for two resident query blocks
// (d*sizeof > 512 bytes).  The kernel runs as clusters of two CTAs that walk the SAME token range; CTA r keeps query
// block r in its tensor memory, loads HALF of every document tile (64 tokens) and multicasts it into both CTAs'
// shared memory, so the pair reads each embedding from L2/HBM once and each SM contracts it against its own 128 rows.
// A stage is shared state: it is refilled only when BOTH CTAs' tensor pipes have read it (the `empty` barriers count two
// arrivals, each CTA's tcgen05.commit is multicast to both).  Everything else -- MMA issue, segmenter, epilogue, max->sum
// -- is per CTA and unchanged (Thm 1's ceil(Nq/BQ) factor stays 1).
// ALT (with NSET = 2): the two epilogue sets take alternate TILES instead of column halves -- every warp reduces whole
// 128-column rows but only of every other tile, so it has two tile periods for a tile's segmented reduction; the running
// maximum crosses tiles through the same mailbox (one hop per tile).
template <int MB, int KBS, bool F32, bool PQD, int NSET, bool PAIR = false, bool ALT = false>
__global__ void __launch_bounds__(128 + NSET * 128 * MB + (F32 ? 128 : 0), 1)
dense_tc_kernel(const __grid_constant__ CUtensorMap map_docs, const Params p) {
    static_assert(!ALT || (NSET == 2 && !F32 && !PAIR), "alternate-tile epilogue sets: two sets, 16-bit inputs");
    static_assert(!PAIR || (MB == 1 && !F32 && !PQD), "CTA pairs: one query block per CTA, 16-bit inputs");
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    // 128-byte-swizzled operand tiles need 1024-byte alignment in the shared window
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    // layout: [operand stages: NS * KBS*16 KB] [F32: raw stages: NR * 32 KB] [SegInfo x NSEG] [park buffers] [barriers]
    // PQD with fp16 operands has no lo parts: its stages hold one 16 KB block and its codebook one 64 KB plane, which
    // leaves room for eight operand stages instead of two (the decode then runs ahead of the tensor pipe).
    const bool pq_half = PQD && p.half_mode != 0;
    const uint32_t stage_bytes = pq_half ? (uint32_t)KB_TILE_BYTES : (uint32_t)KBS * KB_TILE_BYTES;
    constexpr uint32_t raw_bytes = PQD ? BN * 16u : 2u * KB_TILE_BYTES;  // PQD: 16 code bytes per token
    const uint32_t cb_bytes = PQD ? (pq_half ? 16u * 256u * 8u * 2u : 16u * 256u * 8u * 4u) : 0u;  // PQD: the codebook [16][256][8], as two bf16 planes (or one fp16 plane)
    constexpr int n_epi_warps = 4 * MB;            // epilogue warps of one set (one set reduces a tile)
    static_assert(NSET == 1 || (NSET == 2 && !F32), "two epilogue sets exist for 16-bit inputs only");
    uint8_t* st_ptr = smem;
    uint8_t* rw_ptr = st_ptr + (size_t)p.NS * stage_bytes;
    uint8_t* cb_ptr = rw_ptr + (F32 ? (size_t)p.NR * raw_bytes : 0);
    SegInfo* seg = reinterpret_cast<SegInfo*>(cb_ptr + cb_bytes);
    uint32_t* docring = reinterpret_cast<uint32_t*>(seg + NSEG);                    // [DOCRING]
    float* pend_all = reinterpret_cast<float*>(docring + DOCRING);                         // [warps]{[PEND][PEND_PITCH] maxima, [PEND] ids}
    float* mail = pend_all + NSET * n_epi_warps * PEND * (PEND_PITCH + 1);         // [NSET][warps][32] carries between the sets
    uint64_t* bars = reinterpret_cast<uint64_t*>(mail + 2 * 8 * 32);
    uint64_t* full = bars;                       // [NS]   operand stage filled (TMA, or the splitter warps) -> MMA
    uint64_t* empty = full + MAX_STAGES;         // [NS]   operand stage read by the tensor pipe -> TMA / splitter
    uint64_t* tfull = empty + MAX_STAGES;        // [4*MB] MMA -> epilogue: accumulator of (tile t, block mb), ring t & 3
    uint64_t* tempty = tfull + 8;                // [NACC] epilogue -> MMA (4 warps each)
    uint64_t* sfull = tempty + MAX_ACC;          // [NSEG] segmenter -> epilogue
    uint64_t* sempty = sfull + NSEG;             // [NSEG] epilogue -> segmenter
    uint64_t* rfull = sempty + NSEG;             // [NR]   F32: TMA -> splitter
    uint64_t* rempty = rfull + MAX_RAW;          // [NR]   F32: splitter -> TMA (4 warps)
    uint64_t* aready = rempty + MAX_RAW;         // [1]    query rows are in TMEM
    uint64_t* turn = aready + 1;                 // [2]    MMA issuer w may start its next tile (the other one is done issuing)
    uint64_t* carry = turn + 2;                  // [2][8] epilogue set -> the other set: running maxima at the end of a tile
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(carry + 16);
    int64_t* range = reinterpret_cast<int64_t*>(carry + 17);  // b_lo, b_hi, t_lo, t_hi

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = PAIR ? cluster_ctarank() : 0u;  // which query block (and which half of every tile) is this CTA's

    // ---- one-time setup ------------------------------------------------------------------------------------
    if (warp == 0) {
        if (lane == 0) {
            for (int s = 0; s < p.NS; ++s) { mbar_init(smem_u32(full + s), F32 ? 4 : 1); mbar_init(smem_u32(empty + s), PAIR ? 2 : 1); }
            for (int s = 0; s < 8; ++s) mbar_init(smem_u32(tfull + s), 1);
            for (int s = 0; s < MAX_ACC; ++s) mbar_init(smem_u32(tempty + s), 4 * (ALT ? 1 : NSET));
            for (int s = 0; s < MAX_RAW; ++s) { mbar_init(smem_u32(rfull + s), 1); mbar_init(smem_u32(rempty + s), 4); }
            for (int s = 0; s < NSEG; ++s) { mbar_init(smem_u32(sfull + s), 1); mbar_init(smem_u32(sempty + s), (ALT ? 1 : NSET) * n_epi_warps); }
            mbar_init(smem_u32(aready), n_epi_warps);
            mbar_init(smem_u32(turn), 1);
            mbar_init(smem_u32(turn + 1), 1);
            for (int s = 0; s < 16; ++s) mbar_init(smem_u32(carry + s), 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            if (!PQD) asm volatile("prefetch.tensormap [%0];" ::"l"(&map_docs) : "memory");
        }
        // work partition (a3): documents [b_lo, b_hi) whose first tokens lie in [c*T/G, (c+1)*T/G)
        const int64_t G = PAIR ? gridDim.x >> 1 : gridDim.x, c = PAIR ? blockIdx.x >> 1 : blockIdx.x;  // a pair shares its range
        const int64_t tgt_lo = p.tok0 + (c * p.Tseg) / G, tgt_hi = p.tok0 + ((c + 1) * p.Tseg) / G;
        int64_t b_lo, b_hi, o_lo, o_hi;
        warp_lower_bound2(p.offsets, p.B, p.T, tgt_lo, tgt_hi, lane, b_lo, o_lo, b_hi, o_hi);
        if (c == 0 && p.seg_first) { b_lo = 0; o_lo = 0; }          // offsets[0] = 0
        if (c == G - 1 && p.seg_last) { b_hi = p.B; o_hi = p.T; }  // offsets[B] = T
        if (lane == 0) {
            range[0] = b_lo;
            range[1] = b_hi;
            range[2] = o_lo;
            range[3] = o_hi;
        }
    } else if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                     "r"((uint32_t)TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    if constexpr (PAIR) cluster_sync_all();  // the peer's barriers are initialised before anything is sent to them
    else __syncthreads();
    tc_fence_after();

    const uint32_t tmem_base = *tmem_slot;
    const int64_t b_lo = range[0], b_hi = range[1], t_lo = range[2], t_hi = range[3];
    const int64_t ntiles = (t_hi - t_lo + BN - 1) / BN;
    const int nchunks = F32 ? p.NKB : p.NKB / KBS;  // operand stages consumed per tile

    if (warp == 0) {
        // ===== TMA producer =====
        // The whole warp runs the loop and waits on the barriers; one elected lane issues the copies, so that the
        // compiler emits the uniform-datapath instructions straight-line (no per-active-thread loop).
        const uint64_t pol_docs = policy_evict_first();  // streamed once
        uint32_t s = 0, ph = 0;  // ring slot and its phase bit (F32: the raw ring)
        const uint32_t nring = F32 ? (uint32_t)p.NR : (uint32_t)p.NS;
        for (int64_t t = 0; PQD && t < ntiles; ++t) {  // one raw stage per tile: the tile's code rows
            const int64_t tok = t_lo + t * BN;
            const uint32_t bytes = (uint32_t)((p.T - tok < BN ? p.T - tok : BN) * 16);
            mbar_wait(smem_u32(rempty + s), ph ^ 1);
            if (elect_one()) {
                mbar_expect_tx(smem_u32(rfull + s), bytes);
                bulk_load(smem_u32(rw_ptr + (size_t)s * raw_bytes), p.codes + tok * 16, bytes, smem_u32(rfull + s));
            }
            __syncwarp();
            if (++s == nring) { s = 0; ph ^= 1; }
        }
        for (int64_t t = 0; !PQD && t < ntiles; ++t) {
            const int tok = (int)(t_lo - p.tok0 + t * BN);  // row of this launch's tensor map
            for (int ch = 0; ch < nchunks; ++ch) {
                if constexpr (F32) {
                    mbar_wait(smem_u32(rempty + s), ph ^ 1);
                    if (elect_one()) {
                        mbar_expect_tx(smem_u32(rfull + s), raw_bytes);
#pragma unroll
                        for (int k = 0; k < 2; ++k)  // 64 fp32 of every token = two 128-byte dimension blocks
                            tma_load_2d(smem_u32(rw_ptr + (size_t)s * raw_bytes + k * KB_TILE_BYTES), &map_docs,
                                        smem_u32(rfull + s), (ch * 2 + k) * p.kb_elems, tok, pol_docs);
                    }
                } else {
                    mbar_wait(smem_u32(empty + s), ph ^ 1);
    
#ifdef TMS_PROBES
                    if (PROBE(p, 8)) {  // probe: one linear 1-D bulk copy per stage instead of the 2-D tensor copies (wrong data layout, timing only)
                        if (elect_one()) {
                            mbar_expect_tx(smem_u32(full + s), stage_bytes);
                            bulk_load(smem_u32(st_ptr + (size_t)s * stage_bytes), (const uint8_t*)p.docs_raw + (size_t)tok * p.row_bytes, stage_bytes, smem_u32(full + s));
                        }
                    } else
#endif
                    if (elect_one()) {
                        mbar_expect_tx(smem_u32(full + s), stage_bytes);  // both halves land here: mine and the peer's
#pragma unroll
                        for (int k = 0; k < KBS; ++k) {
                            if constexpr (PAIR)  // token rows [64*rank, +64) of the tile, into both CTAs
                                tma_load_2d_multicast(smem_u32(st_ptr + (size_t)s * stage_bytes + k * KB_TILE_BYTES) + rank * (KB_TILE_BYTES / 2),
                                                      &map_docs, smem_u32(full + s), (ch * KBS + k) * p.kb_elems,
                                                      tok + (int)rank * (BN / 2), (uint16_t)3, pol_docs);
                            else
                                tma_load_2d(smem_u32(st_ptr + (size_t)s * stage_bytes + k * KB_TILE_BYTES), &map_docs,
                                            smem_u32(full + s), (ch * KBS + k) * p.kb_elems, tok, pol_docs);
                        }
                    }
                }
                __syncwarp();

                if (++s == nring) { s = 0; ph ^= 1; }
            }
        }
    } else if (warp == 1 || warp == 3) {
        // ===== MMA issuers =====
        // Two warps issue alternate tiles (warp 1 the even ones, warp 3 the odd ones).  Why two: the thread that issues
        // tcgen05.mma blocks while the MMA queue is full, so it reaches the code after a tile's last MMA with only a
        // few MMAs (~250 clk of tensor work) still queued; the barrier waits, ring arithmetic and descriptor set-up
        // of the next tile take a lone warp longer than that and the tensor pipe ran dry at every tile boundary
        // (traced: 1,024 clk of MMAs per 1,380 clk tile period).  With two issuers all of that happens while the
        // other warp is issuing; what is left on the critical path is the hand-over: one mbarrier arrive after the
        // last MMA of a tile has been accepted, and the waiting warp's wake-up.  MMAs of different tiles are never
        // interleaved (switching accumulators between consecutive MMAs costs tensor-pipe time).
        // Inside a tile one elected lane issues everything; the rest of the warp follows the barriers, so the ring
        // arithmetic stays warp-uniform (uniform datapath, descriptors are the previous one plus a constant).
        const uint32_t w = (uint32_t)warp >> 1;  // 0: even tiles, 1: odd tiles
        mbar_wait(smem_u32(aready), 0);
        tc_fence_after();
        // Everything below is computed by the whole warp (warp-uniform values stay in the uniform datapath, where a
        // descriptor is the previous one plus a constant); only the tcgen05 instructions sit in elect_one() regions.
        const uint32_t b_lo0 = ((smem_u32(st_ptr) & 0x3FFFFu) >> 4) | DESC_LO;
        const uint32_t idesc = p.idesc;
        const bool skip = PROBE(p, 2), skip_alo = p.skip_alo != 0, skip_blo = PQD && p.half_mode != 0;
        const uint32_t nacc = (uint32_t)p.NACC, NS = (uint32_t)p.NS, nch = (uint32_t)nchunks;
        const uint32_t acc0 = tmem_base + (uint32_t)p.acc_col0;
        // TMEM columns of one query block's rows (F32: hi halves of all units, then lo halves)
        const uint32_t a_lo_off = (uint32_t)p.NKB * KB_WORDS;
        // split paths: a block's hi plane is followed by its lo plane -- unless every lo part is zero (skip_alo), in which
        // case no lo plane exists and the columns go to a third accumulator instead
        const uint32_t a_mb_step = (F32 && !skip_alo) ? 2 * a_lo_off : a_lo_off;
        const bool epi_frees_stage = !F32 && !PAIR && nchunks == 1;
        const uint32_t full0 = smem_u32(full), empty0 = smem_u32(empty), tempty0 = smem_u32(tempty), tfull0 = smem_u32(tfull);
        const uint32_t my_turn = smem_u32(turn + w), other_turn = smem_u32(turn + (w ^ 1));
        // ring positions of this warp's first tile (tile w): operand stage w*nchunks, accumulator jobs w*MB + mb
        uint32_t s = w * nch, ph = 0;
        while (s >= NS) { s -= NS; ph ^= 1; }
        uint32_t slot[MB], tph[MB];
#pragma unroll
        for (int mb = 0; mb < MB; ++mb) {
            slot[mb] = w * MB + mb; tph[mb] = 0;
            while (slot[mb] >= nacc) { slot[mb] -= nacc; tph[mb] ^= 1; }
        }
        // The tile's first stage and first accumulator are awaited BEFORE the hand-over when that is safe: a parity
        // wait is only meaningful once the barrier's previous phase has completed, which is certain when that phase
        // belongs to a tile <= t-2 (issued before this warp's previous hand-over), i.e. when the ring is longer
        // than one tile's worth (NS > nchunks, NACC > MB).  Otherwise they are awaited after it.
        const bool early_full = NS > nch, early_acc = nacc > (uint32_t)MB;
        uint32_t tp = 0;             // parity of `turn` to wait for; tile 0 needs no hand-over
        uint32_t tq = w;             // t & 3 of this warp's tile: the tfull ring
        const int nt = (int)ntiles;
        for (int t = (int)w; t < nt; t += 2) {
            if (early_full) mbar_wait(full0 + s * 8, ph);
            if (early_acc) mbar_wait(tempty0 + slot[0] * 8, tph[0] ^ 1);  // the epilogue has drained block 0's accumulator
            if (t != 0) { mbar_wait(my_turn, tp); tp ^= 1; }
            TRACE(1, t, 0);
#ifdef TMS_PROBES
            if (blockIdx.x == TRACE_CTA && lane == 0 && t >= TRACE_T0 && t < TRACE_T0 + TRACE_NT) {
                uint64_t gt;
                asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
                g_trace[(1 * TRACE_NT + (int)(t - TRACE_T0)) * TRACE_EV + 7] = (long long)gt;
            }
#endif
            uint32_t a_col = tmem_base;  // this chunk's first dimension block of query block 0
            // PQ decode with room for several tiles of operand stages (fp16 operands: eight 16 KB stages): ONE issue
            // region per tile, block-major -- both 64-dimension units of a block back to back (one accumulator switch
            // per tile, block 0's accumulator handed to the epilogue half a tile early), then the next block.
            const bool whole_tile = PQD && NS >= 4;
            // ... and with only one tile's worth of stages (split bf16 operands: two 32 KB stages): still one region per
            // tile, but unit-major, the issuing lane awaiting the second unit's stage itself and releasing each stage as
            // soon as its MMAs are queued, so the next tile's decode starts as early as before.
            const bool unit_major_tile = F32 && !whole_tile && nch == 2 && NS >= 2;
            // CTA pairs (one query block, d > 256: three to six 256-byte chunks per tile): one region per tile as well -- the
            // issuing lane awaits each later chunk's stage itself, so a tile's 24-48 MMAs are queued without the per-region
            // overhead between every eight of them (ncu: tensor pipe 78 % -> see profiles).
            const bool pair_tile = PAIR && !F32;
            if (pair_tile) {
                if (!early_full) mbar_wait(full0 + s * 8, ph);
                if (!early_acc) mbar_wait(tempty0 + slot[0] * 8, tph[0] ^ 1);
                tc_fence_after();
                if (elect_one()) {
                    uint32_t sc = s, phc = ph, ac = a_col;
                    const uint32_t d_tmem = acc0 + slot[0] * BN;
                    for (uint32_t ch = 0; ch < nch; ++ch) {
                        if (ch != 0) {
                            mbar_wait(full0 + sc * 8, phc);
                            tc_fence_after();
                        }
                        const uint32_t b_lo = b_lo0 + sc * (stage_bytes >> 4);
                        if (!skip) {
#pragma unroll
                            for (int k = 0; k < KBS; ++k) {
#pragma unroll
                                for (int kk = 0; kk < 4; ++kk) {
                                    const uint64_t bd = ((uint64_t)DESC_HI << 32) | (b_lo + k * (KB_TILE_BYTES >> 4) + kk * 2);
                                    tc_mma_ts(d_tmem, ac + k * KB_WORDS + kk * 8, bd, idesc, (ch != 0 || k != 0 || kk != 0) ? 1u : 0u);
                                }
                            }
                        }
                        tc_commit_multicast(empty0 + sc * 8, (uint16_t)3);  // the stage is the pair's
                        ac += KBS * KB_WORDS;
                        if (++sc == NS) { sc = 0; phc ^= 1; }
                    }
                    tc_commit(tfull0 + (tq * MB) * 8);  // accumulator -> epilogue
                    mbar_arrive(other_turn);            // the other issuer may start its tile
                }
                __syncwarp();
                s += nch;
                while (s >= NS) { s -= NS; ph ^= 1; }
            }
            if (unit_major_tile) {
                uint32_t s1 = s + 1, ph1 = ph;
                if (s1 == NS) { s1 = 0; ph1 ^= 1; }
                if (!early_full) mbar_wait(full0 + s * 8, ph);
                if (!early_acc) mbar_wait(tempty0 + slot[0] * 8, tph[0] ^ 1);
                tc_fence_after();
                if (elect_one()) {
#pragma unroll
                    for (int ch = 0; ch < 2; ++ch) {
                        if (ch == 1) {
                            mbar_wait(full0 + s1 * 8, ph1);
                            tc_fence_after();
                        }
                        const uint32_t b_lo = b_lo0 + (ch ? s1 : s) * (stage_bytes >> 4);
#pragma unroll
                        for (int mb = 0; mb < MB; ++mb) {
                            if (ch == 0 && mb != 0) {
                                mbar_wait(tempty0 + slot[mb] * 8, tph[mb] ^ 1);
                                tc_fence_after();
                            }
                            const uint32_t d_tmem = acc0 + slot[mb] * BN;
                            if (!skip) {
#pragma unroll
                                for (int kk = 0; kk < 4; ++kk) {
                                    const uint64_t b_hi = ((uint64_t)DESC_HI << 32) | (b_lo + kk * 2);
                                    const uint64_t b_lw = ((uint64_t)DESC_HI << 32) | (b_lo + (KB_TILE_BYTES >> 4) + kk * 2);
                                    const uint32_t a_hi = a_col + ch * KB_WORDS + mb * a_mb_step + kk * 8;
                                    tc_mma_ts(d_tmem, a_hi, b_hi, idesc, (ch != 0 || kk != 0) ? 1u : 0u);
                                    if (!skip_blo) tc_mma_ts(d_tmem, a_hi, b_lw, idesc, 1u);
                                    if (!skip_alo) tc_mma_ts(d_tmem, a_hi + a_lo_off, b_hi, idesc, 1u);
                                }
                            }
                            if (ch == 1) tc_commit(tfull0 + (tq * MB + mb) * 8);  // accumulator -> epilogue
                        }
                        tc_commit(empty0 + (ch ? s1 : s) * 8);  // the stage goes back to the splitter warps
                    }
                    mbar_arrive(other_turn);  // the other issuer may start its tile
                }
                __syncwarp();
                s += 2;
                while (s >= NS) { s -= NS; ph ^= 1; }
            }
            if (whole_tile) {
                uint32_t s1 = s + 1, ph1 = ph;
                if (s1 == NS) { s1 = 0; ph1 ^= 1; }
                if (!early_full) mbar_wait(full0 + s * 8, ph);
                mbar_wait(full0 + s1 * 8, ph1);
                if (!early_acc) mbar_wait(tempty0 + slot[0] * 8, tph[0] ^ 1);
                tc_fence_after();
                if (elect_one()) {
#pragma unroll
                    for (int mb = 0; mb < MB; ++mb) {
                        if (mb != 0) {
                            mbar_wait(tempty0 + slot[mb] * 8, tph[mb] ^ 1);
                            tc_fence_after();
                        }
                        const uint32_t d_tmem = acc0 + slot[mb] * BN;
                        if (!skip) {
#pragma unroll
                            for (int ch = 0; ch < 2; ++ch) {
                                const uint32_t b_lo = b_lo0 + (ch ? s1 : s) * (stage_bytes >> 4);
#pragma unroll
                                for (int kk = 0; kk < 4; ++kk) {
                                    const uint64_t b_hi = ((uint64_t)DESC_HI << 32) | (b_lo + kk * 2);
                                    const uint64_t b_lw = ((uint64_t)DESC_HI << 32) | (b_lo + (KB_TILE_BYTES >> 4) + kk * 2);
                                    const uint32_t a_hi = a_col + ch * KB_WORDS + mb * a_mb_step + kk * 8;
                                    tc_mma_ts(d_tmem, a_hi, b_hi, idesc, (ch != 0 || kk != 0) ? 1u : 0u);
                                    if (!skip_blo) tc_mma_ts(d_tmem, a_hi, b_lw, idesc, 1u);
                                    if (!skip_alo) tc_mma_ts(d_tmem, a_hi + a_lo_off, b_hi, idesc, 1u);
                                }
                            }
                        }
                        tc_commit(tfull0 + (tq * MB + mb) * 8);  // accumulator -> epilogue
                    }
                    tc_commit(empty0 + s * 8);   // both stages go back to the splitter warps
                    tc_commit(empty0 + s1 * 8);
                    mbar_arrive(other_turn);     // the other issuer may start its tile
                }
                __syncwarp();
                s += 2;
                while (s >= NS) { s -= NS; ph ^= 1; }
            }
            for (uint32_t ch = 0; !whole_tile && !unit_major_tile && !pair_tile && ch < nch; ++ch) {
                if (ch != 0 || !early_full) mbar_wait(full0 + s * 8, ph);
                const uint32_t b_lo = b_lo0 + s * (stage_bytes >> 4);
                const bool last_chunk = ch == nch - 1;
                if constexpr (F32) {
                    // Split paths: ONE issue region per 64-element unit covering every query block.  A region costs the
                    // issuing warp ~300 clk of waits, fences, election and commits next to its MMAs, and the MMA queue
                    // holds only ~4 instructions: with a region per (unit, block) the PQ decode variant issued 4 (fp16
                    // operands) or 8 MMAs per region and the tensor pipe ran dry between regions (probe build: the
                    // barrier skeleton alone took 1,220 clk per tile and the MMAs added their full 1,024 / 2,048 clk).
                    if (ch == 0 && !early_acc) mbar_wait(tempty0 + slot[0] * 8, tph[0] ^ 1);
                    tc_fence_after();
                    if (elect_one()) {
#pragma unroll
                        for (int mb = 0; mb < MB; ++mb) {
                            // a later block's accumulator is awaited by the issuing lane itself, with the earlier
                            // blocks' MMAs already queued (waiting for it up front would idle the pipe)
                            if (ch == 0 && mb != 0) {
                                mbar_wait(tempty0 + slot[mb] * 8, tph[mb] ^ 1);
                                tc_fence_after();
                            }
                            const uint32_t d_tmem = acc0 + slot[mb] * BN;
                            if (!skip) {
#pragma unroll
                                for (int kk = 0; kk < 4; ++kk) {  // four 16-element K steps per 64-element unit
                                    const uint64_t b_hi = ((uint64_t)DESC_HI << 32) | (b_lo + kk * 2);
                                    const uint64_t b_lw = ((uint64_t)DESC_HI << 32) | (b_lo + (KB_TILE_BYTES >> 4) + kk * 2);
                                    const uint32_t a_hi = a_col + mb * a_mb_step + kk * 8;
                                    tc_mma_ts(d_tmem, a_hi, b_hi, idesc, (ch != 0 || kk != 0) ? 1u : 0u);
                                    if (!skip_blo) tc_mma_ts(d_tmem, a_hi, b_lw, idesc, 1u);
                                    if (!skip_alo) tc_mma_ts(d_tmem, a_hi + a_lo_off, b_hi, idesc, 1u);
                                }
                            }
                            if (last_chunk) tc_commit(tfull0 + (tq * MB + mb) * 8);  // accumulator -> epilogue
                        }
                        tc_commit(empty0 + s * 8);                      // the stage goes back to the splitter warps
                        if (last_chunk) mbar_arrive(other_turn);         // the other issuer may start its tile
                    }
                    __syncwarp();
                }
#pragma unroll
                for (int mb = 0; !F32 && mb < MB; ++mb) {
                    if (ch == 0 && !(mb == 0 && early_acc)) mbar_wait(tempty0 + slot[mb] * 8, tph[mb] ^ 1);
                    tc_fence_after();
                    const uint32_t d_tmem = acc0 + slot[mb] * BN;
                    if (elect_one()) {
                        if (!skip) {
                            if constexpr (F32) {
#pragma unroll
                                for (int kk = 0; kk < 4; ++kk) {  // four 16-element K steps per 64-element unit
                                    const uint64_t b_hi = ((uint64_t)DESC_HI << 32) | (b_lo + kk * 2);
                                    const uint64_t b_lw = ((uint64_t)DESC_HI << 32) | (b_lo + (KB_TILE_BYTES >> 4) + kk * 2);
                                    const uint32_t a_hi = a_col + mb * a_mb_step + kk * 8;
                                    tc_mma_ts(d_tmem, a_hi, b_hi, idesc, (ch != 0 || kk != 0) ? 1u : 0u);
                                    if (!skip_blo) tc_mma_ts(d_tmem, a_hi, b_lw, idesc, 1u);
                                    if (!skip_alo) tc_mma_ts(d_tmem, a_hi + a_lo_off, b_hi, idesc, 1u);
                                }
                            } else {
#pragma unroll
                                for (int k = 0; k < KBS; ++k) {
#pragma unroll
                                    for (int kk = 0; kk < 4; ++kk) {  // four 32-byte K steps per 128-byte dimension block
                                        const uint64_t bd =
                                            ((uint64_t)DESC_HI << 32) | (b_lo + k * (KB_TILE_BYTES >> 4) + kk * 2);
                                        const uint32_t at = a_col + mb * a_mb_step + k * KB_WORDS + kk * 8;
                                        if (k == 0 && kk == 0)
                                            tc_mma_ts(d_tmem, at, bd, idesc, ch != 0);
                                        else
                                            tc_mma_ts(d_tmem, at, bd, idesc, 1u);
                                    }
                                }
                            }
                        }
                        // accumulator -> epilogue.  When a tile is a single stage, the last block's barrier also tells
                        // the epilogue that the stage has been read (it hands the stage back to the producer): one
                        // tcgen05.commit fewer per tile.
                        if (last_chunk) tc_commit(tfull0 + (tq * MB + mb) * 8);
                        if (mb == MB - 1 && !epi_frees_stage) {
                            if constexpr (PAIR) tc_commit_multicast(empty0 + s * 8, (uint16_t)3);  // the stage is the pair's
                            else tc_commit(empty0 + s * 8);
                        }
                        if (last_chunk && mb == MB - 1) mbar_arrive(other_turn);  // the other issuer may start its tile
                    }
                    __syncwarp();
                }
                a_col += (F32 ? 1 : KBS) * KB_WORDS;
                if (++s == NS) { s = 0; ph ^= 1; }
            }
            TRACED(1, t, 4);
            // this warp's next tile is two tiles on: skip the other warp's stages and accumulators
            s += nch;
            while (s >= NS) { s -= NS; ph ^= 1; }
#pragma unroll
            for (int mb = 0; mb < MB; ++mb) {
                slot[mb] += 2 * MB;
                while (slot[mb] >= nacc) { slot[mb] -= nacc; tph[mb] ^= 1; }
            }
            tq ^= 2;
        }
    } else if (warp == 2) {
        // ===== document segmenter =====
        // Lane l holds the end offset of document wb + l (a 32-document window in registers); the next window is
        // loaded one window ahead, so no tile waits on a global load.  A document's start is its predecessor's end.
        const uint32_t lt_mask = (1u << lane) - 1u;
        const float ninf = -INFINITY;
        // the queries whose scores this CTA writes: all of the launch's, or (CTA pairs) those of its own query block
        const int q_first = PAIR ? (int)rank * (128 / p.Nq_pad) : 0;
        const int q_end = PAIR ? (p.Q < q_first + 128 / p.Nq_pad ? p.Q : q_first + 128 / p.Nq_pad) : p.Q;
        const int64_t never = INT64_MAX;
        auto load_ends = [&](int64_t base) -> int64_t {
            const int64_t idx = base + lane;
            return idx < b_hi ? p.offsets[idx + 1] : never;
        };
        int64_t wb = b_lo;
        int64_t e_cur = load_ends(wb), e_nxt = load_ends(wb + 32);
        int64_t s_first = t_lo;  // start of document wb
        int consumed = 0;        // documents of the current window already assigned to a tile
        uint32_t ord = 0;        // non-empty documents of this CTA seen so far (DOCRING ordinals)
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
                    docring[(ord + nseg + __popc(nb & lt_mask)) & (DOCRING - 1)] = (uint32_t)(idx - b_lo);
                    const uint32_t bit = 1u << (col & 31);
                    w0 = (col >> 5) == 0 ? bit : 0; w1 = (col >> 5) == 1 ? bit : 0;
                    w2 = (col >> 5) == 2 ? bit : 0; w3 = (col >> 5) == 3 ? bit : 0;
                } else if (in_tile) {
                    for (int q = q_first; q < q_end; ++q) p.scores[(int64_t)q * p.B + idx] = ninf;  // empty document (A2)
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
            if (lane == 0) { seg[g].mask[0] = m0; seg[g].mask[1] = m1; seg[g].mask[2] = m2; seg[g].mask[3] = m3; seg[g].ord0 = ord; }
            ord += nseg;
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(sfull + g));
        }
        // documents after the last token of the range can only be empty
        for (int64_t idx = wb + consumed + lane; idx < b_hi; idx += 32)
            for (int q = q_first; q < q_end; ++q) p.scores[(int64_t)q * p.B + idx] = ninf;
    } else if (F32 && warp >= 4 + NSET * n_epi_warps) {
        // ===== fp32 splitter (F32 only): raw fp32 stage -> bf16 hi block + bf16 lo block of an operand stage =====
        // Thread r owns token row r of the tile.  Both layouts are the 128-byte swizzle (16-byte piece index XOR
        // row % 8), so the eight rows a quarter-warp touches in one instruction fall into eight different bank groups.
        const int r = threadIdx.x - 32 * (4 + NSET * n_epi_warps);
        const uint32_t sw = (uint32_t)(r & 7);
        uint32_t s = 0, ph = 0, rs = 0, rph = 0;
        const int64_t nunits = ntiles * nchunks;
        if constexpr (PQD) {
            // The codebook goes to shared memory once per CTA, already split: plane 0 holds every centroid slice's
            // eight bf16 hi parts (16 bytes per (m, k)), plane 1 the lo parts.  Decoding a token is then a pure gather:
            // token row r's 16 codes -> per 64-dimension unit, eight 16-byte hi pieces and eight lo pieces.
            // Layout [m / 8][k][m % 8][16 bytes]: sub-quantiser m lives in bank group m % 8 whatever the code is.  At
            // step oc thread r handles m % 8 = A(r % 8) ^ oc, A = multiplication by x in GF(8) (x^3 + x + 1): A and A + I
            // are both bijections, so the eight lanes of a quarter-warp READ eight different bank groups (m % 8) and
            // WRITE eight different ones (the operand swizzle puts piece m % 8 of row r into group (m % 8) ^ (r % 8)) --
            // a random gather with no bank conflicts at all.
            const uint32_t ar = ((sw << 1) ^ ((sw & 4u) ? 0xbu : 0u)) & 7u;  // A(r % 8)
            const bool half_mode = p.half_mode != 0;
            {
                const uint4* g = reinterpret_cast<const uint4*>(p.codebooks);
                for (int e0 = r; e0 < 16 * 256; e0 += 128) {
                    const int m_ = e0 >> 8, k_ = e0 & 255;
                    const int e = (((m_ >> 3) * 256 + k_) << 3) + (m_ & 7);
                    const uint4 y0 = ldg_nc16(g + 2 * e0), y1 = ldg_nc16(g + 2 * e0 + 1);
                    uint4 hi, lo;
                    encode_pair(__uint_as_float(y0.x), __uint_as_float(y0.y), hi.x, lo.x, half_mode);
                    encode_pair(__uint_as_float(y0.z), __uint_as_float(y0.w), hi.y, lo.y, half_mode);
                    encode_pair(__uint_as_float(y1.x), __uint_as_float(y1.y), hi.z, lo.z, half_mode);
                    encode_pair(__uint_as_float(y1.z), __uint_as_float(y1.w), hi.w, lo.w, half_mode);
                    *reinterpret_cast<uint4*>(cb_ptr + e * 16) = hi;
                    if (!half_mode) *reinterpret_cast<uint4*>(cb_ptr + cb_bytes / 2 + e * 16) = lo;
                }
                asm volatile("bar.sync 1, 128;" ::: "memory");  // the four splitter warps
            }
            for (int64_t t = 0; t < ntiles; ++t) {
                mbar_wait(smem_u32(rfull + rs), rph);
                const uint4 cw = *reinterpret_cast<const uint4*>(rw_ptr + (size_t)rs * raw_bytes + r * 16);
                const uint32_t cword[4] = {cw.x, cw.y, cw.z, cw.w};
#pragma unroll
                for (int ch = 0; ch < 2; ++ch) {  // d = 128: two 64-dimension units per tile (compile-time: cword stays in registers)
                    mbar_wait(smem_u32(empty + s), ph ^ 1);
                    uint8_t* op = st_ptr + (size_t)s * stage_bytes + r * KB_BYTES;
#pragma unroll
                    for (int oc = 0; oc < 8; ++oc) {  // sub-quantiser m = 8*ch + mm fills 16-byte piece mm of the unit
                        const uint32_t mm = ar ^ (uint32_t)oc;
                        const uint32_t wsel = (mm & 4u) ? cword[2 * ch + 1] : cword[2 * ch];
                        const uint32_t code = __byte_perm(wsel, 0u, 0x4440u | (mm & 3u));
                        const uint8_t* e = cb_ptr + ((size_t)(((uint32_t)ch * 256u + code) * 8u + mm) << 4);
                        const uint32_t o = (mm ^ sw) << 4;
                        *reinterpret_cast<uint4*>(op + o) = *reinterpret_cast<const uint4*>(e);
                        if (!half_mode)
                            *reinterpret_cast<uint4*>(op + KB_TILE_BYTES + o) = *reinterpret_cast<const uint4*>(e + cb_bytes / 2);
                    }
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    __syncwarp();
                    if (lane == 0) mbar_arrive(smem_u32(full + s));
                    if (++s == (uint32_t)p.NS) { s = 0; ph ^= 1; }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(rempty + rs));
                if (++rs == (uint32_t)p.NR) { rs = 0; rph ^= 1; }
            }
        }
        for (int64_t u = 0; !PQD && u < nunits; ++u) {
            mbar_wait(smem_u32(rfull + rs), rph);
            mbar_wait(smem_u32(empty + s), ph ^ 1);
            const uint8_t* raw = rw_ptr + (size_t)rs * raw_bytes + r * KB_BYTES;
            uint8_t* op = st_ptr + (size_t)s * stage_bytes + r * KB_BYTES;
#pragma unroll
            for (int oc = 0; oc < 8; ++oc) {  // 8 fp32 (two 16-byte pieces) in -> 8 bf16 hi (one piece) + 8 bf16 lo out
                const uint8_t* blk = raw + (oc >> 2) * KB_TILE_BYTES;
                const uint32_t c0 = (uint32_t)(2 * (oc & 3));
                const float4 x0 = *reinterpret_cast<const float4*>(blk + ((c0 ^ sw) << 4));
                const float4 x1 = *reinterpret_cast<const float4*>(blk + (((c0 + 1) ^ sw) << 4));
                uint4 hi, lo;
                split_pair(x0.x, x0.y, hi.x, lo.x);
                split_pair(x0.z, x0.w, hi.y, lo.y);
                split_pair(x1.x, x1.y, hi.z, lo.z);
                split_pair(x1.z, x1.w, hi.w, lo.w);
                const uint32_t o = ((uint32_t)oc ^ sw) << 4;
                *reinterpret_cast<uint4*>(op + o) = hi;
                *reinterpret_cast<uint4*>(op + KB_TILE_BYTES + o) = lo;
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> tensor-pipe reads
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(smem_u32(full + s));
                mbar_arrive(smem_u32(rempty + rs));
            }
            if (++s == (uint32_t)p.NS) { s = 0; ph ^= 1; }
            if (++rs == (uint32_t)p.NR) { rs = 0; rph ^= 1; }
        }
    } else if (warp >= 4) {
        // ===== epilogue: running rowmax, segmented by document; max -> sum =====
        int set = (warp - 4) / n_epi_warps;                  // which half of every tile's columns is this warp's (NSET == 2)
        if (NSET == 2) asm volatile("" : "+r"(set));           // opaque: otherwise re-derived from %tid.x (S2R) at every use
        const int ew = (warp - 4) % n_epi_warps, mb = ew >> 2, quad = warp & 3;
        const int row = ((int)rank + mb) * 128 + quad * 32 + lane;   // this thread's query row = TMEM lane quad*32+lane of block mb
        const int q = row / p.Nq_pad, i = row - q * p.Nq_pad;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(quad * 32) << 16);

        // a2: the thread's query row -> TMEM, two 16-bit elements per column: columns [mb*NKB*32, +NKB*32), or for
        // F32 the bf16 hi halves in [mb*2*NKB*32, +NKB*32) followed by the lo halves.  Rows no query token owns
        // are zero (finite similarities that never reach a score, A5).  Done by the first set only.
        if (set == 0)
        {
            const bool row_valid = (q < p.Q) && (i < p.Nq);
            const bool half_mode = PQD && p.half_mode != 0;
            const uint8_t* src = static_cast<const uint8_t*>(p.queries) + ((int64_t)q * p.Nq + i) * p.row_bytes;
            for (int kb = 0; kb < p.NKB; ++kb) {
                if constexpr (F32) {
#pragma unroll 1
                    for (int half = 0; half < 2; ++half) {  // 32 fp32 -> 16 columns of hi, 16 columns of lo
                        uint32_t hi[16], lo[16];
                        if (p.q_fmt == 0) {  // fp32 query rows
#pragma unroll
                            for (int j = 0; j < 8; ++j) {
                                uint4 x = make_uint4(0, 0, 0, 0);
                                if (row_valid) x = ldg_nc16(src + kb * 256 + half * 128 + j * 16);
                                encode_pair(__uint_as_float(x.x), __uint_as_float(x.y), hi[2 * j], lo[2 * j], half_mode);
                                encode_pair(__uint_as_float(x.z), __uint_as_float(x.w), hi[2 * j + 1], lo[2 * j + 1], half_mode);
                            }
                        } else {             // 16-bit query rows (PQD): widened exactly to fp32 first
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                uint4 x = make_uint4(0, 0, 0, 0);
                                if (row_valid) x = ldg_nc16(src + kb * 128 + half * 64 + j * 16);
                                const uint32_t w4[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                                for (int e = 0; e < 4; ++e) {
                                    float f0, f1;
                                    if (p.q_fmt == 2) {  // bf16: the upper half of an fp32
                                        f0 = __uint_as_float(w4[e] << 16);
                                        f1 = __uint_as_float(w4[e] & 0xffff0000u);
                                    } else {
                                        const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w4[e]));
                                        f0 = f.x;
                                        f1 = f.y;
                                    }
                                    encode_pair(f0, f1, hi[4 * j + e], lo[4 * j + e], half_mode);
                                }
                            }
                        }
                        const int planes = p.skip_alo ? 1 : 2;
                        const uint32_t col = (uint32_t)((mb * planes * p.NKB + kb) * KB_WORDS + half * 16);
                        tmem_st16(lane_addr + col, hi);
                        if (planes == 2) tmem_st16(lane_addr + col + (uint32_t)(p.NKB * KB_WORDS), lo);
                    }
                } else {
                    uint32_t w[KB_WORDS];
#pragma unroll
                    for (int j = 0; j < KB_WORDS / 4; ++j) {
                        uint4 x = make_uint4(0, 0, 0, 0);
                        if (row_valid && kb * KB_BYTES + j * 16 < p.row_bytes) x = ldg_nc16(src + kb * KB_BYTES + j * 16);
                        w[4 * j] = x.x; w[4 * j + 1] = x.y; w[4 * j + 2] = x.z; w[4 * j + 3] = x.w;
                    }
                    tmem_st32(lane_addr + (uint32_t)((mb * p.NKB + kb) * KB_WORDS), w);
                }
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(aready));
        }

        // max -> sum constants of this warp: its 32 rows hold 32/Nq_pad queries, the first one being q0
        const int q0 = (((int)rank + mb) * 128 + quad * 32) / p.Nq_pad;
        const int nsub = 32 / p.Nq_pad;
        const int nvalid = p.Q - q0 < 0 ? 0 : (p.Q - q0 < nsub ? p.Q - q0 : nsub);
        const uint32_t cfg = pack_cfg(p.Nq, p.Nq_pad, nvalid);
        float* out = p.scores + (int64_t)q0 * p.B + b_lo;
        const uint32_t pend = smem_u32(pend_all) + (uint32_t)(warp - 4) * (PEND_IDS + PEND * 4);
        const bool skip_math = PROBE(p, 1);
        const int64_t B = p.B;
        const uint32_t ring = smem_u32(docring);
        const bool frees_stage = !F32 && !PAIR && nchunks == 1 && (ALT || set == 0) && ew == 4 * (MB - 1);  // see the MMA warps

        // Two sets (16-bit inputs): set 0 reduces columns 0..63 of every tile, set 1 columns 64..127.  A tcgen05.ld
        // blocks the issuing warp until its data are in registers (measured: two loads "in flight" from one warp take
        // as long as two in sequence, ~90 clk per 32 columns), so a warp cannot overlap its own TMEM reads with its
        // own arithmetic; a second warp on the same sub-partition and TMEM lanes can, and the accumulator goes back to
        // the MMA warps after two loads per warp instead of four.  The running maximum crosses a range boundary through a
        // 32-float mailbox: a range is reduced from -inf, the first document it closes is parked provisionally, and only
        // at the END of the range is the previous range's carry awaited and folded in (into that parked value, or into
        // the still open segment), after which the range's own carry goes to the other set.  The serial chain per
        // tile is therefore two mailbox hops, not two range reductions.
        const uint32_t mail_out = smem_u32(mail) + (uint32_t)((set * 8 + ew) * 32 + lane) * 4;
        const uint32_t mail_in = smem_u32(mail) + (uint32_t)(((set ^ 1) * 8 + ew) * 32 + lane) * 4;
        const uint32_t carry_out = smem_u32(carry + set * 8 + ew), carry_in = smem_u32(carry + (set ^ 1) * 8 + ew);
        uint32_t cph = 0;

        EpiState st;
        st.m = -INFINITY;  // Alg. 3 line 4
        st.ord = 0;
        st.np = 0;
        st.unresolved = false;
        st.first = NONE;
        st.head = 0.f;
        auto resolve = [&]() {
            if constexpr (NSET == 2) {
                mbar_wait(carry_in, cph);
                cph ^= 1;
                const float cin = lds_f32(mail_in);
                if (st.first != NONE) sts_f32(pend + (st.first * PEND_PITCH + lane) * 4, fmaxf(st.head, cin));
                else st.m = fmaxf(st.m, cin);  // nothing closed yet: the open segment continues the previous tile's
                st.unresolved = false;
            }
        };
        const uint32_t nacc = (uint32_t)p.NACC, NS = (uint32_t)p.NS;
        const uint32_t acc0 = lane_addr + (uint32_t)p.acc_col0;
        // ring positions of this warp's first tile (ALT: set s starts at tile s and advances two tiles at a time)
        constexpr uint32_t TSTEP = ALT ? 2u : 1u;
        uint32_t slot = (uint32_t)mb + (ALT ? (uint32_t)(set * MB) : 0u), g = ALT ? (uint32_t)set : 0u, gph = 0, rs = ALT ? (uint32_t)set : 0u;
        while (slot >= nacc) slot -= nacc;
        while (rs >= NS) rs -= NS;
        uint32_t ord_tile = 0;  // (two sets) non-empty documents that ended in earlier tiles
        const bool tr = quad == 0 && (set == 0 || mb == 0);  // (probe builds) the warps whose clocks are traced
        const int trole = set == 0 ? 2 + mb : 0;
        const int nt = (int)ntiles;
        for (int t = ALT ? set : 0; t < nt; t += (int)TSTEP) {
            if (tr) TRACED(trole, t, 0);
            mbar_wait(smem_u32(tfull + (uint32_t)(t & 3) * MB + mb), (uint32_t)(t >> 2) & 1u);
            tc_fence_after();
            if (frees_stage) {  // the tile's only stage has been read by the tensor pipe: back to the producer
                if (lane == 0) mbar_arrive(smem_u32(empty + rs));
                rs += TSTEP;
                while (rs >= NS) rs -= NS;
            }
            if (tr) TRACED(trole, t, 1);
            const uint32_t taddr = acc0 + slot * BN;
            if constexpr (F32) {
                // 512 threads leave 128 registers each: the accumulator is read in two halves of 64 columns.  A tile
                // costs the tensor pipe three MMAs per K step here, so the later release is off the critical path.
                float v[64];
                tmem_ld32(taddr, v);
                tmem_ld32(taddr + 32, v + 32);
                mbar_wait(smem_u32(sfull + g), gph);
                const uint4 mask = *reinterpret_cast<const uint4*>(seg[g].mask);
                tmem_ld_wait32(v);
                tmem_ld_pin32(v + 32);
                process32(v, mask.x, st, pend, ring, out, B, cfg, lane, skip_math, resolve);
                process32(v + 32, mask.y, st, pend, ring, out, B, cfg, lane, skip_math, resolve);
                tmem_ld32(taddr + 64, v);
                tmem_ld32(taddr + 96, v + 32);
                tmem_ld_wait32(v);
                tmem_ld_pin32(v + 32);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(tempty + slot));
                process32(v, mask.z, st, pend, ring, out, B, cfg, lane, skip_math, resolve);
                process32(v + 32, mask.w, st, pend, ring, out, B, cfg, lane, skip_math, resolve);
            } else {
                float v[32];
                constexpr int NW = ALT ? 4 : 4 / NSET;         // 32-column words of a tile that are this warp's
                const uint32_t c0 = ALT ? 0u : (uint32_t)set * (NW * 32);  // its first column
                tmem_ld32(taddr + c0, v);
                mbar_wait(smem_u32(sfull + g), gph);
                const uint4 mask = *reinterpret_cast<const uint4*>(seg[g].mask);
                const uint32_t wds[4] = {mask.x, mask.y, mask.z, mask.w};
                if (ALT) {  // ordinal of the first document that ends in this tile: the segmenter's running count
                    st.ord = seg[g].ord0;
                } else if (NSET == 2) {  // ordinal of the first document that ends in this warp's columns
                    const uint32_t lo = __popc(mask.x) + __popc(mask.y);
                    st.ord = ord_tile + (set ? lo : 0);
                    ord_tile += lo + __popc(mask.z) + __popc(mask.w);
                }
                if (NSET == 2 && (set != 0 || t != 0)) {  // reduced from -inf; the previous range's carry is folded in at the end
                    st.m = -INFINITY;
                    st.unresolved = true;
                    st.first = NONE;
                }
#pragma unroll
                for (int i = 0; i < NW; ++i) {
                    if (i) tmem_ld32(taddr + c0 + 32 * i, v);
                    tmem_ld_wait32(v);
                    if (i == NW - 1) {  // this warp's columns are in registers
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(smem_u32(tempty + slot));
                    }
                    if (tr) TRACED(trole, t, 2 + i);
                    process32(v, wds[(NSET == 2 && !ALT && set ? 2 : 0) + i], st, pend, ring, out, B, cfg, lane, skip_math, resolve);
                }
                if constexpr (NSET == 2) {
                    if (st.unresolved) resolve();
                    if ((!ALT && set == 0) || t + 1 < nt) {  // this range's carry -> the other set
                        sts_f32(mail_out, st.m);
                        __syncwarp();
                        if (lane == 0) mbar_arrive(carry_out);
                    }
                }
                if (tr) TRACED(trole, t, 6);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(sempty + g));
            slot += MB * TSTEP;
            while (slot >= nacc) slot -= nacc;
            g += TSTEP;
            if (g >= NSEG) { g -= NSEG; gph ^= 1; }
        }
        if (st.np) drain(pend, st.np, out, B, cfg, lane);
    }

    // ---- teardown --------------------------------------------------------------------------------------------
    tc_fence_before();
    if constexpr (PAIR) cluster_sync_all();  // no CTA leaves while its peer can still signal its barriers
    else __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"((uint32_t)TMEM_COLS)
                     : "memory");
    }
}

// scores[q,b] = sum_j parts[q*nparts + j, b], j ascending (queries longer than 32 tokens)
__global__ void sum_parts_kernel(const float* __restrict__ parts, float* __restrict__ scores, int Q, int nparts,
                                 int64_t B) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (int64_t)Q * B) return;
    const int64_t q = i / B, b = i - q * B;
    float acc = parts[(q * nparts) * B + b];
    for (int j = 1; j < nparts; ++j) acc += parts[(q * nparts + j) * B + b];
    scores[i] = acc;
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

// Small-batch latency: encoding a tensor map and setting a kernel attribute cost microseconds of host time per call, as
// much as a 1,000-document batch takes on the device.  Both depend only on (store address, shape, dtype) / (kernel,
// device), so recent results are kept per process.  A tensor map holds no data, only the address and the geometry.
struct MapKey {
    const void* base;
    uint64_t rows, cols;
    uint32_t box_cols, box_rows;
    int dtype, device;
};
struct MapEntry {
    MapKey key;
    CUtensorMap map;
    bool valid;
};
std::mutex g_cache_mu;
MapEntry g_maps[8];
int g_map_next = 0;

bool cached_map_2d(CUtensorMap* map, int device, tms_dtype dtype, const void* base, uint64_t rows, uint64_t cols,
                   uint32_t box_cols, uint32_t box_rows) {
    MapKey key;
    memset(&key, 0, sizeof(key));  // padding bytes take part in the comparison
    key.base = base; key.rows = rows; key.cols = cols; key.box_cols = box_cols; key.box_rows = box_rows;
    key.dtype = (int)dtype; key.device = device;
    std::lock_guard<std::mutex> lock(g_cache_mu);
    for (const MapEntry& e : g_maps)
        if (e.valid && memcmp(&e.key, &key, sizeof(key)) == 0) { *map = e.map; return true; }
    if (!make_map_2d(map, dtype, base, rows, cols, box_cols, box_rows)) return false;
    MapEntry& e = g_maps[g_map_next];
    g_map_next = (g_map_next + 1) % 8;
    e.key = key; e.map = *map; e.valid = true;
    return true;
}

struct AttrEntry {
    const void* kern;
    int device;
    uint32_t smem;
};
AttrEntry g_attrs[32];
int g_nattrs = 0;

// cudaFuncAttributeMaxDynamicSharedMemorySize >= smem for this kernel on this device (set once per growth)
bool ensure_smem_attr(const void* kern, int device, uint32_t smem) {
    std::lock_guard<std::mutex> lock(g_cache_mu);
    for (int i = 0; i < g_nattrs; ++i)
        if (g_attrs[i].kern == kern && g_attrs[i].device == device) {
            if (g_attrs[i].smem >= smem) return true;
            if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return false;
            g_attrs[i].smem = smem;
            return true;
        }
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return false;
    if (g_nattrs < 32) g_attrs[g_nattrs++] = AttrEntry{kern, device, smem};
    return true;
}

int next_pow2(int v) {
    int p = 1;
    while (p < v) p <<= 1;
    return p;
}

// Number of equal parts a query of Nq tokens is scored in: the smallest n with Nq % n == 0 and Nq / n <= 32
// (1 for Nq <= 32; Nq / 32 for multiples of 32; 2 x 24 for Nq = 48; Nq parts of one token for a prime Nq > 32).
int query_parts(int Nq) {
    for (int n = 1; n <= Nq; ++n)
        if (Nq % n == 0 && Nq / n <= 32) return n;
    return Nq;
}

struct Plan {
    Params p;           // per-launch fields (queries, scores, Q) are filled in by the launcher
    int MB, KBS;        // query blocks per launch, dimension blocks per stage
    bool f32;           // fp32 inputs: split into bf16 pairs on the fly
    bool pqd;           // decode-and-contract PQ variant
    int nparts;         // equal parts a query is scored in (1 unless Nq > 32)
    int Qg;             // queries per launch
    int nset;           // epilogue warp sets
    bool pair;          // clusters of two CTAs, one query block each, document tiles multicast to both
    bool alt;           // two epilogue sets on alternate tiles instead of column halves
    uint32_t smem_bytes;
};

uint32_t fixed_smem(int MB, int nset) {
    const uint32_t warps = (uint32_t)nset * 4u * MB;
    return (uint32_t)sizeof(SegInfo) * NSEG + DOCRING * 4 + warps * PEND * (PEND_PITCH + 1) * 4 +
           2 * 8 * 32 * 4 + 8u * (2 * MAX_STAGES + 8 + MAX_ACC + 2 * NSEG + 2 * MAX_RAW + 4 + 16) + 4 * 8 + 1024 /* alignment slack */;
}

// Shape -> kernel parameters; false when the tcgen05 path does not cover it.
bool plan(const DenseArgs& a, Plan& pl) {
    if (a.B <= 0 || a.T <= 0) return false;
    const bool pqd = a.codes != nullptr;  // decode-and-contract PQ: fp32-split machinery, 16-bit or fp32 queries
    if (pqd && (a.d != 128 || !a.codebooks)) return false;
    const bool f32 = pqd || a.dtype == TMS_DTYPE_F32;
    const int esize = (int)dtype_size(a.dtype);
    const int row_bytes = a.d * esize;  // of a query row; also of a document row unless pqd
    // fp32: whole 64-element units (256 bytes).  16-bit: any 16-byte multiple -- TMA zero-fills the part of the last
    // 128-byte dimension block that lies beyond the row, and the query rows are zero-padded the same way.
    if (!pqd && row_bytes % (f32 ? 2 * KB_BYTES : 16) != 0) return false;
    // A query's rows must sit inside one warp's 32 TMEM lanes.  Longer queries are scored as n equal parts of Nq/n <= 32
    // tokens -- queries[Q,Nq,d] read as [Q*n, Nq/n, d] -- into a workspace of partial scores that
    // sum_parts_kernel adds up (Eq. 1's outer sum is associative over query tokens, pin P9).
    const int nparts = query_parts(a.Nq);
    if (nparts > 1 && (!a.workspace || a.workspace_bytes < dense_tc_workspace_bytes(a.Q, a.Nq, a.B))) return false;
    if ((int64_t)a.Q * nparts > (1 << 20)) return false;
    const int Nq_part = a.Nq / nparts;
    const int nqp = next_pow2(Nq_part);
    const int NKB = f32 ? a.d / 64 : (row_bytes + KB_BYTES - 1) / KB_BYTES;  // fp32: 64-element units
    // TMEM budget: query rows (fp32: bf16 hi and lo halves) + at least MB accumulators of 128 columns
    // bf16 queries split into (x, 0) and fp16 mode has no lo parts: no lo plane, and one more accumulator fits
    const bool skip_alo = pqd && (a.dtype == TMS_DTYPE_BF16 || a.pq_half);
    const int a_cols_per_block = ((f32 && !skip_alo) ? 2 : 1) * NKB * KB_WORDS;
    int MB = 2;
    if (MB * a_cols_per_block + MB * BN > TMEM_COLS) MB = 1;
    if (MB * a_cols_per_block + MB * BN > TMEM_COLS) return false;  // d too large for a resident query block
    const int per_block = 128 / nqp;  // queries per 128-row block
    // two query blocks wanted but only one fits tensor memory (16-bit d in (256, 768]): a CTA pair holds one block each
    // and shares the document tiles by multicast, so the store is still read once per 256 rows
    const bool pair = !f32 && MB == 1 && a.Q * nparts > per_block;
    if (a.Q * nparts <= per_block) MB = 1;
    Params& p = pl.p;
    p.offsets = a.offsets;
    p.B = a.B;
    p.T = a.T;
    p.tok0 = 0;
    p.Tseg = a.T;
    p.seg_first = p.seg_last = 1;
    p.Nq = Nq_part;
    p.Nq_pad = nqp;
    p.row_bytes = row_bytes;
    p.NKB = NKB;
    p.kb_elems = KB_BYTES / esize;
    p.codes = a.codes;
    p.codebooks = a.codebooks;
    p.q_fmt = (int)a.dtype;  // tms_dtype: 0 fp32, 1 fp16, 2 bf16
    p.half_mode = pqd && a.pq_half;
    p.skip_alo = skip_alo;
    p.NACC = (TMEM_COLS - MB * a_cols_per_block) / BN;
    if (p.NACC > MAX_ACC) p.NACC = MAX_ACC;
    p.acc_col0 = TMEM_COLS - p.NACC * BN;
#ifdef TMS_PROBES
    {
        static const int dbg = [] { const char* e = getenv("TMS_DEBUG"); return e ? atoi(e) : 0; }();
        p.debug = dbg;
        p.docs_raw = a.docs;
    }
#endif
    const uint32_t fmt = ((!f32 && a.dtype == TMS_DTYPE_F16) || (pqd && a.pq_half)) ? 0u : 1u;  // the split paths feed bf16 pairs
    // instruction descriptor: fp32 accumulate, A/B format, both K-major, N = 128, M = 128
    p.idesc = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    pl.MB = MB;
    pl.pair = pair;
    pl.Qg = (pair ? 2 : MB) * per_block;
    pl.nparts = nparts;
    pl.f32 = f32;
    pl.pqd = pqd;
    // two epilogue sets when documents are short on average (< 100 tokens: most tiles then hold a document boundary
    // or several, and the segmented reduction binds), measured on config 3 (mean 72 tokens) against config 2 (128)
    pl.nset = (!f32 && a.T < 100 * a.B) ? 2 : 1;
    // one query block and long documents: a lone epilogue warp per scheduler cannot keep up with the stream (TMEM loads
    // and the reduction are one latency chain: ~870 clk per tile against 634 clk of HBM time at d = 64), so two sets take
    // alternate tiles (measured: c4-d64 -24 %, c2-q4 -6 %; with two blocks or short documents it does not pay)
    pl.alt = !f32 && !pair && MB == 1 && pl.nset == 1;
    if (pl.alt) pl.nset = 2;
#ifdef TMS_PROBES
    if (const char* e = getenv("TMS_NSET")) { const int n = atoi(e); if (!f32 && (n == 1 || n == 2)) pl.nset = n; }
    if (const char* e = getenv("TMS_ALT")) { pl.alt = !f32 && !pair && atoi(e) != 0; if (pl.alt) pl.nset = 2; else if (MB == 1 && a.T >= 100 * a.B) pl.nset = 1; }
#endif
    pl.KBS = f32 ? 2 : ((NKB % 2 == 0) ? 2 : 1);
    const uint32_t fixed = fixed_smem(MB, pl.nset);
    const uint32_t stage_bytes = (uint32_t)pl.KBS * KB_TILE_BYTES;
    int ns = (int)((SMEM_LIMIT - fixed) / stage_bytes);
    p.NR = 0;
    if (pqd) {  // 128 KB codebook + four 2 KB code stages, the rest for 32 KB operand stages (hi + lo block); with fp16
                // operands there are no lo parts: 64 KB codebook, 16 KB stages
        const uint32_t cb = p.half_mode ? 16u * 256u * 8u * 2u : 16u * 256u * 8u * 4u, raw = MAX_RAW * BN * 16u;
        const uint32_t sb = p.half_mode ? (uint32_t)KB_TILE_BYTES : stage_bytes;
        if (fixed + cb + raw + sb > SMEM_LIMIT) return false;
        p.NR = MAX_RAW;
        ns = (int)((SMEM_LIMIT - fixed - cb - raw) / sb);
        p.NS = ns > MAX_STAGES ? MAX_STAGES : ns;
        pl.smem_bytes = (uint32_t)p.NS * sb + raw + cb + fixed;
        return p.NS >= 1;
    }
    if (f32) {  // 32 KB raw stages and 32 KB operand stages share the budget
        p.NR = ns / 2 > MAX_RAW ? MAX_RAW : ns / 2;
        ns -= p.NR;
        if (p.NR < 1) return false;
    }
    p.NS = ns > MAX_STAGES ? MAX_STAGES : ns;
    pl.smem_bytes = (uint32_t)(p.NS + p.NR) * stage_bytes + fixed;
    return p.NS >= (f32 ? 1 : 2);
}

}  // namespace

#ifdef TMS_PROBES
// probe builds only: copies the clock trace of CTA TRACE_CTA to the host ([role][tile][event])
extern "C" int tms_trace_read(long long* host, int* roles, int* tiles, int* events) {
    *roles = TRACE_ROLES; *tiles = TRACE_NT; *events = TRACE_EV;
    return cudaMemcpyFromSymbol(host, g_trace, sizeof(long long) * TRACE_ROLES * TRACE_NT * TRACE_EV) == cudaSuccess ? 0 : 1;
}
#endif

size_t dense_tc_workspace_bytes(int Q, int Nq, int64_t B) {
    if (Nq <= 32) return 0;
    return sizeof(float) * (size_t)Q * (size_t)query_parts(Nq) * (size_t)B;
}

bool dense_tc_shape_ok(const DenseArgs& a) {
    Plan pl;
    return plan(a, pl) && pl.smem_bytes <= SMEM_LIMIT;
}

bool dense_tc_supports(const DenseArgs& a) {
    const DeviceInfo* di = device_info();
    if (!di || di->cc_major != 10) return false;
    Plan pl;
    return plan(a, pl) && pl.smem_bytes <= (uint32_t)di->max_smem_optin;
}

int launch_dense_tc(const DenseArgs& a) {
    const DeviceInfo* di = device_info();
    if (!di) return TMS_ERR_CUDA;
    Plan pl;
    if (di->cc_major != 10 || !plan(a, pl) || pl.smem_bytes > (uint32_t)di->max_smem_optin) return TMS_ERR_UNSUPPORTED;

    void (*kern)(const CUtensorMap, const Params) = nullptr;
    if (pl.pqd) kern = pl.MB == 1 ? dense_tc_kernel<1, 2, true, true, 1> : dense_tc_kernel<2, 2, true, true, 1>;
    else if (pl.f32) kern = pl.MB == 1 ? dense_tc_kernel<1, 2, true, false, 1> : dense_tc_kernel<2, 2, true, false, 1>;
    else if (pl.pair) {
        if (pl.nset == 1) kern = pl.KBS == 1 ? dense_tc_kernel<1, 1, false, false, 1, true> : dense_tc_kernel<1, 2, false, false, 1, true>;
        else kern = pl.KBS == 1 ? dense_tc_kernel<1, 1, false, false, 2, true> : dense_tc_kernel<1, 2, false, false, 2, true>;
    } else if (pl.alt) {
        if (pl.MB == 1) kern = pl.KBS == 1 ? dense_tc_kernel<1, 1, false, false, 2, false, true> : dense_tc_kernel<1, 2, false, false, 2, false, true>;
        else kern = pl.KBS == 1 ? dense_tc_kernel<2, 1, false, false, 2, false, true> : dense_tc_kernel<2, 2, false, false, 2, false, true>;
    } else if (pl.nset == 1) {
        if (pl.MB == 1) kern = pl.KBS == 1 ? dense_tc_kernel<1, 1, false, false, 1> : dense_tc_kernel<1, 2, false, false, 1>;
        else kern = pl.KBS == 1 ? dense_tc_kernel<2, 1, false, false, 1> : dense_tc_kernel<2, 2, false, false, 1>;
    } else {
        if (pl.MB == 1) kern = pl.KBS == 1 ? dense_tc_kernel<1, 1, false, false, 2> : dense_tc_kernel<1, 2, false, false, 2>;
        else kern = pl.KBS == 1 ? dense_tc_kernel<2, 1, false, false, 2> : dense_tc_kernel<2, 2, false, false, 2>;
    }
    if (!ensure_smem_attr(reinterpret_cast<const void*>(kern), di->device, pl.smem_bytes)) return TMS_ERR_CUDA;
    // TMA tile coordinates are 32-bit: a store of 2^31 - 128 tokens or more is scored in token segments of 2^30 tokens,
    // one launch per segment (and query group), each with a tensor map that starts at the segment's first token.  A
    // document belongs to the segment its first token lies in and may reach into the next one (by contract no document
    // of such a store is longer than 2^30 - 128 tokens: one that starts on a segment's last token then still ends
    // inside map_rows below).  Smaller stores are one segment.
    const int64_t SEG = 1ll << 30;
    const int64_t nseg = a.T < (1ll << 31) - BN ? 1 : (a.T + SEG - 1) / SEG;
    // one launch per group of Qg queries (up to 256 query rows): the store is streamed once per group
    const int Qeff = a.Q * pl.nparts;  // queries as the kernel sees them (32-token parts of long queries)
    float* dst = pl.nparts > 1 ? static_cast<float*>(a.workspace) : a.scores;
    for (int64_t sg = 0; sg < nseg; ++sg)
    for (int q0 = 0; q0 < Qeff; q0 += pl.Qg) {
        const int64_t tok0 = nseg == 1 ? 0 : sg * SEG;
        const int64_t Tseg = nseg == 1 ? a.T : (a.T - tok0 < SEG ? a.T - tok0 : SEG);
        int64_t map_rows = a.T - tok0;  // rows the segment's documents can touch: its own tokens + one more segment
        if (map_rows > 2 * SEG - BN) map_rows = 2 * SEG - BN;
        CUtensorMap map_docs = {};  // unused by the PQ decode variant
        if (!pl.pqd && !cached_map_2d(&map_docs, di->device, a.dtype,
                                      static_cast<const uint8_t*>(a.docs) + (size_t)tok0 * pl.p.row_bytes,
                                      (uint64_t)map_rows, (uint64_t)a.d, (uint32_t)pl.p.kb_elems,
                                      pl.pair ? BN / 2 : BN))  // a pair's CTAs load half a tile each
            return TMS_ERR_CUDA;
        // no more CTAs than 128-token tiles; one CTA per SM
        int64_t grid = (Tseg + BN - 1) / BN;
        if (grid > di->num_sms) grid = di->num_sms;
        if (pl.pair) {  // one range per pair of CTAs (the two SMs of a TPC)
            int64_t pairs = (Tseg + BN - 1) / BN;
            if (pairs > di->num_sms / 2) pairs = di->num_sms / 2;
            grid = 2 * pairs;
        }
#ifdef TMS_PROBES
        if (const char* e = getenv("TMS_GRID")) { const int g = atoi(e); if (g > 0 && g < grid) grid = g; }
        if (const char* e = getenv("TMS_NS")) { const int n = atoi(e); if (n > 0 && n < pl.p.NS) pl.p.NS = n; }
#endif
        Params p = pl.p;
        p.tok0 = tok0;
        p.Tseg = Tseg;
        p.seg_first = sg == 0;
        p.seg_last = sg == nseg - 1;
        p.Q = Qeff - q0 < pl.Qg ? Qeff - q0 : pl.Qg;
        p.queries = static_cast<const uint8_t*>(a.queries) + (size_t)q0 * p.Nq * p.row_bytes;
        p.scores = dst + (int64_t)q0 * a.B;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)grid);
        cfg.blockDim = dim3(128 + pl.nset * 128 * pl.MB + (pl.f32 ? 128 : 0));
        cfg.dynamicSmemBytes = pl.smem_bytes;
        cfg.stream = a.stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = pl.pair ? 2 : 1;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        const cudaError_t err = cudaLaunchKernelEx(&cfg, kern, map_docs, p);
        count_launch();
        if (err != cudaSuccess || cudaGetLastError() != cudaSuccess) return TMS_ERR_CUDA;
    }
    if (pl.nparts > 1) {
        const int64_t n = (int64_t)a.Q * a.B;
        sum_parts_kernel<<<(unsigned)((n + 255) / 256), 256, 0, a.stream>>>(dst, a.scores, a.Q, pl.nparts, a.B);
        count_launch();
        if (cudaGetLastError() != cudaSuccess) return TMS_ERR_CUDA;
    }
    return TMS_OK;
}

}  // namespace tms
