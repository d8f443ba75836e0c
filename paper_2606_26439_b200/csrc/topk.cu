// topk.cu -- per-query top-k over scores[Q, B]: the step right after scoring ("followed by torch.topk ... adding
// < 0.1 ms").  Order: score descending, ties by lower document index first; -inf
// (empty documents) sorts last.
//
// A score and its document index are packed into one 64-bit key whose unsigned order IS the ranking order:
// high word = the float's bits mapped monotonically to uint32, low word = ~index.  Level 0 cuts every query's
// scores into chunks of 4096, sorts each chunk in shared memory (bitonic, descending) and keeps its k best keys;
// the following levels do the same on the surviving keys until one chunk is left, whose k best are unpacked into
// values[Q, k] and indices[Q, k].  With k <= 1024 every level shrinks the list at least four-fold.
#include <mutex>

#include "tms_internal.h"

// Built-in scratch of tms_topk_static (include/tms.h): the two ping-pong key buffers of the selection levels, for
// callers that have no device memory to hand over as a workspace.  It is part of the library's device image, so every
// GPU that loads libtms.so carries these TMS_TOPK_STATIC_SCRATCH_BYTES until the process exits, whether or not
// tms_topk_static is ever called.  On the host this name is only a handle for the runtime's symbol lookup -- it is NOT
// a device address and must never be passed to a kernel; static_scratch() below asks the runtime for the real one.
static __device__ __align__(256) unsigned char g_tms_topk_static_scratch[TMS_TOPK_STATIC_SCRATCH_BYTES];

namespace tms {
namespace {

constexpr int CHUNK = 4096;
constexpr int THREADS = 1024;

__device__ __forceinline__ uint64_t make_key(float score, uint32_t idx) {
    uint32_t b = __float_as_uint(score);
    if (b == 0x80000000u) b = 0;  // -0.0 ties with +0.0 (equal values are ranked by index)
    const uint32_t u = (b & 0x80000000u) ? ~b : (b | 0x80000000u);  // monotone: larger float -> larger u
    return ((uint64_t)u << 32) | (uint64_t)(~idx);                   // lower index wins a tie
}
__device__ __forceinline__ float key_score(uint64_t key) {
    const uint32_t u = (uint32_t)(key >> 32);
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}

// One CTA sorts one chunk of one query's list and emits its `keep` best keys.
//   scores != nullptr: level 0, the list is scores[q, 0..n)       keys_in == nullptr
//   else             : the list is keys_in[q, 0..n)
//   values != nullptr: last level (one chunk): unpack into values / indices instead of keys_out
__global__ void __launch_bounds__(THREADS)
topk_level_kernel(const float* __restrict__ scores, const uint64_t* __restrict__ keys_in, int64_t n, int64_t in_pitch,
                  int keep, uint64_t* __restrict__ keys_out, int64_t out_pitch, float* __restrict__ values,
                  int64_t* __restrict__ indices, int k) {
    __shared__ uint64_t key[CHUNK];
    const int q = blockIdx.y;
    const int64_t base = (int64_t)blockIdx.x * CHUNK;
    for (int i = threadIdx.x; i < CHUNK; i += THREADS) {
        const int64_t j = base + i;
        uint64_t kk = 0;  // below every real key (a real key's low word is ~index != 0 only for index < 2^32-1;
                          // its high word is >= 0x007fffff for any non-NaN float)
        if (j < n) kk = scores ? make_key(scores[(int64_t)q * in_pitch + j], (uint32_t)j) : keys_in[(int64_t)q * in_pitch + j];
        key[i] = kk;
    }
    __syncthreads();
    // bitonic sort, descending
    for (int size = 2; size <= CHUNK; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int t = threadIdx.x; t < CHUNK / 2; t += THREADS) {
                const int lo = 2 * t - (t & (stride - 1));  // index of the pair's first element
                const int hi = lo + stride;
                const bool desc = (lo & size) == 0;
                const uint64_t a = key[lo], b = key[hi];
                if ((a < b) == desc) { key[lo] = b; key[hi] = a; }
            }
            __syncthreads();
        }
    }
    if (values) {
        for (int i = threadIdx.x; i < k; i += THREADS) {
            const uint64_t kk = key[i];
            values[(int64_t)q * k + i] = key_score(kk);
            indices[(int64_t)q * k + i] = (int64_t)(uint32_t)(~(uint32_t)kk);
        }
    } else {
        for (int i = threadIdx.x; i < keep; i += THREADS)
            keys_out[(int64_t)q * out_pitch + (int64_t)blockIdx.x * keep + i] = key[i];
    }
}

// ---- k <= 128 (the paper's top-100): the same chunk -> `keep` best keys step without sorting the whole chunk ---------
// A chunk is 32 runs of 128 keys, one run per warp, four keys per thread in registers (logical position p = 4*lane + j).
//   1. every warp sorts its run with a bitonic network that never leaves the warp: strides 1 and 2 are exchanges between a
//      thread's own registers, strides 4..64 are shuffles with lane ^ (stride / 4).  Even runs end descending, odd runs
//      ascending (the network's usual direction rule on the chunk-wide position).
//   2. five halving steps: run pairs (descending, ascending) are combined position by position with max(), which leaves
//      a bitonic run holding exactly the 128 largest of the 256 keys; one bitonic merge (again inside the warp) sorts it in
//      the direction its new run index asks for.  The absorbed run travels through shared memory; every warp writes its
//      own 1 KB region at most once, so a step costs one __syncthreads and there is no write-after-read hazard.
// 5 block-wide barriers instead of the 78 of the full sort; keys are unique (the index is part of the key), so the
// result is the same set in the same order as the sorting kernel's, bit for bit.
__device__ __forceinline__ void cmpx(uint64_t& a, uint64_t& b, bool desc) {  // a at the lower position
    const uint64_t lo = a < b ? a : b, hi = a < b ? b : a;
    a = desc ? hi : lo;
    b = desc ? lo : hi;
}
// The network's stages for this thread's four keys (position p = 4*lane + j).  Strides 1 and 2 pair a thread's own
// registers; a stride >= 4 pairs lane with lane ^ (stride / 4), same register.  desc: direction of the stage.
__device__ __forceinline__ void stage_regs(uint64_t (&e)[4], bool desc) {  // stride 2, then stride 1
    cmpx(e[0], e[2], desc);
    cmpx(e[1], e[3], desc);
    cmpx(e[0], e[1], desc);
    cmpx(e[2], e[3], desc);
}
__device__ __forceinline__ void stage_lanes(uint64_t (&e)[4], int lm, bool desc, int lane) {
    const bool take_max = ((lane & lm) == 0) == desc;  // the lower position of a pair keeps the larger key iff descending
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint64_t o = __shfl_xor_sync(0xffffffffu, e[j], lm);
        e[j] = take_max ? (e[j] > o ? e[j] : o) : (e[j] < o ? e[j] : o);
    }
}
// all stages of one merge of `size` keys (strides size/2 .. 1).  The lane loop is NOT unrolled: the fully unrolled kernel
// was 40 KB of straight-line code that every one of the 32 warps streamed through once, and ran at the instruction
// fetch rate (19 us for a single chunk); as loops it is a few KB.
__device__ __forceinline__ void merge(uint64_t (&e)[4], int size, bool desc, int lane) {
#pragma unroll 1
    for (int lm = size >> 3; lm > 0; lm >>= 1) stage_lanes(e, lm, desc, lane);
    stage_regs(e, desc);
}

constexpr int RUN = 128;  // keys per warp; the small-k kernel serves keep <= RUN

__global__ void __launch_bounds__(THREADS)
topk_level_small_kernel(const float* __restrict__ scores, const uint64_t* __restrict__ keys_in, int64_t n,
                        int64_t in_pitch, int keep, uint64_t* __restrict__ keys_out, int64_t out_pitch,
                        float* __restrict__ values, int64_t* __restrict__ indices, int k) {
    __shared__ uint64_t xch[CHUNK];
    const int q = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t base = (int64_t)blockIdx.x * CHUNK + warp * RUN;
    uint64_t e[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {  // any placement will do (the run is sorted next): coalesced rows of 32
        const int64_t i = base + j * 32 + lane;
        uint64_t kk = 0;  // below every real key
        if (i < n) kk = scores ? make_key(scores[(int64_t)q * in_pitch + i], (uint32_t)i) : keys_in[(int64_t)q * in_pitch + i];
        e[j] = kk;
    }
    // 1. sort the run; direction of a merge = the usual (P & size) == 0 on the chunk-wide position P = 128*warp + 4*lane + j:
    //    size 2 is a register bit, sizes 4..64 a lane bit, 128 the warp's parity
    cmpx(e[0], e[1], true);   // size 2: pair (0,1) descending, pair (2,3) ascending
    cmpx(e[2], e[3], false);
    stage_regs(e, (lane & 1) == 0);  // size 4
#pragma unroll 1
    for (int size = 8; size <= RUN; size <<= 1)
        merge(e, size, size == RUN ? (warp & 1) == 0 : (lane & (size >> 2)) == 0, lane);
    // 2. halving steps: warp w absorbs warp w + 2^s
#pragma unroll 1
    for (int s = 0; s < 5; ++s) {
        const int step = 1 << s;
        const bool alive = (warp & (step - 1)) == 0;
        if (alive && (warp & step)) {
#pragma unroll
            for (int j = 0; j < 4; ++j) xch[warp * RUN + j * 32 + lane] = e[j];
        }
        __syncthreads();
        if (alive && !(warp & step)) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint64_t o = xch[(warp + step) * RUN + j * 32 + lane];
                e[j] = e[j] > o ? e[j] : o;
            }
            merge(e, RUN, ((warp >> (s + 1)) & 1) == 0, lane);  // direction: parity of the new run's index
        }
    }
    if (warp == 0) {  // the chunk's 128 best, descending, at positions p = 4*lane + j
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int p = 4 * lane + j;
            if (values) {
                if (p < k) {
                    values[(int64_t)q * k + p] = key_score(e[j]);
                    indices[(int64_t)q * k + p] = (int64_t)(uint32_t)(~(uint32_t)e[j]);
                }
            } else if (p < keep) {
                keys_out[(int64_t)q * out_pitch + (int64_t)blockIdx.x * keep + p] = e[j];
            }
        }
    }
}

int64_t chunks_of(int64_t n) { return (n + CHUNK - 1) / CHUNK; }

constexpr int MAX_SHARDS = 64;
struct ShardBases { int64_t base[MAX_SHARDS]; };

// keys[q, g*k_in + r] = key(values[g, q, r], shard_base[g] + indices[g, q, r]): the candidates of a k-way merge
__global__ void merge_keys_kernel(const float* __restrict__ values, const int64_t* __restrict__ indices, int G, int Q,
                                  int k_in, const ShardBases bases, uint64_t* __restrict__ keys) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t per_q = (int64_t)G * k_in;
    if (i >= (int64_t)Q * per_q) return;
    const int q = (int)(i / per_q);
    const int64_t c = i - (int64_t)q * per_q;
    const int g = (int)(c / k_in), r = (int)(c - (int64_t)g * k_in);
    const int64_t src = ((int64_t)g * Q + q) * k_in + r;
    keys[i] = make_key(values[src], (uint32_t)(bases.base[g] + indices[src]));
}

// runs the selection levels over keys_in[q, 0..n) (or scores when keys_in == nullptr) down to values / indices
int run_levels(const float* scores, const uint64_t* keys_in, int64_t n, int64_t in_pitch, int Q, int k, uint64_t* buf0,
               uint64_t* buf1, int64_t pitch1, float* values, int64_t* indices, cudaStream_t stream) {
    uint64_t* buf[2] = {buf0, buf1};
    const float* s_in = scores;
    const uint64_t* k_in = keys_in;
    int level = 0;
    while (true) {
        const int64_t nch = chunks_of(n);
        const bool last = nch == 1;
        dim3 grid((unsigned)nch, (unsigned)Q);
        auto* kern = k <= RUN ? topk_level_small_kernel : topk_level_kernel;
        kern<<<grid, THREADS, 0, stream>>>(s_in, k_in, n, in_pitch, k, last ? nullptr : buf[level & 1], pitch1,
                                           last ? values : nullptr, last ? indices : nullptr, k);
        count_launch();
        if (cudaGetLastError() != cudaSuccess) return TMS_ERR_CUDA;
        if (last) break;
        s_in = nullptr;
        k_in = buf[level & 1];
        in_pitch = pitch1;
        n = nch * k;
        ++level;
    }
    return TMS_OK;
}

}  // namespace

// two ping-pong key buffers, each sized for level 1's survivors
size_t topk_workspace_bytes(int Q, int64_t B, int k) {
    if (B <= CHUNK) return 0;
    return 2 * sizeof(uint64_t) * (size_t)Q * (size_t)chunks_of(B) * (size_t)k;
}

int launch_topk(const float* scores, int Q, int64_t B, int k, float* values, int64_t* indices, void* workspace,
                cudaStream_t stream) {
    const int64_t pitch1 = chunks_of(B) * k;  // keys per query in either buffer (level 1 is the largest)
    uint64_t* b0 = static_cast<uint64_t*>(workspace);
    return run_levels(scores, nullptr, B, B, Q, k, b0, b0 ? b0 + (size_t)Q * pitch1 : nullptr, pitch1, values, indices,
                      stream);
}

// candidates [Q, G*k_in] followed by the two ping-pong buffers of the selection levels
size_t topk_merge_workspace_bytes(int G, int Q, int k_in, int k) {
    const int64_t n = (int64_t)G * k_in;
    size_t bytes = sizeof(uint64_t) * (size_t)Q * (size_t)n;
    if (n > CHUNK) bytes += 2 * sizeof(uint64_t) * (size_t)Q * (size_t)chunks_of(n) * (size_t)k;
    return bytes;
}

int launch_topk_merge(const float* values, const int64_t* indices, const int64_t* shard_base, int G, int Q, int k_in,
                      int k, float* out_values, int64_t* out_indices, void* workspace, cudaStream_t stream) {
    if (G > MAX_SHARDS) return TMS_ERR_UNSUPPORTED;
    ShardBases bases = {};
    for (int g = 0; g < G; ++g) bases.base[g] = shard_base[g];
    const int64_t n = (int64_t)G * k_in;
    uint64_t* keys = static_cast<uint64_t*>(workspace);
    const int64_t total = (int64_t)Q * n;
    merge_keys_kernel<<<(unsigned)((total + 255) / 256), 256, 0, stream>>>(values, indices, G, Q, k_in, bases, keys);
    count_launch();
    if (cudaGetLastError() != cudaSuccess) return TMS_ERR_CUDA;
    const int64_t pitch1 = chunks_of(n) * k;
    uint64_t* b0 = keys + (size_t)total;
    return run_levels(nullptr, keys, n, n, Q, k, b0, b0 + (size_t)Q * pitch1, pitch1, out_values, out_indices, stream);
}

// Device address of g_tms_topk_static_scratch on the CURRENT device, looked up once per device (the array exists once
// per GPU, at a different address on each) and cached.  The lookup may make the runtime load the library's device image
// onto that GPU, which is why the first tms_topk_static call on a device belongs outside any stream capture.
static int static_scratch(uint64_t** out) {
    constexpr int MAX_DEVICES = 64;
    static std::mutex mu;
    static uint64_t* cached[MAX_DEVICES] = {};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) {
        cudaGetLastError();
        return TMS_ERR_CUDA;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (!cached[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_tms_topk_static_scratch) != cudaSuccess || !p) {
            cudaGetLastError();
            return TMS_ERR_CUDA;
        }
        cached[dev] = static_cast<uint64_t*>(p);
    }
    *out = cached[dev];
    return TMS_OK;
}

// tms_topk with the key buffers in the built-in array: same kernels, same launch sequence, no allocation of any kind.
// Nothing in the array has to start from a known state: every level writes all nch*k keys of its output buffer
// (chunks with fewer than k live keys pad with the all-zero key) before the next level reads exactly those.
int launch_topk_static(const float* scores, int Q, int64_t B, int k, float* values, int64_t* indices,
                       cudaStream_t stream) {
    const size_t need = topk_workspace_bytes(Q, B, k);
    if (need > (size_t)TMS_TOPK_STATIC_SCRATCH_BYTES) return TMS_ERR_STATIC_SCRATCH;
    uint64_t* b0 = nullptr;
    if (need) {
        const int st = static_scratch(&b0);
        if (st != TMS_OK) return st;
    }
    const int64_t pitch1 = chunks_of(B) * k;
    return run_levels(scores, nullptr, B, B, Q, k, b0, b0 ? b0 + (size_t)Q * pitch1 : nullptr, pitch1, values, indices,
                      stream);
}

}  // namespace tms
