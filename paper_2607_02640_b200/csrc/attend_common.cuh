// attend_common.cuh -- work-list item, small device helpers and the split merge (rows a6, a8).
#pragma once
#include <cuda_bf16.h>

#include "layout.cuh"

namespace metronome {

// One batch item of an attend_frame call, filled by the host from its shadow counts (row a8).
// A "tile" is one resident KV block (16 tokens) of the session: first the pinned sink blocks,
// then the window blocks that hold any key some query of this call may attend
// ("the tile loop gains ceil(S/tile) extra leading iterations remapped onto the
// sink tiles ... in segmented-decode mode only segment 0 takes them").
struct AttendItem {
    int32_t sid;
    int32_t len;              // session length (the newest query sits at len-1)
    int32_t q_len;            // queries = positions len-q_len .. len-1
    int32_t q_row_off;        // exclusive prefix sum of q_len (row of this item's first query)
    int32_t n_sink_tiles;     // min(ceil(S/16), ceil(len/16))
    int32_t first_blk;        // first window logical block needed (>= ceil(S/16))
    int32_t n_tiles;          // n_sink_tiles + window tiles
    int32_t n_splits;         // split-KV segments of this item
    int32_t split_off;        // exclusive prefix sum of n_splits (first CTA of this item)
    int32_t tiles_per_split;
    int32_t tile_off;         // exclusive prefix sum of n_tiles over the items of this launch
    int32_t class_row_off;    // exclusive prefix sum of q_len over the items of this launch
    int32_t fresh_blk;        // early mode: first logical block an append kernel may still be writing (see wait_work_list)
    int32_t pad0, pad1, pad2; // 64 bytes: the list travels in 16-byte chunks
};
static_assert(sizeof(AttendItem) == 64, "AttendItem is copied in 16-byte chunks");

struct AttendParams {
    const AttendItem* items;
    int32_t n_items;
    const int32_t* table;
    int32_t tbl_width, n_sink, ring;
    const __nv_bfloat16* q;
    __nv_bfloat16* out;
    const uint8_t* kv_layer;
    KvLayout L;
    int32_t S, W;             // sinks, window (W = INT32_MAX/2 in the unbounded arm)
    float scale_log2;         // softmax_scale * log2(e): scores live in the log2 domain
    int32_t Hq, G;
    float* ws_acc;            // [row][Hq][max_splits][D]   unnormalised partial outputs
    float* ws_ml;             // [row][Hq][max_splits][2]   running max (log2 domain), running sum
    int32_t max_splits;
    int32_t pdl_early;        // let the next kernel on the stream start launching right away (PDL)
    const int32_t* items_flag; // work list of epoch items_epoch is on the device once *items_flag == items_epoch
    int32_t items_epoch;      // -1: the list came by a copy / plain launch: wait for the predecessor at the top
    const int32_t* range_item; // GQA decode: item that holds the first tile of each range (null: binary search)
    int32_t* gqa_ctr;         // [2] claim / exit counters of the GQA decode kernel's dynamic ranges (zero between launches)
    const uint8_t* sm_class;  // [SM id] 1: an SM that streams slower than the rest (GqaPlan::sm_mode; its claim counters: gqa_ctr[4], [5])
    int32_t* tickets;         // [item][Hkv] arrival counters of the stream-K pieces (zero between launches)
    int32_t* pastwait_flag;    // tensor-core kernels: <- pastwait_epoch once past griddepcontrol.wait, i.e. once this step's append
    int32_t pastwait_epoch;    // kernel is complete (the NEXT append kernel may then do its bookkeeping while this kernel runs); null: off
    unsigned long long* stamp; // measurement aid (null: off): [0] <- min over CTAs of %globaltimer at start, [1] <- max at exit
};

// Measurement aid (metronome_pool_set_profiling mode 2): the kernel's own span in %globaltimer ns, first CTA
// in to last CTA out, without events between the launches (those would break the programmatic launch edges).
__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void stamp_begin(const AttendParams& p) { if (p.stamp) atomicMin(p.stamp, global_ns()); }
__device__ __forceinline__ void stamp_end(const AttendParams& p) { if (p.stamp) atomicMax(p.stamp + 1, global_ns()); }

// Start of an attention kernel.  In early mode (items_epoch >= 0: launched programmatically behind an
// append kernel that triggered its dependents at once) the kernel may run NEXT TO the kernels before
// it: it only waits for its work list here, streams every block the append does not touch, and calls
// pdl_wait() before the first FRESH block of an item (AttendItem::fresh_blk, from the host: the block
// that holds the oldest row appended in this step OR in the step before it -- the append kernel of
// step e-1 is only known to be past its own wait when this kernel starts, not to be complete) and
// before it writes anything.  Otherwise the predecessor is waited for right away.  One thread per
// CTA; the caller syncs.  (Event-free host steps: q comes from a copy stream; the append kernel waits for the copies' flag
// before it publishes the epoch this function waits for, so q is complete here as well.)
__device__ __forceinline__ void wait_work_list(const AttendParams& p) {
    if (p.items_epoch < 0) { pdl_wait(); return; }
    int32_t seen;                       // (>=: a later step's list may already be out, in the other buffer)
    do {
        asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(p.items_flag) : "memory");
        if (seen - p.items_epoch < 0) __nanosleep(64);
    } while (seen - p.items_epoch < 0);
}

// (one thread of the grid, right after pdl_wait)
__device__ __forceinline__ void publish_past_wait(const AttendParams& p) {
    if (p.pastwait_flag) asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p.pastwait_flag), "r"(p.pastwait_epoch) : "memory");
}

__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// largest i in [0,n) with key(items[i]) <= x, keys ascending and key(items[0]) == 0
template <typename F>
__device__ __forceinline__ int32_t find_item(int32_t n, int32_t x, F key) {
    int32_t lo = 0, hi = n - 1;
    while (lo < hi) {
        const int32_t mid = (lo + hi + 1) >> 1;
        if (key(mid) <= x) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// admit(j,t) = j<=t and (j<S or t-j<W)   PAPER.md:L103, L258 (window = W keys including t)
__device__ __forceinline__ bool admit(int32_t j, int32_t t, int32_t S, int32_t W) {
    return j <= t && (j < S || t - j < W);
}

__device__ __forceinline__ float bf16lo(uint32_t x) { return __uint_as_float(x << 16); }
__device__ __forceinline__ float bf16hi(uint32_t x) { return __uint_as_float(x & 0xFFFF0000u); }

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
    __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}

// packed fp32 x 2 arithmetic (sm_100: FFMA2 / FADD2): half the issue slots of the inner loops
__device__ __forceinline__ uint64_t f2_pack(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void f2_unpack(uint64_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ uint64_t f2_fma(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ uint64_t f2_add(uint64_t a, uint64_t b) {
    uint64_t d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ uint64_t f2_sub(uint64_t a, uint64_t b) {
    uint64_t d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ uint64_t f2_mul(uint64_t a, uint64_t b) {
    uint64_t d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// Event-free host steps: publishes "the kernels of step `seq` are complete" in a flag (device memory; the read-back stream
// waits for it with a stream wait-value operation) once everything before it on the stream is complete and flushed (it is launched programmatically right behind the step's last attention kernel, whose
// griddepcontrol.wait chain reaches back to the step's append kernel).  It triggers its own dependents at once, so the
// next step's append kernel still starts under the attention kernel's tail.  grid = 1, block = 32.
__global__ void step_done_kernel(int32_t* done_flag, int32_t seq) {
    pdl_launch_dependents();
    pdl_wait();
    if (threadIdx.x == 0) {
        __threadfence_system();
        asm volatile("st.release.sys.global.s32 [%0], %1;" ::"l"(done_flag), "r"(seq) : "memory");
    }
}

// Row a6: log-sum-exp combine of the split-KV partials of one (query row, q head); sinks were
// counted once, by segment 0 ("merged exactly once").
// grid = (rows of this launch's items, Hq), block = D/4 threads.
template <int D>
__global__ void __launch_bounds__(D / 4)
merge_kernel(AttendParams p) {
    if (p.pdl_early) pdl_launch_dependents();
    pdl_wait();
    const int32_t h = blockIdx.y;
    const int32_t i = find_item(p.n_items, (int32_t)blockIdx.x, [&](int32_t k) { return p.items[k].class_row_off; });
    const int32_t ns = p.items[i].n_splits;
    if (ns <= 1) return;      // the attention kernel already wrote the final output
    const int64_t row = p.items[i].q_row_off + ((int32_t)blockIdx.x - p.items[i].class_row_off);
    const int64_t base = (row * p.Hq + h) * p.max_splits;
    float M = -INFINITY;
    for (int s = 0; s < ns; ++s) M = fmaxf(M, p.ws_ml[(base + s) * 2]);
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    float l = 0.f;
    for (int s = 0; s < ns; ++s) {
        const float m = p.ws_ml[(base + s) * 2];
        if (m == -INFINITY) continue;                 // this segment admitted no key for this row
        const float w = ex2(m - M);
        l += w * p.ws_ml[(base + s) * 2 + 1];
        const float4 a = reinterpret_cast<const float4*>(p.ws_acc + (base + s) * D)[threadIdx.x];
        acc.x += w * a.x; acc.y += w * a.y; acc.z += w * a.z; acc.w += w * a.w;
    }
    const float inv = l > 0.f ? 1.f / l : 0.f;
    uint2 o;
    o.x = pack_bf16(acc.x * inv, acc.y * inv);
    o.y = pack_bf16(acc.z * inv, acc.w * inv);
    reinterpret_cast<uint2*>(p.out + (row * p.Hq + h) * D)[threadIdx.x] = o;
}

}  // namespace metronome
