// kv_append.cuh -- SURVEY.md sec. 8 row a4: scatter the new K,V rows into their paged slots, and
// the inverse gather used to verify it (metronome_read_kv).
//
// k_new / v_new are [sum n_new, Hkv, D] bf16, rows in batch order ("prefill the new
// chunk").  Token p of a session lives in logical block p / 16, row p % 16; the physical id comes
// from the block table.  Each thread moves one 16-byte chunk of K and one of V: reads are fully
// coalesced, writes are 128-byte segments (layout.cuh).  Bytes are tiny next to attention
// (one row per token vs W rows read), so the kernel is latency-bound; it is sized so that a
// decode step (n_new = 1) of 128-512 sessions still fills the machine.
#pragma once
#include "bookkeeping.cuh"
#include "kv_fp8.cuh"

namespace metronome {

// ------------------------------------------------------------------------------------------------
// One launch per append_kv call: rows a2 + a3 (bookkeeping) and a4 (KV scatter) fused, and the
// attention work list of the same step (row a8) carried to the device on the way.
//
// grid = (ceil(max_n_new * Hkv * D/8 / 256), n_items + 1), block = 256.
//   CTA (0, 0)    the bookkeeping CTA: the two phases of bookkeeping.cuh over the whole batch, then
//                 it publishes `epoch` in *bk_flag (release).  It is the first CTA in dispatch
//                 order and waits on nobody.  It also copies the step's AttendItems host -> device.
//   CTA (x, y>0)  scatter CTAs of item y-1.  Only items that allocate a block in this call
//                 (n_alloc > 0) read a table entry the bookkeeping CTA writes: they spin on the flag.
// `items` (and `attend_src`) point into the pool's PINNED HOST staging ring: the kernel reads the
// per-call metadata over the bus itself, so there is no separate H2D copy on the stream, and those
// reads are issued BEFORE griddepcontrol.wait, i.e. while the previous kernel is still running when
// the launch is programmatic (PDL).
struct AppendParams {
    const AppendItem* items;
    int32_t n_items;
    int32_t* table;
    int32_t tbl_width, n_sink, ring;
    int32_t* free_stack;
    int32_t n_free0, total_freed;
    int32_t do_bookkeeping;        // 0: layers > 0, or nothing to free / allocate, or done by bookkeeping_kernel
    int32_t* bk_flag;
    int32_t epoch;
    int32_t pdl_early;             // early mode: let the dependent (attention) kernel launch right away
    int32_t* items_flag;           // [0] <- epoch once the AttendItems are on the device; [4] <- epoch once past the wait
    int32_t gate_epoch;            // early mode: items_flag[4] must have reached this before the buffer is reused
    int32_t early_bk;              // bookkeeping (and the work-list copy) BEFORE griddepcontrol.wait, i.e. while the previous
    const int32_t* pastwait_flag;  // step's attention kernel still runs, as soon as *pastwait_flag has reached pastwait_gate
    int32_t pastwait_gate;         // (= that kernel is past its own wait = the previous append kernel is complete)
    const uint4* attend_src;       // AttendItems of this step (host), attend_n16 x 16 bytes; may be null
    uint4* attend_dst;
    int32_t attend_n16;
    const uint4* k_new;
    const uint4* v_new;
    uint8_t* kv_layer;             // null: metadata only
    KvLayout L;
    // event-free host steps (metronome_step_host_async, direct mode): k_new / v_new are filled by copies on ANOTHER stream
    // that end with a 4-byte copy of h2d_seq into *h2d_flag; the scatter CTAs wait for it (null: inputs are stream-ordered)
    const int32_t* h2d_flag;
    int32_t h2d_seq;
};

constexpr int kAppendSmemItems = 1024;       // AppendItems the bookkeeping CTA stages in shared memory

// The two phases of bookkeeping.cuh over the whole batch by ONE CTA (any block size), then the call's
// epoch is published in *bk_flag (release): table entries of blocks allocated in this call are valid
// for whoever has seen it (acquire).
__device__ __forceinline__ void bookkeeping_phases(const AppendParams& a, const AppendItem* items) {
    // phase 1: evict (a2) -- PAPER.md:L256 "frees blocks that fall entirely behind the window"
    for (int i = threadIdx.x; i < a.n_items; i += blockDim.x) {
        const AppendItem it = items[i];
        const int32_t* row = a.table + (int64_t)it.sid * a.tbl_width;
        for (int k = 0; k < it.n_freed; ++k)
            a.free_stack[a.n_free0 + it.free_off + k] = row[table_slot(it.free_lo + k, a.n_sink, a.ring)];
    }
    __syncthreads();
    // phase 2: allocate (a3) -- pops from the top of the stack, batch order, ascending logical block
    const int32_t top = a.n_free0 + a.total_freed - 1;
    for (int i = threadIdx.x; i < a.n_items; i += blockDim.x) {
        const AppendItem it = items[i];
        int32_t* row = a.table + (int64_t)it.sid * a.tbl_width;
        for (int k = 0; k < it.n_alloc; ++k)
            row[table_slot(it.alloc_lo + k, a.n_sink, a.ring)] = a.free_stack[top - (it.alloc_off + k)];
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(a.bk_flag), "r"(a.epoch) : "memory");
}

__global__ void __launch_bounds__(256)
append_fused_kernel(const AppendParams a) {
    extern __shared__ __align__(16) uint8_t smem_items[];
    if (a.pdl_early) pdl_launch_dependents();
    if (blockIdx.y == 0) {
        if (blockIdx.x != 0) return;
        // ---- bookkeeping CTA ----
        constexpr int kPre = 8;                        // 8 x 256 x 16 B = 682 AttendItems in registers
        uint4 pre[kPre];
#pragma unroll
        for (int k = 0; k < kPre; ++k) {
            const int32_t idx = k * 256 + (int32_t)threadIdx.x;
            if (idx < a.attend_n16) pre[k] = a.attend_src[idx];
        }
        const bool staged = a.do_bookkeeping && a.n_items <= kAppendSmemItems;
        if (staged) {
            const uint4* src = reinterpret_cast<const uint4*>(a.items);
            uint4* dst = reinterpret_cast<uint4*>(smem_items);
            const int32_t n16 = a.n_items * (int32_t)(sizeof(AppendItem) / 16);
            for (int32_t idx = threadIdx.x; idx < n16; idx += 256) dst[idx] = src[idx];
        }
        // The attention work list goes to the device, then *items_flag <- epoch (release).
        //  - early mode (pdl_early: the row kernel may start before this kernel has passed its own
        //    wait, to overlap its ramp-up with the previous attention kernel's tail): the copy is made
        //    BEFORE the wait, into one of two buffers (epoch parity).  The reader of that buffer was the
        //    attention kernel two steps back; it is over once the previous append kernel got past ITS
        //    wait, which an early-mode kernel publishes in items_flag[4] (gate_epoch: the previous append's
        //    epoch if it ran in early mode, else 0 = no gate: a kernel that is not in early mode lets its
        //    attention kernel start only when it has completed).
        //  - otherwise: after the wait.
        auto copy_items = [&]() {
#pragma unroll
            for (int k = 0; k < kPre; ++k) {
                const int32_t idx = k * 256 + (int32_t)threadIdx.x;
                if (idx < a.attend_n16) a.attend_dst[idx] = pre[k];
            }
            for (int32_t idx = kPre * 256 + threadIdx.x; idx < a.attend_n16; idx += 256) a.attend_dst[idx] = a.attend_src[idx];
        };
        if (a.pdl_early) {
            if (threadIdx.x == 0) {
                int32_t seen;
                do {
                    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(a.items_flag + 4) : "memory");
                    if (seen - a.gate_epoch < 0) __nanosleep(64);
                } while (seen - a.gate_epoch < 0);
                // event-free host steps: the early-mode row kernel reads q as soon as it has seen this step's epoch below, so
                // the input copies (k_new, v_new, q: one flag behind all three) must have landed before it is published --
                // one system-scope wait per launch here instead of one per CTA of the row kernel
                if (a.h2d_flag) spin_until_reached_sys(a.h2d_flag, a.h2d_seq);
            }
            __syncthreads();
            copy_items();
            __threadfence();
            __syncthreads();
            if (threadIdx.x == 0)
                asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(a.items_flag), "r"(a.epoch) : "memory");
        }
        if (a.early_bk) {
            // Rows a2 / a3 need nothing the previous step's ATTENTION kernel produces, only the tables and the free
            // stack as the previous APPEND kernel left them: ~4 dependent round trips (table -> stack -> table -> flag)
            // that used to sit between two attention kernels now run under the tail of the first.  What that kernel may
            // still read is untouched: freed ids are only pushed, a new block's table slot is one that no block of any
            // window it reads maps to (checked on the host), and K/V rows are written by the scatter CTAs AFTER the wait.
            if (threadIdx.x == 0) {
                int32_t seen;
                do {
                    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(a.pastwait_flag) : "memory");
                    if (seen - a.pastwait_gate < 0) __nanosleep(64);
                } while (seen - a.pastwait_gate < 0);
            }
            __syncthreads();
            copy_items();          // (buffer of this epoch's parity: last read two steps back)
            if (a.do_bookkeeping) bookkeeping_phases(a, staged ? reinterpret_cast<const AppendItem*>(smem_items) : a.items);
            pdl_wait();
            return;
        }
        pdl_wait();
        if (a.pdl_early) {
            if (threadIdx.x == 0)
                asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(a.items_flag + 4), "r"(a.epoch) : "memory");
        } else {
            copy_items();          // (the kernel boundary publishes it: the attention kernel waits for this kernel at its top)
        }
        if (!a.do_bookkeeping) return;
        __syncthreads();          // the staged AppendItems are complete in shared memory
        bookkeeping_phases(a, staged ? reinterpret_cast<const AppendItem*>(smem_items) : a.items);
        return;
    }
    // ---- scatter CTAs (a4) ----
    if (!a.kv_layer) return;
    const AppendItem it = a.items[blockIdx.y - 1];
    const int32_t chunks_per_row = a.L.head_dim >> 3;
    const int32_t chunks_per_tok = a.L.n_kv_heads * chunks_per_row;
    const int32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (blockIdx.x * (int32_t)blockDim.x >= it.n_new * chunks_per_tok) return;      // CTA-uniform
    const bool active = idx < it.n_new * chunks_per_tok;
    const int32_t tok = idx / chunks_per_tok;
    const int32_t rem = idx - tok * chunks_per_tok;
    const int32_t h = rem / chunks_per_row;
    const int32_t c = rem - h * chunks_per_row;
    const int64_t src = (int64_t)(it.row_off + tok) * chunks_per_tok + rem;
    pdl_wait();                                       // k_new / v_new may come from the previous kernel
    uint4 kk = make_uint4(0u, 0u, 0u, 0u), vv = kk;
    if (a.h2d_flag) {                                 // (kernel-uniform) ... or from a copy stream: wait for its flag,
        if (threadIdx.x == 0) spin_until_reached_sys(a.h2d_flag, a.h2d_seq);
        __syncthreads();
        if (active) {                                 // and read past L1 (the rows landed while this grid was resident)
            kk = __ldcg(a.k_new + src);
            vv = __ldcg(a.v_new + src);
        }
    } else if (active) {
        kk = __ldg(a.k_new + src);
        vv = __ldg(a.v_new + src);
    }
    if (a.do_bookkeeping && it.n_alloc > 0) {
        if (threadIdx.x == 0) {
            int32_t seen;
            do {
                asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(a.bk_flag) : "memory");
                if (seen != a.epoch) __nanosleep(100);
            } while (seen != a.epoch);
        }
        __syncthreads();
    }
    if (!active) return;
    const int32_t pos = it.len0 + tok;
    const int32_t blk = pos / kBlockTokens, r = pos % kBlockTokens;
    const int32_t phys = __ldcg(a.table + (int64_t)it.sid * a.tbl_width + table_slot(blk, a.n_sink, a.ring));
    uint8_t* tile = a.kv_layer + (int64_t)phys * a.L.block_bytes + (int64_t)h * a.L.head_bytes;
    if (a.L.fp8) {
        // (the chunks_per_row threads of a row are consecutive lanes of one warp, all active or all not)
        const uint2 kq = quantize_chunk_e4m3(kk, chunks_per_row, c == 0 ? reinterpret_cast<float*>(tile + 2 * a.L.tile_bytes) + r : nullptr);
        const uint2 vq = quantize_chunk_e4m3(vv, chunks_per_row, c == 0 ? reinterpret_cast<float*>(tile + 2 * a.L.tile_bytes) + kBlockTokens + r : nullptr);
        const int32_t off8 = fp8_unit_offset(a.L.head_dim, r, c);
        *reinterpret_cast<uint2*>(tile + off8) = kq;
        *reinterpret_cast<uint2*>(tile + a.L.tile_bytes + off8) = vq;
        return;
    }
    const int32_t off = tile_chunk_offset(r, c);
    *reinterpret_cast<uint4*>(tile + off) = kk;
    *reinterpret_cast<uint4*>(tile + a.L.tile_bytes + off) = vv;
}

// grid = ceil(n * Hkv * D/8 / 256); positions whose block is not resident give bf16 NaN.
__global__ void __launch_bounds__(256)
kv_read_kernel(const int32_t* __restrict__ row, int32_t n_sink, int32_t ring, int32_t n_sink_res,
               int32_t first_live, int32_t n_blk, int32_t pos0, int32_t n, const uint8_t* __restrict__ kv_layer,
               KvLayout L, uint4* __restrict__ k_out, uint4* __restrict__ v_out) {
    const int32_t chunks_per_row = L.head_dim >> 3;
    const int32_t chunks_per_tok = L.n_kv_heads * chunks_per_row;
    const int32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n * chunks_per_tok) return;
    const int32_t tok = idx / chunks_per_tok;
    const int32_t rem = idx - tok * chunks_per_tok;
    const int32_t h = rem / chunks_per_row;
    const int32_t c = rem - h * chunks_per_row;
    const int32_t pos = pos0 + tok;
    const int32_t blk = pos / kBlockTokens, r = pos % kBlockTokens;
    const bool resident = blk < n_blk && (blk < n_sink_res || blk >= first_live);
    uint4 kk = make_uint4(0x7FC07FC0u, 0x7FC07FC0u, 0x7FC07FC0u, 0x7FC07FC0u), vv = kk;
    if (resident) {
        const int32_t phys = row[table_slot(blk, n_sink, ring)];
        const uint8_t* tile = kv_layer + (int64_t)phys * L.block_bytes + (int64_t)h * L.head_bytes;
        const int32_t off = tile_chunk_offset(r, c);
        kk = *reinterpret_cast<const uint4*>(tile + off);
        vv = *reinterpret_cast<const uint4*>(tile + L.tile_bytes + off);
    }
    k_out[idx] = kk;
    v_out[idx] = vv;
}

// The same for an fp8 pool: what the stored codes decode to, float32 [n, Hkv, D] (bit-exact check of the quantiser).
__global__ void __launch_bounds__(256)
kv_read_fp8_kernel(const int32_t* __restrict__ row, int32_t n_sink, int32_t ring, int32_t n_sink_res,
                   int32_t first_live, int32_t n_blk, int32_t pos0, int32_t n, const uint8_t* __restrict__ kv_layer,
                   KvLayout L, float* __restrict__ k_out, float* __restrict__ v_out) {
    const int32_t chunks_per_row = L.head_dim >> 3;
    const int32_t chunks_per_tok = L.n_kv_heads * chunks_per_row;
    const int32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n * chunks_per_tok) return;
    const int32_t tok = idx / chunks_per_tok;
    const int32_t rem = idx - tok * chunks_per_tok;
    const int32_t h = rem / chunks_per_row;
    const int32_t c = rem - h * chunks_per_row;
    const int32_t pos = pos0 + tok;
    const int32_t blk = pos / kBlockTokens, r = pos % kBlockTokens;
    const bool resident = blk < n_blk && (blk < n_sink_res || blk >= first_live);
    float kf[8], vf[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) kf[k] = vf[k] = __int_as_float(0x7FC00000);
    if (resident) {
        const int32_t phys = row[table_slot(blk, n_sink, ring)];
        const uint8_t* tile = kv_layer + (int64_t)phys * L.block_bytes + (int64_t)h * L.head_bytes;
        const float* scales = reinterpret_cast<const float*>(tile + 2 * L.tile_bytes);
        const int32_t off8 = fp8_unit_offset(L.head_dim, r, c);
        dequant8_e4m3(*reinterpret_cast<const uint2*>(tile + off8), scales[r], kf);
        dequant8_e4m3(*reinterpret_cast<const uint2*>(tile + L.tile_bytes + off8), scales[kBlockTokens + r], vf);
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) { k_out[(int64_t)idx * 8 + k] = kf[k]; v_out[(int64_t)idx * 8 + k] = vf[k]; }
}

// Read-only stream over n16 x 16 bytes: 4 independent 16-byte loads in flight per thread, grid-stride.
// (metronome_stream_read_gbs: the read-only HBM ceiling next to the copy figure.)
__global__ void __launch_bounds__(512)
stream_read_kernel(const uint4* __restrict__ buf, int64_t n16, unsigned int* __restrict__ sink) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int acc = 0;
    for (; i + 3 * stride < n16; i += 4 * stride) {
        const uint4 a = __ldcs(buf + i), b = __ldcs(buf + i + stride), c = __ldcs(buf + i + 2 * stride),
                    d = __ldcs(buf + i + 3 * stride);
        acc ^= a.x ^ a.y ^ a.z ^ a.w ^ b.x ^ b.y ^ b.z ^ b.w ^ c.x ^ c.y ^ c.z ^ c.w ^ d.x ^ d.y ^ d.z ^ d.w;
    }
    for (; i < n16; i += stride) {
        const uint4 a = __ldcs(buf + i);
        acc ^= a.x ^ a.y ^ a.z ^ a.w;
    }
    if (acc == 0x9E3779B9u) *sink = acc;                 // never true for the 0x01 fill: keeps the loads alive
}

}  // namespace metronome
