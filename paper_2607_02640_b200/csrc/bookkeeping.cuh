// bookkeeping.cuh -- device-side block table / free list updates.
//
// The host keeps only COUNTS (length, first live block, free count: pure functions of the call
// history) and uses them to validate a call and to pre-compute, per batch item, how many blocks it
// frees / allocates and the exclusive prefix sums of those counts.  The physical block ids live
// only on the device.  Because every offset is known up front, the sequential rule
//   "all frees in batch order, then all allocations in batch order, LIFO"   (reading R6)
// becomes two data-parallel phases over disjoint stack slots:
//   phase 1  item i pushes its freed ids at   stack[n_free0 + free_off[i] + k]
//   phase 2  item i pops                      stack[n_free0 + F - 1 - (alloc_off[i] + k)]
// One CTA does both with a barrier in between (N <= max_sessions items, 0-2 blocks each: the
// kernel is latency-bound, a few microseconds).
#pragma once
#include "layout.cuh"

namespace metronome {

// Per batch item of an append call; filled by the host from its shadow counts.
struct AppendItem {
    int32_t sid;
    int32_t len0;       // L0: length before this call
    int32_t n_new;      // tokens appended
    int32_t row_off;    // exclusive prefix sum of n_new (row of this item's first token in k_new)
    int32_t free_lo;    // first logical block to free (old first_live)
    int32_t n_freed;    // blocks [free_lo, free_lo + n_freed) fall entirely behind the window (L256)
    int32_t free_off;   // exclusive prefix sum of n_freed
    int32_t alloc_lo;   // first new logical block = ceil(L0 / B)
    int32_t n_alloc;    // ceil(L1/B) - ceil(L0/B)
    int32_t alloc_off;  // exclusive prefix sum of n_alloc
    int32_t pad0, pad1;
};

__global__ void __launch_bounds__(512)
bookkeeping_kernel(const AppendItem* __restrict__ items, int32_t n_items, int32_t* __restrict__ table,
                   int32_t tbl_width, int32_t n_sink, int32_t ring, int32_t* __restrict__ free_stack,
                   int32_t n_free0, int32_t total_freed) {
    // phase 1: evict (a2) -- PAPER.md:L256 "frees blocks that fall entirely behind the window"
    for (int i = threadIdx.x; i < n_items; i += blockDim.x) {
        const AppendItem it = items[i];
        const int32_t* row = table + (int64_t)it.sid * tbl_width;
        for (int k = 0; k < it.n_freed; ++k)
            free_stack[n_free0 + it.free_off + k] = row[table_slot(it.free_lo + k, n_sink, ring)];
    }
    __syncthreads();
    // phase 2: allocate (a3) -- pops from the top of the stack, batch order, ascending logical block
    const int32_t top = n_free0 + total_freed - 1;
    for (int i = threadIdx.x; i < n_items; i += blockDim.x) {
        const AppendItem it = items[i];
        int32_t* row = table + (int64_t)it.sid * tbl_width;
        for (int k = 0; k < it.n_alloc; ++k)
            row[table_slot(it.alloc_lo + k, n_sink, ring)] = free_stack[top - (it.alloc_off + k)];
    }
}

// session_close (a1): push sink blocks [0, n_sink_res) then window blocks [first_live, n_blk),
// ascending logical order, onto the stack at n_free0.
__global__ void __launch_bounds__(256)
close_session_kernel(const int32_t* __restrict__ row, int32_t n_sink, int32_t ring, int32_t n_sink_res,
                     int32_t first_live, int32_t n_blk, int32_t* __restrict__ free_stack, int32_t n_free0) {
    const int32_t n_win = n_blk > first_live ? n_blk - first_live : 0;
    for (int k = threadIdx.x; k < n_sink_res + n_win; k += blockDim.x) {
        const int32_t b = k < n_sink_res ? k : first_live + (k - n_sink_res);
        free_stack[n_free0 + k] = row[table_slot(b, n_sink, ring)];
    }
}

// METRONOME_FLAG_POISON_ON_FREE ("freed blocks NaN-poisoned"): fill the blocks whose
// ids sit in stack[lo, lo+count) with bf16 NaN in every layer.  grid = (count, n_layers).
__global__ void __launch_bounds__(256)
poison_blocks_kernel(const int32_t* __restrict__ free_stack, int32_t lo, uint8_t* __restrict__ kv,
                     int64_t block_bytes, int64_t layer_bytes) {
    const int32_t id = free_stack[lo + blockIdx.x];
    uint4* dst = reinterpret_cast<uint4*>(kv + (int64_t)blockIdx.y * layer_bytes + (int64_t)id * block_bytes);
    const uint4 nan4 = make_uint4(0x7FC07FC0u, 0x7FC07FC0u, 0x7FC07FC0u, 0x7FC07FC0u);
    for (int64_t i = threadIdx.x; i < block_bytes / 16; i += blockDim.x) dst[i] = nan4;
}

// Whole-pool fill used once at pool_create when POISON_ON_FREE is set (never-written storage is
// poison too).
__global__ void fill_nan_kernel(uint4* __restrict__ dst, int64_t n16) {
    const uint4 nan4 = make_uint4(0x7FC07FC0u, 0x7FC07FC0u, 0x7FC07FC0u, 0x7FC07FC0u);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (int64_t)gridDim.x * blockDim.x)
        dst[i] = nan4;
}

// Initial free stack: pop order 0,1,2,... => stack[i] = n_blocks-1-i.
__global__ void init_free_stack_kernel(int32_t* __restrict__ free_stack, int32_t n_blocks) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_blocks; i += gridDim.x * blockDim.x)
        free_stack[i] = n_blocks - 1 - i;
}

}  // namespace metronome
