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

namespace metronome {

// grid = (ceil(max_n_new * Hkv * D/8 / 256), n_items), block = 256
__global__ void __launch_bounds__(256)
kv_append_kernel(const AppendItem* __restrict__ items, const int32_t* __restrict__ table, int32_t tbl_width,
                 int32_t n_sink, int32_t ring, const uint4* __restrict__ k_new, const uint4* __restrict__ v_new,
                 uint8_t* __restrict__ kv_layer, KvLayout L) {
    const AppendItem it = items[blockIdx.y];
    const int32_t chunks_per_row = L.head_dim >> 3;
    const int32_t chunks_per_tok = L.n_kv_heads * chunks_per_row;
    const int32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= it.n_new * chunks_per_tok) return;
    const int32_t tok = idx / chunks_per_tok;
    const int32_t rem = idx - tok * chunks_per_tok;
    const int32_t h = rem / chunks_per_row;
    const int32_t c = rem - h * chunks_per_row;
    const int32_t pos = it.len0 + tok;
    const int32_t blk = pos / kBlockTokens, r = pos % kBlockTokens;
    const int32_t phys = table[(int64_t)it.sid * tbl_width + table_slot(blk, n_sink, ring)];
    const int64_t src = (int64_t)(it.row_off + tok) * chunks_per_tok + rem;
    uint8_t* tile = kv_layer + (int64_t)phys * L.block_bytes + (int64_t)h * L.head_bytes;
    const int32_t off = tile_chunk_offset(r, c);
    const uint4 kk = __ldg(k_new + src);
    const uint4 vv = __ldg(v_new + src);
    *reinterpret_cast<uint4*>(tile + off) = kk;
    *reinterpret_cast<uint4*>(tile + L.tile_bytes + off) = vv;
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

}  // namespace metronome
