// attend_rows.cuh -- row a5: split-KV flash-decoding over sink + window blocks on CUDA cores.
//
// One CTA = one (split-KV segment, q head, query row).  It is THE kernel for multi-head decode
// (G = 1, q_len = 1: BASELINE.json config 2), where the work is a pure HBM stream at 1 flop/byte
// and tensor cores have nothing to contract; for G > 1 or q_len > 1 it is the general
// (re-reading) fallback behind the tensor-core tile kernel in attend_mma.cuh.
//
// Mapping (D = 128): a K/V row of 256 bytes is read by 16 lanes x 16 bytes, so a warp covers two
// tokens per step and one 16-token tile in 8 steps; all 16 loads of a tile (8 K + 8 V, 16 bytes
// per lane each = 8 KiB per warp) are issued before the first use, which with 4 warps per CTA and
// several CTAs per SM keeps far more than the ~44 KiB/SM in flight that 6.5 TB/s at ~1 us needs.
// Score = 8 FMAs per lane + a 4-step xor-shuffle reduction over the 16 lanes of a token
// ("warp-shuffle softmax", north_star); online softmax per half-warp in the log2 domain; the
// halves, then the 4 warps, are combined once at the end.  The four warps take tiles
// round-robin, so there is no barrier inside the tile loop.
#pragma once
#include "attend_common.cuh"
#include "kv_fp8.cuh"

namespace metronome {

__device__ __forceinline__ void merge_state(float& m, float& l, float (&acc)[8], float m2, float l2,
                                            const float (&acc2)[8]) {
    const float M = fmaxf(m, m2);
    if (M == -INFINITY) return;
    const float a = ex2(m - M), b = ex2(m2 - M);   // ex2(-inf) = 0
    l = l * a + l2 * b;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = acc[i] * a + acc2[i] * b;
    m = M;
}

// 8 consecutive elements of a K / V row as the lane holds them: 16 bytes of bf16, or 8 E4M3 codes (fp8 KV, NEXT row
// f4: the row's float32 scale is applied to the finished dot product / folded into the softmax weight)
template <bool FP8> struct RowChunk { using type = uint4; };
template <> struct RowChunk<true> { using type = uint2; };
// elements 2 k, 2 k + 1 of the chunk as a packed float pair
__device__ __forceinline__ uint64_t chunk_pair(const uint4& c, int k) {
    const uint32_t w = k == 0 ? c.x : k == 1 ? c.y : k == 2 ? c.z : c.w;
    return f2_pack(bf16lo(w), bf16hi(w));
}
__device__ __forceinline__ uint64_t chunk_pair(const uint2& c, int k) {
    const uint32_t w = (k < 2 ? c.x : c.y) >> (16 * (k & 1));
    uint32_t h2;
    asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"((uint16_t)w));
    const __half2 hv = *reinterpret_cast<const __half2*>(&h2);
    return f2_pack(__low2float(hv), __high2float(hv));
}

// grid = (Hq, total_splits, max_q_len), block = 128
template <int D, bool FP8>
__global__ void __launch_bounds__(128)
attend_rows_kernel(AttendParams p) {
    using Chunk = typename RowChunk<FP8>::type;
    if (p.pdl_early) pdl_launch_dependents();
    if (threadIdx.x == 0) { stamp_begin(p); wait_work_list(p); }
    __syncthreads();
    if (p.items_epoch < 0) pdl_wait();
    constexpr int LPT = D / 8;         // lanes per token (16-byte chunks per row)
    constexpr int TPS = 32 / LPT;      // tokens per warp step
    constexpr int STEPS = kBlockTokens / TPS;
    // heads vary fastest across the grid: CTAs that run together read neighbouring 8 KiB tiles of the same
    // KV blocks
    const int32_t seg = (int32_t)blockIdx.y;
    const int32_t i = find_item(p.n_items, seg, [&](int32_t k) { return p.items[k].split_off; });
    const AttendItem it = p.items[i];
    const int32_t r = blockIdx.z;
    if (r >= it.q_len) return;
    const int32_t split = seg - it.split_off;
    const int32_t h = blockIdx.x, kvh = h / p.G;
    const int32_t t = it.len - it.q_len + r;          // absolute position of this query (reading R2)
    const int32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t sub = lane % LPT, grp = lane / LPT;
    const int64_t qrow = (int64_t)(it.q_row_off + r) * p.Hq + h;

    float qf[8];
    {
        const uint4 qv = *reinterpret_cast<const uint4*>(p.q + qrow * D + sub * 8);
        const uint32_t w[4] = {qv.x, qv.y, qv.z, qv.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            qf[2 * k] = bf16lo(w[k]) * p.scale_log2;
            qf[2 * k + 1] = bf16hi(w[k]) * p.scale_log2;
        }
    }

    float m = -INFINITY, l = 0.f, acc[8];
    uint64_t acc2[4] = {0ull, 0ull, 0ull, 0ull}, q2[4];           // packed (even, odd) accumulators / query
#pragma unroll
    for (int k = 0; k < 4; ++k) q2[k] = f2_pack(qf[2 * k], qf[2 * k + 1]);

    const int32_t* trow = p.table + (int64_t)it.sid * p.tbl_width;
    const int32_t tl0 = split * it.tiles_per_split;
    const int32_t tl1 = min(it.n_tiles, tl0 + it.tiles_per_split);

    // Software pipeline: the K rows of the NEXT tile are requested as soon as the scores of the current
    // tile are out of the K registers, its V rows as soon as P V is done with the V registers, so a
    // warp keeps ~8 KiB in flight through its whole compute phase (not only while it waits).
    auto block_of = [&](int32_t tile) { return tile < it.n_sink_tiles ? tile : it.first_blk + (tile - it.n_sink_tiles); };
    // next tile >= `tile` (stride 4) with at least one admitted key for this row; tl1 if none.  Later chunk
    // rows leave early window tiles behind, earlier chunk rows do not see the newest tile.
    auto next_valid = [&](int32_t tile) {
        for (; tile < tl1; tile += 4) {
            const int32_t p0 = block_of(tile) * kBlockTokens;
            if (!(p0 > t || (p0 >= p.S && t - (p0 + kBlockTokens - 1) >= p.W))) break;
        }
        return tile;
    };
    const int32_t fresh = it.fresh_blk;
    auto tile_ptr = [&](int32_t tile) {
        if (block_of(tile) >= fresh) pdl_wait();        // rows (and maybe the block) of this step's append
        const int32_t phys = __ldg(trow + table_slot(block_of(tile), p.n_sink, p.ring));
        return p.kv_layer + (int64_t)phys * p.L.block_bytes + (int64_t)kvh * p.L.head_bytes;
    };
    Chunk kr[STEPS], vr[STEPS];
    float ks[FP8 ? STEPS : 1], vs[FP8 ? STEPS : 1];                 // fp8: the rows' scales
    // fp8 code tiles are XOR-swizzled in 128-byte lines (layout.cuh: fp8_chunk_offset, for the tensor-core kernels'
    // ldmatrix); this thread's offsets take four distinct swizzle patterns (step j and j + 4 are eight rows apart: the
    // same pattern, 4 TPS D bytes further), computed once instead of per load -- the fp8 arm of this kernel is issue-bound
    int32_t xo[4] = {0, 0, 0, 0};
    if (FP8) {
#pragma unroll
        for (int jj = 0; jj < (STEPS < 4 ? STEPS : 4); ++jj) xo[jj] = fp8_unit_offset(D, jj * TPS + grp, sub);
    }
    auto chunk_off_j = [&](int j) {
        return FP8 ? xo[j & 3] + (j >> 2) * (4 * TPS * D) : tile_chunk_offset(j * TPS + grp, sub);
    };
    auto load_k = [&](const uint8_t* kt) {
#pragma unroll
        for (int j = 0; j < STEPS; ++j) {
            kr[j] = __ldg(reinterpret_cast<const Chunk*>(kt + chunk_off_j(j)));
            if (FP8) ks[j] = __ldg(reinterpret_cast<const float*>(kt + 2 * p.L.tile_bytes) + j * TPS + grp);
        }
    };
    auto load_v = [&](const uint8_t* kt) {
#pragma unroll
        for (int j = 0; j < STEPS; ++j) {
            vr[j] = __ldg(reinterpret_cast<const Chunk*>(kt + p.L.tile_bytes + chunk_off_j(j)));
            if (FP8) vs[j] = __ldg(reinterpret_cast<const float*>(kt + 2 * p.L.tile_bytes) + kBlockTokens + j * TPS + grp);
        }
    };
    int32_t tile = next_valid(tl0 + warp);
    if (tile < tl1) {
        const uint8_t* kt = tile_ptr(tile);
        load_k(kt);
        load_v(kt);
    }
    while (tile < tl1) {
        const int32_t p0 = block_of(tile) * kBlockTokens;
        const int32_t nxt = next_valid(tile + 4);
        const uint8_t* kt_next = nxt < tl1 ? tile_ptr(nxt) : nullptr;
        float s[STEPS];
#pragma unroll
        for (int j = 0; j < STEPS; ++j) {
            uint64_t d2 = 0ull;                                   // (even, odd) partial sums, FFMA2
#pragma unroll
            for (int k = 0; k < 4; ++k) d2 = f2_fma(q2[k], chunk_pair(kr[j], k), d2);
            float de, dodd;
            f2_unpack(d2, de, dodd);
            float d = de + dodd;
#pragma unroll
            for (int o = LPT / 2; o >= 1; o >>= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
            s[j] = FP8 ? d * ks[j] : d;
        }
        if (kt_next) load_k(kt_next);
        const bool full = (p0 + kBlockTokens - 1 <= t) &&
                          (p0 + kBlockTokens - 1 < p.S || t - p0 < p.W);
        if (!full) {
            // boundary tile: token-exact mask; rows that are not admitted may hold stale or
            // poisoned bytes (0 * NaN = NaN), so their V is zeroed, not multiplied by p = 0
#pragma unroll
            for (int j = 0; j < STEPS; ++j) {
                const int32_t pos = p0 + j * TPS + grp;
                if (!admit(pos, t, p.S, p.W)) {
                    s[j] = -INFINITY;
                    vr[j] = Chunk{};
                    if (FP8) vs[j] = 0.f;
                }
            }
        }
        float tmax = s[0];
#pragma unroll
        for (int j = 1; j < STEPS; ++j) tmax = fmaxf(tmax, s[j]);
        const float mn = fmaxf(m, tmax);
        if (mn != -INFINITY) {            // (uniform inside a token group)
            const float corr = ex2(m - mn);
            l *= corr;
            const uint64_t corr2 = f2_pack(corr, corr);
#pragma unroll
            for (int k = 0; k < 4; ++k) acc2[k] = f2_mul(acc2[k], corr2);
#pragma unroll
            for (int j = 0; j < STEPS; ++j) {
                const float pj = ex2(s[j] - mn);
                l += pj;
                const float pv = FP8 ? pj * vs[j] : pj;
                const uint64_t pj2 = f2_pack(pv, pv);
#pragma unroll
                for (int k = 0; k < 4; ++k) acc2[k] = f2_fma(pj2, chunk_pair(vr[j], k), acc2[k]);
            }
            m = mn;
        }
        if (kt_next) load_v(kt_next);
        tile = nxt;
    }

    pdl_wait();       // nothing is written before the predecessor (and the kernels before it) are over
#pragma unroll
    for (int k = 0; k < 4; ++k) f2_unpack(acc2[k], acc[2 * k], acc[2 * k + 1]);
    // combine the token groups of the warp
#pragma unroll
    for (int o = 16; o >= LPT; o >>= 1) {
        const float m2 = __shfl_xor_sync(0xffffffffu, m, o);
        const float l2 = __shfl_xor_sync(0xffffffffu, l, o);
        float a2[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) a2[k] = __shfl_xor_sync(0xffffffffu, acc[k], o);
        merge_state(m, l, acc, m2, l2, a2);
    }
    // combine the 4 warps
    __shared__ float sm_m[4], sm_l[4], sm_acc[4][D];
    if (lane < LPT) {
        if (sub == 0) { sm_m[warp] = m; sm_l[warp] = l; }
#pragma unroll
        for (int k = 0; k < 8; ++k) sm_acc[warp][sub * 8 + k] = acc[k];
    }
    __syncthreads();
    if (threadIdx.x < LPT) {
        m = sm_m[0]; l = sm_l[0];
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k] = sm_acc[0][sub * 8 + k];
        for (int w = 1; w < 4; ++w) {
            float a2[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) a2[k] = sm_acc[w][sub * 8 + k];
            merge_state(m, l, acc, sm_m[w], sm_l[w], a2);
        }
        if (it.n_splits == 1) {
            const float inv = l > 0.f ? 1.f / l : 0.f;
            uint4 o;
            o.x = pack_bf16(acc[0] * inv, acc[1] * inv);
            o.y = pack_bf16(acc[2] * inv, acc[3] * inv);
            o.z = pack_bf16(acc[4] * inv, acc[5] * inv);
            o.w = pack_bf16(acc[6] * inv, acc[7] * inv);
            *reinterpret_cast<uint4*>(p.out + qrow * D + sub * 8) = o;
        } else {
            const int64_t slot = qrow * p.max_splits + split;
            float4* dst = reinterpret_cast<float4*>(p.ws_acc + slot * D + sub * 8);
            dst[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
            dst[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
            if (sub == 0) { p.ws_ml[slot * 2] = m; p.ws_ml[slot * 2 + 1] = l; }
        }
    }
    if (threadIdx.x == 0) stamp_end(p);
}

}  // namespace metronome
