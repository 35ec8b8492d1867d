// attend_mma.cuh -- row a5 (+ a6) for grouped-query decode, on the tensor cores (mma.sync).
//
// The R = G x q_len <= 16 query rows that share one KV head ("grouped-query
// attention") form one m16 row tile, so the KV stream is read from HBM ONCE for the whole group.
//
//   attend_gqa_kernel   HBM-bound at G flop/byte.  The flattened list of (item, KV head, tile)
//                       work is cut into EQUAL contiguous ranges, one per CTA of a single wave of
//                       n_SM x 3 CTAs ("stream-K": ragged session ages cannot unbalance the SMs);
//                       inside a CTA four warps take tiles round-robin, each with a PRIVATE ring
//                       of bulk async copies (no CTA barrier in the tile loop), and are merged
//                       through shared memory once per (item, head) piece.
//
// Data movement: one cp.async.bulk (SASS UBLKCP) of 2*16*D*2 bytes per (block, head) -- layout.cuh
// keeps K|V of a block-head contiguous and pre-swizzled -- completion counted on an mbarrier.
// Sinks go first ("extra leading iterations remapped onto the sink tiles ...
// accumulating them first is exact"); in split mode only the piece that holds them takes them.
//
// Per 16-key tile (WarpTile): S = Q K^T (mma.sync m16n8k16 bf16, K fragments by ldmatrix),
// token-exact union mask on boundary tiles only, online softmax in the log2 domain with a
// warp-uniform skip of the rescale, O += P V (V fragments by ldmatrix.trans).  Two accuracy devices,
// both on the tensor core:
//   * the softmax denominator is accumulated from the SAME rounded P that multiplies V (an extra n8
//     tile against a ones matrix), so numerator and denominator see identical weights;
//   * P is split into bf16 hi + lo parts, and the lo MMA is issued only for tiles that hold a key
//     whose weight exceeds 1/256 of the running sum (warp-uniform vote; the MMA is free in a
//     bandwidth-bound kernel): peaky softmax rows (config 4's x20 outlier channels) get ~2^-17
//     weights, flat rows pay almost nothing.
//
// Why mma.sync here and tcgen05 only for the chunk (attend_umma.cuh): decode is ONE m16 tile per KV
// head at G flop/byte; a 128-row UMMA tile would be > 87 % padding.  The shared helpers of this file
// (mbarrier / bulk-copy wrappers, tile_block) are used by the chunk kernel too.
#pragma once
#include <type_traits>

#include "attend_common.cuh"

namespace metronome {

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
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// generic-proxy accesses to shared memory before, async-proxy (bulk copy / UMMA) accesses after
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& d0, uint32_t& d1, uint32_t& d2, uint32_t& d3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(d0), "=r"(d1), "=r"(d2), "=r"(d3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t& d0, uint32_t& d1, uint32_t& d2, uint32_t& d3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(d0), "=r"(d1), "=r"(d2), "=r"(d3) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mma_f16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// two E4M3 codes (low byte -> low half) as two fp16 values: exact, E4M3 is a subset of fp16
__device__ __forceinline__ uint32_t e4m3x2_f16x2(uint16_t v) {
    uint32_t d;
    asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(d) : "h"(v));
    return d;
}
__device__ __forceinline__ uint32_t pack_f16(float lo, float hi) {
    __half2 v = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float2 lds_f2(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds_u4(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint2 lds_u2(uint32_t addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}

// ------------------------------------------------------------------------------------------------
// One m16 row tile, per-thread view.  Row rho = 16*mtile + lane/4 (a) and +8 (b); rho = r*G + g:
// query row r of the call (position t_first + r), member g of the GQA group.
template <int D>
struct WarpTile {
    static constexpr int KSTEPS = D / 16;   // k-steps of Q K^T
    static constexpr int NT = D / 8;        // n8 tiles of P V
    uint32_t qa[KSTEPS][4];
    float o[NT][4];
    float m_a, m_b;                          // running max per row, log2 domain (-inf: nothing admitted yet)
    float lsum[4];                           // [0] row a, [2] row b: running sum, accumulated by the tensor core
    int32_t ta, tb;                          // absolute position of rows a / b (-1: padding row, admits nothing)
    int32_t t_min, t_max;                    // positions spanned by the tile's valid rows (warp-uniform)
    bool va, vb;
    int64_t qrow_a, qrow_b;                  // (query row, q head) flattened: row of q / out

    template <typename Item>                 // AttendItem, or the fused step kernel's StepGeo (same field names)
    __device__ __forceinline__ void init(const AttendParams& p, const Item& it, int32_t kvh, int32_t mtile,
                                         int32_t lane) {
        const int32_t R = it.q_len * p.G;
        const int32_t t_first = it.len - it.q_len;            // reading R15: the last q_len positions
        const int32_t rho_a = 16 * mtile + (lane >> 2), rho_b = rho_a + 8;
        va = rho_a < R; vb = rho_b < R;
        const int32_t ra = rho_a / p.G, rb = rho_b / p.G;
        ta = va ? t_first + ra : -1;
        tb = vb ? t_first + rb : -1;
        qrow_a = (int64_t)(it.q_row_off + ra) * p.Hq + kvh * p.G + (rho_a - ra * p.G);
        qrow_b = (int64_t)(it.q_row_off + rb) * p.Hq + kvh * p.G + (rho_b - rb * p.G);
        t_min = t_first + (16 * mtile) / p.G;
        t_max = t_first + (min(R, 16 * mtile + 16) - 1) / p.G;
        const uint32_t* pa = reinterpret_cast<const uint32_t*>(p.q + qrow_a * D);
        const uint32_t* pb = reinterpret_cast<const uint32_t*>(p.q + qrow_b * D);
        const int32_t c = lane & 3;
#pragma unroll
        for (int kk = 0; kk < KSTEPS; ++kk) {
            qa[kk][0] = va ? __ldg(pa + kk * 8 + c) : 0u;
            qa[kk][1] = vb ? __ldg(pb + kk * 8 + c) : 0u;
            qa[kk][2] = va ? __ldg(pa + kk * 8 + 4 + c) : 0u;
            qa[kk][3] = vb ? __ldg(pb + kk * 8 + 4 + c) : 0u;
        }
        reset();
    }
    __device__ __forceinline__ void reset() {
#pragma unroll
        for (int n = 0; n < NT; ++n) { o[n][0] = o[n][1] = o[n][2] = o[n][3] = 0.f; }
        m_a = m_b = -INFINITY;
        lsum[0] = lsum[1] = lsum[2] = lsum[3] = 0.f;
    }

    // true when no key of the 16-token tile at position p0 is admitted for any row (warp-uniform)
    __device__ __forceinline__ bool skips(const AttendParams& p, int32_t p0) const {
        return p0 > t_max || (p0 >= p.S && t_min - (p0 + kBlockTokens - 1) >= p.W);
    }

    // one 16-key tile: kt / vt are shared-memory addresses of the swizzled K and V tiles
    // kLoInv: the lo part of P is issued when some key's weight exceeds 1/kLoInv of the running sum
    template <int kLoInv>
    __device__ __forceinline__ void step(const AttendParams& p, int32_t len, uint32_t kt, uint32_t vt, int32_t p0,
                                         int32_t lane) {
        const int32_t mat = lane >> 3, r8 = lane & 7;
        const int32_t k_row = r8 + ((mat >> 1) << 3), k_cs = mat & 1;   // K: (rows 0-7 | 8-15) x (chunk, chunk+1)
        const int32_t v_row = r8 + ((mat & 1) << 3), v_cs = mat >> 1;   // V: (chunk, chunk+1) x (rows 0-7 | 8-15)
        const int32_t col0 = (lane & 3) * 2;
        // ---- S = Q K^T: two n8 tiles ----
        float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int kk = 0; kk < KSTEPS; ++kk) {
            uint32_t b0, b1, b2, b3;
            ldsm_x4(kt + tile_chunk_offset(k_row, 2 * kk + k_cs), b0, b1, b2, b3);
            mma_bf16(s0, qa[kk], b0, b1);
            mma_bf16(s1, qa[kk], b2, b3);
        }
        // ---- union mask, boundary tiles only ----
        const bool full = (p0 + kBlockTokens - 1 <= t_min) && (p0 + kBlockTokens - 1 < p.S || t_max - p0 < p.W);
        if (!full) {
            const int32_t ja = p0 + col0, jb = ja + 8;
            s0[0] = admit(ja, ta, p.S, p.W) ? s0[0] : -INFINITY;
            s0[1] = admit(ja + 1, ta, p.S, p.W) ? s0[1] : -INFINITY;
            s0[2] = admit(ja, tb, p.S, p.W) ? s0[2] : -INFINITY;
            s0[3] = admit(ja + 1, tb, p.S, p.W) ? s0[3] : -INFINITY;
            s1[0] = admit(jb, ta, p.S, p.W) ? s1[0] : -INFINITY;
            s1[1] = admit(jb + 1, ta, p.S, p.W) ? s1[1] : -INFINITY;
            s1[2] = admit(jb, tb, p.S, p.W) ? s1[2] : -INFINITY;
            s1[3] = admit(jb + 1, tb, p.S, p.W) ? s1[3] : -INFINITY;
        }
        // ---- online softmax (log2 domain) ----
        float mx_a = fmaxf(fmaxf(s0[0], s0[1]), fmaxf(s1[0], s1[1]));
        float mx_b = fmaxf(fmaxf(s0[2], s0[3]), fmaxf(s1[2], s1[3]));
        mx_a = fmaxf(mx_a, __shfl_xor_sync(0xffffffffu, mx_a, 1));
        mx_a = fmaxf(mx_a, __shfl_xor_sync(0xffffffffu, mx_a, 2));
        mx_b = fmaxf(mx_b, __shfl_xor_sync(0xffffffffu, mx_b, 1));
        mx_b = fmaxf(mx_b, __shfl_xor_sync(0xffffffffu, mx_b, 2));
        const float mn_a = fmaxf(m_a, mx_a * p.scale_log2), mn_b = fmaxf(m_b, mx_b * p.scale_log2);
        if (__any_sync(0xffffffffu, (mn_a != m_a) || (mn_b != m_b))) {
            const float ca = mn_a == -INFINITY ? 1.f : ex2(m_a - mn_a);
            const float cb = mn_b == -INFINITY ? 1.f : ex2(m_b - mn_b);
            lsum[0] *= ca; lsum[1] *= ca; lsum[2] *= cb; lsum[3] *= cb;
#pragma unroll
            for (int n = 0; n < NT; ++n) { o[n][0] *= ca; o[n][1] *= ca; o[n][2] *= cb; o[n][3] *= cb; }
            m_a = mn_a; m_b = mn_b;
        }
        // a row with nothing admitted so far keeps m = -inf: subtract 0 instead (its p are all 0)
        const float sub_a = m_a == -INFINITY ? 0.f : m_a, sub_b = m_b == -INFINITY ? 0.f : m_b;
        float pr[8];
        pr[0] = ex2(fmaf(s0[0], p.scale_log2, -sub_a)); pr[1] = ex2(fmaf(s0[1], p.scale_log2, -sub_a));
        pr[2] = ex2(fmaf(s0[2], p.scale_log2, -sub_b)); pr[3] = ex2(fmaf(s0[3], p.scale_log2, -sub_b));
        pr[4] = ex2(fmaf(s1[0], p.scale_log2, -sub_a)); pr[5] = ex2(fmaf(s1[1], p.scale_log2, -sub_a));
        pr[6] = ex2(fmaf(s1[2], p.scale_log2, -sub_b)); pr[7] = ex2(fmaf(s1[3], p.scale_log2, -sub_b));
        uint32_t hi[4], lo[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            hi[k] = pack_bf16(pr[2 * k], pr[2 * k + 1]);     // [0] row a keys col0.., [1] row b, [2] row a keys 8+col0.., [3] row b
            lo[k] = pack_bf16(pr[2 * k] - bf16lo(hi[k]), pr[2 * k + 1] - bf16hi(hi[k]));
        }
        // lo part only where a key carries more than 1/kLoInv of the running sum (warp-uniform)
        const float pm_a = fmaxf(fmaxf(pr[0], pr[1]), fmaxf(pr[4], pr[5]));
        const float pm_b = fmaxf(fmaxf(pr[2], pr[3]), fmaxf(pr[6], pr[7]));
        const bool need_lo = __any_sync(0xffffffffu, (pm_a * (float)kLoInv > lsum[0]) || (pm_b * (float)kLoInv > lsum[2]));
        constexpr uint32_t kOnes = 0x3F803F80u;              // bf16 (1, 1)
        mma_bf16(lsum, hi, kOnes, kOnes);
        if (need_lo) mma_bf16(lsum, lo, kOnes, kOnes);
        // ---- O += P V; V rows past the session's length hold stale / poisoned bytes (0 * NaN) ----
        const int32_t nvalid = len - p0;                     // < 16 only in the session's last block
        uint32_t mk0 = 0xFFFFFFFFu, mk1 = 0xFFFFFFFFu;
        if (nvalid < kBlockTokens) {
            mk0 = (col0 < nvalid ? 0x0000FFFFu : 0u) | (col0 + 1 < nvalid ? 0xFFFF0000u : 0u);
            mk1 = (col0 + 8 < nvalid ? 0x0000FFFFu : 0u) | (col0 + 9 < nvalid ? 0xFFFF0000u : 0u);
        }
#pragma unroll
        for (int n = 0; n < NT; n += 2) {
            uint32_t b0, b1, b2, b3;
            ldsm_x4_t(vt + tile_chunk_offset(v_row, n + v_cs), b0, b1, b2, b3);
            if (nvalid < kBlockTokens) { b0 &= mk0; b1 &= mk1; b2 &= mk0; b3 &= mk1; }
            mma_bf16(o[n], hi, b0, b1);
            mma_bf16(o[n + 1], hi, b2, b3);
            if (need_lo) {
                mma_bf16(o[n], lo, b0, b1);
                mma_bf16(o[n + 1], lo, b2, b3);
            }
        }
    }

    // this warp's state of the rows < R_rows into the CTA's merge scratch: [R][D + 2] floats = acc | m | l
    __device__ __forceinline__ void to_scratch(float* scratch, int32_t R_rows, int32_t lane) const {
        const int32_t ra = lane >> 2, c = (lane & 3) * 2;
        const bool wa = ra < R_rows, wb = ra + 8 < R_rows;
#pragma unroll
        for (int n = 0; n < NT; ++n) {
            if (wa) *reinterpret_cast<float2*>(scratch + ra * (D + 2) + n * 8 + c) = make_float2(o[n][0], o[n][1]);
            if (wb) *reinterpret_cast<float2*>(scratch + (ra + 8) * (D + 2) + n * 8 + c) = make_float2(o[n][2], o[n][3]);
        }
        if ((lane & 3) == 0) {
            if (wa) { scratch[ra * (D + 2) + D] = m_a; scratch[ra * (D + 2) + D + 1] = lsum[0]; }
            if (wb) { scratch[(ra + 8) * (D + 2) + D] = m_b; scratch[(ra + 8) * (D + 2) + D + 1] = lsum[2]; }
        }
    }

    // final bf16 output (the piece covered every tile of this (item, head))
    __device__ __forceinline__ void store_final(const AttendParams& p, int32_t lane) const {
        const float ia = lsum[0] > 0.f ? 1.f / lsum[0] : 0.f, ib = lsum[2] > 0.f ? 1.f / lsum[2] : 0.f;
        uint32_t* oa = reinterpret_cast<uint32_t*>(p.out + qrow_a * D);
        uint32_t* ob = reinterpret_cast<uint32_t*>(p.out + qrow_b * D);
#pragma unroll
        for (int n = 0; n < NT; ++n) {
            if (va) oa[n * 4 + (lane & 3)] = pack_bf16(o[n][0] * ia, o[n][1] * ia);
            if (vb) ob[n * 4 + (lane & 3)] = pack_bf16(o[n][2] * ib, o[n][3] * ib);
        }
    }
    // unnormalised partial (acc, m, l) of one split-KV piece
    __device__ __forceinline__ void store_partial(const AttendParams& p, int32_t piece, int32_t lane) const {
        const int64_t slot_a = qrow_a * p.max_splits + piece, slot_b = qrow_b * p.max_splits + piece;
        float2* wa = reinterpret_cast<float2*>(p.ws_acc + slot_a * D);
        float2* wb = reinterpret_cast<float2*>(p.ws_acc + slot_b * D);
#pragma unroll
        for (int n = 0; n < NT; ++n) {
            if (va) wa[n * 4 + (lane & 3)] = make_float2(o[n][0], o[n][1]);
            if (vb) wb[n * 4 + (lane & 3)] = make_float2(o[n][2], o[n][3]);
        }
        if ((lane & 3) == 0) {
            if (va) { p.ws_ml[slot_a * 2] = m_a; p.ws_ml[slot_a * 2 + 1] = lsum[0]; }
            if (vb) { p.ws_ml[slot_b * 2] = m_b; p.ws_ml[slot_b * 2 + 1] = lsum[2]; }
        }
    }
};

// ------------------------------------------------------------------------------------------------
// The same m16 row tile over an fp8 (E4M3) KV pool (NEXT row f4, "the two compose"; DESIGN.md reading
// R18: code x one float32 scale per (token, KV head) row).  The codes go to the tensor core as fp16 -- E4M3 is a subset
// of fp16, so `cvt.rn.f16x2.e4m3x2` is exact -- and the scales never touch an operand:
//   * S = (Q' C_K^T) * ks_j * qs_row: the K scale of key j multiplies the finished fp32 dot product; Q' is the bf16
//     query row times a power of two that brings its largest element into [1, 2) (exact, undone by qs_row), rounded
//     to fp16 (exact for every element within 2^-14 of the row's maximum, 2^-25 absolute below);
//   * O = sum_j (p_j * vs_j / vref) C_V[j] * vref: the V scale of key j is folded into the softmax weight before it
//     is rounded to fp16 (11 bits: no hi / lo split as in the bf16 tile), relative to a running reference vref >= every
//     V scale seen so far and times 2^9, so the weights stay in [0, 2^15] whatever the magnitude of V (p_j reaches 2^6
//     under the lazily updated row maximum, vs_j / vref reaches 1) and keep full fp16 precision down to p_j vs_j = 2^-23 vref (a one-hot row
//     on a key whose V is 10^5 times smaller than its neighbours' still comes out to 11 bits); O is rescaled when vref grows (warp-uniform, rare: vref is raised with
//     a factor 4 of headroom); the denominator is summed in fp32 from the unrounded p_j, each thread its own four
//     keys of a tile, reduced over the quad once at the end.
// Fragments without a transposing load: a k16 step of Q K^T takes 16-byte chunk c of the K rows (ldmatrix on code
// bytes gives a thread 4 consecutive codes = its k = 2t, 2t+1 | 2t+8, 2t+9 operands, the Q fragment is fetched in the
// same order); for P V a thread reads D/8 code bytes of rows 2t, 2t+1, 2t+8, 2t+9 and byte-permutes row pairs together,
// so n8 tile j, column g is dim (D/8) g + j: the thread ends up with D/4 CONSECUTIVE dims of its two rows.
template <int D>
struct WarpTileF8 {
    static constexpr int KSTEPS = D / 16;
    static constexpr int NT = D / 8;
    static constexpr int kTileBytes = kBlockTokens * D;
    // fp16 weight = p (<= 2^6, lazy reference) x vs / vref (<= 1: vref is only raised when a scale exceeds it)
    // x kWScale <= 2^15 < 65504; full fp16 precision down to p vs / vref = 2^-23
    static constexpr float kWScale = 512.f;
    uint32_t qa[KSTEPS][4];
    float o[NT][4];                          // [j][e] rows a (e = 0, 1) / b (e = 2, 3): dim (D/4) t + (e & 1) NT + j, in units of vref / 2^9
    float m_a, m_b;
    float lsum[4];                           // [0] row a, [2] row b: this thread's own keys only (see quad_sum)
    float qs_a, qs_b;                        // scale_log2 * 2^e of the row's Q prescale
    float vref, inv_vref;
    int32_t ta, tb, t_min, t_max;
    bool va, vb;
    int64_t qrow_a, qrow_b;

    template <typename Item>
    __device__ __forceinline__ void init(const AttendParams& p, const Item& it, int32_t kvh, int32_t mtile,
                                         int32_t lane) {
        const int32_t R = it.q_len * p.G;
        const int32_t t_first = it.len - it.q_len;            // reading R15: the last q_len positions
        const int32_t rho_a = 16 * mtile + (lane >> 2), rho_b = rho_a + 8;
        va = rho_a < R; vb = rho_b < R;
        const int32_t ra = rho_a / p.G, rb = rho_b / p.G;
        ta = va ? t_first + ra : -1;
        tb = vb ? t_first + rb : -1;
        qrow_a = (int64_t)(it.q_row_off + ra) * p.Hq + kvh * p.G + (rho_a - ra * p.G);
        qrow_b = (int64_t)(it.q_row_off + rb) * p.Hq + kvh * p.G + (rho_b - rb * p.G);
        t_min = t_first + (16 * mtile) / p.G;
        t_max = t_first + (min(R, 16 * mtile + 16) - 1) / p.G;
        // dims 16 kk + 4 t .. + 3 of the row: k = 2t, 2t+1 (first word) and 2t+8, 2t+9 (second word) of k-step kk
        const uint2* pa = reinterpret_cast<const uint2*>(p.q + qrow_a * D);
        const uint2* pb = reinterpret_cast<const uint2*>(p.q + qrow_b * D);
        const int32_t c = lane & 3;
        uint2 xa[KSTEPS], xb[KSTEPS];
        float amax_a = 0.f, amax_b = 0.f;
#pragma unroll
        for (int kk = 0; kk < KSTEPS; ++kk) {
            xa[kk] = va ? __ldg(pa + kk * 4 + c) : make_uint2(0u, 0u);
            xb[kk] = vb ? __ldg(pb + kk * 4 + c) : make_uint2(0u, 0u);
            amax_a = fmaxf(fmaxf(amax_a, fmaxf(fabsf(bf16lo(xa[kk].x)), fabsf(bf16hi(xa[kk].x)))),
                           fmaxf(fabsf(bf16lo(xa[kk].y)), fabsf(bf16hi(xa[kk].y))));
            amax_b = fmaxf(fmaxf(amax_b, fmaxf(fabsf(bf16lo(xb[kk].x)), fabsf(bf16hi(xb[kk].x)))),
                           fmaxf(fabsf(bf16lo(xb[kk].y)), fabsf(bf16hi(xb[kk].y))));
        }
        amax_a = fmaxf(amax_a, __shfl_xor_sync(0xffffffffu, amax_a, 1));
        amax_a = fmaxf(amax_a, __shfl_xor_sync(0xffffffffu, amax_a, 2));
        amax_b = fmaxf(amax_b, __shfl_xor_sync(0xffffffffu, amax_b, 1));
        amax_b = fmaxf(amax_b, __shfl_xor_sync(0xffffffffu, amax_b, 2));
        // 2^(127 - E) brings the row's largest element into [1, 2); E = its biased exponent (a zero row: factor 1)
        int32_t Ea = (__float_as_int(amax_a) >> 23) & 0xff, Eb = (__float_as_int(amax_b) >> 23) & 0xff;
        Ea = Ea == 0 ? 127 : min(Ea, 253);
        Eb = Eb == 0 ? 127 : min(Eb, 253);
        const float da = __int_as_float((254 - Ea) << 23), db = __int_as_float((254 - Eb) << 23);
        qs_a = p.scale_log2 * __int_as_float(Ea << 23);
        qs_b = p.scale_log2 * __int_as_float(Eb << 23);
#pragma unroll
        for (int kk = 0; kk < KSTEPS; ++kk) {
            qa[kk][0] = pack_f16(bf16lo(xa[kk].x) * da, bf16hi(xa[kk].x) * da);
            qa[kk][1] = pack_f16(bf16lo(xb[kk].x) * db, bf16hi(xb[kk].x) * db);
            qa[kk][2] = pack_f16(bf16lo(xa[kk].y) * da, bf16hi(xa[kk].y) * da);
            qa[kk][3] = pack_f16(bf16lo(xb[kk].y) * db, bf16hi(xb[kk].y) * db);
        }
        reset();
    }
    __device__ __forceinline__ void reset() {
#pragma unroll
        for (int n = 0; n < NT; ++n) { o[n][0] = o[n][1] = o[n][2] = o[n][3] = 0.f; }
        m_a = m_b = -INFINITY;
        lsum[0] = lsum[1] = lsum[2] = lsum[3] = 0.f;
        vref = 0.f; inv_vref = 0.f;
    }
    __device__ __forceinline__ bool skips(const AttendParams& p, int32_t p0) const {
        return p0 > t_max || (p0 >= p.S && t_min - (p0 + kBlockTokens - 1) >= p.W);
    }

    // one 16-key tile at shared-memory address kt: [K codes][V codes][16 K scales][16 V scales]
    template <int kLoInv>
    __device__ __forceinline__ void step(const AttendParams& p, int32_t len, uint32_t kt, uint32_t vt, int32_t p0,
                                         int32_t lane) {
        const uint32_t sc = kt + 2 * kTileBytes;
        const int32_t mat = lane >> 3, r8 = lane & 7;
        const int32_t k_row = r8 + ((mat & 1) << 3), k_cs = mat >> 1;   // K: (rows 0-7 | 8-15) x (chunk, chunk+1)
        const int32_t g = lane >> 2, t = lane & 3, col0 = 2 * t;
        // ---- S = Q' C_K^T: two n8 tiles (keys 0-7 | 8-15) ----
        float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int kk = 0; kk < KSTEPS; kk += 2) {
            uint32_t d0, d1, d2, d3;
            ldsm_x4(kt + fp8_chunk_offset(D, k_row, kk + k_cs), d0, d1, d2, d3);
            mma_f16(s0, qa[kk], e4m3x2_f16x2((uint16_t)d0), e4m3x2_f16x2((uint16_t)(d0 >> 16)));
            mma_f16(s1, qa[kk], e4m3x2_f16x2((uint16_t)d1), e4m3x2_f16x2((uint16_t)(d1 >> 16)));
            mma_f16(s0, qa[kk + 1], e4m3x2_f16x2((uint16_t)d2), e4m3x2_f16x2((uint16_t)(d2 >> 16)));
            mma_f16(s1, qa[kk + 1], e4m3x2_f16x2((uint16_t)d3), e4m3x2_f16x2((uint16_t)(d3 >> 16)));
        }
        // ---- the rows' scales: keys col0, col0+1 (.x, .y of *_lo) and col0+8, col0+9 (*_hi) ----
        const float2 ks_lo = lds_f2(sc + col0 * 4), ks_hi = lds_f2(sc + (col0 + 8) * 4);
        float2 vs_lo = lds_f2(sc + (kBlockTokens + col0) * 4), vs_hi = lds_f2(sc + (kBlockTokens + col0 + 8) * 4);
        float sv[8];                            // log2 domain: [0] [1] row a, [2] [3] row b keys col0, col0+1; [4..7] keys col0+8, +9
        sv[0] = s0[0] * (ks_lo.x * qs_a); sv[1] = s0[1] * (ks_lo.y * qs_a);
        sv[2] = s0[2] * (ks_lo.x * qs_b); sv[3] = s0[3] * (ks_lo.y * qs_b);
        sv[4] = s1[0] * (ks_hi.x * qs_a); sv[5] = s1[1] * (ks_hi.y * qs_a);
        sv[6] = s1[2] * (ks_hi.x * qs_b); sv[7] = s1[3] * (ks_hi.y * qs_b);
        // ---- union mask, boundary tiles only (a masked score may be anything, NaN included: it is replaced) ----
        const bool full = (p0 + kBlockTokens - 1 <= t_min) && (p0 + kBlockTokens - 1 < p.S || t_max - p0 < p.W);
        if (!full) {
            const int32_t ja = p0 + col0, jb = ja + 8;
            sv[0] = admit(ja, ta, p.S, p.W) ? sv[0] : -INFINITY;
            sv[1] = admit(ja + 1, ta, p.S, p.W) ? sv[1] : -INFINITY;
            sv[2] = admit(ja, tb, p.S, p.W) ? sv[2] : -INFINITY;
            sv[3] = admit(ja + 1, tb, p.S, p.W) ? sv[3] : -INFINITY;
            sv[4] = admit(jb, ta, p.S, p.W) ? sv[4] : -INFINITY;
            sv[5] = admit(jb + 1, ta, p.S, p.W) ? sv[5] : -INFINITY;
            sv[6] = admit(jb, tb, p.S, p.W) ? sv[6] : -INFINITY;
            sv[7] = admit(jb + 1, tb, p.S, p.W) ? sv[7] : -INFINITY;
        }
        // ---- online softmax (log2 domain) ----
        float mx_a = fmaxf(fmaxf(sv[0], sv[1]), fmaxf(sv[4], sv[5]));
        float mx_b = fmaxf(fmaxf(sv[2], sv[3]), fmaxf(sv[6], sv[7]));
        mx_a = fmaxf(mx_a, __shfl_xor_sync(0xffffffffu, mx_a, 1));
        mx_a = fmaxf(mx_a, __shfl_xor_sync(0xffffffffu, mx_a, 2));
        mx_b = fmaxf(mx_b, __shfl_xor_sync(0xffffffffu, mx_b, 1));
        mx_b = fmaxf(mx_b, __shfl_xor_sync(0xffffffffu, mx_b, 2));
        // lazy reference: a row keeps its stale maximum while the true one is within 2^kLazy of it (its weights then
        // reach 2^kLazy instead of 1, which the fp16 weight factor below leaves room for); the 4 NT accumulators are
        // rescaled on ~1 tile in 20 instead of 2 in 3 (8 rows, each with a new maximum every few tiles)
        constexpr float kLazy = 6.f;
        const bool need_a = mx_a > m_a + kLazy, need_b = mx_b > m_b + kLazy;        // (-inf + 6 = -inf: the first key counts)
        const float mn_a = need_a ? mx_a : m_a, mn_b = need_b ? mx_b : m_b;
        // ---- V scales: rows past the session's length hold stale / poisoned bytes ----
        const int32_t nvalid = len - p0;                     // < 16 only in the session's last block
        if (nvalid < kBlockTokens) {
            vs_lo.x = col0 < nvalid ? vs_lo.x : 0.f; vs_lo.y = col0 + 1 < nvalid ? vs_lo.y : 0.f;
            vs_hi.x = col0 + 8 < nvalid ? vs_hi.x : 0.f; vs_hi.y = col0 + 9 < nvalid ? vs_hi.y : 0.f;
        }
        float vmax = fmaxf(fmaxf(vs_lo.x, vs_lo.y), fmaxf(vs_hi.x, vs_hi.y));
        vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, 1));
        vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, 2));       // (the same in every quad: warp-uniform)
        const bool grow = vmax > vref;
        if (grow || __any_sync(0xffffffffu, need_a || need_b)) {
            float ca = mn_a == -INFINITY ? 1.f : ex2(m_a - mn_a);
            float cb = mn_b == -INFINITY ? 1.f : ex2(m_b - mn_b);
            lsum[0] *= ca; lsum[2] *= cb;
            if (grow) {
                const float nv = vmax * 4.f, f = vref / nv;
                ca *= f; cb *= f;
                vref = nv; inv_vref = kWScale / nv;
            }
#pragma unroll
            for (int n = 0; n < NT; ++n) { o[n][0] *= ca; o[n][1] *= ca; o[n][2] *= cb; o[n][3] *= cb; }
            m_a = mn_a; m_b = mn_b;
        }
        const float sub_a = m_a == -INFINITY ? 0.f : m_a, sub_b = m_b == -INFINITY ? 0.f : m_b;
        float pr[8];
        pr[0] = ex2(sv[0] - sub_a); pr[1] = ex2(sv[1] - sub_a); pr[2] = ex2(sv[2] - sub_b); pr[3] = ex2(sv[3] - sub_b);
        pr[4] = ex2(sv[4] - sub_a); pr[5] = ex2(sv[5] - sub_a); pr[6] = ex2(sv[6] - sub_b); pr[7] = ex2(sv[7] - sub_b);
        lsum[0] += (pr[0] + pr[1]) + (pr[4] + pr[5]);
        lsum[2] += (pr[2] + pr[3]) + (pr[6] + pr[7]);
        const float w0 = vs_lo.x * inv_vref, w1 = vs_lo.y * inv_vref, w8 = vs_hi.x * inv_vref, w9 = vs_hi.y * inv_vref;
        uint32_t pw[4];                          // A fragment of P V: [0] row a keys col0.., [1] row b, [2] row a keys 8+col0.., [3] row b
        pw[0] = pack_f16(pr[0] * w0, pr[1] * w1);
        pw[1] = pack_f16(pr[2] * w0, pr[3] * w1);
        pw[2] = pack_f16(pr[4] * w8, pr[5] * w9);
        pw[3] = pack_f16(pr[6] * w8, pr[7] * w9);
        // ---- O += P' C_V: code bytes (D/8) g .. of rows 2t, 2t+1 | 2t+8, 2t+9, row pairs zipped with byte permutes ----
        uint32_t mk0 = 0xFFFFFFFFu, mk1 = 0xFFFFFFFFu;
        if (nvalid < kBlockTokens) {
            mk0 = (col0 < nvalid ? 0x00FF00FFu : 0u) | (col0 + 1 < nvalid ? 0xFF00FF00u : 0u);
            mk1 = (col0 + 8 < nvalid ? 0x00FF00FFu : 0u) | (col0 + 9 < nvalid ? 0xFF00FF00u : 0u);
        }
        constexpr int WPR = D / 32;              // 32-bit words a thread takes from each row
        uint32_t r0[WPR], r1[WPR], r2[WPR], r3[WPR];
        if constexpr (D == 128) {
            const uint4 a0 = lds_u4(vt + fp8_chunk_offset(D, col0, g)), a1 = lds_u4(vt + fp8_chunk_offset(D, col0 + 1, g));
            const uint4 a2 = lds_u4(vt + fp8_chunk_offset(D, col0 + 8, g)), a3 = lds_u4(vt + fp8_chunk_offset(D, col0 + 9, g));
            r0[0] = a0.x; r0[1] = a0.y; r0[2] = a0.z; r0[3] = a0.w;
            r1[0] = a1.x; r1[1] = a1.y; r1[2] = a1.z; r1[3] = a1.w;
            r2[0] = a2.x; r2[1] = a2.y; r2[2] = a2.z; r2[3] = a2.w;
            r3[0] = a3.x; r3[1] = a3.y; r3[2] = a3.z; r3[3] = a3.w;
        } else {
            static_assert(D == 64 || D == 128, "head_dim");
            const uint2 a0 = lds_u2(vt + fp8_unit_offset(D, col0, g)), a1 = lds_u2(vt + fp8_unit_offset(D, col0 + 1, g));
            const uint2 a2 = lds_u2(vt + fp8_unit_offset(D, col0 + 8, g)), a3 = lds_u2(vt + fp8_unit_offset(D, col0 + 9, g));
            r0[0] = a0.x; r0[1] = a0.y; r1[0] = a1.x; r1[1] = a1.y;
            r2[0] = a2.x; r2[1] = a2.y; r3[0] = a3.x; r3[1] = a3.y;
        }
#pragma unroll
        for (int i = 0; i < WPR; ++i) {
            uint32_t x01 = __byte_perm(r0[i], r1[i], 0x5140), x23 = __byte_perm(r0[i], r1[i], 0x7362);
            uint32_t y01 = __byte_perm(r2[i], r3[i], 0x5140), y23 = __byte_perm(r2[i], r3[i], 0x7362);
            if (nvalid < kBlockTokens) { x01 &= mk0; x23 &= mk0; y01 &= mk1; y23 &= mk1; }
            mma_f16(o[4 * i], pw, e4m3x2_f16x2((uint16_t)x01), e4m3x2_f16x2((uint16_t)y01));
            mma_f16(o[4 * i + 1], pw, e4m3x2_f16x2((uint16_t)(x01 >> 16)), e4m3x2_f16x2((uint16_t)(y01 >> 16)));
            mma_f16(o[4 * i + 2], pw, e4m3x2_f16x2((uint16_t)x23), e4m3x2_f16x2((uint16_t)y23));
            mma_f16(o[4 * i + 3], pw, e4m3x2_f16x2((uint16_t)(x23 >> 16)), e4m3x2_f16x2((uint16_t)(y23 >> 16)));
        }
    }

    __device__ __forceinline__ static float quad_sum(float x) {
        x += __shfl_xor_sync(0xffffffffu, x, 1);
        return x + __shfl_xor_sync(0xffffffffu, x, 2);
    }
    // this warp's state of the rows < R_rows into the CTA's merge scratch: [R][D + 2] floats = acc | m | l
    // (all 32 lanes call it; acc in true units, dims in their natural order)
    __device__ __forceinline__ void to_scratch(float* scratch, int32_t R_rows, int32_t lane) const {
        const float la = quad_sum(lsum[0]), lb = quad_sum(lsum[2]);
        const float vu = vref * (1.f / kWScale);
        const int32_t ra = lane >> 2, d0 = (lane & 3) * (D / 4);
        const bool wa = ra < R_rows, wb = ra + 8 < R_rows;
#pragma unroll
        for (int n = 0; n < NT; n += 2) {
            if (wa) {
                *reinterpret_cast<float2*>(scratch + ra * (D + 2) + d0 + n) = make_float2(o[n][0] * vu, o[n + 1][0] * vu);
                *reinterpret_cast<float2*>(scratch + ra * (D + 2) + d0 + NT + n) = make_float2(o[n][1] * vu, o[n + 1][1] * vu);
            }
            if (wb) {
                *reinterpret_cast<float2*>(scratch + (ra + 8) * (D + 2) + d0 + n) = make_float2(o[n][2] * vu, o[n + 1][2] * vu);
                *reinterpret_cast<float2*>(scratch + (ra + 8) * (D + 2) + d0 + NT + n) = make_float2(o[n][3] * vu, o[n + 1][3] * vu);
            }
        }
        if ((lane & 3) == 0) {
            if (wa) { scratch[ra * (D + 2) + D] = m_a; scratch[ra * (D + 2) + D + 1] = la; }
            if (wb) { scratch[(ra + 8) * (D + 2) + D] = m_b; scratch[(ra + 8) * (D + 2) + D + 1] = lb; }
        }
    }
};

// logical block and first token position of tile `tile` of an item (sinks first, then the window)
template <typename Item>
__device__ __forceinline__ int32_t tile_block(const Item& it, int32_t tile) {
    return tile < it.n_sink_tiles ? tile : it.first_blk + (tile - it.n_sink_tiles);
}

// ================================================================================================
// GQA decode (R <= 16): stream-K partition of the flattened (item, KV head, tile) list.
template <int D, bool FP8>
struct GqaCfg {
    static constexpr int NWARP = 4;
    // private stages per warp, one 16-key tile each (fp8 tiles are half the bytes: twice the stages keep the same
    // number of bytes in flight)
    static constexpr int NS = FP8 ? 4 : 2;
    static constexpr int kPre = NS - 1;                 // the stage that takes the NEXT pair's first tile during a merge
    static constexpr int kTileBytes = kBlockTokens * D * (FP8 ? 1 : 2);                   // K (or V) of one block-head
    static constexpr int kHeadBytes = 2 * kTileBytes + (FP8 ? 2 * kBlockTokens * 4 : 0);   // = KvLayout::head_bytes
    static constexpr int kWarpBytes = NS * kHeadBytes;
    static constexpr int kSmemBytes = NWARP * kWarpBytes + NWARP * NS * 8 + 128;
    static constexpr int kThreads = 32 * NWARP;
    // the merge of the 4 warps reuses the rings: 16 rows x (D + 2) floats per warp must fit
    static_assert(16 * (D + 2) * 4 <= kWarpBytes, "merge scratch does not fit a warp's ring");
    static_assert(kHeadBytes % 128 == 0, "stages stay 128-byte aligned");
};

// The flattened tile list [0, total_tiles) is cut into RANGES in two regimes:
//   static   ranges 0 .. n_static-1, q1 tiles each, cover [0, g1): range r belongs to CTA r
//   dynamic  ranges n_static .. n_total-1, q2 (< q1) tiles each, cover [g1, total): claimed with an
//            atomic counter by whichever CTA finishes early.  SMs do not stream at the same speed
//            (equal static shares finished 63..95 us apart on a B200), so the last ~20 % of the
//            work is handed out in small pieces.
struct GqaPlan {
    int32_t n_kv_heads;
    int32_t bnd;              // cost of starting an (item, head) pair, in tiles (see make_gqa_plan)
    int64_t total_tiles;      // Hkv * sum of (the items' n_tiles + bnd): the list is cut in these COST units
    int64_t q1, g1;           // static regime
    int64_t q2;               // dynamic regime
    int32_t n_static, n_total;
    int32_t sm_mode;          // 1: ranges 0 .. n_static-1 are for CTAs on fast SMs, the rest (shorter) for CTAs on slow SMs: one range
                              // per CTA, claimed from the list of the CTA's SM class (make_gqa_plan_smclass)
    __host__ __device__ int64_t range_lo(int32_t r) const { return r < n_static ? r * q1 : g1 + (int64_t)(r - n_static) * q2; }
    __host__ __device__ int64_t range_hi(int32_t r) const {
        const int64_t hi = r < n_static ? (r + 1) * q1 : g1 + (int64_t)(r - n_static + 1) * q2;
        const int64_t cap = r < n_static ? g1 : total_tiles;
        return hi < cap ? hi : cap;
    }
    __host__ __device__ int32_t range_of(int64_t g) const {
        return g < g1 ? (int32_t)(g / q1) : n_static + (int32_t)((g - g1) / q2);
    }
    // upper bound on the pieces one (item, head) pair of n tiles can be cut into
    // (the shorter of the two range lengths: a forced dynamic plan of tiny shares has q2 = 8 > q1)
    __host__ __device__ int32_t max_pieces(int32_t n) const {
        const int64_t q = q1 < q2 ? q1 : q2;
        return (int32_t)((n + q - 1) / q) + 2;
    }
};

// Host: cut `total_tiles` into one static range per CTA and, when `dynamic`, keep the last 10 % for
// small ranges (a sixth of a static one, at least 8 tiles) that the CTAs claim as they finish.
// The list is measured in COST units: pair (item i, head h) occupies n_tiles_i + bnd units starting at
// (tile_off_i + bnd * i) * Hkv + h * (n_tiles_i + bnd); its first `bnd` units stand for the work of starting a pair
// (item, table and Q fetch, merge of the four warps, write-out: ~4 us per pair on a B200, during which the CTA
// streams nothing), the rest are its tiles.  Equal TILE shares ended 62 / 71 / 74 / 78 / 84 us after the wait for CTAs
// that held 1 / 2 / 3 / 4 / 6 pairs (config 3), and the kernel ends with the last one.
inline GqaPlan make_gqa_plan(int32_t n_kv_heads, int64_t total_tiles, int64_t ctas, bool dynamic, int32_t bnd) {
    GqaPlan g{};
    g.n_kv_heads = n_kv_heads;
    g.bnd = bnd;
    g.total_tiles = total_tiles;
    const int64_t share = (total_tiles + ctas - 1) / ctas;
    g.q1 = dynamic ? (share * 9 + 9) / 10 : share;
    g.n_static = (int32_t)(dynamic ? ctas : (total_tiles + g.q1 - 1) / g.q1);
    g.g1 = g.q1 * g.n_static < total_tiles ? g.q1 * g.n_static : total_tiles;
    g.q2 = dynamic ? (g.q1 / 6 > 8 ? g.q1 / 6 : 8) : g.q1;
    g.n_total = g.n_static + (int32_t)((total_tiles - g.g1 + g.q2 - 1) / g.q2);
    return g;
}

// The same list cut for a GPU whose SMs do not stream at the same speed (on a B200 the same ~26-40 SMs run at ~0.9 of the
// others' rate, launch after launch, and a launch ends with its slowest CTA): n_fast long ranges of q1 units for the CTAs
// that land on fast SMs, then n_slow ranges shorter by `ratio` for those on slow SMs.  Which CTA lands where is the
// hardware's choice: a CTA reads %smid and CLAIMS a range from its class's list (or from the other one if its own is
// used up, which keeps any placement correct: there are exactly as many ranges as CTAs).
inline GqaPlan make_gqa_plan_smclass(int32_t n_kv_heads, int64_t total_tiles, int64_t n_fast, int64_t n_slow, double ratio, int32_t bnd) {
    GqaPlan g{};
    g.n_kv_heads = n_kv_heads;
    g.bnd = bnd;
    g.total_tiles = total_tiles;
    g.sm_mode = 1;
    const double weight = (double)n_fast + ratio * (double)n_slow;
    g.q1 = (int64_t)((double)total_tiles / weight) + 1;
    g.g1 = g.q1 * n_fast < total_tiles ? g.q1 * n_fast : total_tiles;
    g.n_static = (int32_t)((g.g1 + g.q1 - 1) / g.q1);
    const int64_t rem = total_tiles - g.g1;
    g.q2 = rem > 0 ? (rem + n_slow - 1) / n_slow : g.q1;
    g.n_total = g.n_static + (int32_t)((rem + g.q2 - 1) / g.q2);
    return g;
}

// The piece of pair (item i, the head that holds unit g) that a range ending at unit g_end takes: tiles [a, b) of the
// pair (b <= a: the range ends inside the pair's start-up units), pair_lo = the unit of the pair's tile 0.  A walk over a
// range goes g -> pair_lo + b (and on to item i + 1 after the last head); tests/native/gqa_plan_check.cu walks every
// range of random plans with this same function and checks that each tile is visited exactly once.
struct GqaPiece { int32_t kvh, a, b; int64_t pair_lo; };
__host__ __device__ inline GqaPiece gqa_piece(const GqaPlan& plan, int32_t i, int32_t tile_off, int32_t n_tiles, int64_t g, int64_t g_end) {
    GqaPiece pc;
    const int64_t item_lo = ((int64_t)tile_off + (int64_t)plan.bnd * i) * plan.n_kv_heads;
    pc.kvh = (int32_t)((g - item_lo) / (n_tiles + plan.bnd));
    pc.pair_lo = item_lo + (int64_t)pc.kvh * (n_tiles + plan.bnd) + plan.bnd;
    const int64_t a = g - pc.pair_lo, b = g_end - pc.pair_lo;
    pc.a = (int32_t)(a > 0 ? a : 0);
    pc.b = (int32_t)(b < n_tiles ? b : n_tiles);
    return pc;
}

// grid = n_SM * CTAs/SM (<= total tiles), block = 128.  items[].tile_off = exclusive prefix of n_tiles.
template <int D, bool FP8>
__global__ void __launch_bounds__(GqaCfg<D, FP8>::kThreads)
attend_gqa_kernel(AttendParams p, GqaPlan plan) {
    using C = GqaCfg<D, FP8>;
    using Tile = typename std::conditional<FP8, WarpTileF8<D>, WarpTile<D>>::type;
    if (p.pdl_early) pdl_launch_dependents();
    if (threadIdx.x == 0) stamp_begin(p);
    pdl_wait();                  // the work list and this step's K/V rows come from the append kernel
    if (blockIdx.x == 0 && threadIdx.x == 0) publish_past_wait(p);
    extern __shared__ __align__(128) uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 127u) & ~127u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    const int32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t ring = smem_base + warp * C::kWarpBytes;
    const uint32_t bars = smem_base + C::NWARP * C::kWarpBytes + warp * C::NS * 8;
    if (lane == 0) {
        for (int s = 0; s < C::NS; ++s) mbar_init(bars + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __shared__ int32_t s_range;
    if (plan.sm_mode && threadIdx.x == 0) {
        // one range per CTA, from the list of this SM's class (GqaPlan::sm_mode); if that list is used up (the hardware
        // placed the CTAs otherwise than 3 per SM) from the other one: ranges and CTAs are equally many, so one of the
        // two claims succeeds
        unsigned int smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        int32_t cls = __ldg(p.sm_class + smid) ? 1 : 0;
        int32_t idx = atomicAdd(p.gqa_ctr + 4 + cls, 1);
        if (idx >= (cls ? plan.n_total - plan.n_static : plan.n_static)) {
            cls ^= 1;
            idx = atomicAdd(p.gqa_ctr + 4 + cls, 1);
        }
        const bool got = idx < (cls ? plan.n_total - plan.n_static : plan.n_static);
        s_range = got ? (cls ? plan.n_static + idx : idx) : plan.n_total;
    }
    __syncthreads();
    uint32_t phase_bits = 0;                             // parity of each private stage

    const int32_t Hkv = plan.n_kv_heads;
    int32_t range = plan.sm_mode ? s_range : (int32_t)blockIdx.x;   // first the CTA's static range, then claimed ones
    const int32_t bnd = plan.bnd;
    while (range < plan.n_total) {
    int64_t g = plan.range_lo(range);                    // (cost units, see make_gqa_plan)
    const int64_t g_end = plan.range_hi(range);
    // the item that holds the range's first unit: from the host's table, else by binary search
    // (largest i with (tile_off[i] + bnd * i) * Hkv <= g); later pairs of the range follow without a search
    int32_t i = 0;
    if (p.range_item) {
        i = p.range_item[range];
    } else {
        int32_t lo = 0, hi = p.n_items - 1;
        while (lo < hi) {
            const int32_t mid = (lo + hi + 1) >> 1;
            if (((int64_t)p.items[mid].tile_off + (int64_t)bnd * mid) * Hkv <= g) lo = mid; else hi = mid - 1;
        }
        i = lo;
    }
    int32_t pre = 0;        // 1: the first tile of the coming pair is already in flight, in stage kPre
    while (g < g_end) {
        // ---- the (item, head) pair that holds unit g, and this CTA's piece of it: tiles [a, b) ----
        const AttendItem it = p.items[i];
        const GqaPiece pc = gqa_piece(plan, i, it.tile_off, it.n_tiles, g, g_end);
        const int32_t kvh = pc.kvh, a = pc.a, b = pc.b;
        const int64_t pair_lo = pc.pair_lo;                                    // unit of the pair's tile 0
        if (b <= a) break;                               // the range ends inside this pair's start-up units
        const int32_t first_cta = plan.range_of(pair_lo);                      // first / last range of this pair
        const int32_t last_cta = plan.range_of(pair_lo + it.n_tiles - 1);

        const int32_t* trow = p.table + (int64_t)it.sid * p.tbl_width;
        const uint8_t* head_base = p.kv_layer + (int64_t)kvh * p.L.head_bytes;
        // this warp's tiles: a + warp, a + warp + 4, ...   (private ring, prologue fills NS stages)
        const int32_t n_mine = (b - a - warp + C::NWARP - 1) / C::NWARP;
        const int32_t sbase = pre ? C::kPre : 0;   // k-th tile of this warp -> stage (k + sbase) % NS
        // Physical block ids of this warp's tiles, fetched 32 at a time (lane j: the warp's tiles j and 32 + j of the
        // piece) and handed out by shuffle: a refill is then shuffle -> bulk copy instead of logical block -> table slot
        // (an integer modulo) -> dependent table load (an L2 round trip) -> bulk copy, by one lane, for every tile.
        // A piece of more than 64 tiles per warp (W > 4096) looks the rest up one by one.
        auto lookup = [&](int32_t k) {
            return __ldg(trow + table_slot(tile_block(it, a + warp + k * C::NWARP), p.n_sink, p.ring));
        };
        const int32_t phys_c0 = lane < n_mine ? lookup(lane) : 0;
        const int32_t phys_c1 = lane + 32 < n_mine ? lookup(lane + 32) : 0;
        auto issue = [&](int32_t k) {                      // (all lanes)
            int32_t phys = __shfl_sync(0xffffffffu, (k & 32) ? phys_c1 : phys_c0, k & 31);
            if (k >= 64) phys = lookup(k);
            if (lane == 0) {
                const int32_t st = (k + sbase) % C::NS;
                const uint32_t bar = bars + 8 * st;
                mbar_expect_tx(bar, C::kHeadBytes);
                bulk_g2s(ring + st * C::kHeadBytes, head_base + (int64_t)phys * p.L.block_bytes, C::kHeadBytes, bar);
            }
        };
        for (int32_t k = pre; k < min(n_mine, C::NS); ++k) issue(k);
        Tile wt;                                          // (Q rows are fetched while the first tiles fly)
        wt.init(p, it, kvh, 0, lane);
        for (int32_t k = 0; k < n_mine; ++k) {
            const int32_t st = (k + sbase) % C::NS;
            mbar_wait(bars + 8 * st, (phase_bits >> st) & 1u);
            phase_bits ^= 1u << st;
            const int32_t p0 = tile_block(it, a + warp + k * C::NWARP) * kBlockTokens;
            const uint32_t kt = ring + st * C::kHeadBytes;
            if (!wt.skips(p, p0)) wt.template step<256>(p, it.len, kt, kt + C::kTileBytes, p0, lane);
            __syncwarp();                                  // every lane is done reading the stage
            if (k + C::NS < n_mine) issue(k + C::NS);
        }
        // ---- while the warps are merged below, the first tile of the NEXT pair of this range is
        // already on its way: when the merge scratch of the R rows fits the stages below kPre, stage kPre
        // takes that tile now (saves the table -> HBM round trip after every (item, head) boundary) ----
        const int32_t R_rows = it.q_len * p.G;
        pre = 0;
        if (R_rows * (D + 2) * 4 <= C::kPre * C::kHeadBytes && b == it.n_tiles && pair_lo + b + bnd < g_end) {
            const bool same = kvh + 1 < Hkv;
            const int32_t i2 = same ? i : i + 1;
            const int32_t sid2 = same ? it.sid : p.items[i2].sid;
            const int32_t nt2 = same ? it.n_tiles : p.items[i2].n_tiles;
            const int32_t sink2 = same ? it.n_sink_tiles : p.items[i2].n_sink_tiles;
            const int32_t first2 = same ? it.first_blk : p.items[i2].first_blk;
            const int32_t b2 = (int32_t)min((int64_t)nt2, g_end - (pair_lo + b + bnd));
            if (warp < b2) {
                if (lane == 0) {
                    const int32_t blk = warp < sink2 ? warp : first2 + (warp - sink2);
                    const int32_t phys = __ldg(p.table + (int64_t)sid2 * p.tbl_width + table_slot(blk, p.n_sink, p.ring));
                    const uint32_t bar = bars + 8 * C::kPre;
                    mbar_expect_tx(bar, C::kHeadBytes);
                    bulk_g2s(ring + C::kPre * C::kHeadBytes,
                             p.kv_layer + (int64_t)phys * p.L.block_bytes + (int64_t)(same ? kvh + 1 : 0) * p.L.head_bytes,
                             C::kHeadBytes, bar);
                }
                pre = 1;
            }
        }
        // ---- merge the four warps through shared memory (their rings are idle now) ----
        __syncthreads();
        wt.to_scratch(reinterpret_cast<float*>(smem_gen + warp * C::kWarpBytes), R_rows, lane);   // [R][D + 2], rows < R only
        __syncthreads();
        {
            // 128 threads: row = tid / 8 (16 rows), 8 threads x (D/8) consecutive dims each
            const int32_t row = threadIdx.x >> 3, sub = threadIdx.x & 7;
            const int32_t R = it.q_len * p.G;
            if (row < R) {
                const float* sc = reinterpret_cast<const float*>(smem_gen);
                float M = -INFINITY;
#pragma unroll
                for (int w = 0; w < C::NWARP; ++w) M = fmaxf(M, sc[w * (C::kWarpBytes / 4) + row * (D + 2) + D]);
                float wgt[C::NWARP], l = 0.f;
#pragma unroll
                for (int w = 0; w < C::NWARP; ++w) {
                    const float mw = sc[w * (C::kWarpBytes / 4) + row * (D + 2) + D];
                    wgt[w] = (mw == -INFINITY) ? 0.f : ex2(mw - M);
                    l += wgt[w] * sc[w * (C::kWarpBytes / 4) + row * (D + 2) + D + 1];
                }
                const int32_t r = row / p.G, gq = row - r * p.G;
                const int64_t qrow = (int64_t)(it.q_row_off + r) * p.Hq + kvh * p.G + gq;
                constexpr int DPT = D / 8;                    // dims per thread
                float acc[DPT];
#pragma unroll
                for (int d = 0; d < DPT; ++d) {
                    float v = 0.f;
#pragma unroll
                    for (int w = 0; w < C::NWARP; ++w) v += wgt[w] * sc[w * (C::kWarpBytes / 4) + row * (D + 2) + sub * DPT + d];
                    acc[d] = v;
                }
                if (first_cta == last_cta) {
                    const float inv = l > 0.f ? 1.f / l : 0.f;
                    uint32_t* dst = reinterpret_cast<uint32_t*>(p.out + qrow * D + sub * DPT);
#pragma unroll
                    for (int d = 0; d < DPT; d += 2) dst[d >> 1] = pack_bf16(acc[d] * inv, acc[d + 1] * inv);
                } else {
                    const int64_t slot = qrow * p.max_splits + (range - first_cta);
                    float4* dst = reinterpret_cast<float4*>(p.ws_acc + slot * D + sub * DPT);
#pragma unroll
                    for (int d = 0; d < DPT; d += 4) __stcg(dst + (d >> 2), make_float4(acc[d], acc[d + 1], acc[d + 2], acc[d + 3]));
                    if (sub == 0) __stcg(reinterpret_cast<float2*>(p.ws_ml + slot * 2), make_float2(M, l));
                }
            }
            // ---- row a6, fused: the LAST piece of this (item, head) to arrive combines them all
            // ("merged exactly once"); the ticket counter resets itself ----
            if (first_cta != last_cta) {                       // CTA-uniform
                __shared__ int32_t s_ticket;
                int32_t* ticket = p.tickets + (int64_t)i * Hkv + kvh;
                __threadfence();
                __syncthreads();
                if (threadIdx.x == 0) s_ticket = atomicAdd(ticket, 1);
                __syncthreads();
                const int32_t ns = last_cta - first_cta + 1;
                if (s_ticket == ns - 1) {
                    __threadfence();
                    if (row < R) {
                        const int32_t r = row / p.G, gq = row - r * p.G;
                        const int64_t qrow = (int64_t)(it.q_row_off + r) * p.Hq + kvh * p.G + gq;
                        const int64_t base = qrow * p.max_splits;
                        constexpr int DPT = D / 8;
                        float Mx = -INFINITY;
                        for (int32_t s2 = 0; s2 < ns; ++s2) Mx = fmaxf(Mx, __ldcg(p.ws_ml + (base + s2) * 2));
                        float acc[DPT], l = 0.f;
#pragma unroll
                        for (int d = 0; d < DPT; ++d) acc[d] = 0.f;
                        for (int32_t s2 = 0; s2 < ns; ++s2) {
                            const float2 ml = __ldcg(reinterpret_cast<const float2*>(p.ws_ml + (base + s2) * 2));
                            if (ml.x == -INFINITY) continue;      // this piece admitted no key for this row
                            const float w = ex2(ml.x - Mx);
                            l += w * ml.y;
                            const float4* src = reinterpret_cast<const float4*>(p.ws_acc + (base + s2) * D + sub * DPT);
#pragma unroll
                            for (int d = 0; d < DPT; d += 4) {
                                const float4 a = __ldcg(src + (d >> 2));
                                acc[d] += w * a.x; acc[d + 1] += w * a.y; acc[d + 2] += w * a.z; acc[d + 3] += w * a.w;
                            }
                        }
                        const float inv = l > 0.f ? 1.f / l : 0.f;
                        uint32_t* dst = reinterpret_cast<uint32_t*>(p.out + qrow * D + sub * DPT);
#pragma unroll
                        for (int d = 0; d < DPT; d += 2) dst[d >> 1] = pack_bf16(acc[d] * inv, acc[d + 1] * inv);
                    }
                    if (threadIdx.x == 0) *ticket = 0;
                }
            }
        }
        // scratch (generic-proxy stores) is dead before the rings are refilled by the async proxy
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        g = pair_lo + b;
        if (kvh + 1 == Hkv) ++i;                          // (a pair left unfinished ends the range anyway)
    }
    // ---- next range: one of the small dynamic ones, first come first served ----
    if (plan.n_total == plan.n_static || plan.sm_mode) break;
    if (threadIdx.x == 0) s_range = plan.n_static + atomicAdd(p.gqa_ctr, 1);
    __syncthreads();
    range = s_range;
    }
    // every CTA leaves through exactly one failed claim: the last one out zeroes the counters for
    // the next launch
    if (plan.sm_mode) {
        if (threadIdx.x == 0 && atomicAdd(p.gqa_ctr + 1, 1) == (int32_t)gridDim.x - 1) { p.gqa_ctr[1] = 0; p.gqa_ctr[4] = 0; p.gqa_ctr[5] = 0; }
    } else if (plan.n_total != plan.n_static && threadIdx.x == 0) {
        if (atomicAdd(p.gqa_ctr + 1, 1) == (int32_t)gridDim.x - 1) { p.gqa_ctr[0] = 0; p.gqa_ctr[1] = 0; }
    }
    if (threadIdx.x == 0) stamp_end(p);
}

// ------------------------------------------------------------------------------------------------
inline cudaError_t configure_attend_mma_kernels() {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(attend_gqa_kernel<128, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  GqaCfg<128, false>::kSmemBytes)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(attend_gqa_kernel<64, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  GqaCfg<64, false>::kSmemBytes)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(attend_gqa_kernel<128, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  GqaCfg<128, true>::kSmemBytes)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(attend_gqa_kernel<64, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                GqaCfg<64, true>::kSmemBytes);
}

// decode-class items (R <= 16); `fp8`: the pool holds E4M3 codes + row scales (KvLayout::fp8)
inline cudaError_t launch_attend_gqa(const AttendParams& p, const GqaPlan& plan, int32_t D, int32_t n_ctas, cudaStream_t st,
                                     bool pdl = false) {
    if (p.L.fp8) {
        if (D == 128) return launch_kernel(attend_gqa_kernel<128, true>, dim3(n_ctas), GqaCfg<128, true>::kThreads, GqaCfg<128, true>::kSmemBytes, st, pdl, p, plan);
        return launch_kernel(attend_gqa_kernel<64, true>, dim3(n_ctas), GqaCfg<64, true>::kThreads, GqaCfg<64, true>::kSmemBytes, st, pdl, p, plan);
    }
    if (D == 128) return launch_kernel(attend_gqa_kernel<128, false>, dim3(n_ctas), GqaCfg<128, false>::kThreads, GqaCfg<128, false>::kSmemBytes, st, pdl, p, plan);
    return launch_kernel(attend_gqa_kernel<64, false>, dim3(n_ctas), GqaCfg<64, false>::kThreads, GqaCfg<64, false>::kSmemBytes, st, pdl, p, plan);
}
}  // namespace metronome
