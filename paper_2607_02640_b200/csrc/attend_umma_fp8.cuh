// attend_umma_fp8.cuh -- row a7 (chunk prefill, causal inside the chunk) over an fp8 (E4M3) KV pool, on tcgen05 + TMEM.
//
// NEXT row f4 (sec. 4.1 "Orthogonal to KV compression, which shrinks each token ...:
// we bound which tokens stay resident, and the two compose"; format = DESIGN.md reading R18: E4M3 codes + one float32
// scale per (token, KV head) row).  Same decomposition as attend_umma.cuh (one CTA per (KV head, item segment),
// R = G x q_len <= 256 query rows as one or two M = 128 row tiles, S = Q K^T into double-buffered TMEM columns, one
// thread per query row for the softmax, O += P V with P read from TMEM), with these differences:
//
//   * The tensor-core operands are fp16, not bf16: E4M3 is a subset of fp16, so the codes convert EXACTLY and no scale
//     ever touches an operand.  The K scale of key j multiplies the finished fp32 score (softmax thread), the V scale is
//     folded into the softmax weight before it is rounded to fp16 -- relative to a running reference vref >= every V
//     scale seen so far, times 2^7: weights stay at or below 2^15 < 65504 even with the lazily updated row maximum
//     (p <= 2^8) and a key whose scale equals the reference (vref is only raised when a scale exceeds it), and keep
//     full fp16 precision down to p vs = 2^-21 vref.  fp16's 11 bits replace the bf16 hi + lo pair of the bf16 kernel:
//     ONE P V instruction per block instead of two.
//   * Q is staged as fp16 after an exact power-of-two prescale per row (its largest element into [1, 2)), undone in the
//     softmax's scale factor: |q| > 65504 and tiny rows both survive.
//   * Four CONVERTER warps sit between the producer and the MMA issuers: the producer bulk-copies whole (block, head)
//     units (K codes | V codes | scales, 4224 B at D = 128, contiguous in HBM) into a staging ring; the converters turn
//     the code tiles into the K-major / MN-major SWIZZLE_128B fp16 operands the MMAs read, zero V rows past the
//     session's length, and publish the half-stage's scales (ks_j, vs_j 2^7 / vref, vref) for the softmax threads.
//     HBM traffic per key and KV head: 2 D + 8 bytes instead of 4 D.
//   * A row tile count of one (R <= 128) runs on slot 0 alone (the bf16 kernel alternates half-stages between the two
//     softmax warpgroups there).
#pragma once
#include "attend_umma.cuh"

namespace metronome {

template <int D>
struct UmmaF8Cfg {
    static constexpr int KS = 4;                                  // KV blocks per half-stage (64 keys)
    static constexpr int NH = D / 64;
    static constexpr int kCodeTile = kBlockTokens * D;            // K or V codes of one (block, head)
    static constexpr int kStageBlk = 2 * kCodeTile + 2 * kBlockTokens * 4;   // = KvLayout::head_bytes of an fp8 pool
    static constexpr int kStageBytes = KS * kStageBlk;            // one half-stage as it arrives from HBM
    static constexpr int NSTAGE = 4;                              // staging entries
    static constexpr int kOpTile = kBlockTokens * D * 2;          // fp16 K or V operand of one block
    static constexpr int kBufBytes = KS * kOpTile;                // one K or one V half-stage, fp16
    static constexpr int kKHalfBytes = KS * kBlockTokens * 128;   // [64 keys][64 dims]
    static constexpr int kQHalfBytes = 128 * 128;                 // [128 rows][64 dims]
    static constexpr int kQBytes = 128 * D * 2;                   // Q rows of one slot
    static constexpr int NBUF = 5;                                // operand ring buffers
    static constexpr int NSC = 16;                                // scale slots (one per half-stage in flight)
    static constexpr int kScFloats = 136;                         // 64 ks | 64 vs 2^7 / vref | vref | pad
    static constexpr int kRingOff = 2 * kQBytes;
    static constexpr int kStageOff = kRingOff + NBUF * kBufBytes;
    static constexpr int kScOff = kStageOff + NSTAGE * kStageBytes;
    static constexpr int kQsOff = kScOff + NSC * kScFloats * 4;   // 256 floats: the rows' Q prescale
    static constexpr int kBarOff = kQsOff + 1024;
    static constexpr int kSmemBytes = kBarOff + 512 + 1024;       // + alignment slack
    static constexpr int kThreads = 512;                          // 16 warps: producer, 3 MMA issuers, 2 x 4 softmax, 4 converters
    static constexpr int kTmemCols = 512;
    static constexpr int kColS = 0, kColO = 256;
    static constexpr float kPScale = 128.f;                       // 2^7 (see the header)
    static_assert(kSmemBytes <= 232448, "shared memory budget");
    static_assert(kStageBlk % 128 == 0, "staging units stay 128-byte aligned");
};

// instruction descriptor, kind::f16: fp16 A x fp16 B -> f32, M = 128
__host__ __device__ constexpr uint32_t umma_idesc_f16(int n, bool b_mn_major) {
    return (1u << 4) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
__device__ __forceinline__ void sts_u4(uint32_t addr, uint4 v) {
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ float4 lds_f4(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float lds_f1(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
// 16 E4M3 codes -> 16 fp16 values (two 16-byte chunks)
__device__ __forceinline__ void e4m3x16_f16(uint4 x, uint4& lo, uint4& hi) {
    lo.x = e4m3x2_f16x2((uint16_t)x.x); lo.y = e4m3x2_f16x2((uint16_t)(x.x >> 16));
    lo.z = e4m3x2_f16x2((uint16_t)x.y); lo.w = e4m3x2_f16x2((uint16_t)(x.y >> 16));
    hi.x = e4m3x2_f16x2((uint16_t)x.z); hi.y = e4m3x2_f16x2((uint16_t)(x.z >> 16));
    hi.z = e4m3x2_f16x2((uint16_t)x.w); hi.w = e4m3x2_f16x2((uint16_t)(x.w >> 16));
}

// grid = (Hkv, total segments of the chunk-class items), block = 512, one CTA per SM
template <int D>
__global__ void __launch_bounds__(UmmaF8Cfg<D>::kThreads, 1)
attend_umma_fp8_kernel(AttendParams p) {
    using C = UmmaF8Cfg<D>;
    if (p.pdl_early) pdl_launch_dependents();
    if (threadIdx.x == 0) stamp_begin(p);
    pdl_wait();                  // the work list and this step's K/V rows come from the append kernel
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) publish_past_wait(p);
    extern __shared__ __align__(1024) uint8_t smem_umma8[];
    const uint32_t base = (smem_u32(smem_umma8) + 1023u) & ~1023u;      // swizzle atoms are 1024-byte aligned
    uint8_t* gen = smem_umma8 + (base - smem_u32(smem_umma8));
    const uint32_t sQ = base, sRing = base + C::kRingOff, sStage = base + C::kStageOff, sSc = base + C::kScOff,
                   sQs = base + C::kQsOff, sBar = base + C::kBarOff;
    auto bar_full = [&](int b) { return sBar + 8u * b; };                                   // operand ready (converters -> MMA)
    auto bar_empty = [&](int b) { return sBar + 8u * (C::NBUF + b); };                      // operand consumed (MMA -> converters)
    auto bar_stf = [&](int s) { return sBar + 8u * (2 * C::NBUF + s); };                    // staging full (bulk copy -> converters)
    auto bar_ste = [&](int s) { return sBar + 8u * (2 * C::NBUF + C::NSTAGE + s); };        // staging free (converters -> producer)
    constexpr int kB0 = 2 * C::NBUF + 2 * C::NSTAGE;
    auto bar_s = [&](int s, int buf) { return sBar + 8u * (kB0 + 2 * s + buf); };           // S ready  (MMA -> softmax)
    auto bar_p = [&](int s, int buf) { return sBar + 8u * (kB0 + 4 + 2 * s + buf); };       // P written (softmax -> MMA)
    auto bar_pv = [&](int s, int buf) { return sBar + 8u * (kB0 + 8 + 2 * s + buf); };      // P V out of that buffer done
    auto bar_o = [&](int s) { return sBar + 8u * (kB0 + 12 + s); };                         // last P V of slot s done
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(gen + C::kBarOff + 8 * (kB0 + 14));

    const int32_t kvh = blockIdx.x;
    const int32_t i = (int32_t)gridDim.y == p.n_items
                          ? (int32_t)blockIdx.y
                          : find_item(p.n_items, (int32_t)blockIdx.y, [&](int32_t k) { return p.items[k].split_off; });
    const AttendItem it = p.items[i];
    const int32_t split = (int32_t)blockIdx.y - it.split_off;
    const int32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t R = it.q_len * p.G;
    const bool two = R > 128;
    const int32_t n_slots = two ? 2 : 1;
    const int32_t tl0 = split * it.tiles_per_split;
    const int32_t tl1 = min(it.n_tiles, tl0 + it.tiles_per_split);
    const int32_t n_half = (tl1 - tl0 + C::KS - 1) / C::KS;             // half-stages of this segment
    const int32_t t_first = it.len - it.q_len;                          // reading R15: the last q_len positions
    // operand ring entry of K / V of half-stage h: K0 K1 V0 K2 V1 ... K(n-1) V(n-2) V(n-1)
    auto entry_k = [&](int32_t h) { return umma_seq_k(h); };
    auto entry_v = [&](int32_t h) { return umma_seq_v(h, n_half); };

    // Register budget per warpgroup (setmaxnreg; 512 threads launch with 128 each): producer + MMA issuers 72,
    // converters 104, the two softmax warpgroups 168 (one thread per query row holds 64 scores + 64 weights:
    // at 128 it spilled ~200 bytes per thread into the half-stage loop).  4 x 32 x (72 + 104 + 2 x 168) = 65536.
    if (warp < 4) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 72;");
        if (warp == 0) {
            // ================================ producer ================================
            if (lane == 0) {
                for (int b = 0; b < C::NBUF; ++b) { mbar_init(bar_full(b), 4); mbar_init(bar_empty(b), n_slots); }
                for (int s = 0; s < C::NSTAGE; ++s) { mbar_init(bar_stf(s), 1); mbar_init(bar_ste(s), 4); }
                for (int s = 0; s < 2; ++s) {
                    for (int buf = 0; buf < 2; ++buf) { mbar_init(bar_s(s, buf), 1); mbar_init(bar_p(s, buf), 4); mbar_init(bar_pv(s, buf), 1); }
                    mbar_init(bar_o(s), 1);
                }
                asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            }
            __syncwarp();
            named_arrive(1, C::kThreads);
            const int32_t* trow = p.table + (int64_t)it.sid * p.tbl_width;
            const uint8_t* head_base = p.kv_layer + (int64_t)kvh * p.L.head_bytes;
            // physical block ids of this segment's tiles, fetched ONCE (lane l holds tiles l, l+32, ...)
            constexpr int kPhysPre = 8;                               // 256 tiles; longer segments look up the rest
            int32_t phys_pre[kPhysPre];
    #pragma unroll
            for (int j = 0; j < kPhysPre; ++j) {
                const int32_t t = tl0 + j * 32 + lane;
                phys_pre[j] = t < tl1 ? __ldg(trow + table_slot(tile_block(it, t), p.n_sink, p.ring)) : 0;
            }
            auto phys_of = [&](int32_t rel) {                         // rel = tile - tl0; rel >> 5 is warp-uniform
                const int32_t j = rel >> 5;
                int32_t v = phys_pre[0];
    #pragma unroll
                for (int q = 1; q < kPhysPre; ++q) v = j == q ? phys_pre[q] : v;
                v = __shfl_sync(0xffffffffu, v, rel & 31);
                if (j >= kPhysPre) v = __ldg(trow + table_slot(tile_block(it, tl0 + rel), p.n_sink, p.ring));
                return v;
            };
            for (int32_t h = 0; h < n_half; ++h) {
                const int32_t st = h % C::NSTAGE, k = h / C::NSTAGE;
                if (k >= 1) mbar_wait(bar_ste(st), (k - 1) & 1);
                const int32_t t0 = tl0 + h * C::KS;
                const int32_t nt = min(C::KS, tl1 - t0);
                if (lane == 0) mbar_expect_tx(bar_stf(st), (uint32_t)nt * C::kStageBlk);
                __syncwarp();
                const int32_t phys = phys_of(h * C::KS + min(lane, nt - 1));        // (every lane takes part in the shuffle)
                if (lane < nt)
                    bulk_g2s(sStage + st * C::kStageBytes + lane * C::kStageBlk, head_base + (int64_t)phys * p.L.block_bytes,
                             C::kStageBlk, bar_stf(st));
            }
            return;
        }
        {
            // ================================ MMA issuers ================================
            // Warp 1 issues Q K^T for both slots, warps 2 / 3 issue P V of slot 0 / 1 (as in attend_umma.cuh).
            const bool is_pv = warp >= 2;
            const int32_t slot = is_pv ? warp - 2 : 0;
            if (warp == 1) {
                asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                             ::"r"(smem_u32(const_cast<uint32_t*>(tmem_slot))), "r"(C::kTmemCols));
                asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
            }
            tc_fence_before();
            named_sync(1, C::kThreads);
            tc_fence_after();
            const uint32_t tmem = *tmem_slot;
            constexpr uint32_t idesc_qk = umma_idesc_f16(C::KS * kBlockTokens, false);
            constexpr uint32_t idesc_pv = umma_idesc_f16(D, true);
            const uint32_t tSbase = tmem + C::kColS + 128 * slot, tOacc = tmem + C::kColO + D * slot;      // (P V warps)
            auto wait_full = [&](int32_t e) {
                mbar_wait(bar_full(e % C::NBUF), (e / C::NBUF) & 1);
                tc_fence_after();
            };
            auto release = [&](int32_t e) { if (lane == 0) umma_commit(bar_empty(e % C::NBUF)); };
            const uint32_t elect = lane == 0 ? 1u : 0u;
            // S[buf] = Q K^T over the K half-stage in ring entry e
            auto issue_qk = [&](int32_t qslot, int32_t buf, int32_t e) {
                const uint64_t dq0 = umma_desc(sQ + qslot * C::kQBytes, 16, 1024);
                const uint64_t dk0 = umma_desc(sRing + (e % C::NBUF) * C::kBufBytes, 16, 1024);
                const uint32_t ts = tmem + C::kColS + 128 * qslot + 64 * buf;
    #pragma unroll
                for (int kk = 0; kk < D / 16; ++kk)
                    umma_ss_e(ts, dq0 + (uint64_t)(((kk >> 2) * C::kQHalfBytes + (kk & 3) * 32) >> 4),
                              dk0 + (uint64_t)(((kk >> 2) * C::kKHalfBytes + (kk & 3) * 32) >> 4), idesc_qk, kk > 0 ? 1u : 0u, elect);
                if (lane == 0) umma_commit(bar_s(qslot, buf));
                __syncwarp();
            };
            // O (+)= P V over the V half-stage in ring entry e: one K = 16 MMA per valid block; the fp16 P of block b
            // sits in columns 32 (b / 2) + 8 (b % 2) .. + 7 of the S buffer
            auto issue_pv = [&](int32_t buf, int32_t e, int32_t nt, bool accumulate) {
                const uint64_t vd0 = umma_desc(sRing + (e % C::NBUF) * C::kBufBytes, 2048, 1024);
                const uint32_t pa0 = tSbase + 64 * buf;
    #pragma unroll
                for (int b = 0; b < C::KS; ++b) {
                    if (b < nt) {                             // (warp-uniform)
                        const uint32_t pa = pa0 + 32 * (b >> 1) + 8 * (b & 1);
                        const uint64_t vd = vd0 + (uint64_t)((b * C::kOpTile) >> 4);
                        umma_ts_e(tOacc, pa, vd, idesc_pv, (accumulate || b > 0) ? 1u : 0u, elect);
                    }
                }
                if (lane == 0) umma_commit(bar_pv(slot, buf));
                __syncwarp();
            };
            if (!is_pv) {
                // ---- Q K^T of every half-stage, for every slot: into S buffer h & 1 of the slot, as soon as P V of
                // h - 2 has drained that buffer ----
                for (int32_t h = 0; h < n_half; ++h) {
                    const int32_t e = entry_k(h);
                    wait_full(e);
                    for (int32_t qs = 0; qs < n_slots; ++qs) {
                        const int32_t buf = h & 1;
                        if (h >= 2) {
                            mbar_wait(bar_pv(qs, buf), ((h >> 1) - 1) & 1);
                            tc_fence_after();
                        }
                        issue_qk(qs, buf, e);
                        release(e);                          // (one arrival per consuming slot)
                    }
                }
            } else if (slot < n_slots) {
                // ---- P V: half-stage h out of S buffer h & 1, once the softmax has written P there ----
                for (int32_t h = 0; h < n_half; ++h) {
                    const int32_t e = entry_v(h), buf = h & 1;
                    const int32_t nt = min(C::KS, tl1 - (tl0 + h * C::KS));
                    wait_full(e);
                    mbar_wait(bar_p(slot, buf), (h >> 1) & 1);
                    tc_fence_after();
                    issue_pv(buf, e, nt, h > 0);
                    release(e);
                    if (h == n_half - 1 && lane == 0) umma_commit(bar_o(slot));
                }
            }
            if (warp == 1) {
                // every softmax warp has finished reading TMEM
                named_sync(2, 32 + 256);
                tc_fence_after();
                asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(C::kTmemCols));
            }
            return;
        }
    }
    if (warp >= 12) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 104;");
        // ================================ converters ================================
        // Operand ring entry e = K or V of a half-stage, in the order the MMA issuers consume them.  The staging
        // entry of half-stage j is awaited at K(j) (always before V(j)) and handed back after V(j).
        named_sync(1, C::kThreads);
        const int32_t cw = warp - 12, ctid = threadIdx.x - 384;
        constexpr int CPR = D / 16;                               // 16-code chunks per row
        float vref = 0.f;
        const int32_t n_entries = 2 * n_half;
        const int32_t last_tile = it.n_tiles - 1, last_valid = it.len & (kBlockTokens - 1);   // rows of the last block (0: all 16)
        for (int32_t e = 0; e < n_entries; ++e) {
            bool is_v;
            int32_t j;
            if (e == 0) { is_v = false; j = 0; }
            else if (e == n_entries - 1) { is_v = true; j = n_half - 1; }
            else if (e & 1) { is_v = false; j = (e + 1) >> 1; }
            else { is_v = true; j = (e >> 1) - 1; }
            const int32_t b = e % C::NBUF, k = e / C::NBUF;
            const int32_t st = j % C::NSTAGE;
            if (!is_v) mbar_wait(bar_stf(st), (j / C::NSTAGE) & 1);
            if (k >= 1) mbar_wait(bar_empty(b), (k - 1) & 1);
            const int32_t t0 = tl0 + j * C::KS;
            const int32_t nt = min(C::KS, tl1 - t0);
            const uint32_t src = sStage + st * C::kStageBytes, dst = sRing + b * C::kBufBytes;
            if (!is_v) {
                // ---- the half-stage's scales: key kk = 16 blk + r; keys past the segment or the session: 0 ----
                float ksv[2], vsv[2];
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const int32_t kk = lane + 32 * q, blk = kk >> 4, r = kk & 15;
                    const bool ok = blk < nt && (t0 + blk != last_tile || last_valid == 0 || r < last_valid);
                    const uint32_t a = src + blk * C::kStageBlk + 2 * C::kCodeTile + r * 4;
                    ksv[q] = ok ? lds_f1(a) : 0.f;
                    vsv[q] = ok ? lds_f1(a + kBlockTokens * 4) : 0.f;
                }
                float vmax = fmaxf(vsv[0], vsv[1]);
#pragma unroll
                for (int o = 16; o >= 1; o >>= 1) vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
                if (vmax > vref) vref = vmax * 4.f;               // (every converter warp keeps the same vref)
                if (cw == 0) {
                    const float inv = vref > 0.f ? C::kPScale / vref : 0.f;
                    float* sc = reinterpret_cast<float*>(gen + C::kScOff) + (j % C::NSC) * C::kScFloats;
                    sc[lane] = ksv[0]; sc[lane + 32] = ksv[1];
                    sc[64 + lane] = vsv[0] * inv; sc[96 + lane] = vsv[1] * inv;
                    if (lane == 0) sc[128] = vref;
                }
            }
            // ---- code tiles -> fp16 operand: K rows into [half][64 keys][128 B] (K-major), V tiles as in the bf16
            // layout ([half][16 keys][128 B] per block: MN-major operand of one K = 16 MMA); 16-byte chunks swizzled ----
            const int32_t n_task = nt * kBlockTokens * CPR;
            for (int32_t task = ctid; task < n_task; task += 128) {
                const int32_t blk = task / (kBlockTokens * CPR), rem = task - blk * (kBlockTokens * CPR);
                const int32_t r = rem / CPR, c = rem - r * CPR;
                uint4 x = lds_u4(src + blk * C::kStageBlk + (is_v ? C::kCodeTile : 0) + fp8_chunk_offset(D, r, c));
                if (is_v && t0 + blk == last_tile && last_valid != 0 && r >= last_valid) x = make_uint4(0u, 0u, 0u, 0u);
                uint4 lo, hi;
                e4m3x16_f16(x, lo, hi);
                const int32_t c0 = 2 * c, c1 = 2 * c + 1;         // 8-element chunks of the fp16 row
                if (is_v) {
                    sts_u4(dst + blk * C::kOpTile + tile_chunk_offset(r, c0), lo);
                    sts_u4(dst + blk * C::kOpTile + tile_chunk_offset(r, c1), hi);
                } else {
                    const int32_t row = blk * kBlockTokens + r;
                    sts_u4(dst + (c0 >> 3) * C::kKHalfBytes + row * 128 + (((c0 & 7) ^ (r & 7)) << 4), lo);
                    sts_u4(dst + (c1 >> 3) * C::kKHalfBytes + row * 128 + (((c1 & 7) ^ (r & 7)) << 4), hi);
                }
            }
            fence_async_smem();                                   // generic-proxy stores before the MMA's async-proxy reads
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(bar_full(b));
                if (is_v) mbar_arrive(bar_ste(st));
            }
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 168;");

    // ================================ softmax warps (4 .. 11) ================================
    const int32_t slot = (warp - 4) >> 2, quarter = warp & 3;       // TMEM lanes 32 (warp % 4) .. + 31
    const int32_t row = quarter * 32 + lane;
    const int32_t tile_row0 = 128 * slot;
    const int32_t rho = tile_row0 + row;                              // rho = r * G + g
    const bool valid = rho < R;
    const int32_t rq = rho / p.G, gq = rho - rq * p.G;
    const int32_t t = valid ? t_first + rq : -1;                      // -1: padding row, admits nothing
    const bool warp_active = tile_row0 + quarter * 32 < R;
    const int32_t t_wmin = t_first + (tile_row0 + quarter * 32) / p.G;
    const int32_t t_wmax = t_first + (min(R, tile_row0 + quarter * 32 + 32) - 1) / p.G;

    // ---- Q rows -> shared memory as fp16, K-major SWIZZLE_128B, one [128][64] region per 64-dim half.  A row's
    // D / 8 chunks sit in consecutive lanes: its largest magnitude by shuffles, 2^(127 - E) brings it into [1, 2)
    // (exact), the inverse goes to sQs[row] for the thread that owns the row in the softmax ----
    {
        const int32_t tid2 = threadIdx.x - 128;
        const int32_t n_rows = two ? 256 : 128;
        constexpr int CPR = D / 8;                                    // 8-element chunks per row
        constexpr int kBatch = 8;
        for (int32_t idx0 = tid2; idx0 < n_rows * CPR; idx0 += 256 * kBatch) {
            uint4 x[kBatch];
#pragma unroll
            for (int u = 0; u < kBatch; ++u) {
                const int32_t idx = idx0 + 256 * u, rr = idx / CPR, c = idx % CPR;
                x[u] = make_uint4(0u, 0u, 0u, 0u);
                if (idx < n_rows * CPR && rr < R) {
                    const int32_t r2 = rr / p.G, g2 = rr - r2 * p.G;
                    x[u] = __ldg(reinterpret_cast<const uint4*>(p.q + ((int64_t)(it.q_row_off + r2) * p.Hq + kvh * p.G + g2) * D + c * 8));
                }
            }
#pragma unroll
            for (int u = 0; u < kBatch; ++u) {
                const int32_t idx = idx0 + 256 * u, rr = idx / CPR, c = idx % CPR;      // (idx < n_rows * CPR for every lane or none)
                const uint32_t w[4] = {x[u].x, x[u].y, x[u].z, x[u].w};
                float amax = 0.f;
#pragma unroll
                for (int q = 0; q < 4; ++q) amax = fmaxf(amax, fmaxf(fabsf(bf16lo(w[q])), fabsf(bf16hi(w[q]))));
#pragma unroll
                for (int o = CPR / 2; o >= 1; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
                int32_t E = (__float_as_int(amax) >> 23) & 0xff;
                E = E == 0 ? 127 : min(E, 253);
                const float down = __int_as_float((254 - E) << 23);
                if (idx < n_rows * CPR) {
                    uint4 y;
                    y.x = pack_f16(bf16lo(w[0]) * down, bf16hi(w[0]) * down);
                    y.y = pack_f16(bf16lo(w[1]) * down, bf16hi(w[1]) * down);
                    y.z = pack_f16(bf16lo(w[2]) * down, bf16hi(w[2]) * down);
                    y.w = pack_f16(bf16lo(w[3]) * down, bf16hi(w[3]) * down);
                    sts_u4(sQ + (rr >> 7) * C::kQBytes + (c >> 3) * C::kQHalfBytes + (rr & 127) * 128 + (((c & 7) ^ (rr & 7)) << 4), y);
                    if (c == 0) reinterpret_cast<float*>(gen + C::kQsOff)[rr] = __int_as_float(E << 23);
                }
            }
        }
        fence_async_smem();
    }
    named_sync(1, C::kThreads);
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t lane_base = (uint32_t)(quarter * 32) << 16;
    const uint32_t tS = tmem + lane_base + C::kColS + 128 * slot;     // two 64-column S buffers; fp16 P goes over S
    const uint32_t tO = tmem + lane_base + C::kColO + D * slot;
    const float qsl = lds_f1(sQs + 4 * rho) * p.scale_log2;            // log2-domain scale of this row's raw scores

    // One half-stage per thread = per query row: 64 raw scores read ONCE into registers, times the keys' K scales,
    // row max, exp2, and P (times the keys' V weights, fp16) written back over the columns just read.
    float m_run = -INFINITY, m_used = -INFINITY;
    float l0 = 0.f, l1 = 0.f, l2 = 0.f, l3 = 0.f;                     // four partial sums (ILP)
    float my_vref = 0.f;                                              // the V reference O is accumulated in
    const int32_t n_mine = slot < n_slots ? n_half : 0;
    for (int32_t k = 0; k < n_mine; ++k) {
        const int32_t h = k, buf = k & 1;
        mbar_wait(bar_s(slot, buf), (k >> 1) & 1);
        tc_fence_after();
        if (warp_active) {
            const uint32_t tSb = tS + 64 * buf;
            const uint32_t sc = sSc + (h % C::NSC) * (C::kScFloats * 4);
            uint32_t sa[32], sb[32];
            tmem_ld32(tSb, sa);
            tmem_ld32(tSb + 32, sb);
            const float vref_h = lds_f1(sc + 128 * 4);
            const int32_t t0 = tl0 + h * C::KS;
            const int32_t nt = min(C::KS, tl1 - t0);
            const int32_t p_first = tile_block(it, t0) * kBlockTokens;
            const bool full = nt == C::KS && t0 >= it.n_sink_tiles && p_first + C::KS * kBlockTokens - 1 <= t_wmin &&
                              t_wmax - p_first < p.W;
            tmem_wait_ld();
            // ---- raw score x K scale of its key ----
            auto scale_chunk = [&](uint32_t (&s)[32], int c) {
#pragma unroll
                for (int kk = 0; kk < 32; kk += 4) {
                    const float4 ks = lds_f4(sc + (32 * c + kk) * 4);
                    float a0, a1, a2, a3;
                    f2_unpack(f2_mul(f2_pack(__uint_as_float(s[kk]), __uint_as_float(s[kk + 1])), f2_pack(ks.x, ks.y)), a0, a1);
                    f2_unpack(f2_mul(f2_pack(__uint_as_float(s[kk + 2]), __uint_as_float(s[kk + 3])), f2_pack(ks.z, ks.w)), a2, a3);
                    s[kk] = __float_as_uint(a0); s[kk + 1] = __float_as_uint(a1);
                    s[kk + 2] = __float_as_uint(a2); s[kk + 3] = __float_as_uint(a3);
                }
            };
            scale_chunk(sa, 0);
            scale_chunk(sb, 1);
            if (!full) {
                auto mask_chunk = [&](uint32_t (&s)[32], int c) {
#pragma unroll
                    for (int bb = 0; bb < 2; ++bb) {
                        const int32_t b = 2 * c + bb;
                        const int32_t p0 = b < nt ? tile_block(it, t0 + b) * kBlockTokens : INT32_MAX / 2;
#pragma unroll
                        for (int kk = 0; kk < kBlockTokens; ++kk)
                            if (!admit(p0 + kk, t, p.S, p.W)) s[bb * kBlockTokens + kk] = 0xFF800000u;   // -inf
                    }
                };
                mask_chunk(sa, 0);
                mask_chunk(sb, 1);
            }
            float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
            for (int kk = 0; kk < 32; kk += 2) {
                mx0 = fmaxf(mx0, __uint_as_float(sa[kk]));
                mx1 = fmaxf(mx1, __uint_as_float(sa[kk + 1]));
                mx2 = fmaxf(mx2, __uint_as_float(sb[kk]));
                mx3 = fmaxf(mx3, __uint_as_float(sb[kk + 1]));
            }
            const float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * qsl;
            m_run = fmaxf(m_run, mx);
            if (k == 0) {
                m_used = m_run;                                       // O is still empty
                my_vref = vref_h;
            } else {
                // lazy rescale: keep the stale reference max while it is within 2^8 of the true one; a raised V
                // reference (the same for every row: warp-uniform) rescales O as well
                const bool need = (m_run - m_used) > 8.f;             // (-inf) - (-inf) = NaN -> false
                const bool grow = vref_h != my_vref;
                if (grow || __any_sync(0xffffffffu, need)) {
                    // S is double buffered, so P V of the previous half-stage may still be running
                    mbar_wait(bar_pv(slot, (k - 1) & 1), ((k - 1) >> 1) & 1);
                    tc_fence_after();
                    const float f = (need && m_used != -INFINITY) ? ex2(m_used - m_run) : 1.f;
                    l0 *= f; l1 *= f; l2 *= f; l3 *= f;
                    const float fo = grow ? f * (my_vref / vref_h) : f;
#pragma unroll
                    for (int c = 0; c < D / 32; ++c) {
                        uint32_t o[32];
                        tmem_ld32(tO + 32 * c, o);
                        tmem_wait_ld();
#pragma unroll
                        for (int kk = 0; kk < 32; ++kk) o[kk] = __float_as_uint(__uint_as_float(o[kk]) * fo);
                        tmem_st32(tO + 32 * c, o);
                    }
                    if (need) m_used = m_run;
                    my_vref = vref_h;
                }
            }
            const float sub = m_used == -INFINITY ? 0.f : m_used;     // nothing admitted yet: every p is 0
            const uint64_t scale2 = f2_pack(qsl, qsl), nsub2 = f2_pack(-sub, -sub);
            uint64_t lA = f2_pack(l0, l1), lB = f2_pack(l2, l3);
            auto exp_chunk = [&](uint32_t (&cur)[32], int c) {
                uint32_t pk[16];
#pragma unroll
                for (int kk = 0; kk < 32; kk += 4) {
                    const float4 vw = lds_f4(sc + (64 + 32 * c + kk) * 4);
                    float x0, x1, x2, x3;
                    f2_unpack(f2_fma(f2_pack(__uint_as_float(cur[kk]), __uint_as_float(cur[kk + 1])), scale2, nsub2), x0, x1);
                    f2_unpack(f2_fma(f2_pack(__uint_as_float(cur[kk + 2]), __uint_as_float(cur[kk + 3])), scale2, nsub2), x2, x3);
                    const uint64_t pa = f2_pack(ex2(x0), ex2(x1)), pb = f2_pack(ex2(x2), ex2(x3));
                    lA = f2_add(lA, pa);
                    lB = f2_add(lB, pb);
                    float w0, w1, w2, w3;
                    f2_unpack(f2_mul(pa, f2_pack(vw.x, vw.y)), w0, w1);
                    f2_unpack(f2_mul(pb, f2_pack(vw.z, vw.w)), w2, w3);
                    pk[kk >> 1] = pack_f16(w0, w1);
                    pk[(kk >> 1) + 1] = pack_f16(w2, w3);
                }
                tmem_st16(tSb + 32 * c, pk);
            };
            exp_chunk(sa, 0);
            exp_chunk(sb, 1);
            f2_unpack(lA, l0, l1);
            f2_unpack(lB, l2, l3);
            tmem_wait_st();
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_p(slot, buf));
    }
    const float l = (l0 + l1) + (l2 + l3);

    // ---- epilogue: O (in units of vref / 2^7) -> bf16 output, or the unnormalised partial of a split, 32 columns at a time ----
    if (n_mine > 0) {
        mbar_wait(bar_o(slot), 0);
        tc_fence_after();
        if (warp_active) {
            const int64_t qrow = (int64_t)(it.q_row_off + rq) * p.Hq + kvh * p.G + gq;
            const float vu = my_vref * (1.f / C::kPScale);
            const float fin = it.n_splits == 1 ? (l > 0.f ? vu / l : 0.f) : vu;
            const int64_t ws = qrow * p.max_splits + split;
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
                uint32_t ou[32];
                tmem_ld32(tO + 32 * c, ou);
                tmem_wait_ld();
                float o[32];
#pragma unroll
                for (int kk = 0; kk < 32; ++kk) o[kk] = __uint_as_float(ou[kk]) * fin;
                if (!valid) continue;
                if (it.n_splits == 1) {
                    uint4* dst = reinterpret_cast<uint4*>(p.out + qrow * D + 32 * c);
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        dst[q] = make_uint4(pack_bf16(o[8 * q], o[8 * q + 1]), pack_bf16(o[8 * q + 2], o[8 * q + 3]),
                                            pack_bf16(o[8 * q + 4], o[8 * q + 5]), pack_bf16(o[8 * q + 6], o[8 * q + 7]));
                } else {
                    float4* dst = reinterpret_cast<float4*>(p.ws_acc + ws * D + 32 * c);
#pragma unroll
                    for (int q = 0; q < 8; ++q) dst[q] = make_float4(o[4 * q], o[4 * q + 1], o[4 * q + 2], o[4 * q + 3]);
                }
            }
            if (valid && it.n_splits != 1) {
                p.ws_ml[ws * 2] = m_used;
                p.ws_ml[ws * 2 + 1] = l;
            }
        }
    }
    tc_fence_before();
    named_arrive(2, 32 + 256);
    if (threadIdx.x == 128) stamp_end(p);
}

// ------------------------------------------------------------------------------------------------
inline cudaError_t configure_attend_umma_fp8_kernels() {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(attend_umma_fp8_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  UmmaF8Cfg<128>::kSmemBytes)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(attend_umma_fp8_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                UmmaF8Cfg<64>::kSmemBytes);
}

// chunk-class items (16 < R <= 256) of an fp8 pool: p.items / p.n_items must point at them
inline cudaError_t launch_attend_umma_fp8(const AttendParams& p, int32_t D, int32_t Hkv, int32_t total_splits, cudaStream_t st,
                                          bool pdl = false) {
    dim3 grid(Hkv, total_splits);
    if (D == 128) return launch_kernel(attend_umma_fp8_kernel<128>, grid, UmmaF8Cfg<128>::kThreads, UmmaF8Cfg<128>::kSmemBytes, st, pdl, p);
    return launch_kernel(attend_umma_fp8_kernel<64>, grid, UmmaF8Cfg<64>::kThreads, UmmaF8Cfg<64>::kSmemBytes, st, pdl, p);
}

}  // namespace metronome
