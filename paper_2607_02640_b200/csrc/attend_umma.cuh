// attend_umma.cuh -- row a7 (chunk prefill) on the 5th-generation tensor cores: tcgen05.mma with
// TMEM accumulators (SASS UTCHMMA / LDTM / STTM), operands staged by bulk async copies (UBLKCP).
//
// The R = G x q_len query rows that share one KV head ("grouped-query attention",
// "mixed prefill/decode"; L46 "prefill the new chunk") are a real dense contraction against the
// session's sink + window keys: S = Q K^T and O = P V with M = 128-row tiles.  One CTA owns one
// (item, KV head, split-KV segment) and streams its KV ONCE from HBM in half-stages of 4 blocks
// (64 keys):
//
//   warp 0      producer (the segment's physical block ids are fetched once): per half-stage, bulk
//               copies of the K tiles (one 2 KB copy per 64-dim half,
//               so the halves of 4 blocks form one UMMA K-major operand) and of the V tiles (a V
//               tile as laid out in HBM already IS a SWIZZLE_128B MN-major operand of one K=16
//               MMA), into a ring of 16 KB buffers, mbarrier complete_tx
//   warps 1-3   MMA issuers (warp 1 also allocates TMEM): warp 1 issues Q K^T for both slots, warps
//               2 / 3 issue P V of slot 0 / 1 -- one thread only gets a tcgen05.mma out every ~110-130
//               cycles, so the 32 MMAs of a half-stage are spread over three threads; per half-stage h:
//                 S = Q K_h^T   (SS form, D/16 instructions 128x64x16)   -> one of TWO S buffers
//                 O += P_h V_h  (TS form: P read from TMEM, V from shared memory; hi and lo parts)
//               S is double buffered, so Q K^T of half-stage h+1 is issued BEFORE P V of h (it only
//               waits for P V of h-1 to have drained the buffer): the softmax warps never wait for
//               the tensor pipe in steady state
//   warps 4-7   softmax warpgroup of slot 0, warps 8-11 of slot 1: ONE THREAD PER QUERY ROW
//               (tcgen05.ld 32x32b, 64 scores in registers): token-exact union mask on boundary
//               half-stages, row max and row sum without any shuffle, exp2 in the log2 domain, P split
//               into bf16 hi + lo and written back over the S buffer (tcgen05.st), lazy rescale of
//               O (only when the max moved by > 2^8, after the previous P V has completed)
//
// Two slots (TMEM: 2 x (2 x 64 S/P + D O) columns of the 512):
//   R > 128  : slot s = rows [128 s, 128 s + 128), both slots see every half-stage
//   R <= 128 : both slots hold the same rows; slot s takes half-stages h = s (mod 2); the two
//              partial (O, m, l) are merged through shared memory at the end
// Sinks go first, in segment 0 only; a single segment writes the final bf16 output,
// several write unnormalised partials for merge_kernel (row a6).
#pragma once
#include "attend_mma.cuh"

namespace metronome {

// HALF: the variant for items of R <= 128 rows (one row tile): one softmax warpgroup, 256 TMEM columns and a ring of 4
// buffers, so that TWO CTAs fit an SM and each runs under the other's prologue (Q staging, TMEM allocation, first tiles)
// and epilogue (O read-out, normalisation, store): ~7 us of a ~22 us (item, head) pair on config 4.
template <int D, bool HALF = false>
struct UmmaCfg {
    static constexpr int KS = 4;                          // KV blocks per half-stage (64 keys)
    static constexpr int NH = D / 64;                     // 64-dim halves (128-byte swizzle span)
    static constexpr int kTileBytes = kBlockTokens * D * 2;   // K or V of one (block, head)
    static constexpr int kBufBytes = KS * kTileBytes;     // 16 KB at D = 128: one K or one V half-stage
    static constexpr int kKHalfBytes = KS * kBlockTokens * 128;   // [64 keys][64 dims]
    static constexpr int kQHalfBytes = 128 * 128;         // [128 rows][64 dims]
    static constexpr int kQBytes = 128 * D * 2;           // Q rows of one slot
    static constexpr int NQ = HALF ? 1 : 2;               // row tiles (slots) a CTA can hold
    static constexpr int NBUF = HALF ? 4 : (D == 128 ? 10 : 12);       // ring buffers
    static constexpr int kBarOff = NQ * kQBytes + NBUF * kBufBytes;
    static constexpr int kMlOff = kBarOff + 512;          // (m, l) of slot 1 for the in-CTA merge
    static constexpr int kSmemBytes = kMlOff + 1024 + 1024;   // + alignment slack
    static constexpr int kThreads = HALF ? 256 : 384;     // 12 warps: producer, 3 MMA issuers, 2 x 4 softmax (HALF: 8 warps, one softmax warpgroup)
    static constexpr int kSoftmaxThreads = HALF ? 128 : 256;
    static constexpr int kTmemCols = HALF ? 256 : 512;
    static constexpr int kColS = 0, kColO = HALF ? 128 : 256;   // S buffers of slot s at 128 s + {0, 64}; O_s at kColO + D s
    static_assert(kSmemBytes <= (HALF ? 115712 : 232448), "shared memory budget");
    static_assert(!HALF || kColO + D <= kTmemCols, "TMEM budget of the half-size variant");
};

// ---- tcgen05 / UMMA primitives --------------------------------------------------------------
// shared-memory matrix descriptor, SWIZZLE_128B (cute::UMMA::SmemDescriptor bit layout)
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((saddr >> 4) & 0x3FFFu) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
// instruction descriptor, kind::f16: (bf16 | fp16) A x bf16 B -> f32, M = 128
__host__ __device__ constexpr uint32_t umma_idesc(int n, bool b_mn_major, bool a_fp16 = false) {
    return (1u << 4) | ((a_fp16 ? 0u : 1u) << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) |
           ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint64_t a, uint64_t b, uint32_t idesc, uint32_t accum) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(a), "l"(b), "r"(idesc), "r"(accum) : "memory");
}
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b, uint32_t idesc, uint32_t accum) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_tmem), "l"(b), "r"(idesc), "r"(accum) : "memory");
}
// The same, issued by the lane whose `elect` is non-zero while EVERY lane of the warp carries the
// (warp-uniform) operands: the descriptor arithmetic then stays on the uniform datapath instead of
// running as a dependent chain of one lane plus R2UR moves (measured: ~130 -> ~45 cycles per MMA issued).
__device__ __forceinline__ void umma_ss_e(uint32_t d_tmem, uint64_t a, uint64_t b, uint32_t idesc, uint32_t accum, uint32_t elect) {
    asm volatile("{\n\t.reg .pred p, e;\n\tsetp.ne.b32 p, %4, 0;\n\tsetp.ne.b32 e, %5, 0;\n\t"
                 "@e tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(a), "l"(b), "r"(idesc), "r"(accum), "r"(elect) : "memory");
}
__device__ __forceinline__ void umma_ts_e(uint32_t d_tmem, uint32_t a_tmem, uint64_t b, uint32_t idesc, uint32_t accum, uint32_t elect) {
    asm volatile("{\n\t.reg .pred p, e;\n\tsetp.ne.b32 p, %4, 0;\n\tsetp.ne.b32 e, %5, 0;\n\t"
                 "@e tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "r"(a_tmem), "l"(b), "r"(idesc), "r"(accum), "r"(elect) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void named_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void named_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// 32 lanes x 32 consecutive 32-bit columns: thread i of the warp gets lane (quarter base + i)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t* r) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                 "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
                   "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
                   "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr));
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t* r) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
                 "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
                 ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
                   "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]),
                   "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]),
                   "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
                 : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
                 "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
                   "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
                 : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }


// Order in which the ring is filled and drained.  Each slot runs Q K^T one half-stage ahead of P V:
//   R > 128  (both slots consume every entry): K0 K1 V0 K2 V1 ... K(n-1) V(n-2) V(n-1)
//   R <= 128 (slot s consumes half-stages h = s mod 2): the same order over PAIRS (2j, 2j+1), each
//            pair entry expanded into its two half-stages; a missing last half-stage is a phantom
//            entry (no bytes) so that the indices stay closed-form
__device__ __forceinline__ int32_t umma_seq_k(int32_t j) { return j == 0 ? 0 : 2 * j - 1; }
__device__ __forceinline__ int32_t umma_seq_v(int32_t j, int32_t n) { return j == n - 1 ? 2 * n - 1 : 2 * j + 2; }

// grid = (Hkv, total segments of the chunk-class items), block = 384, one CTA per SM
template <int D, bool HALF>
__global__ void __launch_bounds__(UmmaCfg<D, HALF>::kThreads, HALF ? 2 : 1)
attend_umma_kernel(AttendParams p) {
    using C = UmmaCfg<D, HALF>;
    if (p.pdl_early) pdl_launch_dependents();
    if (threadIdx.x == 0) stamp_begin(p);
    pdl_wait();                  // the work list and this step's K/V rows come from the append kernel
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) publish_past_wait(p);
    extern __shared__ __align__(1024) uint8_t smem_umma[];
    const uint32_t base = (smem_u32(smem_umma) + 1023u) & ~1023u;       // swizzle atoms are 1024-byte aligned
    uint8_t* gen = smem_umma + (base - smem_u32(smem_umma));
    const uint32_t sQ = base, sRing = base + C::NQ * C::kQBytes, sBar = base + C::kBarOff;
    auto bar_full = [&](int b) { return sBar + 8u * b; };
    auto bar_empty = [&](int b) { return sBar + 8u * (C::NBUF + b); };
    auto bar_s = [&](int s, int buf) { return sBar + 8u * (2 * C::NBUF + 2 * s + buf); };       // S ready  (MMA -> softmax)
    auto bar_p = [&](int s, int buf) { return sBar + 8u * (2 * C::NBUF + 4 + 2 * s + buf); };   // P written (softmax -> MMA)
    auto bar_pv = [&](int s, int buf) { return sBar + 8u * (2 * C::NBUF + 8 + 2 * s + buf); };  // P V out of that buffer done
    auto bar_o = [&](int s) { return sBar + 8u * (2 * C::NBUF + 12 + s); };                     // last P V of slot s done
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(gen + C::kBarOff + 8 * (2 * C::NBUF + 14));

    // HALF: an item of more than 128 rows is run as several CTAs of 128 rows each (gridDim.x = Hkv x row tiles, the row
    // tile fastest: the CTAs that stream the same K / V tiles are dispatched next to each other, the second pass hits L2)
    const int32_t n_rt = HALF ? (int32_t)gridDim.x / p.L.n_kv_heads : 1;
    const int32_t kvh = (int32_t)blockIdx.x / n_rt, r0 = ((int32_t)blockIdx.x % n_rt) * 128;
    // (no item is split when the grid has one row per item: no search)
    const int32_t i = (int32_t)gridDim.y == p.n_items
                          ? (int32_t)blockIdx.y
                          : find_item(p.n_items, (int32_t)blockIdx.y, [&](int32_t k) { return p.items[k].split_off; });
    const AttendItem it = p.items[i];
    const int32_t split = (int32_t)blockIdx.y - it.split_off;
    const int32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t R_all = it.q_len * p.G;
    if (HALF && r0 >= R_all) return;                                    // (CTA-uniform, before anything is set up)
    const int32_t R = HALF ? min(128, R_all - r0) : R_all;              // rows of THIS CTA: global rows r0 .. r0 + R - 1
    const bool two = !HALF && R > 128;
    const bool seq = two || HALF;                                       // every consuming slot takes every half-stage, in order
    const int32_t tl0 = split * it.tiles_per_split;
    const int32_t tl1 = min(it.n_tiles, tl0 + it.tiles_per_split);
    const int32_t n_half = (tl1 - tl0 + C::KS - 1) / C::KS;             // half-stages of this segment
    const int32_t n_pair = (n_half + 1) >> 1;
    const int32_t t_first = it.len - it.q_len;                          // reading R15: the last q_len positions
    // ring entry of K / V of half-stage h (see umma_seq_k / umma_seq_v)
    auto entry_k = [&](int32_t h) { return seq ? umma_seq_k(h) : 2 * umma_seq_k(h >> 1) + (h & 1); };
    auto entry_v = [&](int32_t h) { return seq ? umma_seq_v(h, n_half) : 2 * umma_seq_v(h >> 1, n_pair) + (h & 1); };

    // HALF: two CTAs of 256 threads share an SM (128 registers each at launch): the producer / MMA warpgroup keeps 64,
    // the softmax warpgroup (one thread per query row, 64 scores + P in registers) takes 192.  4 x 32 x (64 + 192) = 32768.
    if (warp < 4) {
        if constexpr (HALF) asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
        if (warp == 0) {
            // ================================ producer ================================
            if (lane == 0) {
                for (int b = 0; b < C::NBUF; ++b) { mbar_init(bar_full(b), 1); mbar_init(bar_empty(b), two ? 2 : 1); }
                for (int s = 0; s < C::NQ; ++s) {
                    for (int buf = 0; buf < 2; ++buf) { mbar_init(bar_s(s, buf), 1); mbar_init(bar_p(s, buf), 4); mbar_init(bar_pv(s, buf), 1); }
                    mbar_init(bar_o(s), 1);
                }
                asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            }
            __syncwarp();
            named_arrive(1, C::kThreads);
            const int32_t* trow = p.table + (int64_t)it.sid * p.tbl_width;
            const uint8_t* head_base = p.kv_layer + (int64_t)kvh * p.L.head_bytes;
            const int32_t n_entries = seq ? 2 * n_half : 4 * n_pair;
            // Physical block ids of this segment's tiles, fetched ONCE (lane l holds tiles l, l+32, ...): a
            // table lookup inside the loop is a dependent L2 round trip per ring entry and made the producer,
            // not the tensor pipe or the softmax, set the pace of the whole kernel.
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
            for (int32_t e = 0; e < n_entries; ++e) {
                // invert the order: which (K | V, half-stage) is entry e
                const int32_t es = seq ? e : e >> 1, ns = seq ? n_half : n_pair;
                bool is_v;
                int32_t j;
                if (es == 0) { is_v = false; j = 0; }
                else if (es == 2 * ns - 1) { is_v = true; j = ns - 1; }
                else if (es & 1) { is_v = false; j = (es + 1) >> 1; }
                else { is_v = true; j = (es >> 1) - 1; }
                const int32_t h = seq ? j : 2 * j + (e & 1);
                const int32_t b = e % C::NBUF, k = e / C::NBUF;
                if (k >= 1) mbar_wait(bar_empty(b), (k - 1) & 1);
                if (h >= n_half) {                                        // phantom half-stage of an odd count
                    if (lane == 0) mbar_arrive(bar_full(b));
                    continue;
                }
                const int32_t t0 = tl0 + h * C::KS;
                const int32_t nt = min(C::KS, tl1 - t0);
                if (lane == 0) mbar_expect_tx(bar_full(b), (uint32_t)nt * C::kTileBytes);
                __syncwarp();
                const uint32_t dst = sRing + b * C::kBufBytes;
                const int32_t blk = is_v ? lane : lane / C::NH, hh = lane % C::NH;
                const int32_t phys = phys_of(h * C::KS + min(blk, C::KS - 1));      // (every lane takes part in the shuffle)
                if (is_v) {
                    if (lane < nt)
                        bulk_g2s(dst + lane * C::kTileBytes, head_base + (int64_t)phys * p.L.block_bytes + p.L.tile_bytes,
                                 C::kTileBytes, bar_full(b));
                } else if (lane < nt * C::NH) {
                    bulk_g2s(dst + hh * C::kKHalfBytes + blk * 2048, head_base + (int64_t)phys * p.L.block_bytes + hh * 2048, 2048,
                             bar_full(b));
                }
            }
            return;
        }
        {
            // ================================ MMA issuers ================================
            // Warp 1 issues Q K^T for both slots, warps 2 / 3 issue P V of slot 0 / 1.  A single thread
            // gets one tcgen05.mma out every ~110-130 cycles (measured), so the 32 MMAs of a half-stage
            // are spread over three issuing threads (a fourth warp would put 4 warps on one SM
            // sub-partition and cap everyone at 128 registers).
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
            constexpr uint32_t idesc_qk = umma_idesc(C::KS * kBlockTokens, false);
            constexpr uint32_t idesc_pv = umma_idesc(D, true);
            const uint32_t tSbase = tmem + C::kColS + 128 * slot, tOacc = tmem + C::kColO + D * slot;      // (P V warps)
            if (HALF && warp == 3) return;                    // (one row tile: no second P V issuer; warp 1 frees the TMEM)

            auto wait_full = [&](int32_t e) {
                mbar_wait(bar_full(e % C::NBUF), (e / C::NBUF) & 1);
                tc_fence_after();
            };
            auto release = [&](int32_t e) { if (lane == 0) umma_commit(bar_empty(e % C::NBUF)); };
            // S[buf] = Q K^T over the K half-stage in ring entry e
            const uint32_t elect = lane == 0 ? 1u : 0u;
            auto issue_qk = [&](int32_t qslot, int32_t buf, int32_t e) {
                // descriptors = base + (byte offset >> 4) in the address field (no carry: shared memory < 256 KB)
                const uint64_t dq0 = umma_desc(sQ + (two ? qslot : 0) * C::kQBytes, 16, 1024);
                const uint64_t dk0 = umma_desc(sRing + (e % C::NBUF) * C::kBufBytes, 16, 1024);
                const uint32_t ts = tmem + C::kColS + 128 * qslot + 64 * buf;
    #pragma unroll
                for (int kk = 0; kk < D / 16; ++kk)
                    umma_ss_e(ts, dq0 + (uint64_t)(((kk >> 2) * C::kQHalfBytes + (kk & 3) * 32) >> 4),
                              dk0 + (uint64_t)(((kk >> 2) * C::kKHalfBytes + (kk & 3) * 32) >> 4), idesc_qk, kk > 0 ? 1u : 0u, elect);
                if (lane == 0) umma_commit(bar_s(qslot, buf));
                __syncwarp();
            };
            // O (+)= P V over the V half-stage in ring entry e: per valid block one K=16 MMA for the hi part of P
            // and one for the lo part (per 32-column chunk of the S buffer: hi in columns 0-15, lo in 16-31)
            auto issue_pv = [&](int32_t buf, int32_t e, int32_t nt, bool accumulate) {
                const uint64_t vd0 = umma_desc(sRing + (e % C::NBUF) * C::kBufBytes, 2048, 1024);
                const uint32_t pa0 = tSbase + 64 * buf;
    #pragma unroll
                for (int b = 0; b < C::KS; ++b) {
                    if (b < nt) {                             // (warp-uniform)
                        const uint32_t pa = pa0 + 32 * (b >> 1) + 8 * (b & 1);
                        const uint64_t vd = vd0 + (uint64_t)((b * C::kTileBytes) >> 4);
                        umma_ts_e(tOacc, pa, vd, idesc_pv, (accumulate || b > 0) ? 1u : 0u, elect);
                        umma_ts_e(tOacc, pa + 16, vd, idesc_pv, 1u, elect);
                    }
                }
                if (lane == 0) umma_commit(bar_pv(slot, buf));
                __syncwarp();
            };
            // V rows past the session's length hold stale or poisoned bytes (0 * NaN = NaN): zero them
            auto fix_ragged_v = [&](int32_t e, int32_t t0, int32_t nt) {
                const int32_t last = it.n_tiles - 1, nvalid = it.len & (kBlockTokens - 1);
                if (nvalid == 0 || last < t0 || last >= t0 + nt) return;
                uint8_t* vt = gen + C::NQ * C::kQBytes + (e % C::NBUF) * C::kBufBytes + (last - t0) * C::kTileBytes;
                const int32_t per_row = C::NH * 8;
                for (int32_t idx = lane; idx < (kBlockTokens - nvalid) * per_row; idx += 32) {
                    const int32_t row = nvalid + idx / per_row, rem = idx % per_row;
                    *reinterpret_cast<uint4*>(vt + (rem >> 3) * 2048 + row * 128 + (rem & 7) * 16) = make_uint4(0u, 0u, 0u, 0u);
                }
                fence_async_smem();
                __syncwarp();
            };
            // this slot's half-stages: h(k) = k (two) or 2 k + slot
            const int32_t n_mine = seq ? n_half : (n_half - slot + 1) >> 1;
            auto half_of = [&](int32_t k) { return seq ? k : 2 * k + slot; };
            if (!is_pv) {
                // ---- Q K^T of every half-stage h, for both slots (R > 128) or for slot h & 1: into S buffer
                // k & 1 of the slot (k = the slot's own count), as soon as P V of k - 2 has drained that buffer ----
                for (int32_t h = 0; h < n_half; ++h) {
                    const int32_t e = entry_k(h);
                    wait_full(e);
                    for (int32_t qs = seq ? 0 : (h & 1); qs < (two ? 2 : HALF ? 1 : (h & 1) + 1); ++qs) {
                        const int32_t k = seq ? h : h >> 1, buf = k & 1;
                        if (k >= 2) {
                            mbar_wait(bar_pv(qs, buf), ((k >> 1) - 1) & 1);
                            tc_fence_after();
                        }
                        issue_qk(qs, buf, e);
                        release(e);                          // (one arrival per consuming slot)
                    }
                }
                if (!seq && (n_half & 1)) {                   // phantom half-stage of an odd count: hand the entry back
                    const int32_t ek = entry_k(n_half);
                    wait_full(ek); if (lane == 0) mbar_arrive(bar_empty(ek % C::NBUF));
                }
            } else {
                // ---- P V: half-stage k out of S buffer k & 1, once the softmax has written P there ----
                for (int32_t k = 0; k < n_mine; ++k) {
                    const int32_t h = half_of(k), e = entry_v(h), buf = k & 1;
                    const int32_t t0 = tl0 + h * C::KS, nt = min(C::KS, tl1 - t0);
                    wait_full(e);
                    fix_ragged_v(e, t0, nt);
                    mbar_wait(bar_p(slot, buf), (k >> 1) & 1);
                    tc_fence_after();
                    issue_pv(buf, e, nt, k > 0);
                    release(e);
                    if (k == n_mine - 1 && lane == 0) umma_commit(bar_o(slot));
                }
                if (!seq && slot == 1 && (n_half & 1)) {
                    const int32_t ev = entry_v(n_half);
                    wait_full(ev); if (lane == 0) mbar_arrive(bar_empty(ev % C::NBUF));
                }
            }
            if (warp == 1) {
                // every softmax warp has finished reading TMEM
                named_sync(2, 32 + C::kSoftmaxThreads);
                tc_fence_after();
                asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(C::kTmemCols));
            }
            return;
        }
    }
    if constexpr (HALF) asm volatile("setmaxnreg.inc.sync.aligned.u32 192;");

    // ================================ softmax warps ================================
    const int32_t slot = (warp - 4) >> 2, quarter = warp & 3;       // TMEM lanes 32 (warp % 4) .. + 31
    const int32_t row = quarter * 32 + lane;
    const int32_t tile_row0 = two ? 128 * slot : 0;                   // (HALF: slot is always 0)
    const int32_t rho = r0 + tile_row0 + row;                         // (global row) rho = r * G + g
    const bool valid = tile_row0 + row < R;
    const int32_t rq = rho / p.G, gq = rho - rq * p.G;
    const int32_t t = valid ? t_first + rq : -1;                      // -1: padding row, admits nothing
    const bool warp_active = tile_row0 + quarter * 32 < R;
    const int32_t t_wmin = t_first + (r0 + tile_row0 + quarter * 32) / p.G;
    const int32_t t_wmax = t_first + (r0 + min(R, tile_row0 + quarter * 32 + 32) - 1) / p.G;

    // ---- Q rows -> shared memory, K-major SWIZZLE_128B, one [128][64] region per 64-dim half ----
    {
        const int32_t tid2 = threadIdx.x - 128;
        const int32_t n_rows = two ? 256 : 128;                       // (HALF: 128, one Q region)
        constexpr int CPR = D / 8;                                    // 16-byte chunks per row
        // 16-byte cp.async per chunk: all of a thread's copies are in flight together
        for (int32_t idx = tid2; idx < n_rows * CPR; idx += C::kSoftmaxThreads) {
            const int32_t rr = idx / CPR, c = idx % CPR;
            const uint32_t dst = (rr >> 7) * C::kQBytes + (c >> 3) * C::kQHalfBytes + (rr & 127) * 128 + (((c & 7) ^ (rr & 7)) << 4);
            if (rr < R) {
                const int32_t r2 = (r0 + rr) / p.G, g2 = (r0 + rr) - r2 * p.G;
                const __nv_bfloat16* src = p.q + ((int64_t)(it.q_row_off + r2) * p.Hq + kvh * p.G + g2) * D + c * 8;
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sQ + dst), "l"(src) : "memory");
            } else {
                *reinterpret_cast<uint4*>(gen + dst) = make_uint4(0u, 0u, 0u, 0u);
            }
        }
        asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
        fence_async_smem();
    }
    named_sync(1, C::kThreads);
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t lane_base = (uint32_t)(quarter * 32) << 16;
    const uint32_t tS = tmem + lane_base + C::kColS + 128 * slot;     // two 64-column S buffers; P (bf16 hi | lo) goes over S
    const uint32_t tO = tmem + lane_base + C::kColO + D * slot;

    // One half-stage of one slot, per thread = per query row: 64 scores, read ONCE into registers
    // (two tcgen05.ld of 32 columns), row max, exp2, and P written back over the columns just read.
    float m_run = -INFINITY, m_used = -INFINITY;
    float l0 = 0.f, l1 = 0.f, l2 = 0.f, l3 = 0.f;                     // four partial sums (ILP)
    const int32_t n_mine = seq ? n_half : (n_half - slot + 1) >> 1;
    for (int32_t k = 0; k < n_mine; ++k) {
        const int32_t h = seq ? k : 2 * k + slot, buf = k & 1;
        mbar_wait(bar_s(slot, buf), (k >> 1) & 1);
        tc_fence_after();
        if (warp_active) {
            const uint32_t tSb = tS + 64 * buf;
            uint32_t sa[32], sb[32];
            tmem_ld32(tSb, sa);
            tmem_ld32(tSb + 32, sb);
            const int32_t t0 = tl0 + h * C::KS;
            const int32_t nt = min(C::KS, tl1 - t0);
            // a half-stage needs no mask when every key of it is admitted for every row of this warp
            // (window tiles are consecutive logical blocks; one that holds sink tiles takes the mask)
            const int32_t p_first = tile_block(it, t0) * kBlockTokens;
            const bool full = nt == C::KS && t0 >= it.n_sink_tiles && p_first + C::KS * kBlockTokens - 1 <= t_wmin &&
                              t_wmax - p_first < p.W;
            tmem_wait_ld();
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
            const float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * p.scale_log2;
            m_run = fmaxf(m_run, mx);
            if (k == 0) {
                m_used = m_run;                                       // O is still empty
            } else {
                // lazy rescale: keep the stale reference max while it is within 2^8 of the true one
                const bool need = (m_run - m_used) > 8.f;             // (-inf) - (-inf) = NaN -> false
                if (__any_sync(0xffffffffu, need)) {
                    // S is double buffered, so P V of the previous half-stage may still be running
                    mbar_wait(bar_pv(slot, (k - 1) & 1), ((k - 1) >> 1) & 1);
                    tc_fence_after();
                    const float f = (need && m_used != -INFINITY) ? ex2(m_used - m_run) : 1.f;
                    l0 *= f; l1 *= f; l2 *= f; l3 *= f;
#pragma unroll
                    for (int c = 0; c < D / 32; ++c) {
                        uint32_t o[32];
                        tmem_ld32(tO + 32 * c, o);
                        tmem_wait_ld();
#pragma unroll
                        for (int kk = 0; kk < 32; ++kk) o[kk] = __float_as_uint(__uint_as_float(o[kk]) * f);
                        tmem_st32(tO + 32 * c, o);
                    }
                    if (need) m_used = m_run;
                }
            }
            const float sub = m_used == -INFINITY ? 0.f : m_used;     // nothing admitted yet: every p is 0
            // p = 2^(s * scale - m); P = bf16 hi + bf16 lo (2^-17 weights: the x20 outlier channels of
            // config 4 need more than bf16's 2^-9); hi | lo of chunk c over S columns [32c, +16) | [32c+16, +32)
            const uint64_t scale2 = f2_pack(p.scale_log2, p.scale_log2), nsub2 = f2_pack(-sub, -sub);
            uint64_t lA = f2_pack(l0, l1), lB = f2_pack(l2, l3);
            auto exp_chunk = [&](uint32_t (&cur)[32], int c) {
                uint32_t pk[32];
#pragma unroll
                for (int kk = 0; kk < 16; kk += 2) {
                    float x0, x1, x2, x3;
                    f2_unpack(f2_fma(f2_pack(__uint_as_float(cur[2 * kk]), __uint_as_float(cur[2 * kk + 1])), scale2, nsub2), x0, x1);
                    f2_unpack(f2_fma(f2_pack(__uint_as_float(cur[2 * kk + 2]), __uint_as_float(cur[2 * kk + 3])), scale2, nsub2), x2, x3);
                    const float p0 = ex2(x0), p1 = ex2(x1), p2 = ex2(x2), p3 = ex2(x3);
                    pk[kk] = pack_bf16(p0, p1);
                    pk[kk + 1] = pack_bf16(p2, p3);
                    const uint64_t pa = f2_pack(p0, p1), pb = f2_pack(p2, p3);
                    float d0, d1, d2, d3;
                    f2_unpack(f2_sub(pa, f2_pack(bf16lo(pk[kk]), bf16hi(pk[kk]))), d0, d1);
                    f2_unpack(f2_sub(pb, f2_pack(bf16lo(pk[kk + 1]), bf16hi(pk[kk + 1]))), d2, d3);
                    pk[16 + kk] = pack_bf16(d0, d1);
                    pk[17 + kk] = pack_bf16(d2, d3);
                    lA = f2_add(lA, pa);
                    lB = f2_add(lB, pb);
                }
                tmem_st32(tSb + 32 * c, pk);
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
    float l = (l0 + l1) + (l2 + l3);
    const int32_t n_it = n_mine;

    // ---- epilogue ----
    const int64_t qrow = (int64_t)(it.q_row_off + rq) * p.Hq + kvh * p.G + gq;
    float* ml1 = reinterpret_cast<float*>(gen + C::kMlOff);
    auto store_row = [&](const float (&o)[D], float m, float lsum) {
        if (!valid) return;
        if (it.n_splits == 1) {
            const float inv = lsum > 0.f ? 1.f / lsum : 0.f;
            uint4* dst = reinterpret_cast<uint4*>(p.out + qrow * D);
#pragma unroll
            for (int c = 0; c < D / 8; ++c)
                dst[c] = make_uint4(pack_bf16(o[8 * c] * inv, o[8 * c + 1] * inv), pack_bf16(o[8 * c + 2] * inv, o[8 * c + 3] * inv),
                                    pack_bf16(o[8 * c + 4] * inv, o[8 * c + 5] * inv), pack_bf16(o[8 * c + 6] * inv, o[8 * c + 7] * inv));
        } else {
            const int64_t ws = qrow * p.max_splits + split;
            float4* dst = reinterpret_cast<float4*>(p.ws_acc + ws * D);
#pragma unroll
            for (int c = 0; c < D / 4; ++c) dst[c] = make_float4(o[4 * c], o[4 * c + 1], o[4 * c + 2], o[4 * c + 3]);
            p.ws_ml[ws * 2] = m;
            p.ws_ml[ws * 2 + 1] = lsum;
        }
    };
    auto load_o = [&](float (&o)[D]) {
#pragma unroll
        for (int c = 0; c < D / 32; ++c) tmem_ld32(tO + 32 * c, reinterpret_cast<uint32_t*>(o) + 32 * c);
        tmem_wait_ld();
    };
    if (seq) {
        if (n_it > 0) {
            mbar_wait(bar_o(slot), 0);
            tc_fence_after();
            if (warp_active) {
                float o[D];
                load_o(o);
                store_row(o, m_used, l);
            }
        }
    } else {
        // both slots' MMAs are complete before the Q region is reused for the exchange
        mbar_wait(bar_o(0), 0);
        if (n_half >= 2) mbar_wait(bar_o(1), 0);
        tc_fence_after();
        constexpr int NCH = D / 4;                                     // float4 chunks per row
        float4* ex = reinterpret_cast<float4*>(gen) + row * NCH;
        if (slot == 1) {
            if (n_it > 0 && warp_active) {
                float o[D];
                load_o(o);
#pragma unroll
                for (int c = 0; c < NCH; ++c) ex[(c ^ row) & (NCH - 1)] = make_float4(o[4 * c], o[4 * c + 1], o[4 * c + 2], o[4 * c + 3]);
                ml1[2 * row] = m_used;
                ml1[2 * row + 1] = l;
            }
            __threadfence_block();
            named_arrive(3, 256);
        } else {
            float o[D];
            if (warp_active) load_o(o);
            named_sync(3, 256);
            if (warp_active) {
                if (n_half >= 2) {
                    const float m1 = ml1[2 * row], l1 = ml1[2 * row + 1];
                    const float M = fmaxf(m_used, m1);
                    const float a0 = m_used == -INFINITY ? 0.f : ex2(m_used - M);
                    const float a1 = m1 == -INFINITY ? 0.f : ex2(m1 - M);
#pragma unroll
                    for (int c = 0; c < NCH; ++c) {
                        const float4 b = ex[(c ^ row) & (NCH - 1)];
                        o[4 * c] = a0 * o[4 * c] + a1 * b.x;
                        o[4 * c + 1] = a0 * o[4 * c + 1] + a1 * b.y;
                        o[4 * c + 2] = a0 * o[4 * c + 2] + a1 * b.z;
                        o[4 * c + 3] = a0 * o[4 * c + 3] + a1 * b.w;
                    }
                    l = a0 * l + a1 * l1;
                    m_used = M;
                }
                store_row(o, m_used, l);
            }
        }
    }
    tc_fence_before();
    named_arrive(2, 32 + C::kSoftmaxThreads);
    if (threadIdx.x == 128) stamp_end(p);
}

// ------------------------------------------------------------------------------------------------
constexpr int kUmmaMaxRows = 256;

inline bool attend_umma_supported(int32_t G, int32_t max_q) { return (int64_t)G * max_q <= kUmmaMaxRows; }

inline cudaError_t configure_attend_umma_kernels() {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(attend_umma_kernel<128, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  UmmaCfg<128, false>::kSmemBytes)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(attend_umma_kernel<64, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  UmmaCfg<64, false>::kSmemBytes)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(attend_umma_kernel<128, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  UmmaCfg<128, true>::kSmemBytes)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(attend_umma_kernel<128, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 100)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(attend_umma_kernel<64, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  UmmaCfg<64, true>::kSmemBytes)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(attend_umma_kernel<64, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
}

// chunk-class items (16 < R <= 256): p.items / p.n_items must point at them.  `half`: the half-size variant, two CTAs
// per SM (UmmaCfg<D, true>), `row_tiles` = ceil(largest R / 128) CTAs of 128 rows per (item, head) segment
inline cudaError_t launch_attend_umma(const AttendParams& p, int32_t D, int32_t Hkv, int32_t total_splits, cudaStream_t st,
                                      bool pdl = false, bool half = false, int32_t row_tiles = 1) {
    dim3 grid(Hkv, total_splits);
    if (half) {
        grid.x = Hkv * row_tiles;                        // (row tile fastest)
        if (D == 128) return launch_kernel(attend_umma_kernel<128, true>, grid, UmmaCfg<128, true>::kThreads, UmmaCfg<128, true>::kSmemBytes, st, pdl, p);
        return launch_kernel(attend_umma_kernel<64, true>, grid, UmmaCfg<64, true>::kThreads, UmmaCfg<64, true>::kSmemBytes, st, pdl, p);
    }
    if (D == 128) return launch_kernel(attend_umma_kernel<128, false>, grid, UmmaCfg<128, false>::kThreads, UmmaCfg<128, false>::kSmemBytes, st, pdl, p);
    return launch_kernel(attend_umma_kernel<64, false>, grid, UmmaCfg<64, false>::kThreads, UmmaCfg<64, false>::kSmemBytes, st, pdl, p);
}

}  // namespace metronome
