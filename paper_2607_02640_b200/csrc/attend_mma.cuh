// attend_mma.cuh -- rows a5 (GQA decode) and a7 (chunk prefill): tensor-core tile kernel.
//
// One CTA = one (split-KV segment, KV head).  The R = G x q_len query rows that share this KV head
// (GQA group x chunk rows; "grouped-query attention", "mixed prefill/decode") form
// up to 13 m16 row tiles, one per compute warp; the KV stream is read from HBM ONCE for all of
// them.  A producer warp streams the sink tiles first and then the window tiles
// ("extra leading iterations remapped onto the sink tiles ... accumulating them
// first is exact") into a shared-memory ring with bulk async copies (cp.async.bulk -> UBLKCP, one
// 8 KiB copy per (block, head) because layout.cuh keeps K|V of a block-head contiguous and
// pre-swizzled), completion counted on mbarriers; compute warps release stages on "empty"
// mbarriers.  Per 16-key tile a warp does S = Q K^T (mma.sync m16n8k16 bf16, K fragments by
// ldmatrix), the token-exact union mask on boundary tiles only, an online softmax in the log2
// domain with a warp-uniform skip of the rescale, and O += P V (V fragments by ldmatrix.trans).
//
// Why mma.sync and not tcgen05 here (round 1): decode has R <= 16 rows, one m16 tile at AI = G
// flop/byte, far below what needs UMMA; the chunk tiles (R <= 208) are the candidate for a
// tcgen05 path ("next").  The HBM layout is already UMMA's SWIZZLE_128B K-major.
#pragma once
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

template <int D, int NW>
struct MmaCfg {
    static constexpr int KS = NW == 1 ? 2 : 4;          // key tiles (blocks) per pipeline stage
    static constexpr int NS = NW == 1 ? 4 : 3;          // stages
    static constexpr int kHeadBytes = 2 * kBlockTokens * D * 2;
    static constexpr int kStageBytes = KS * kHeadBytes;
    static constexpr int kSmemBytes = NS * kStageBytes + 2 * NS * 8 + 128;
    static constexpr int kThreads = 32 * (NW + 1);
};

// grid = (total_splits, Hkv); block = 32 * (NW + 1): NW compute warps + 1 producer warp.
template <int D, int NW>
__global__ void __launch_bounds__(MmaCfg<D, NW>::kThreads, 1)
attend_mma_kernel(AttendParams p) {
    using C = MmaCfg<D, NW>;
    constexpr int KSTEPS = D / 16;       // k-steps of Q K^T
    constexpr int NT = D / 8;            // n-tiles of P V
    extern __shared__ __align__(128) uint8_t smem_raw[];
    // 128-byte aligned stage buffers (rows of a tile are 128-byte swizzle atoms)
    const uint32_t smem_base = (smem_u32(smem_raw) + 127u) & ~127u;
    const uint32_t bar_full = smem_base + C::NS * C::kStageBytes;
    const uint32_t bar_empty = bar_full + C::NS * 8;

    const int32_t i = find_item(p.n_items, (int32_t)blockIdx.x, [&](int32_t k) { return p.items[k].split_off; });
    const AttendItem it = p.items[i];
    const int32_t split = blockIdx.x - it.split_off;
    const int32_t kvh = blockIdx.y;
    const int32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t R = it.q_len * p.G;                       // query rows sharing this KV head
    const int32_t nw_active = (R + 15) >> 4;                // compute warps with at least one row
    const int32_t tl0 = split * it.tiles_per_split;
    const int32_t tl1 = min(it.n_tiles, tl0 + it.tiles_per_split);
    const int32_t n_stage = (tl1 - tl0 + C::KS - 1) / C::KS;

    if (threadIdx.x == 0) {
        for (int s = 0; s < C::NS; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, nw_active);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NW) {
        // ------------------------------ producer warp ------------------------------
        const int32_t* trow = p.table + (int64_t)it.sid * p.tbl_width;
        for (int32_t s = 0; s < n_stage; ++s) {
            const int32_t slot = s % C::NS;
            if (s >= C::NS) mbar_wait(bar_empty + 8 * slot, ((s / C::NS) - 1) & 1);
            const int32_t t0 = tl0 + s * C::KS;
            const int32_t nt = min(C::KS, tl1 - t0);
            if (lane == 0) mbar_expect_tx(bar_full + 8 * slot, (uint32_t)nt * C::kHeadBytes);
            __syncwarp();
            if (lane < nt) {
                const int32_t tile = t0 + lane;
                const int32_t blk = tile < it.n_sink_tiles ? tile : it.first_blk + (tile - it.n_sink_tiles);
                const int32_t phys = __ldg(trow + table_slot(blk, p.n_sink, p.ring));
                const uint8_t* src = p.kv_layer + (int64_t)phys * p.L.block_bytes + (int64_t)kvh * p.L.head_bytes;
                bulk_g2s(smem_base + slot * C::kStageBytes + lane * C::kHeadBytes, src, C::kHeadBytes, bar_full + 8 * slot);
            }
        }
        return;
    }
    if (warp >= nw_active) return;

    // -------------------------------- compute warps --------------------------------
    // rows of this warp's m16 tile: rho_a = 16*warp + lane/4, rho_b = rho_a + 8; rho = r*G + g
    const int32_t t_first = it.len - it.q_len;              // position of query row 0 (reading R15)
    const int32_t rho_a = 16 * warp + (lane >> 2), rho_b = rho_a + 8;
    const bool va = rho_a < R, vb = rho_b < R;
    const int32_t ra = rho_a / p.G, rb = rho_b / p.G;
    const int32_t ta = va ? t_first + ra : -1, tb = vb ? t_first + rb : -1;   // -1: admits nothing
    const int64_t qrow_a = (int64_t)(it.q_row_off + ra) * p.Hq + kvh * p.G + (rho_a - ra * p.G);
    const int64_t qrow_b = (int64_t)(it.q_row_off + rb) * p.Hq + kvh * p.G + (rho_b - rb * p.G);
    // positions spanned by the valid rows of this warp (warp-uniform)
    const int32_t r_lo = (16 * warp) / p.G, r_hi = (min(R, 16 * warp + 16) - 1) / p.G;
    const int32_t t_min = t_first + r_lo, t_max = t_first + r_hi;

    uint32_t qa[KSTEPS][4];
    {
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
    }

    float o[NT][4];
#pragma unroll
    for (int n = 0; n < NT; ++n) { o[n][0] = o[n][1] = o[n][2] = o[n][3] = 0.f; }
    // running max per row (log2 domain) and running sum.  The sum is accumulated BY THE TENSOR CORE
    // from the same bf16-rounded P that multiplies V (one extra n8 tile against a ones matrix), so
    // numerator and denominator see identical weights: with one dominant key (outlier channels,
    // config 4) the rounding of P cancels instead of scaling the output.
    float m_a = -INFINITY, m_b = -INFINITY;
    float lsum[4] = {0.f, 0.f, 0.f, 0.f};
    constexpr uint32_t kOnes = 0x3F803F80u;   // bf16 (1, 1)

    // ldmatrix lane roles
    const int32_t mat = lane >> 3, r8 = lane & 7;
    const int32_t k_row = r8 + ((mat >> 1) << 3), k_cs = mat & 1;      // K: matrices (rows 0-7|8-15) x (chunk, chunk+1)
    const int32_t v_row = r8 + ((mat & 1) << 3), v_cs = mat >> 1;      // V: matrices (chunk, chunk+1) x (rows 0-7|8-15)
    const int32_t col0 = (lane & 3) * 2;

    for (int32_t s = 0; s < n_stage; ++s) {
        const int32_t slot = s % C::NS;
        mbar_wait(bar_full + 8 * slot, (s / C::NS) & 1);
        const int32_t tbase = tl0 + s * C::KS;
        const int32_t nt = min(C::KS, tl1 - tbase);
        for (int32_t j = 0; j < nt; ++j) {
            const int32_t tile = tbase + j;
            const int32_t blk = tile < it.n_sink_tiles ? tile : it.first_blk + (tile - it.n_sink_tiles);
            const int32_t p0 = blk * kBlockTokens;
            // no admitted key for any row of this warp: skip (warp-uniform)
            if (p0 > t_max || (p0 >= p.S && t_min - (p0 + kBlockTokens - 1) >= p.W)) continue;
            const uint32_t kt = smem_base + slot * C::kStageBytes + j * C::kHeadBytes;
            const uint32_t vt = kt + kBlockTokens * D * 2;

            // ---- S = Q K^T over this 16-key tile: two n8 tiles ----
            float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int kk = 0; kk < KSTEPS; ++kk) {
                uint32_t b0, b1, b2, b3;
                ldsm_x4(kt + tile_chunk_offset(k_row, 2 * kk + k_cs), b0, b1, b2, b3);
                mma_bf16(s0, qa[kk], b0, b1);
                mma_bf16(s1, qa[kk], b2, b3);
            }
            // ---- mask (boundary tiles only) ----
            const bool full = (p0 + kBlockTokens - 1 <= t_min) &&
                              (p0 + kBlockTokens - 1 < p.S || t_max - p0 < p.W);
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
            const bool grow = (mn_a != m_a) || (mn_b != m_b);
            if (__any_sync(0xffffffffu, grow)) {
                const float ca = mn_a == -INFINITY ? 1.f : ex2(m_a - mn_a);
                const float cb = mn_b == -INFINITY ? 1.f : ex2(m_b - mn_b);
                lsum[0] *= ca; lsum[1] *= ca; lsum[2] *= cb; lsum[3] *= cb;
#pragma unroll
                for (int n = 0; n < NT; ++n) { o[n][0] *= ca; o[n][1] *= ca; o[n][2] *= cb; o[n][3] *= cb; }
                m_a = mn_a; m_b = mn_b;
            }
            // a row with nothing admitted so far keeps m = -inf: use 0 as the subtrahend (p = 0)
            const float sub_a = m_a == -INFINITY ? 0.f : m_a, sub_b = m_b == -INFINITY ? 0.f : m_b;
            const float p00 = ex2(fmaf(s0[0], p.scale_log2, -sub_a)), p01 = ex2(fmaf(s0[1], p.scale_log2, -sub_a));
            const float p02 = ex2(fmaf(s0[2], p.scale_log2, -sub_b)), p03 = ex2(fmaf(s0[3], p.scale_log2, -sub_b));
            const float p10 = ex2(fmaf(s1[0], p.scale_log2, -sub_a)), p11 = ex2(fmaf(s1[1], p.scale_log2, -sub_a));
            const float p12 = ex2(fmaf(s1[2], p.scale_log2, -sub_b)), p13 = ex2(fmaf(s1[3], p.scale_log2, -sub_b));
            uint32_t pa[4];
            pa[0] = pack_bf16(p00, p01);   // row a, keys col0..col0+1
            pa[1] = pack_bf16(p02, p03);   // row b
            pa[2] = pack_bf16(p10, p11);   // row a, keys 8+col0..
            pa[3] = pack_bf16(p12, p13);   // row b
            mma_bf16(lsum, pa, kOnes, kOnes);
            // ---- O += P V ; rows of V past the session's length hold stale / poisoned bytes ----
            const int32_t nvalid = it.len - p0;           // < 16 only in the session's last block
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
                mma_bf16(o[n], pa, b0, b1);
                mma_bf16(o[n + 1], pa, b2, b3);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * slot);
    }

    // ---- epilogue ----
    const float l_a = lsum[0], l_b = lsum[2];     // every column of the ones tile holds the row sum
    if (it.n_splits == 1) {
        const float ia = l_a > 0.f ? 1.f / l_a : 0.f, ib = l_b > 0.f ? 1.f / l_b : 0.f;
        uint32_t* oa = reinterpret_cast<uint32_t*>(p.out + qrow_a * D);
        uint32_t* ob = reinterpret_cast<uint32_t*>(p.out + qrow_b * D);
#pragma unroll
        for (int n = 0; n < NT; ++n) {
            if (va) oa[n * 4 + (lane & 3)] = pack_bf16(o[n][0] * ia, o[n][1] * ia);
            if (vb) ob[n * 4 + (lane & 3)] = pack_bf16(o[n][2] * ib, o[n][3] * ib);
        }
    } else {
        const int64_t slot_a = qrow_a * p.max_splits + split, slot_b = qrow_b * p.max_splits + split;
        float2* wa = reinterpret_cast<float2*>(p.ws_acc + slot_a * D);
        float2* wb = reinterpret_cast<float2*>(p.ws_acc + slot_b * D);
#pragma unroll
        for (int n = 0; n < NT; ++n) {
            if (va) wa[n * 4 + (lane & 3)] = make_float2(o[n][0], o[n][1]);
            if (vb) wb[n * 4 + (lane & 3)] = make_float2(o[n][2], o[n][3]);
        }
        if ((lane & 3) == 0) {
            if (va) { p.ws_ml[slot_a * 2] = m_a; p.ws_ml[slot_a * 2 + 1] = l_a; }
            if (vb) { p.ws_ml[slot_b * 2] = m_b; p.ws_ml[slot_b * 2 + 1] = l_b; }
        }
    }
}

constexpr int kMmaMaxRows = 13 * 16;

inline bool attend_mma_supported(int32_t G, int32_t max_q) { return (int64_t)G * max_q <= kMmaMaxRows; }

template <int D, int NW>
inline cudaError_t configure_one() {
    return cudaFuncSetAttribute(attend_mma_kernel<D, NW>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                MmaCfg<D, NW>::kSmemBytes);
}

inline cudaError_t configure_attend_mma_kernels() {
    cudaError_t e;
    if ((e = configure_one<128, 1>()) != cudaSuccess) return e;
    if ((e = configure_one<128, 4>()) != cudaSuccess) return e;
    if ((e = configure_one<128, 8>()) != cudaSuccess) return e;
    if ((e = configure_one<128, 13>()) != cudaSuccess) return e;
    if ((e = configure_one<64, 1>()) != cudaSuccess) return e;
    if ((e = configure_one<64, 4>()) != cudaSuccess) return e;
    if ((e = configure_one<64, 8>()) != cudaSuccess) return e;
    if ((e = configure_one<64, 13>()) != cudaSuccess) return e;
    return cudaSuccess;
}

template <int D>
inline int launch_attend_mma_d(const AttendParams& p, int32_t Hkv, int32_t total_splits, int32_t max_rows,
                               cudaStream_t st) {
    dim3 grid(total_splits, Hkv);
    if (max_rows <= 16) attend_mma_kernel<D, 1><<<grid, MmaCfg<D, 1>::kThreads, MmaCfg<D, 1>::kSmemBytes, st>>>(p);
    else if (max_rows <= 64) attend_mma_kernel<D, 4><<<grid, MmaCfg<D, 4>::kThreads, MmaCfg<D, 4>::kSmemBytes, st>>>(p);
    else if (max_rows <= 128) attend_mma_kernel<D, 8><<<grid, MmaCfg<D, 8>::kThreads, MmaCfg<D, 8>::kSmemBytes, st>>>(p);
    else attend_mma_kernel<D, 13><<<grid, MmaCfg<D, 13>::kThreads, MmaCfg<D, 13>::kSmemBytes, st>>>(p);
    return 0;
}

// returns 0 when a kernel was launched
inline int launch_attend_mma(const AttendParams& p, int32_t D, int32_t Hkv, int32_t total_splits, int32_t max_q,
                             cudaStream_t st) {
    const int32_t max_rows = p.G * max_q;
    if (max_rows > kMmaMaxRows) return 1;
    return D == 128 ? launch_attend_mma_d<128>(p, Hkv, total_splits, max_rows, st)
                    : launch_attend_mma_d<64>(p, Hkv, total_splits, max_rows, st);
}

}  // namespace metronome
