// step_gqa.cuh -- ONE launch for a whole decode sub-step of a grouped-query model: rows a2 a3 a4
// (evict, allocate, KV write) and a5 a6 (attention partials, merge) of SURVEY.md sec. 8(a), behind
// metronome_append_attend ("prefill the new chunk, then decode up to tau output tokens,
// attending over the session's accumulated context ... for all due sessions each tick").
//
// Why one launch.  With two (append kernel, then attention kernel) the attention of step e waits for
// the whole append kernel of step e: a latency chain of ~11 us (host metadata -> block table -> free
// stack -> table -> scatter) in front of ~80 us of streaming.  But the attention of step e needs NOTHING
// the append of step e produces through memory:
//   * the rows appended in this step are in the caller's k_new / v_new: the warp that reaches the tile
//     holding them patches them into the tile in SHARED memory (and is also the one that writes them to
//     their paged slot -- the K/V scatter, row a4, costs no extra read);
//   * a block ALLOCATED in this step holds nothing but rows of this step: it is not read at all, so the
//     table entry the bookkeeping writes is only needed by that same scatter (it waits for the
//     bookkeeping CTA's epoch flag; that CTA is the first of the grid and waits for nobody);
//   * blocks FREED in this step lie entirely behind the window of every query of this step.
// So CTA 0 does the bookkeeping (bookkeeping.cuh's two phases) while all the others stream.
//
// How the stream is cut.  attend_gqa_kernel (attend_mma.cuh) gives each CTA one range of the flattened
// (item, KV head, tile) list and merges its four warps through shared memory at every (item, head)
// boundary: measured on B200 (config 3) every boundary a CTA crosses costs it ~3 us (ring drained, three
// CTA barriers, ticket round trip, restart through item -> table -> HBM), CTAs end 52..82 us apart
// according to how many boundaries they hold, and the kernel ends with the slowest.  Here the WARP is
// the worker: the list is cut into one contiguous range per warp (n_SM x 2 x 4 of them), a warp streams
// its range through a private 3-stage ring of bulk async copies and never meets a CTA barrier; at an
// (item, head) boundary it stores its piece (final output, or an unnormalised partial + ticket, last
// arriver merges: row a6) while its ring is already filling with the next pair's tiles -- the issue
// cursor runs ahead of the consume cursor across boundaries.  The work list is in KERNEL PARAMETER
// space (16 bytes per item, constant bank): no upload, no dependent loads to find or advance an item.
#pragma once
#include "attend_mma.cuh"
#include "kv_append.cuh"

namespace metronome {

constexpr int kStepMaxItems = 1024;          // items whose work list fits the kernel parameters
constexpr int kStepMaxSms = 256;

struct StepItem {
    int32_t sid_q;            // sid | q_len << 16      (sid <= 65533, q_len * G <= 16)
    int32_t len;              // session length AFTER this step's append
    int32_t q_row_off;        // row of the item's first query in q / out == its first new row in k_new / v_new
    int32_t tile_off;         // exclusive prefix sum of n_tiles over the items of the launch
};

struct StepParams {
    AttendParams p;           // (p.items unused: the list is below)
    AppendParams a;           // a.items: pinned host memory, read by the bookkeeping CTA only
    GqaPlan plan;             // two lists of ranges over the flattened (item, head, tile) list: [0, n_static) of q1 tiles
                              // for warps on fast SMs, [n_static, n_total) of q2 <= q1 tiles for warps on slow SMs
    int32_t n_workers;        // warps that take ranges (4 per CTA but the first)
    int32_t n_items;
    int32_t* claim_ctr;       // [0] / [1] next range of either list, [2] warps that have left (all zero between launches)
    uint8_t sm_class[kStepMaxSms];   // 0 fast, 1 slow: measured per SM when the pool was created (step_calibrate_kernel)
    StepItem items[kStepMaxItems];
};
static_assert(sizeof(StepParams) <= 32000, "kernel parameters are limited to 32764 bytes");

// What plan_attend() keeps in an AttendItem, recomputed from the 16 bytes above (same formulas:
// metronome.cu plan_attend; the one-call GPU tests compare the results).
struct StepGeo {
    int32_t sid, len, q_len, q_row_off, n_sink_tiles, first_blk, n_tiles, tile_off;
    int32_t len0;             // length before this step's append: rows [len0, len) are in k_new / v_new
    int32_t alloc_lo;         // first logical block allocated in this step = ceil(len0 / 16)
};
__host__ __device__ __forceinline__ StepGeo step_geo(const StepItem& s, int32_t W, int32_t n_sink) {
    StepGeo g;
    g.sid = s.sid_q & 0xFFFF;
    g.q_len = s.sid_q >> 16;
    g.len = s.len;
    g.q_row_off = s.q_row_off;
    g.tile_off = s.tile_off;
    const int32_t n_blk = (s.len + kBlockTokens - 1) / kBlockTokens;
    g.len0 = s.len - g.q_len;
    const int32_t wfirst = g.len0 - W + 1 > 0 ? g.len0 - W + 1 : 0;       // oldest window key of the oldest query
    g.first_blk = wfirst / kBlockTokens > n_sink ? wfirst / kBlockTokens : n_sink;
    g.n_sink_tiles = n_blk < n_sink ? n_blk : n_sink;
    g.n_tiles = g.n_sink_tiles + (n_blk > g.first_blk ? n_blk - g.first_blk : 0);
    g.alloc_lo = (g.len0 + kBlockTokens - 1) / kBlockTokens;
    return g;
}

// ------------------------------------------------------------------------------------------------
// One 16-key tile against the R <= 8 NQ query rows of a GQA group, TRANSPOSED: the keys are the M = 16
// side of mma.sync m16n8k16 and the query rows the N = 8 side,
//     S^T = K Q^T   (A = K tile [key][dim] by ldmatrix, B = Q^T fragments kept in registers)
//     O^T += V^T P^T (A = V^T by ldmatrix.trans, B = P^T: the S^T accumulators, packed to bf16 and
//                     transposed across the warp by movmatrix)
// so a group of G <= 8 rows costs ONE n8 tile instead of an m16 tile that is at least half padding:
// 8 + 8 (+ 1 for the row sums) tensor instructions per tile and 48 state registers instead of 16 + 32 (+ 2)
// and 96.  Measured on B200 with the m16-rows form (WarpTile): a warp spent ~1.2 us of issue + legacy
// tensor-pipe time per 8 KB tile, 2 warps per SM sub-partition -- the decode step was bound by that, not
// by HBM.  Row statistics (max, sum) live with the lane's two COLUMNS (rows 8 nq + 2 (lane & 3) + {0, 1}),
// replicated over the eight lanes that share them; P gets the same bf16 hi + lo split as WarpTile.
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
    uint32_t d;
    asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
    return d;
}

template <int D, int NQ>
struct WarpTileT {
    static constexpr int KSTEPS = D / 16;
    static constexpr int MT = D / 16;            // m16 tiles of O^T (16 output dims each)
    uint32_t qb[NQ][KSTEPS][2];
    float o[NQ][MT][4];                          // [0],[1]: dim 16 mt + lane/4, rows 2j, 2j+1; [2],[3]: dim + 8
    float m[NQ][2];                              // running max of this lane's two rows, log2 domain
    float lsum[NQ][4];                           // [0],[1]: their running sums (accumulated by the tensor core)
    int32_t t[NQ][2];                            // their absolute positions (-1: padding row, admits nothing)
    int32_t t_min, t_max;                        // positions spanned by the valid rows (warp-uniform)

    template <typename Item>
    __device__ __forceinline__ void init(const AttendParams& p, const Item& it, int32_t kvh, int32_t lane) {
        const int32_t R = it.q_len * p.G;
        const int32_t t_first = it.len - it.q_len;            // reading R15: the last q_len positions
        const int32_t c = lane & 3;
#pragma unroll
        for (int nq = 0; nq < NQ; ++nq) {
            const int32_t rho_b = 8 * nq + (lane >> 2);       // the row whose Q this lane holds as a B fragment
            const bool vb = rho_b < R;
            const int32_t rb = rho_b / p.G;
            const int64_t qrow = (int64_t)(it.q_row_off + rb) * p.Hq + kvh * p.G + (rho_b - rb * p.G);
            const uint32_t* pq = reinterpret_cast<const uint32_t*>(p.q + qrow * D);
#pragma unroll
            for (int kk = 0; kk < KSTEPS; ++kk) {
                qb[nq][kk][0] = vb ? __ldg(pq + kk * 8 + c) : 0u;
                qb[nq][kk][1] = vb ? __ldg(pq + kk * 8 + 4 + c) : 0u;
            }
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int32_t rho = 8 * nq + 2 * c + e;
                t[nq][e] = rho < R ? t_first + rho / p.G : -1;
                m[nq][e] = -INFINITY;
            }
            lsum[nq][0] = lsum[nq][1] = lsum[nq][2] = lsum[nq][3] = 0.f;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) o[nq][mt][0] = o[nq][mt][1] = o[nq][mt][2] = o[nq][mt][3] = 0.f;
        }
        t_min = t_first;
        t_max = t_first + (min(R, 8 * NQ) - 1) / p.G;
    }

    // true when no key of the 16-token tile at position p0 is admitted for any row (warp-uniform)
    __device__ __forceinline__ bool skips(const AttendParams& p, int32_t p0) const {
        return p0 > t_max || (p0 >= p.S && t_min - (p0 + kBlockTokens - 1) >= p.W);
    }

    template <int kLoInv>
    __device__ __forceinline__ void step(const AttendParams& p, int32_t len, uint32_t kt, uint32_t vt, int32_t p0, int32_t lane) {
        const int32_t mat = lane >> 3, r8 = lane & 7;
        const int32_t k_row = r8 + ((mat >> 1) << 3), k_cs = mat & 1;   // K: (keys 0-7 | 8-15) x (chunk, chunk+1)
        const int32_t v_row = r8 + ((mat & 1) << 3), v_cs = mat >> 1;   // V: (chunk, chunk+1) x (keys 0-7 | 8-15)
        // All fragment loads of the tile go out FIRST (K: one ldmatrix per 16 dims; V: one ldmatrix.trans per 16 output
        // dims): in program order "load, multiply, load, multiply" every tensor instruction waited for its own load
        // and a warp needed ~2300 cycles per tile (measured), with 2-3 warps per SM sub-partition that, not HBM, paced
        // the kernel.
        uint32_t kf[KSTEPS][4], vf[MT][4];
#pragma unroll
        for (int kk = 0; kk < KSTEPS; ++kk) ldsm_x4(kt + tile_chunk_offset(k_row, 2 * kk + k_cs), kf[kk][0], kf[kk][1], kf[kk][2], kf[kk][3]);
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) ldsm_x4_t(vt + tile_chunk_offset(v_row, 2 * mt + v_cs), vf[mt][0], vf[mt][1], vf[mt][2], vf[mt][3]);
        // ---- S^T = K Q^T: two independent accumulation chains (even / odd k-steps) ----
        float s[NQ][4], s2[NQ][4];
#pragma unroll
        for (int nq = 0; nq < NQ; ++nq) { s[nq][0] = s[nq][1] = s[nq][2] = s[nq][3] = 0.f; s2[nq][0] = s2[nq][1] = s2[nq][2] = s2[nq][3] = 0.f; }
#pragma unroll
        for (int kk = 0; kk < KSTEPS; ++kk) {
            const uint32_t a[4] = {kf[kk][0], kf[kk][2], kf[kk][1], kf[kk][3]};   // keys 0-7 | 8-15 (rows) x dims 0-7 | 8-15 of the k-step
#pragma unroll
            for (int nq = 0; nq < NQ; ++nq) mma_bf16((kk & 1) ? s2[nq] : s[nq], a, qb[nq][kk][0], qb[nq][kk][1]);
        }
#pragma unroll
        for (int nq = 0; nq < NQ; ++nq) { s[nq][0] += s2[nq][0]; s[nq][1] += s2[nq][1]; s[nq][2] += s2[nq][2]; s[nq][3] += s2[nq][3]; }
        // ---- union mask, boundary tiles only: [0],[1] key p0 + lane/4, [2],[3] key + 8 ----
        const bool full = (p0 + kBlockTokens - 1 <= t_min) && (p0 + kBlockTokens - 1 < p.S || t_max - p0 < p.W);
        if (!full) {
            const int32_t ja = p0 + (lane >> 2), jb = ja + 8;
#pragma unroll
            for (int nq = 0; nq < NQ; ++nq)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    s[nq][e] = admit(ja, t[nq][e], p.S, p.W) ? s[nq][e] : -INFINITY;
                    s[nq][2 + e] = admit(jb, t[nq][e], p.S, p.W) ? s[nq][2 + e] : -INFINITY;
                }
        }
        // ---- online softmax (log2 domain): the 16 keys of a row sit in the 8 lanes with the same lane & 3 ----
        float mn[NQ][2];
        bool moved = false;
#pragma unroll
        for (int nq = 0; nq < NQ; ++nq)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                float mx = fmaxf(s[nq][e], s[nq][2 + e]);
                mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 4));
                mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 8));
                mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 16));
                mn[nq][e] = fmaxf(m[nq][e], mx * p.scale_log2);
                moved |= mn[nq][e] != m[nq][e];
            }
        if (__any_sync(0xffffffffu, moved)) {
#pragma unroll
            for (int nq = 0; nq < NQ; ++nq) {
                const float c0 = mn[nq][0] == -INFINITY ? 1.f : ex2(m[nq][0] - mn[nq][0]);
                const float c1 = mn[nq][1] == -INFINITY ? 1.f : ex2(m[nq][1] - mn[nq][1]);
                lsum[nq][0] *= c0; lsum[nq][1] *= c1; lsum[nq][2] *= c0; lsum[nq][3] *= c1;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) { o[nq][mt][0] *= c0; o[nq][mt][1] *= c1; o[nq][mt][2] *= c0; o[nq][mt][3] *= c1; }
                m[nq][0] = mn[nq][0]; m[nq][1] = mn[nq][1];
            }
        }
        uint32_t bh[NQ][2], bl[NQ][2];
        bool want_lo = false;
#pragma unroll
        for (int nq = 0; nq < NQ; ++nq) {
            // a row with nothing admitted so far keeps m = -inf: subtract 0 instead (its p are all 0)
            const float sub0 = m[nq][0] == -INFINITY ? 0.f : m[nq][0], sub1 = m[nq][1] == -INFINITY ? 0.f : m[nq][1];
            const float p0a = ex2(fmaf(s[nq][0], p.scale_log2, -sub0)), p1a = ex2(fmaf(s[nq][1], p.scale_log2, -sub1));
            const float p0b = ex2(fmaf(s[nq][2], p.scale_log2, -sub0)), p1b = ex2(fmaf(s[nq][3], p.scale_log2, -sub1));
            const uint32_t ha = pack_bf16(p0a, p1a), hb = pack_bf16(p0b, p1b);      // keys 0-7 | 8-15, rows (2j, 2j+1)
            const uint32_t la = pack_bf16(p0a - bf16lo(ha), p1a - bf16hi(ha)), lb = pack_bf16(p0b - bf16lo(hb), p1b - bf16hi(hb));
            // lo part only where a key carries more than 1/kLoInv of the running sum (warp-uniform)
            want_lo |= (fmaxf(p0a, p0b) * (float)kLoInv > lsum[nq][0]) || (fmaxf(p1a, p1b) * (float)kLoInv > lsum[nq][1]);
            bh[nq][0] = movmatrix_trans(ha); bh[nq][1] = movmatrix_trans(hb);       // P^T as a (k16 keys x n8 rows) B operand
            bl[nq][0] = movmatrix_trans(la); bl[nq][1] = movmatrix_trans(lb);
        }
        const bool need_lo = __any_sync(0xffffffffu, want_lo);
        // row sums from the SAME rounded P that multiplies V: A = ones, every M row gets the column sums
        constexpr uint32_t kOnes = 0x3F803F80u;              // bf16 (1, 1)
        const uint32_t ones[4] = {kOnes, kOnes, kOnes, kOnes};
#pragma unroll
        for (int nq = 0; nq < NQ; ++nq) {
            mma_bf16(lsum[nq], ones, bh[nq][0], bh[nq][1]);
            if (need_lo) mma_bf16(lsum[nq], ones, bl[nq][0], bl[nq][1]);
        }
        // ---- O^T += V^T P^T; V rows past the session's length hold stale / poisoned bytes (0 * NaN) ----
        const int32_t nvalid = len - p0;                     // < 16 only in the session's last block
        const int32_t col0 = (lane & 3) * 2;
        uint32_t mk0 = 0xFFFFFFFFu, mk1 = 0xFFFFFFFFu;
        if (nvalid < kBlockTokens) {
            mk0 = (col0 < nvalid ? 0x0000FFFFu : 0u) | (col0 + 1 < nvalid ? 0xFFFF0000u : 0u);
            mk1 = (col0 + 8 < nvalid ? 0x0000FFFFu : 0u) | (col0 + 9 < nvalid ? 0xFFFF0000u : 0u);
        }
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            uint32_t b0 = vf[mt][0], b1 = vf[mt][1], b2 = vf[mt][2], b3 = vf[mt][3];
            if (nvalid < kBlockTokens) { b0 &= mk0; b1 &= mk1; b2 &= mk0; b3 &= mk1; }
            const uint32_t a[4] = {b0, b2, b1, b3};           // dims 0-7 | 8-15 (rows) x keys 0-7 | 8-15 of the tile
#pragma unroll
            for (int nq = 0; nq < NQ; ++nq) {
                mma_bf16(o[nq][mt], a, bh[nq][0], bh[nq][1]);
                if (need_lo) mma_bf16(o[nq][mt], a, bl[nq][0], bl[nq][1]);
            }
        }
    }

    // row of q / out of query row rho of the pair, or -1
    template <typename Item>
    __device__ __forceinline__ int64_t qrow_of(const AttendParams& p, const Item& it, int32_t kvh, int32_t rho) const {
        if (rho >= it.q_len * p.G) return -1;
        const int32_t r = rho / p.G;
        return (int64_t)(it.q_row_off + r) * p.Hq + kvh * p.G + (rho - r * p.G);
    }
    // final bf16 output (the piece covered every tile of this (item, head))
    template <typename Item>
    __device__ __forceinline__ void store_final(const AttendParams& p, const Item& it, int32_t kvh, int32_t lane) const {
#pragma unroll
        for (int nq = 0; nq < NQ; ++nq)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int64_t qrow = qrow_of(p, it, kvh, 8 * nq + 2 * (lane & 3) + e);
                if (qrow < 0) continue;
                const float inv = lsum[nq][e] > 0.f ? 1.f / lsum[nq][e] : 0.f;
                __nv_bfloat16* dst = p.out + qrow * D + (lane >> 2);
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    dst[16 * mt] = __float2bfloat16_rn(o[nq][mt][e] * inv);
                    dst[16 * mt + 8] = __float2bfloat16_rn(o[nq][mt][2 + e] * inv);
                }
            }
    }
    // unnormalised partial (acc, m, l) of one split-KV piece
    template <typename Item>
    __device__ __forceinline__ void store_partial(const AttendParams& p, const Item& it, int32_t kvh, int32_t piece, int32_t lane) const {
#pragma unroll
        for (int nq = 0; nq < NQ; ++nq)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int64_t qrow = qrow_of(p, it, kvh, 8 * nq + 2 * (lane & 3) + e);
                if (qrow < 0) continue;
                const int64_t slot = qrow * p.max_splits + piece;
                float* dst = p.ws_acc + slot * D + (lane >> 2);
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    dst[16 * mt] = o[nq][mt][e];
                    dst[16 * mt + 8] = o[nq][mt][2 + e];
                }
                if ((lane >> 2) == 0) { p.ws_ml[slot * 2] = m[nq][e]; p.ws_ml[slot * 2 + 1] = lsum[nq][e]; }
            }
    }
};

// Row a6 for one (item, head) pair, by ONE warp (the last piece to arrive): log-sum-exp combine of its `ns`
// partials.  Eight rows at a time, four lanes per row (lane j of a row takes the 16-byte chunks j, j+4, ...), and
// the pieces FOUR at a time: all loads of a group (max / sum pairs and accumulators) are issued together, so a
// merge of up to four pieces is ONE L2 round trip (they cost ~1 us each while the other warps stream).
template <int D>
__device__ __forceinline__ void step_merge_pieces(const AttendParams& p, int32_t R, int32_t q_row_off, int32_t kvh, int32_t ns,
                                               int32_t lane) {
    constexpr int NCH = D / 16;                       // float4 chunks per lane
    constexpr int GP = 4;                             // pieces per group
    for (int32_t rb = 0; rb < R; rb += 8) {
        const int32_t rho = rb + (lane >> 2), j = lane & 3;
        if (rho >= R) continue;
        const int32_t r = rho / p.G;
        const int64_t qrow = (int64_t)(q_row_off + r) * p.Hq + kvh * p.G + (rho - r * p.G);
        const int64_t base = qrow * p.max_splits;
        float M = -INFINITY, l = 0.f;
        float4 acc[NCH];
#pragma unroll
        for (int k = 0; k < NCH; ++k) acc[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int32_t s0 = 0; s0 < ns; s0 += GP) {
            float2 ml[GP];
            float4 v4[GP][NCH];
#pragma unroll
            for (int g = 0; g < GP; ++g) {
                const int32_t s2 = min(s0 + g, ns - 1);           // (a repeated piece is dropped below)
                ml[g] = __ldcg(reinterpret_cast<const float2*>(p.ws_ml + (base + s2) * 2));
                const float4* src = reinterpret_cast<const float4*>(p.ws_acc + (base + s2) * D) + j;
#pragma unroll
                for (int k = 0; k < NCH; ++k) v4[g][k] = __ldcg(src + 4 * k);
            }
            float Mn = M;
#pragma unroll
            for (int g = 0; g < GP; ++g)
                if (s0 + g < ns) Mn = fmaxf(Mn, ml[g].x);
            if (Mn == -INFINITY) continue;                        // nothing admitted so far for this row
            const float f = M == -INFINITY ? 0.f : ex2(M - Mn);   // rescale what earlier groups gave
            l *= f;
#pragma unroll
            for (int k = 0; k < NCH; ++k) { acc[k].x *= f; acc[k].y *= f; acc[k].z *= f; acc[k].w *= f; }
            M = Mn;
#pragma unroll
            for (int g = 0; g < GP; ++g) {
                if (s0 + g >= ns || ml[g].x == -INFINITY) continue;   // (a piece that admitted no key for this row)
                const float wgt = ex2(ml[g].x - M);
                l += wgt * ml[g].y;
#pragma unroll
                for (int k = 0; k < NCH; ++k) {
                    acc[k].x += wgt * v4[g][k].x; acc[k].y += wgt * v4[g][k].y;
                    acc[k].z += wgt * v4[g][k].z; acc[k].w += wgt * v4[g][k].w;
                }
            }
        }
        const float inv = l > 0.f ? 1.f / l : 0.f;
        uint2* dst = reinterpret_cast<uint2*>(p.out + qrow * D) + j;
#pragma unroll
        for (int k = 0; k < NCH; ++k)
            dst[4 * k] = make_uint2(pack_bf16(acc[k].x * inv, acc[k].y * inv), pack_bf16(acc[k].z * inv, acc[k].w * inv));
    }
}

// Publishes the partials of `n_pend` cut pairs (records {R | kvh << 8 | pieces << 16, q_row_off, item}, written by
// lane 0 to shared memory) and combines the pairs this warp arrived LAST at ("merged exactly once";
// the ticket counters reset themselves).  Lane l takes the ticket of record l: one round trip for all.
template <int D>
__device__ __forceinline__ void step_flush_pend(const AttendParams& p, const int4* pend, int32_t n_pend, int32_t Hkv, int32_t lane) {
    __threadfence();
    __syncwarp();
    int32_t last = 0;
    if (lane < n_pend) {
        const int4 mine = pend[lane];
        int32_t* ticket = p.tickets + (int64_t)mine.z * Hkv + ((mine.x >> 8) & 0xFF);
        last = atomicAdd(ticket, 1) == (mine.x >> 16) - 1;
        if (last) *ticket = 0;
    }
    uint32_t todo = __ballot_sync(0xffffffffu, last);
    if (todo) __threadfence();
    while (todo) {
        const int32_t k = __ffs(todo) - 1;
        todo &= todo - 1;
        const int4 rec = pend[k];
        step_merge_pieces<D>(p, rec.x & 0xFF, rec.y, (rec.x >> 8) & 0xFF, rec.x >> 16, lane);
    }
    __syncwarp();
}

// Two CTAs of four warps per SM, every warp with a private THREE-stage ring of 8 KB tiles (96 KB per CTA): the same
// 192 KB per SM in flight as attend_gqa_kernel's 3 x 4 x 2, but with up to 255 registers per thread -- the tile loop
// keeps Q fragments, 64 accumulators and the work cursor in registers without a spill.
template <int D, int NQ>
struct StepCfg {
    static constexpr int NWARP = 4;
    static constexpr int NS = 3;
    static constexpr int kCtasPerSm = 2;
    static constexpr int kHeadBytes = 2 * kBlockTokens * D * 2;
    static constexpr int kWarpBytes = NS * kHeadBytes;
    static constexpr int kSmemBytes = NWARP * kWarpBytes + NWARP * NS * 8 + 128;
    static constexpr int kThreads = 32 * NWARP;
    static_assert(kAppendSmemItems * sizeof(AppendItem) <= NWARP * kWarpBytes || D < 128, "the bookkeeping CTA stages its items in the rings");
};

// grid = 1 + ceil(n_workers / 4), block = 128.  CTA 0: bookkeeping.  Warp w of the others: tiles
// [w q1, (w+1) q1) of the flattened list.
template <int D, int NQ>
__global__ void __launch_bounds__(StepCfg<D, NQ>::kThreads, StepCfg<D, NQ>::kCtasPerSm)
step_gqa_kernel(const __grid_constant__ StepParams sp) {
    using C = StepCfg<D, NQ>;
    const AttendParams& p = sp.p;
    const AppendParams& a = sp.a;
    if (p.pdl_early) pdl_launch_dependents();
    extern __shared__ __align__(128) uint8_t smem_raw[];
    if (blockIdx.x == 0) {
        // ---- rows a2 + a3: the bookkeeping CTA (its AppendItems come over the bus BEFORE the wait) ----
        const bool staged = a.do_bookkeeping && (size_t)a.n_items * sizeof(AppendItem) <= (size_t)C::NWARP * C::kWarpBytes;
        if (staged) {
            const uint4* src = reinterpret_cast<const uint4*>(a.items);
            uint4* dst = reinterpret_cast<uint4*>(smem_raw);
            const int32_t n16 = a.n_items * (int32_t)(sizeof(AppendItem) / 16);
            for (int32_t idx = threadIdx.x; idx < n16; idx += blockDim.x) dst[idx] = src[idx];
        }
        pdl_wait();               // tables and free stack: the previous step's kernels are complete
        if (!a.do_bookkeeping) return;
        __syncthreads();
        bookkeeping_phases(a, staged ? reinterpret_cast<const AppendItem*>(smem_raw) : a.items);
        return;
    }
    if (threadIdx.x == 0) stamp_begin(p);
    const uint32_t smem_base = (smem_u32(smem_raw) + 127u) & ~127u;
    const int32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t ring = smem_base + warp * C::kWarpBytes;
    const uint32_t bars = smem_base + C::NWARP * C::kWarpBytes + warp * C::NS * 8;
    if (lane == 0) {
        for (int s = 0; s < C::NS; ++s) mbar_init(bars + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();                                        // (the ring and its barriers are private to the warp)
    const GqaPlan& plan = sp.plan;
    const int32_t Hkv = a.L.n_kv_heads;
    __shared__ int4 s_pend[C::NWARP][2];                 // the (at most two) cut pairs of a range
    int4* pend = s_pend[warp];
    struct Cursor { int32_t i, kvh, t; StepGeo it; };    // item, KV head, tile of the pair, the item's geometry
    // Physical block ids of 32 consecutive tiles of one item (lane l: tile pc_base + l), fetched with ONE
    // coalesced load: a table lookup per tile is a dependent L2 round trip (~1 us under load) in front of
    // every copy.  The table row belongs to the session, so the ids serve all its KV heads.
    int32_t pc_item = -1, pc_base = 0, pc_phys = 0;
    // Request the tile `ahead` places after cursor `x` into ring stage `st` (the issue position is not kept as
    // state: inside a pair it is x.t + ahead; the walk over a pair boundary is the rare path).
    auto issue = [&](const Cursor& x, int32_t ahead, int32_t st) {
        int32_t ii = x.i, kv = x.kvh, d = x.t + ahead;
        int32_t sid = x.it.sid, n_sink_tiles = x.it.n_sink_tiles, first_blk = x.it.first_blk, n_tiles = x.it.n_tiles, alloc_lo = x.it.alloc_lo;
        while (d >= n_tiles) {
            d -= n_tiles;
            if (++kv == Hkv) {
                kv = 0;
                const StepGeo g2 = step_geo(sp.items[++ii], p.W, p.n_sink);
                sid = g2.sid; n_sink_tiles = g2.n_sink_tiles; first_blk = g2.first_blk; n_tiles = g2.n_tiles; alloc_lo = g2.alloc_lo;
            }
        }
        const int32_t blk = d < n_sink_tiles ? d : first_blk + (d - n_sink_tiles);
        const uint32_t bar = bars + 8 * st;
        if (blk >= alloc_lo) {
            // a block allocated in this step: every valid row of it is in k_new / v_new, and its table
            // entry may not be written yet -- nothing to copy, the phase completes at once
            if (lane == 0) mbar_arrive(bar);
            return;
        }
        if (ii != pc_item || d < pc_base || d >= pc_base + 32) {
            pc_item = ii; pc_base = d;
            const int32_t dl = d + lane;
            const int32_t bl = dl < n_sink_tiles ? dl : first_blk + (dl - n_sink_tiles);
            pc_phys = dl < n_tiles ? __ldg(p.table + (int64_t)sid * p.tbl_width + table_slot(bl, p.n_sink, p.ring)) : 0;
        }
        const int32_t phys = __shfl_sync(0xffffffffu, pc_phys, d - pc_base);
        if (lane == 0) {
            mbar_expect_tx(bar, C::kHeadBytes);
            bulk_g2s(ring + st * C::kHeadBytes, p.kv_layer + (int64_t)phys * p.L.block_bytes + (int64_t)kv * p.L.head_bytes,
                     C::kHeadBytes, bar);
        }
    };

    constexpr int CPR = D / 8;                           // 16-byte chunks per K or V row
    uint32_t phase_bits = 0;
    int32_t st = 0;                                      // ring stage of the tile being consumed (cyclic over all ranges)
    // SMs of one B200 do not stream at the same speed: with equal ranges the warps of the same ~40 SMs ended 10 % after
    // the others, launch after launch, and the kernel ends with the slowest.  So a warp takes its range AFTER it knows
    // where it runs: from the list of long ranges on a fast SM, of short ones on a slow SM (the other list when its
    // own is used up: every range is taken whatever the placement of the CTAs).
    uint32_t smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    const int32_t my_list = smid < kStepMaxSms ? sp.sm_class[smid] : 0;
    pdl_wait();                  // older rows, table entries, claim counters: every earlier kernel on the stream is complete
    WarpTileT<D, NQ> wt;
    while (true) {
        int32_t range = -1;
        if (lane == 0) {
            for (int32_t attempt = 0; attempt < 2 && range < 0; ++attempt) {
                const int32_t list = my_list ^ attempt;
                const int32_t lo = list == 0 ? 0 : plan.n_static, hi = list == 0 ? plan.n_static : plan.n_total;
                if (lo >= hi) continue;
                const int32_t k = lo + atomicAdd(sp.claim_ctr + list, 1);
                if (k < hi) range = k;
            }
        }
        range = __shfl_sync(0xffffffffu, range, 0);
        if (range < 0) break;
        const int64_t g0 = plan.range_lo(range);
        const int32_t n_total = (int32_t)(plan.range_hi(range) - g0);
        int32_t n_pend = 0;
        // where the range starts: binary search in the constant bank
        Cursor c;
        {
            int32_t lo = 0, hi = sp.n_items - 1;
            while (lo < hi) {
                const int32_t mid = (lo + hi + 1) >> 1;
                if ((int64_t)sp.items[mid].tile_off * Hkv <= g0) lo = mid; else hi = mid - 1;
            }
            c.i = lo;
            c.it = step_geo(sp.items[lo], p.W, p.n_sink);
            const int32_t rel = (int32_t)(g0 - (int64_t)c.it.tile_off * Hkv);
            c.kvh = rel / c.it.n_tiles;
            c.t = rel - c.kvh * c.it.n_tiles;
        }
        for (int32_t k = 0; k < min(n_total, C::NS); ++k) issue(c, k, (st + k) % C::NS);
        wt.init(p, c.it, c.kvh, lane);                   // (Q rows are fetched while the first tiles fly)
        for (int32_t n = 0; n < n_total; ++n) {
            mbar_wait(bars + 8 * st, (phase_bits >> st) & 1u);
            phase_bits ^= 1u << st;
            const StepGeo& it = c.it;
            const int32_t blk = tile_block(it, c.t), p0 = blk * kBlockTokens;
            const uint32_t kt = ring + st * C::kHeadBytes;
            // ---- rows of this step that live in this tile: from k_new / v_new into the tile in shared memory ----
            const int32_t new_lo = max(it.len0, p0), new_hi = min(it.len, p0 + kBlockTokens);
            const bool fresh = new_lo < new_hi;
            if (fresh) {
                uint8_t* kt_gen = smem_raw + (kt - smem_u32(smem_raw));
#pragma unroll 1
                for (int32_t pos = new_lo; pos < new_hi; ++pos) {
                    const int32_t r = pos - p0;
                    const int64_t src_row = ((int64_t)(it.q_row_off + (pos - it.len0)) * Hkv + c.kvh) * CPR;
#pragma unroll 1
                    for (int32_t idx = lane; idx < 2 * CPR; idx += 32) {
                        const int32_t is_v = idx >= CPR ? 1 : 0, cc = idx - is_v * CPR;
                        const uint4 val = __ldg((is_v ? a.v_new : a.k_new) + src_row + cc);
                        *reinterpret_cast<uint4*>(kt_gen + is_v * (kBlockTokens * D * 2) + tile_chunk_offset(r, cc)) = val;
                    }
                }
                __syncwarp();
            }
            if (!wt.skips(p, p0)) wt.template step<256>(p, it.len, kt, kt + kBlockTokens * D * 2, p0, lane);
            if (fresh) fence_async_smem();               // generic-proxy writes above, async-proxy refill below
            __syncwarp();                                // every lane is done with the stage
            if (n + C::NS < n_total) issue(c, C::NS, st);     // refill the stage
            // ---- row a4: the same rows go to their paged slots ----
            if (fresh && a.kv_layer) {
                if (blk >= it.alloc_lo && a.do_bookkeeping) {
                    if (lane == 0) {
                        int32_t seen;
                        do {
                            asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(a.bk_flag) : "memory");
                            if (seen != a.epoch) __nanosleep(100);
                        } while (seen != a.epoch);
                    }
                    __syncwarp();
                }
                const int32_t phys = __ldcg(a.table + (int64_t)it.sid * a.tbl_width + table_slot(blk, a.n_sink, a.ring));
                uint8_t* tile = a.kv_layer + (int64_t)phys * a.L.block_bytes + (int64_t)c.kvh * a.L.head_bytes;
#pragma unroll 1
                for (int32_t pos = new_lo; pos < new_hi; ++pos) {
                    const int32_t r = pos - p0;
                    const int64_t src_row = ((int64_t)(it.q_row_off + (pos - it.len0)) * Hkv + c.kvh) * CPR;
#pragma unroll 1
                    for (int32_t idx = lane; idx < 2 * CPR; idx += 32) {
                        const int32_t is_v = idx >= CPR ? 1 : 0, cc = idx - is_v * CPR;
                        const uint4 val = __ldg((is_v ? a.v_new : a.k_new) + src_row + cc);
                        *reinterpret_cast<uint4*>(tile + is_v * a.L.tile_bytes + tile_chunk_offset(r, cc)) = val;
                    }
                }
            }
            // ---- end of this warp's piece of the (item, head) pair ----
            const bool pair_end = c.t == it.n_tiles - 1;
            if (pair_end || n == n_total - 1) {
                const int64_t pair_lo = (int64_t)it.tile_off * Hkv + (int64_t)c.kvh * it.n_tiles;
                const int32_t first_r = plan.range_of(pair_lo), last_r = plan.range_of(pair_lo + it.n_tiles - 1);
                if (first_r == last_r) {
                    wt.store_final(p, it, c.kvh, lane);
                } else {
                    // row a6: unnormalised partial, written now and PUBLISHED after the tile loop (step_flush_pend): at
                    // most two pairs of a range are cut (its first and its last) and every piece of a pair is finished
                    // at the end of some warp's range anyway, so one fence and one ticket round trip per warp serve
                    // both -- a fence + ticket at the cut itself stalled the warp ~2-5 us with its ring full
                    wt.store_partial(p, it, c.kvh, range - first_r, lane);
                    if (lane == 0)
                        pend[n_pend] = make_int4(it.q_len * p.G | (c.kvh << 8) | ((last_r - first_r + 1) << 16), it.q_row_off, c.i, 0);
                    ++n_pend;
                }
            }
            // ---- advance the cursor (the ring stage follows the tile count) ----
            st = st + 1 == C::NS ? 0 : st + 1;
            if (pair_end) {
                c.t = 0;
                if (++c.kvh == Hkv) {
                    c.kvh = 0;
                    if (++c.i < sp.n_items) c.it = step_geo(sp.items[c.i], p.W, p.n_sink);
                }
                if (n + 1 < n_total) wt.init(p, c.it, c.kvh, lane);
            } else {
                ++c.t;
            }
        }
        if (n_pend > 0) step_flush_pend<D>(p, pend, n_pend, Hkv, lane);
    }
    // the last warp out zeroes the claim counters for the next launch
    if (lane == 0) {
        if (atomicAdd(sp.claim_ctr + 2, 1) == sp.n_workers - 1) { sp.claim_ctr[0] = 0; sp.claim_ctr[1] = 0; sp.claim_ctr[2] = 0; }
        stamp_end(p);
    }
}

// Measures how fast every SM streams when all of them stream (pool creation): the fused step kernel's launch shape
// (two CTAs of four warps per SM, a private 3-stage ring of 8 KB bulk copies per warp), `n_tiles` tiles per warp from
// pseudo-random blocks of the pool's own KV storage, nothing computed.  out[2 w] = SM of warp w, out[2 w + 1] = its
// time in ns.
template <int D>
__global__ void __launch_bounds__(StepCfg<D, 1>::kThreads, StepCfg<D, 1>::kCtasPerSm)
step_calibrate_kernel(const uint8_t* kv, KvLayout L, int64_t n_blocks, int32_t n_tiles, unsigned long long* out) {
    using C = StepCfg<D, 1>;
    extern __shared__ __align__(128) uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 127u) & ~127u;
    const int32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t ring = smem_base + warp * C::kWarpBytes;
    const uint32_t bars = smem_base + C::NWARP * C::kWarpBytes + warp * C::NS * 8;
    if (lane == 0) {
        for (int s = 0; s < C::NS; ++s) mbar_init(bars + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    const int32_t w = (int32_t)blockIdx.x * C::NWARP + warp;
    auto issue = [&](int32_t n, int32_t st) {
        if (lane == 0) {
            uint32_t h = (uint32_t)w * 2654435761u + (uint32_t)n * 40503u;
            h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
            const int64_t blk = (int64_t)(h % (uint32_t)n_blocks);
            mbar_expect_tx(bars + 8 * st, C::kHeadBytes);
            bulk_g2s(ring + st * C::kHeadBytes, kv + blk * L.block_bytes + (int64_t)(w % L.n_kv_heads) * L.head_bytes, C::kHeadBytes,
                     bars + 8 * st);
        }
    };
    const unsigned long long t0 = global_ns();
    for (int32_t k = 0; k < min(n_tiles, C::NS); ++k) issue(k, k);
    uint32_t phase_bits = 0;
    for (int32_t n = 0, st = 0; n < n_tiles; ++n) {
        mbar_wait(bars + 8 * st, (phase_bits >> st) & 1u);
        phase_bits ^= 1u << st;
        __syncwarp();
        if (n + C::NS < n_tiles) issue(n + C::NS, st);
        st = st + 1 == C::NS ? 0 : st + 1;
    }
    if (lane == 0) {
        uint32_t smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        out[2 * w] = smid;
        out[2 * w + 1] = global_ns() - t0;
    }
}

template <int D, int NQ>
inline cudaError_t configure_step_kernel() {
    return cudaFuncSetAttribute(step_gqa_kernel<D, NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, StepCfg<D, NQ>::kSmemBytes);
}
inline cudaError_t configure_step_kernels() {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(step_calibrate_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  StepCfg<128, 1>::kSmemBytes)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(step_calibrate_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  StepCfg<64, 1>::kSmemBytes)) != cudaSuccess) return e;
    if ((e = configure_step_kernel<128, 1>()) != cudaSuccess) return e;
    if ((e = configure_step_kernel<128, 2>()) != cudaSuccess) return e;
    if ((e = configure_step_kernel<64, 1>()) != cudaSuccess) return e;
    return configure_step_kernel<64, 2>();
}

// CTAs per SM and warps per CTA of the variant that serves rows_max = G x max q_len query rows per pair
inline int step_workers_per_sm(int rows_max) {
    return rows_max <= 8 ? StepCfg<128, 1>::kCtasPerSm * StepCfg<128, 1>::NWARP : StepCfg<128, 2>::kCtasPerSm * StepCfg<128, 2>::NWARP;
}

template <int D, int NQ>
inline cudaError_t launch_step_variant(const StepParams& sp, cudaStream_t st, bool pdl) {
    using C = StepCfg<D, NQ>;
    const dim3 grid(1 + sp.n_workers / C::NWARP);
    return launch_kernel(step_gqa_kernel<D, NQ>, grid, C::kThreads, C::kSmemBytes, st, pdl, sp);
}

// rows_max = G x max q_len over the items (<= 16)
inline cudaError_t launch_step_gqa(const StepParams& sp, int32_t D, int32_t rows_max, cudaStream_t st, bool pdl) {
    if (D == 128) return rows_max <= 8 ? launch_step_variant<128, 1>(sp, st, pdl) : launch_step_variant<128, 2>(sp, st, pdl);
    return rows_max <= 8 ? launch_step_variant<64, 1>(sp, st, pdl) : launch_step_variant<64, 2>(sp, st, pdl);
}

}  // namespace metronome
