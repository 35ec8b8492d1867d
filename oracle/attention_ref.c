/*
 * oracle/attention_ref.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of what Metronome's bounded-window attention
 * computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares no code, header, table or helper with the
 * CUDA path under paper_2607_02640_b200/csrc/.
 *
 * What it computes (the definition; the GPU only reaches it faster):
 *
 *   PAPER.md:L101 (sec. 4.1)  "the most recent W tokens plus the session's first few tokens, kept pinned"
 *   PAPER.md:L103 (sec. 4.1)  "the attention kernel's windowed mask admits [0,S) U [t-W,t]"
 *   PAPER.md:L258 (App. A)    "the windowed mask gains the OR-term k < S"
 *   PAPER.md:L258 (App. A)    "verified against a float32 reference of the union mask (mixed
 *                              prefill/decode, grouped-query attention ...)"
 *
 *   admit(j, t) = (j <= t)  and  ( j < S  or  t - j < W )
 *   s_j   = scale * < q[t,h] , k[j, h / G] >            for admitted j          (G = Hq / Hkv)
 *   p     = softmax over the admitted j (two passes: max, exp, sum, divide)
 *   o[t,h] = sum_j p_j * v[j, h / G]
 *
 * Reading of "[t-W, t]" (reading R1): the window holds W keys INCLUDING the query's own
 * position, i.e. t-W < j <= t.  "[t-W,t]" read literally has W+1 keys, but L101 says "the most
 * recent W tokens", L29 "last W tokens", and the resident-set invariant min(len, S+W) needs W.
 *
 * Precision: the paper fixes a float32 reference (L258), so oracle_attend_f32 is THE oracle.
 * oracle_attend_f64 is the same text in double; tests use it to bound the fp32 oracle's own
 * rounding (it is not what the GPU is compared with).
 *
 * Inputs are bf16 bit patterns (uint16).  Keys carry explicit absolute positions so the same
 * routine serves the "definition layer" (whole unpaged history, positions 0..len-1) and the
 * "paged layer" (only the rows still resident, gathered through a simulated block table).
 * Keys must be given in ascending position so both layers sum in the same order.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static float bf16_bits_to_float(uint16_t b) {
    union { uint32_t u; float f; } x;
    x.u = ((uint32_t)b) << 16; /* bf16 is the top half of an IEEE float32 */
    return x.f;
}

/* admit(j,t): PAPER.md:L103 / L258 union mask, causal, window of W keys including t itself. */
int oracle_admit(int64_t j, int64_t t, int64_t S, int64_t W) {
    if (j > t) return 0;          /* causal */
    if (j < S) return 1;          /* sink term  "k < S"        (L258) */
    if (t - j < W) return 1;      /* window term, W most recent (L101) */
    return 0;
}

static float kv_identity(float x) { return x; }

#define DEFINE_ORACLE_ATTEND(NAME, REAL, EXPF, KVT, KVLOAD)                                       \
    int NAME(const uint16_t* q, const int64_t* q_pos, int64_t n_q,                                \
             const KVT* k, const KVT* v, const int64_t* k_pos, int64_t n_k,                       \
             int32_t Hq, int32_t Hkv, int32_t D, int64_t S, int64_t W, double scale,              \
             float* out, float* weights, int32_t n_threads) {                                     \
        if (Hkv <= 0 || Hq % Hkv != 0) return 1;                                                  \
        const int32_t G = Hq / Hkv;                                                               \
        int failed = 0;                                                                           \
        _Pragma("omp parallel for collapse(2) schedule(dynamic) num_threads(n_threads)")          \
        for (int64_t r = 0; r < n_q; ++r) {                                                       \
            for (int32_t h = 0; h < Hq; ++h) {                                                    \
                const int64_t t = q_pos[r];                                                       \
                const int32_t hk = h / G;                                                         \
                const uint16_t* qv = q + ((size_t)r * Hq + h) * D;                                \
                REAL* s = (REAL*)malloc(sizeof(REAL) * (size_t)(n_k > 0 ? n_k : 1));              \
                if (!s) { failed = 1; continue; }                                                 \
                /* pass 1: scores of admitted keys, and their maximum */                          \
                REAL m = -INFINITY;                                                               \
                int64_t n_adm = 0;                                                                \
                for (int64_t i = 0; i < n_k; ++i) {                                               \
                    if (!oracle_admit(k_pos[i], t, S, W)) continue;                               \
                    const KVT* kv = k + ((size_t)i * Hkv + hk) * D;                               \
                    REAL dot = 0;                                                                 \
                    for (int32_t d = 0; d < D; ++d)                                               \
                        dot += (REAL)bf16_bits_to_float(qv[d]) * (REAL)KVLOAD(kv[d]);             \
                    s[i] = (REAL)scale * dot;                                                     \
                    if (s[i] > m) m = s[i];                                                       \
                    ++n_adm;                                                                      \
                }                                                                                 \
                /* pass 2: exp, sum, divide, weighted sum of V */                                 \
                REAL l = 0;                                                                       \
                for (int64_t i = 0; i < n_k; ++i) {                                               \
                    if (!oracle_admit(k_pos[i], t, S, W)) continue;                               \
                    s[i] = EXPF(s[i] - m);                                                        \
                    l += s[i];                                                                    \
                }                                                                                 \
                for (int64_t i = 0; i < n_k; ++i)                                                 \
                    if (oracle_admit(k_pos[i], t, S, W)) s[i] = s[i] / l;       /* p_i */         \
                REAL* acc = (REAL*)calloc((size_t)D, sizeof(REAL));                               \
                if (!acc) { free(s); failed = 1; continue; }                                      \
                for (int64_t i = 0; i < n_k; ++i) {            /* o = sum_i p_i v_i */            \
                    if (!oracle_admit(k_pos[i], t, S, W)) continue;                               \
                    const KVT* vv = v + ((size_t)i * Hkv + hk) * D;                               \
                    for (int32_t d = 0; d < D; ++d)                                               \
                        acc[d] += s[i] * (REAL)KVLOAD(vv[d]);                                     \
                }                                                                                 \
                float* o = out + ((size_t)r * Hq + h) * D;                                        \
                for (int32_t d = 0; d < D; ++d) o[d] = (n_adm > 0) ? (float)acc[d] : 0.0f;        \
                float* wrow = weights ? weights + ((size_t)r * Hq + h) * n_k : 0;                 \
                if (wrow)                                                                         \
                    for (int64_t i = 0; i < n_k; ++i)                                             \
                        wrow[i] = oracle_admit(k_pos[i], t, S, W) ? (float)s[i] : 0.0f;           \
                free(acc);                                                                        \
                free(s);                                                                          \
            }                                                                                     \
        }                                                                                         \
        return failed;                                                                            \
    }

/* q [n_q][Hq][D], k/v [n_k][Hkv][D] bf16 bits; out [n_q][Hq][D] float32;
 * weights (optional, may be NULL) [n_q][Hq][n_k] float32 softmax weights (0 where not admitted).
 * A query with no admitted key (cannot happen when the query's own key is present) yields 0.
 * Returns 0 on success. */
DEFINE_ORACLE_ATTEND(oracle_attend_f32, float, expf, uint16_t, bf16_bits_to_float)
DEFINE_ORACLE_ATTEND(oracle_attend_f64, double, exp, uint16_t, bf16_bits_to_float)
/* The same text with k / v given as float32 VALUES (q stays bf16 bits): the fp8 KV arm (oracle/kv_fp8.py), whose
 * dequantised keys and values code x scale are not bf16 numbers ("we bound which tokens stay
 * resident, and the two compose"). */
DEFINE_ORACLE_ATTEND(oracle_attend_kvf32_f32, float, expf, float, kv_identity)
DEFINE_ORACLE_ATTEND(oracle_attend_kvf32_f64, double, exp, float, kv_identity)

int32_t oracle_max_threads(void) {
#ifdef _OPENMP
    return (int32_t)omp_get_max_threads();
#else
    return 1;
#endif
}
