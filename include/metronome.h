/*
 * metronome.h -- C ABI of libmetronome.so: bounded-window paged attention for resident streaming
 * sessions on one NVIDIA B200 (sm_100a).
 *
 * The library implements the data-parallel hot path of Metronome's per-frame serving step
 * (arxiv/paper_2607_02640; citations are PAPER.md:L<line>):
 *
 *   "retain each session's first S and last W tokens, freeing everything between -- as an API"
 *                                                                    (sec. 6)
 *   "the KV manager pins each request's first blocks instead of freeing them, and the attention
 *    kernel's windowed mask admits [0,S) U [t-W,t]"                  (sec. 4.1)
 *
 * Conventions
 *   - All functions return an int status (METRONOME_OK = 0).  No exceptions, no aborts.
 *     On ANY error the pool's state (host and device) is unchanged.  (One exception, stated where it
 *     applies: a CUDA launch failure that FOLLOWS a kernel the same call has already enqueued, which
 *     only the poison / bookkeeping-only debug modes can see, leaves the CUDA context in its sticky
 *     error state and the pool unusable.)
 *   - "host" pointers are ordinary CPU memory, read or written before the call returns.
 *     "device" pointers are CUDA global memory on the pool's device; they are consumed
 *     asynchronously on `cuda_stream` (a cudaStream_t passed as void*; NULL = default stream).
 *   - All calls on one pool must be issued from one host thread at a time and on ONE stream (or on
 *     streams the caller has ordered); the library adds no cross-stream synchronisation.
 *   - The pool owns the KV storage (unless the caller provides it), block tables, free list and
 *     split-KV workspace.  The caller owns q / k_new / v_new / out and the stream.
 *   - bf16 = IEEE bfloat16 bit patterns, 2 bytes.  Row-major, innermost index last.
 *   - Positions: the token appended i-th to a session (counting from 0 at session_open) has
 *     absolute position i for ever ("the resident request keeps growing logically", L103).
 *     K arrives position-encoded; the library applies no rotary embedding.
 */
#ifndef METRONOME_H_
#define METRONOME_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define METRONOME_ABI_VERSION 3

/* ---- status codes --------------------------------------------------------------------------- */
enum {
    METRONOME_OK = 0,
    METRONOME_ERR_INVALID_ARG = 1,        /* NULL pointer, negative count, unsupported shape       */
    METRONOME_ERR_INVALID_SESSION = 2,    /* sid not open                                          */
    METRONOME_ERR_DUPLICATE_SESSION = 3,  /* a session may appear once per call (L46: "all due
                                             sessions each tick")                                  */
    METRONOME_ERR_SESSIONS_FULL = 4,      /* max_sessions slots are open                           */
    METRONOME_ERR_POOL_EXHAUSTED = 5,     /* the paper's stall (L60: "the scheduler can no longer
                                             allocate blocks"), surfaced cleanly: nothing changed  */
    METRONOME_ERR_CHUNK_TOO_LARGE = 6,    /* n_new > max_new_tokens                                */
    METRONOME_ERR_QLEN_EXCEEDS_LAST_APPEND = 7, /* older rows' windows may already be freed        */
    METRONOME_ERR_LAYER_SEQUENCE = 8,     /* layer > 0 append that does not repeat layer 0's batch,
                                             or attend on a layer not yet appended this step       */
    METRONOME_ERR_LEN_OVERFLOW = 9,       /* the clean version of the max_model_len crash (L271)   */
    METRONOME_ERR_CUDA = 10,              /* a CUDA runtime call failed; see metronome_last_cuda_error */
    METRONOME_ERR_UNSUPPORTED = 11,       /* e.g. attention on a bookkeeping-only pool             */
    METRONOME_ERR_OUT_OF_MEMORY = 12,
    METRONOME_ERR_SCRATCH_EXCEEDED = 13   /* metronome_attend_frame_static: the call's split-KV partials do not fit
                                             the library's fixed scratch array; nothing was launched             */
};

/* ---- flags ---------------------------------------------------------------------------------- */
/* Fill every freed block with bf16 NaN (L258: "freed blocks NaN-poisoned to prove nothing outside
 * sinks U window is ever read").  Debug / test aid; off by default. */
#define METRONOME_FLAG_POISON_ON_FREE 0x1u
/* No KV storage: only sessions, block tables and the free list (any block_size >= 1).  append_kv
 * must be given k_new = v_new = NULL; attend_frame returns METRONOME_ERR_UNSUPPORTED.  For
 * occupancy studies (Eq. 1, Fig. 5) and bookkeeping tests. */
#define METRONOME_FLAG_BOOKKEEPING_ONLY 0x2u
/* The paper's vanilla arm (L52: "it bounds nothing"): no block is ever freed before close and the
 * mask is plain causal.  W is ignored. */
#define METRONOME_FLAG_UNBOUNDED 0x4u

/* NEXT row f4, sec. 4.1 "Orthogonal to KV compression, which shrinks each token
 * ...: we bound which tokens stay resident, and the two compose": K / V rows are STORED as fp8 -- E4M3 codes plus one
 * float32 scale per (token, KV head) row, scale = max |x| / 448, code = x / scale rounded to nearest even (DESIGN.md
 * reading R18; the paper names no format).  k_new / v_new / q / out stay bf16; attention runs over what the codes
 * decode to (value(code) x scale, float32).  A block-head takes 2 x 16 x D + 128 bytes instead of 2 x 16 x D x 2.
 * All attention of such a pool runs on the CUDA-core row kernel.  metronome_read_kv returns FLOAT32 rows. */
#define METRONOME_FLAG_KV_FP8 0x8u

/* ---- configuration -------------------------------------------------------------------------- */
typedef struct metronome_pool_config {
    int32_t n_layers;        /* >= 1; one block table is shared by all layers (L256: every decoder
                                layer reports the same windowed spec)                              */
    int32_t n_q_heads;       /* Hq                                                                 */
    int32_t n_kv_heads;      /* Hkv; Hq % Hkv == 0; G = Hq / Hkv (grouped-query attention, L258)   */
    int32_t head_dim;        /* D in {64, 128}                                                     */
    int32_t block_size;      /* tokens per KV block; 16 (L149: "S=16 -- one KV block") unless
                                METRONOME_FLAG_BOOKKEEPING_ONLY                                    */
    int32_t n_sinks;         /* S >= 0: pinned attention-sink tokens (L101)                        */
    int32_t window;          /* W >= 1: most recent tokens kept, the query's own included          */
    int32_t max_sessions;    /* session slots, 1..65534                                            */
    int32_t max_new_tokens;  /* largest n_new of one session in one append_kv (chunk length)       */
    int32_t n_blocks;        /* size of the fixed KV block pool (L60)                              */
    float   softmax_scale;   /* 0 -> 1/sqrt(D)                                                     */
    uint32_t flags;          /* METRONOME_FLAG_*                                                   */
    int64_t max_session_len; /* 0 -> 2^31 - 1 - max_new_tokens; longer appends: LEN_OVERFLOW       */
    void*   kv_storage;      /* device; NULL -> the pool allocates metronome_kv_storage_bytes()    */
    size_t  kv_storage_bytes;/* size of kv_storage when provided                                   */
} metronome_pool_config_t;

typedef struct metronome_pool metronome_pool_t; /* opaque */

/* ---- pool ----------------------------------------------------------------------------------- */

/* Bytes of device memory the KV storage of `cfg` needs:
 * n_layers * n_blocks * n_kv_heads * 2 (K,V) * block_size * head_dim * 2  (bf16), or
 * n_layers * n_blocks * n_kv_heads * (2 * block_size * head_dim + 128)     (METRONOME_FLAG_KV_FP8).  0 if cfg is invalid. */
size_t metronome_kv_storage_bytes(const metronome_pool_config_t* cfg);

/* Worst-case resident blocks of one session: ceil(S/B) + floor((W + max_new_tokens - 1)/B) + 2.
 * (L258: "the per-request admission cap counts the pinned blocks so pool sizing stays exact".)
 * Returns -1 on invalid arguments. */
int32_t metronome_max_blocks_per_session(int32_t S, int32_t W, int32_t B, int32_t max_new_tokens);

/* Creates a pool on the current CUDA device.  cfg: host.  *out receives the handle.
 * The free list is a LIFO stack whose initial pop order is 0,1,2,...  (reading R6).
 * Errors: INVALID_ARG, OUT_OF_MEMORY, CUDA. */
int metronome_pool_create(const metronome_pool_config_t* cfg, metronome_pool_t** out);

/* Frees everything the pool owns (synchronises the device first).  NULL is a no-op. */
int metronome_pool_destroy(metronome_pool_t* pool);

/* ---- sessions (L52: a session is one long-lived resident request) ----------------------------- */

/* Claims the LOWEST free session slot; len = 0, no blocks.  *sid_out: host.  No device work.
 * Errors: SESSIONS_FULL. */
int metronome_session_open(metronome_pool_t* pool, int32_t* sid_out);

/* Returns all blocks of `sid` to the free list (sink blocks, then live window blocks, ascending
 * logical order) and releases the slot.  Asynchronous on cuda_stream.
 * Errors: INVALID_SESSION, CUDA. */
int metronome_session_close(metronome_pool_t* pool, int32_t sid, void* cuda_stream);

/* ---- the per-frame hot path (L46: "prefill the new chunk, then decode up to tau output tokens,
 *      attending over the session's accumulated context ... for all due sessions each tick") ---- */

/* Appends n_new[i] tokens to session sids[i], i = 0..n_batch-1 (batch order matters, reading R6).
 *   sids, n_new : host int32 [n_batch]; each session at most once; 0 <= n_new[i] <= max_new_tokens
 *   k_new,v_new : device bf16 [sum(n_new), n_kv_heads, head_dim], rows in batch order
 *   layer == 0  : bookkeeping, then the K/V write:
 *       phase 1  every session frees its non-sink blocks that lie ENTIRELY behind the window of
 *                position L0 (its length before this call) -- block b is freed iff b >= ceil(S/B)
 *                and (b+1)*B <= L0-W+1 (L256: "frees blocks that fall entirely behind the window";
 *                L258: "pins each request's first ceil(S/block) blocks instead of freeing them");
 *       check    free + freed >= needed, else POOL_EXHAUSTED and nothing has changed;
 *       phase 2  every session pops ceil(L1/B) - ceil(L0/B) blocks, ascending logical order.
 *   layer  > 0  : must repeat layer 0's most recent batch exactly; only writes K/V of that layer.
 * One kernel launch (bookkeeping + K/V scatter); k_new / v_new are read by that kernel in stream order,
 * the host arrays before the call returns.  Calls on one pool must be ordered on ONE stream.  The call
 * also plans the usual attend_frame(q_lens = n_new) of this step, so that call needs no upload.
 * Errors: INVALID_ARG, INVALID_SESSION, DUPLICATE_SESSION, CHUNK_TOO_LARGE, LEN_OVERFLOW,
 *         POOL_EXHAUSTED, LAYER_SEQUENCE, CUDA. */
int metronome_append_kv(metronome_pool_t* pool, int32_t layer, int32_t n_batch,
                        const int32_t* sids, const int32_t* n_new,
                        const void* k_new, const void* v_new, void* cuda_stream);

/* Attention of the LAST q_lens[i] positions of session sids[i] over its resident keys under
 *   admit(j,t) = (j <= t) and (j < S or t - j < W)        (L103, L258; window = W keys incl. t)
 *   out[t,h] = softmax_j(scale * <q[t,h], k[j,h/G]>) . v[j,h/G]      fp32 accumulate, bf16 out
 * decode: q_len 1; chunk prefill: q_len n (causal inside the chunk).  One call may mix both (L258).
 *   sids, q_lens : host int32 [n_batch]; 0 <= q_lens[i] <= n_new of that session's last append
 *   q, out       : device bf16 [sum(q_lens), n_q_heads, head_dim], rows in batch order
 * The layer must have been appended in the current step (since the last layer-0 append).
 * q must be complete on cuda_stream when the call is enqueued; when it repeats the batch of this
 * step's append_kv (the usual case) its kernel may begin -- reading q and blocks no append is still
 * writing -- while that append kernel runs, so q must not be produced by work enqueued on another
 * stream without an event the caller has waited on.
 * Errors: INVALID_ARG, INVALID_SESSION, DUPLICATE_SESSION, QLEN_EXCEEDS_LAST_APPEND,
 *         LAYER_SEQUENCE, UNSUPPORTED, CUDA. */
int metronome_attend_frame(metronome_pool_t* pool, int32_t layer, int32_t n_batch,
                           const int32_t* sids, const int32_t* q_lens,
                           const void* q, void* out, void* cuda_stream);

/* metronome_attend_frame for callers that must not allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same arguments, same result (the union mask
 * [0,S) U (t-W, t]; L258 "segmented-decode ... merged exactly once"), but the call -- unlike attend_frame,
 * whose split-KV workspace is grown with cudaFree / cudaMalloc when a batch needs more -- calls NO cudaMalloc,
 * cudaFree or allocating library routine.  It always runs the split-KV CUDA-core row kernel + the merge kernel
 * (any group size, bf16 and fp8 pools; the tensor-core kernels are not used), and the segments' partial
 * results (acc, m, l) go to ONE fixed array of METRONOME_STATIC_SCRATCH_BYTES that lives in the library image:
 * every GPU that loads libmetronome.so holds those bytes until the process exits.
 *   limit   sum(q_lens) * n_q_heads * max_splits * (head_dim + 2) * 4 <= METRONOME_STATIC_SCRATCH_BYTES, where
 *           max_splits (<= 64) is the largest number of segments the call's split plan gives one session
 *           (segments of >= 8 KV blocks, sized for >= 16 CTAs per SM; 1 = no partials at all).  A call beyond it
 *           returns METRONOME_ERR_SCRATCH_EXCEEDED (metronome_last_cuda_error() says by how much); nothing was
 *           launched and nothing changed.  Config 2's decode step (128 rows x 32 heads x 6 segments) needs 12.2 MiB.
 *   sharing the array is shared by EVERY call in the process (all pools, all streams of one device) and keeps the
 *           previous call's contents.  Nothing in it has to start at zero: a call reads only the slots its own
 *           row kernel wrote.  Two calls whose kernels overlap on the GPU (different streams, different pools)
 *           RACE on it: order such calls yourself (one stream, or an event between them).
 *   set-up  the array's device address is looked up once per device (cudaGetSymbolAddress, no allocation) by the
 *           first call made with that device current; the pool must have been created on the current device.
 * sids, q_lens, q, out, stream ordering and the other errors: as metronome_attend_frame.  The per-call work
 * list travels through the pool's staging ring (allocated at pool creation) with one cudaMemcpyAsync.
 * Errors: those of metronome_attend_frame, SCRATCH_EXCEEDED. */
#define METRONOME_STATIC_SCRATCH_BYTES (16u << 20)
int metronome_attend_frame_static(metronome_pool_t* pool, int32_t layer, int32_t n_batch,
                                  const int32_t* sids, const int32_t* q_lens,
                                  const void* q, void* out, void* cuda_stream);

/* One sub-step of a frame in ONE call: exactly metronome_append_kv(layer, sids, n_new, k_new, v_new)
 * followed by metronome_attend_frame(layer, sids, q_lens = n_new, q, out) -- same arguments, same
 * results, same errors (union of the two; on any error nothing has changed) -- which is the shape of
 * every sub-step of PAPER.md:L46 ("prefill the new chunk, then decode up to tau output tokens": each
 * appends its tokens and attends from them), in one call: one validation, one plan, and the library is free
 * to run both halves in one launch where that pays (a tuning knob of metronome_measure.h; today it runs the
 * two kernels back to back).  k_new / v_new / q are read, out is written, in stream order by the kernels of
 * this call.  Deviation from SURVEY.md sec. 8(b), which lists the two calls only; they remain. */
int metronome_append_attend(metronome_pool_t* pool, int32_t layer, int32_t n_batch,
                            const int32_t* sids, const int32_t* n_new,
                            const void* k_new, const void* v_new,
                            const void* q, void* out, void* cuda_stream);

/* append_kv followed by attend_frame(q_lens = n_new) with HOST buffers: k_new, v_new, q are copied
 * host->device, out device->host, all on cuda_stream, and the stream is synchronised before
 * returning.  Pinned (page-locked) host memory makes the copies asynchronous.  This is the
 * end-to-end entry point bench.py's `e2e` leg times.  Errors: union of the two calls. */
int metronome_step_host(metronome_pool_t* pool, int32_t layer, int32_t n_batch,
                        const int32_t* sids, const int32_t* n_new,
                        const void* k_new_host, const void* v_new_host,
                        const void* q_host, void* out_host, void* cuda_stream);

/* The same step, pipelined: returns once the copies and kernels are ENQUEUED -- k/v/q host->device on a copy
 * stream of the pool's, the step on cuda_stream, out device->host on a second copy stream -- so that the uploads of
 * the next steps and the read-back of the previous ones run next to the kernels of step k.
 *   pinned host buffers (out_host page-locked): three staging slots and NO event on cuda_stream between two kernels, so
 *     the kernels keep their programmatic launch edges (one step per tick, back to back): the input copies
 *     end with a 4-byte copy of the step number into a device flag the kernels wait for, a one-thread kernel behind the
 *     step's last kernel publishes "kernels complete", the read-back stream waits for that value (stream wait-value),
 *     copies out and writes the step number to a pinned flag that metronome_step_host_wait polls.  The host may run
 *     two steps ahead: issuing step k blocks until step k-3 is complete.
 *   pageable host buffers (or METRONOME_HOST_STEP_EVENTS=1 in the environment at pool creation, a measurement aid): two
 *     staging slots chained by events; issuing step k blocks until step k-2 is complete.  The library drains one mode
 *     before it switches to the other.
 * The host buffers of a step must stay untouched, and out_host is not valid, until
 * metronome_step_host_wait(pool, keep) has returned with that step among the finished ones: it blocks until at
 * most `keep` (0, 1, 2) of the steps issued so far are still in flight.  Steps complete in issue order.
 * Errors: as metronome_step_host; an error leaves the pool as it was (the step was not enqueued). */
int metronome_step_host_async(metronome_pool_t* pool, int32_t layer, int32_t n_batch,
                              const int32_t* sids, const int32_t* n_new,
                              const void* k_new_host, const void* v_new_host,
                              const void* q_host, void* out_host, void* cuda_stream);
int metronome_step_host_wait(metronome_pool_t* pool, int32_t keep);

/* ---- introspection (bit-exact parity of tables and free list; occupancy signal, L83) ---------- */

/* All out-pointers are host and optional (NULL = skip).  Blocks the host until cuda_stream has
 * finished the pool's earlier work.  block_ids receives the resident physical ids in logical order
 * (sink blocks first); room for metronome_max_blocks_per_session() entries is required.
 * first_live_block = first logical non-sink block still resident.  Errors: INVALID_SESSION, CUDA. */
int metronome_session_query(metronome_pool_t* pool, int32_t sid, void* cuda_stream, int64_t* len,
                            int32_t* first_live_block, int32_t* n_blocks, int32_t* block_ids);

/* n_free and the free ids in POP order (next allocation first); free_ids needs n_blocks entries. */
int metronome_pool_query(metronome_pool_t* pool, void* cuda_stream, int32_t* n_free, int32_t* free_ids);

/* Reads back, through the block table, K and V rows of positions [pos0, pos0+n) of `sid` in
 * `layer` into device bf16 [n, n_kv_heads, head_dim] buffers (verification of the KV write; float32
 * buffers holding the decoded rows for a METRONOME_FLAG_KV_FP8 pool).
 * Positions whose block is not resident return bf16 NaN.  Errors: INVALID_*, UNSUPPORTED, CUDA. */
int metronome_read_kv(metronome_pool_t* pool, int32_t layer, int32_t sid, int64_t pos0, int32_t n,
                      void* k_out, void* v_out, void* cuda_stream);

/* ---- NEXT row f3: deadline-aware admission on the per-frame latency signal ----
 * PAPER.md:L105-111 sec. 4.2: "an AIMD loop on the measured per-frame latency, which lowers the
 * admission cap multiplicatively when latency nears a target fraction of the budget and raises it
 * additively to probe when there is headroom.  Arrivals beyond the cap receive a clean overload
 * rejection."  The paper gives no constants (parity unpinned by the paper; the rule below is this
 * build's reading, R17).  Pure host state, no CUDA, not thread-safe.
 *   observe(latency): cap <- max(cap_min, cap * mult_factor)   if latency >= target_frac * budget_ms
 *                     cap <- min(cap_max, cap + add_step)      otherwise        (one update per frame)
 *   admit(n_live):    1 iff n_live < floor(cap)                (the caller opens the session or sheds)
 * Errors: INVALID_ARG (null pointers; budget_ms <= 0; target_frac not in (0, 1]; add_step <= 0;
 * mult_factor not in (0, 1); cap_min < 1; cap_max < cap_min; cap_init outside [cap_min, cap_max]; a
 * negative or NaN latency; n_live < 0). */
typedef struct metronome_gate metronome_gate_t;
typedef struct {
    float budget_ms;     /* the frame deadline ("80 ms frame")            */
    float target_frac;   /* back off when latency reaches this fraction of the budget  */
    float add_step;      /* additive increase of the cap per frame with headroom       */
    float mult_factor;   /* multiplicative decrease, in (0, 1)                          */
    float cap_min, cap_max, cap_init;
} metronome_gate_config_t;
int metronome_gate_create(const metronome_gate_config_t* cfg, metronome_gate_t** out);
int metronome_gate_destroy(metronome_gate_t* gate);
int metronome_gate_observe(metronome_gate_t* gate, float frame_latency_ms, float* cap_out);
int metronome_gate_admit(metronome_gate_t* gate, int32_t n_live, int32_t* admitted_out);

const char* metronome_strerror(int status);
/* Text of the last CUDA error seen by this pool ("" if none).  Valid until the next call. */
const char* metronome_last_cuda_error(metronome_pool_t* pool);
int metronome_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* METRONOME_H_ */
