// metronome.cu -- the C ABI of libmetronome.so (include/metronome.h) and its host-side state.
//
// Host state is "shadow counts" only: per session {open, len, first_live, last_n}, the free count,
// and the last layer-0 batch.  They are pure functions of the call history, so every error is
// raised synchronously and before anything changes, while the physical block ids (block tables,
// free stack) live on the device and are only ever touched by kernels on the caller's stream.
#include "../../include/metronome.h"
#include "../../include/metronome_measure.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <algorithm>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "attend_common.cuh"
#include "attend_mma.cuh"
#include "attend_rows.cuh"
#include "attend_umma.cuh"
#include "attend_umma_fp8.cuh"
#include "bookkeeping.cuh"
#include "kv_append.cuh"
#include "step_gqa.cuh"

using namespace metronome;

// metronome_attend_frame_static (include/metronome.h): the split-KV partials of a call that must not allocate.
// The name below is a host-side stand-in in host code, NOT a device address: static_scratch_ptr() asks the runtime
// for the address (once per device, with that device current) and only that pointer is ever given to a kernel.
static __device__ __align__(256) unsigned char g_static_scratch[METRONOME_STATIC_SCRATCH_BYTES];

namespace {

struct Session {
    bool open = false;
    int64_t len = 0;
    int32_t first_live = 0;   // first logical non-sink block still resident
    int32_t last_n = 0;       // n_new of this session's most recent append
    int64_t last_epoch = 0;   // pool epoch of that append
    int32_t prev_n = 0;       // the same two for the append before it (early mode: rows the append kernel of
    int64_t prev_epoch = 0;   // step e-1 wrote may still be in flight when the row kernel of step e starts)
};

constexpr int kStagingSlots = 64;      // per-call metadata slots (pinned host + device twin)
constexpr int kStagingGroup = 8;       // one completion event per 8 slots: an event between two kernels
                                       // would break their programmatic (PDL) launch edge
constexpr int kMaxSplits = 64;
constexpr int kUmmaHalfDefault = 2;
constexpr int kGqaSmClassDefault = 0;  // (set to 1 once measured)
constexpr int kDirectSlots = 3;        // device staging slots of the event-free async host steps
constexpr int kStampSlots = 1 << 15;   // attention launches one stamped pass can hold
#ifndef METRONOME_GQA_BND_BYTES
#define METRONOME_GQA_BND_BYTES 65536
#endif
constexpr int kMaxRangeItems = 4096;   // GQA decode ranges whose start item travels with the work list

// Row a8: the launch plan of one attend_frame call (host side of the work list).  Items of class 0
// go to the row kernel or the GQA decode kernel, items of class 1 (placed after them) to the chunk
// kernel.
struct AttendPlan {
    bool valid = false;
    int64_t epoch = -1;               // pool epoch the plan was made for (cached plans only)
    int family = 1;                   // 1 CUDA-core rows, 2 tensor-core (gqa + chunk)
    int32_t n_items = 0;
    int32_t n_cls[2] = {0, 0}, total_splits[2] = {0, 0}, cls_rows[2] = {0, 0}, cls_max_q[2] = {0, 0};
    bool merge_cls[2] = {false, false};
    int32_t max_splits = 1;
    GqaPlan gplan{};
    int32_t gqa_ctas = 0;
    int32_t n_range_items = 0;        // int32 entries after the AttendItems (0: kernels search)
    bool early = false;               // the append kernel of this step runs in early mode (see append_fused_kernel)
    int64_t total_rows = 0;
    // fused decode step (step_gqa.cuh): every item is decode class and the list fits the kernel parameters
    bool step_ok = false;
    GqaPlan step_plan{};              // its two lists of ranges (long: fast SMs, short: slow SMs)
    int32_t step_workers = 0;         // warps of the launch (4 per CTA but the bookkeeping one)
};

}  // namespace

struct metronome_pool {
    metronome_pool_config_t cfg{};
    int32_t n_sink = 0, tbl_width = 0, ring = 0, G = 1, W_eff = 0;
    float scale = 0.f;
    KvLayout L{};
    bool bookkeeping_only = false, poison = false, unbounded = false, own_kv = false, fp8 = false;

    std::vector<Session> sessions;
    std::vector<int32_t> stamp;        // duplicate detection
    int32_t stamp_now = 0;
    int32_t n_open = 0, n_free = 0;

    int64_t epoch = 0;                 // number of layer-0 appends so far
    std::vector<int64_t> layer_epoch;  // epoch of each layer's latest append
    std::vector<int32_t> last_sids, last_n_new;
    AttendPlan cached_plan;            // plan of attend_frame(q_lens = n_new) for the latest layer-0 append
    std::vector<StepItem> step_items;  // the same work list in the fused step kernel's 16-byte form (cached_plan.step_ok)
    std::vector<Session> undo_sessions;          // append_kv's rollback snapshot (members: no allocation per call)
    std::vector<int32_t> undo_sids, undo_n_new;
    int32_t inject_fault = 0;          // metronome_pool_debug_fail_next (one-shot, tests of the error path)

    // device
    int32_t* d_table = nullptr;
    int32_t* d_free = nullptr;
    uint8_t* d_kv = nullptr;
    float* d_ws_acc = nullptr;
    float* d_ws_ml = nullptr;
    int32_t* d_tickets = nullptr;      // [max_sessions][Hkv], zero between launches
    int32_t* d_bk_flag = nullptr;      // [0] bookkeeping epoch, [1] work-list epoch, [2..3] GQA claim counters, [5] past-wait epoch, [6..7] GQA SM-class claims
    int32_t last_early_epoch = 0;      // epoch of the previous append kernel if it ran in early mode, else 0
    int64_t pastwait_launches = -1;    // value of n_launch right after a tensor-core attention launch that publishes its epoch once
    int32_t pastwait_epoch = 0;        // past its wait (d_bk_flag[12]); still equal to n_launch <=> nothing was launched since
    AttendItem* d_attend_items = nullptr;   // 2 x [max_sessions] (+ range items), written by the append kernel (cached plan)
    size_t attend_buf_bytes = 0;
    size_t ws_slots = 0;               // capacity in (row, head, split) slots
    uint8_t* d_io = nullptr;           // staging for metronome_step_host
    size_t io_bytes = 0;
    // metronome_step_host_async: two staging slots, a copy stream per direction, events that chain
    // H2D(k) -> step(k) -> D2H(k) while H2D(k+1) and D2H(k-1) run next to step(k)
    uint8_t* d_io2[3] = {nullptr, nullptr, nullptr};   // (the event-chained mode uses two slots, the event-free mode three)
    size_t io2_bytes[3] = {0, 0, 0};
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    cudaEvent_t ev_h2d[2]{}, ev_comp[2]{}, ev_d2h[2]{};
    bool slot_busy[2] = {false, false};
    int64_t host_seq = 0;              // async steps issued so far (step k uses slot k & 1)
    // event-free mode of the async host steps (out_host pinned): no event sits between two kernels of the compute stream, so
    // their programmatic launch edges survive.  Inputs: copies on s_h2d that end with a 4-byte copy of the step number
    // into d_h2d_flag[0] (kernels spin on it); completion: step_done_kernel stores the step number into d_h2d_flag[32];
    // result: s_d2h waits for that value (stream wait-value), copies the step's output to out_host and then writes the
    // step number into *h_done (stream write-value; pinned, the host polls it).
    typedef int (*memop32_fn)(void* stream, unsigned long long addr, unsigned int value, unsigned int flags);
    memop32_fn fn_wait32 = nullptr, fn_write32 = nullptr;
    int memops_state = 0;              // 0 not looked up yet, 1 available, -1 not available (event-chained mode only)
    unsigned long long h_done_dev = 0; // device address of *h_done
    bool direct_mode = false;
    int32_t direct_seq = 0;            // steps issued in this mode (step n uses slot n & 1)
    int32_t* d_h2d_flag = nullptr;
    int32_t* h_done = nullptr;         // pinned + mapped
    int32_t* h_seq_ring = nullptr;     // pinned: sources of the flag copies (a copy reads its source when it executes)
    const int32_t* cur_h2d_flag = nullptr;   // non-null only while such a step is being enqueued (append_impl passes it to the append kernel)
    int32_t cur_h2d_seq = 0;

    // per-call metadata staging: pinned host ring + matching device ring
    uint8_t* h_stage = nullptr;
    uint8_t* d_stage = nullptr;
    size_t slot_bytes = 0;
    cudaEvent_t ev[kStagingSlots / kStagingGroup]{};
    bool ev_used[kStagingSlots / kStagingGroup]{};
    bool group_dirty[kStagingSlots / kStagingGroup]{};   // slots of the group handed out since its last event
    cudaStream_t last_stream = nullptr;
    bool have_stream = false;
    int next_slot = 0;

    // profiling (metronome_pool_set_profiling): event pairs around the attention kernel
    bool profiling = false;            // mode 1: event brackets (launches are then not programmatic)
    std::vector<cudaEvent_t> prof_ev;  // start, stop, start, stop, ...
    size_t prof_used = 0;
    bool stamping = false;             // mode 2: %globaltimer stamps written by the attention kernels themselves
    unsigned long long* d_stamps = nullptr;    // [kStampSlots][2]
    std::vector<int32_t> stamp_kind;   // per used slot: 1 rows, 2 gqa decode, 3 chunk

    int32_t tune_split_tokens = 0, tune_family = 0, tune_gqa_dynamic = 0, tune_fused_step = 0;
    int tune_umma_half = 1;            // METRONOME_UMMA_HALF: 0 full-size chunk kernel only, 1 half-size kernel (two CTAs per SM) when every
                                       // chunk item of the launch has R <= 128 rows, 2 always (larger items as two CTAs of 128 rows)
    int tune_gqa_smclass = 0;          // GQA decode ranges sized by the SM's streaming speed (METRONOME_GQA_SMCLASS at pool creation)
    uint8_t* d_sm_class = nullptr;     // device copy of sm_class (256 bytes)
    bool tune_host_direct = true;      // false (METRONOME_HOST_STEP_EVENTS=1 at pool creation): async host steps always chain events
    int32_t n_sm = 148;
    int64_t n_launch = 0, n_append = 0, n_attend = 0;
    std::string cuda_err;
    StepParams step_params{};          // launch parameters of the fused step kernel (16 KB: not on the stack)
    uint8_t sm_class[kStepMaxSms] = {};   // 1: an SM that streams slower than the rest (calibrate_sm_speeds)
    int32_t n_slow_sms = 0;
    double slow_ratio = 1.0;           // speed of the slow SMs relative to the fast ones
};

namespace {

int cuda_fail(metronome_pool* p, cudaError_t e, const char* what) {
    if (p) p->cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
    return METRONOME_ERR_CUDA;
}
#define CU(call)                                                     \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) return cuda_fail(pool, e_, #call);    \
    } while (0)

bool valid_cfg(const metronome_pool_config_t* c) {
    if (!c) return false;
    const bool bk = c->flags & METRONOME_FLAG_BOOKKEEPING_ONLY;
    if (c->n_layers < 1 || c->n_q_heads < 1 || c->n_kv_heads < 1 || c->n_q_heads % c->n_kv_heads) return false;
    if (c->block_size < 1 || c->n_sinks < 0 || c->window < 1 || c->max_sessions < 1 || c->max_sessions > 65534)
        return false;
    if (c->max_new_tokens < 1 || c->n_blocks < 1 || c->max_session_len < 0) return false;
    if (!bk && (c->block_size != kBlockTokens || (c->head_dim != 64 && c->head_dim != 128))) return false;
    if ((c->flags & METRONOME_FLAG_UNBOUNDED) && c->max_session_len <= 0) return false;
    if (!(c->softmax_scale >= 0.f)) return false;
    return true;
}

// Stage `bytes` of per-call metadata: returns the host pointer to fill and the device pointer the
// kernels will read; commit_stage() enqueues the copy.
int acquire_stage(metronome_pool* pool, uint8_t** h, uint8_t** d, int* slot) {
    const int s = pool->next_slot;
    pool->next_slot = (s + 1) % kStagingSlots;
    if (s % kStagingGroup == 0) {
        // Entering a group.  (1) Close the group just left: one event on the stream of its last call
        // covers all its slots (calls on a pool are stream-ordered).  Doing it here, not after each
        // call, keeps events from sitting between an append kernel and its attention kernel (that
        // would break their programmatic launch edge) and also covers calls that returned an error.
        const int prev = ((s + kStagingSlots - kStagingGroup) % kStagingSlots) / kStagingGroup;
        if (pool->group_dirty[prev] && pool->have_stream) {
            CU(cudaEventRecord(pool->ev[prev], pool->last_stream));
            pool->ev_used[prev] = true;
            pool->group_dirty[prev] = false;
        }
        // (2) every call that used this group one lap ago must have been consumed by the GPU
        if (pool->ev_used[s / kStagingGroup]) CU(cudaEventSynchronize(pool->ev[s / kStagingGroup]));
    }
    pool->group_dirty[s / kStagingGroup] = true;
    *h = pool->h_stage + (size_t)s * pool->slot_bytes;
    *d = pool->d_stage + (size_t)s * pool->slot_bytes;
    *slot = s;
    return METRONOME_OK;
}
// after the last kernel / copy that reads the slot has been enqueued on `st`
int release_stage(metronome_pool* pool, int slot, cudaStream_t st) {
    (void)slot;
    pool->last_stream = st;
    pool->have_stream = true;
    return METRONOME_OK;
}
int commit_stage(metronome_pool* pool, int slot, size_t bytes, cudaStream_t st) {
    CU(cudaMemcpyAsync(pool->d_stage + (size_t)slot * pool->slot_bytes, pool->h_stage + (size_t)slot * pool->slot_bytes,
                       bytes, cudaMemcpyHostToDevice, st));
    return release_stage(pool, slot, st);
}

int check_batch(metronome_pool* pool, int32_t n_batch, const int32_t* sids, const int32_t* counts) {
    if (n_batch < 0 || n_batch > pool->cfg.max_sessions) return METRONOME_ERR_INVALID_ARG;
    if (n_batch > 0 && (!sids || !counts)) return METRONOME_ERR_INVALID_ARG;
    // duplicates first, then per-item checks (same precedence as the oracle)
    if (++pool->stamp_now == INT32_MAX) {
        std::fill(pool->stamp.begin(), pool->stamp.end(), 0);
        pool->stamp_now = 1;
    }
    for (int i = 0; i < n_batch; ++i) {
        const int32_t s = sids[i];
        if (s < 0 || s >= pool->cfg.max_sessions) continue;
        if (pool->stamp[s] == pool->stamp_now) return METRONOME_ERR_DUPLICATE_SESSION;
        pool->stamp[s] = pool->stamp_now;
    }
    for (int i = 0; i < n_batch; ++i) {
        const int32_t s = sids[i];
        if (s < 0 || s >= pool->cfg.max_sessions || !pool->sessions[s].open) return METRONOME_ERR_INVALID_SESSION;
        if (counts[i] < 0) return METRONOME_ERR_INVALID_ARG;
    }
    return METRONOME_OK;
}

int ensure_workspace(metronome_pool* pool, size_t slots) {
    if (slots <= pool->ws_slots) return METRONOME_OK;
    // cudaFree synchronises the device, so kernels still reading the old workspace are done
    if (pool->d_ws_acc) cudaFree(pool->d_ws_acc);
    if (pool->d_ws_ml) cudaFree(pool->d_ws_ml);
    pool->d_ws_acc = pool->d_ws_ml = nullptr;
    pool->ws_slots = 0;
    const size_t want = slots + slots / 4;
    CU(cudaMalloc(&pool->d_ws_acc, want * pool->cfg.head_dim * sizeof(float)));
    CU(cudaMalloc(&pool->d_ws_ml, want * 2 * sizeof(float)));
    pool->ws_slots = want;
    return METRONOME_OK;
}

// Which SMs stream slower than the rest, and by how much (the fused step kernel cuts its ranges accordingly).
// Three passes of step_calibrate_kernel over the pool's own KV storage; the first warms up.  An SM is "slow" when
// its mean time is more than 4 % above the median SM's.  Leaves "no slow SMs" behind on any failure.
void calibrate_sm_speeds(metronome_pool* pool) {
    const metronome_pool_config_t& c = pool->cfg;
    pool->n_slow_sms = 0;
    pool->slow_ratio = 1.0;
    memset(pool->sm_class, 0, sizeof(pool->sm_class));
    if (pool->n_sm > kStepMaxSms || c.n_blocks < 64) return;
    const int n_ctas = pool->n_sm * StepCfg<128, 1>::kCtasPerSm, n_warps = n_ctas * StepCfg<128, 1>::NWARP;
    unsigned long long* d_out = nullptr;
    if (cudaMalloc(&d_out, (size_t)n_warps * 2 * sizeof(unsigned long long)) != cudaSuccess) { cudaGetLastError(); return; }
    std::vector<unsigned long long> h((size_t)n_warps * 2);
    std::vector<double> t_sm(pool->n_sm, 0.0), n_sm_w(pool->n_sm, 0.0);
    bool ok = true;
    for (int pass = 0; pass < 3 && ok; ++pass) {
        if (c.head_dim == 128)
            step_calibrate_kernel<128><<<n_ctas, StepCfg<128, 1>::kThreads, StepCfg<128, 1>::kSmemBytes>>>(pool->d_kv, pool->L, c.n_blocks, 96, d_out);
        else
            step_calibrate_kernel<64><<<n_ctas, StepCfg<64, 1>::kThreads, StepCfg<64, 1>::kSmemBytes>>>(pool->d_kv, pool->L, c.n_blocks, 96, d_out);
        ok = cudaMemcpy(h.data(), d_out, h.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost) == cudaSuccess;
        if (!ok || pass == 0) continue;
        for (int w = 0; w < n_warps; ++w) {
            const unsigned long long sm = h[2 * (size_t)w];
            if (sm < (unsigned long long)pool->n_sm) { t_sm[sm] += (double)h[2 * (size_t)w + 1]; n_sm_w[sm] += 1.0; }
        }
    }
    cudaFree(d_out);
    if (!ok) { cudaGetLastError(); return; }
    std::vector<double> mean;
    for (int s = 0; s < pool->n_sm; ++s)
        if (n_sm_w[s] > 0) mean.push_back(t_sm[s] / n_sm_w[s]);
    if ((int)mean.size() < pool->n_sm) return;                 // (an SM that got no CTA: leave the ranges equal)
    std::vector<double> sorted = mean;
    std::sort(sorted.begin(), sorted.end());
    const double med = sorted[sorted.size() / 2];
    double t_fast = 0.0, t_slow = 0.0;
    int n_fast = 0, n_slow = 0;
    for (int s = 0; s < pool->n_sm; ++s) {
        const bool slow = mean[s] > 1.04 * med;
        pool->sm_class[s] = slow ? 1 : 0;
        if (slow) { t_slow += mean[s]; ++n_slow; } else { t_fast += mean[s]; ++n_fast; }
    }
    if (n_slow == 0 || n_fast == 0 || n_slow > pool->n_sm / 2) { memset(pool->sm_class, 0, sizeof(pool->sm_class)); return; }
    pool->n_slow_sms = n_slow;
    pool->slow_ratio = std::max(0.75, std::min(1.0, (t_fast / n_fast) / (t_slow / n_slow)));
}

// ---- row a8: the per-call work list, from the shadow counts ------------------------------------
// Kernel families (north_star: "Tensor cores are used only for the GQA-group x chunk QK^T/PV tiles,
// where the work really is a dense contraction"):
//   rows   CUDA-core row kernel: pure multi-head decode (G x q_len < 4 for every item), and the
//          general fallback
//   gqa    tensor-core stream-K decode kernel: items with R = G x q_len <= 16
//   chunk  tcgen05 / TMEM chunk-prefill kernel: items with 16 < R <= 256
// Fills items[0 .. plan.n_items) (host memory) and the plan; grows the split workspace if needed.
// `step_items` (may be null): also plan the fused decode step and leave its work list there.
int plan_attend(metronome_pool* pool, int32_t n_batch, const int32_t* sids, const int32_t* q_lens, AttendItem* items,
                AttendPlan& pl, std::vector<StepItem>* step_items = nullptr) {
    const metronome_pool_config_t& c = pool->cfg;
    pl = AttendPlan();
    int32_t max_q = 0;
    for (int i = 0; i < n_batch; ++i) {
        if (q_lens[i] > max_q) max_q = q_lens[i];
        pl.total_rows += q_lens[i];
    }
    int family = pool->tune_family;
    if (family == 0) family = (pool->G * max_q >= 4) ? 2 : 1;
    // (fp8 KV, NEXT row f4: the same three families -- fp8 rows in the row kernel, an fp8 tile in the GQA decode
    // kernel, attend_umma_fp8_kernel for the chunk class)
    if (family == 2 && !attend_umma_supported(pool->G, max_q))
        family = 1;
    pl.family = family;

    const int32_t W = pool->W_eff;
    int32_t* n_cls = pl.n_cls;
    if (family == 2)
        for (int i = 0; i < n_batch; ++i)
            if (q_lens[i] > 0) ++n_cls[pool->G * q_lens[i] > 16 ? 1 : 0];
    int32_t fill[2] = {0, n_cls[0]};
    int32_t row = 0, n_items = 0;
    for (int i = 0; i < n_batch; ++i) {
        if (q_lens[i] == 0) continue;
        const Session& s = pool->sessions[sids[i]];
        const int cls = (family == 2 && pool->G * q_lens[i] > 16) ? 1 : 0;
        AttendItem& it = items[family == 2 ? fill[cls]++ : n_items];
        ++n_items;
        memset(&it, 0, sizeof(it));
        it.sid = sids[i];
        it.len = (int32_t)s.len;
        it.q_len = q_lens[i];
        it.q_row_off = row;
        row += q_lens[i];
        const int32_t n_blk = (int32_t)((s.len + kBlockTokens - 1) / kBlockTokens);
        const int64_t t0 = s.len - q_lens[i];                      // oldest query of this call
        const int64_t wfirst = t0 - W + 1 > 0 ? t0 - W + 1 : 0;    // its oldest window key
        int32_t first_blk = (int32_t)(wfirst / kBlockTokens);
        if (first_blk < pool->n_sink) first_blk = pool->n_sink;
        it.n_sink_tiles = n_blk < pool->n_sink ? n_blk : pool->n_sink;
        it.first_blk = first_blk;
        it.n_tiles = it.n_sink_tiles + (n_blk > first_blk ? n_blk - first_blk : 0);
        // Early mode: the row kernel of step e may run next to the append kernels of steps e AND e-1 (the
        // one of step e-1 is only known to be past its own wait, not complete), so the first block it must
        // not touch before griddepcontrol.wait is the one holding the oldest row either of them wrote.
        const int64_t exposed = (s.last_epoch == pool->epoch && s.prev_epoch == pool->epoch - 1) ? s.prev_n : 0;
        const int64_t fresh_pos = s.len - std::max<int64_t>(q_lens[i], s.last_epoch == pool->epoch ? s.last_n : 0) - exposed;
        it.fresh_blk = (int32_t)((fresh_pos > 0 ? fresh_pos : 0) / kBlockTokens);
    }
    pl.n_items = n_items;
    if (family != 2) { n_cls[0] = n_items; n_cls[1] = 0; }
    // chunk class: longest first, so the hardware's in-order CTA dispatch packs the short ones last
    if (family == 2 && n_cls[1] > 1)
        std::stable_sort(items + n_cls[0], items + n_cls[0] + n_cls[1],
                         [](const AttendItem& a, const AttendItem& b) { return a.n_tiles > b.n_tiles; });

    // per-class prefix sums, split-KV plan
    int64_t cls_tiles[2] = {0, 0};
    for (int cls = 0; cls < 2; ++cls) {
        AttendItem* its = items + (cls == 0 ? 0 : n_cls[0]);
        const int32_t n = n_cls[cls];
        if (n == 0) continue;
        int64_t units = 0;           // tile visits of this class's CTAs if nothing were split
        for (int i = 0; i < n; ++i) {
            its[i].tile_off = (int32_t)cls_tiles[cls];
            its[i].class_row_off = pl.cls_rows[cls];
            cls_tiles[cls] += its[i].n_tiles;
            pl.cls_rows[cls] += its[i].q_len;
            if (its[i].q_len > pl.cls_max_q[cls]) pl.cls_max_q[cls] = its[i].q_len;
            units += (int64_t)its[i].n_tiles * (family == 2 ? c.n_kv_heads : c.n_q_heads * its[i].q_len);
        }
        if (family == 2 && cls == 0) {
            // stream-K: one wave of n_SM x 3 CTAs, equal static ranges (one per CTA); for long shares the
            // last 10 % of the flattened tile list is cut into small ranges claimed dynamically.
            const int64_t total_tiles = cls_tiles[0] * c.n_kv_heads;
            int64_t ctas = (int64_t)pool->n_sm * 3;
            const int64_t min_tiles = pool->tune_split_tokens > 0 ? (pool->tune_split_tokens + 15) / 16 : 8;
            if (ctas > (total_tiles + min_tiles - 1) / min_tiles) ctas = (total_tiles + min_tiles - 1) / min_tiles;
            if (pool->tune_split_tokens > 0) ctas = (total_tiles + min_tiles - 1) / min_tiles;
            if (ctas < 1) ctas = 1;
            // measured on B200: the dynamic tail pays (-2 % on config 5) only when a CTA's share is long
            // (>= 512 tiles = 4 MB); for shorter shares the restart of a claimed range costs more than the
            // imbalance it removes (configs 3 and 4: +3..7 %), so they stay fully static
            const bool dynamic = pool->tune_gqa_dynamic == 1 ||
                                 (pool->tune_gqa_dynamic == 0 && pool->tune_split_tokens <= 0 && (total_tiles + ctas - 1) / ctas >= 512);
            // ranges are cut in cost units: a pair's tiles + what starting a pair costs (make_gqa_plan), the latter
            // ~4 us of one CTA's share of the stream = METRONOME_GQA_BND_BYTES of K/V tiles
            const int32_t bnd = (int32_t)(METRONOME_GQA_BND_BYTES / pool->L.head_bytes);
            // a full one-wave launch on a GPU with a known set of slow SMs: long ranges for the CTAs that land on fast SMs,
            // ranges shorter by the measured speed ratio for those on slow SMs (each CTA claims from its SM's list)
            const bool smclass = pool->d_sm_class && pool->n_slow_sms > 0 && !dynamic && pool->tune_split_tokens <= 0 &&
                                 pool->tune_gqa_dynamic != 2 && ctas == (int64_t)pool->n_sm * 3;
            if (smclass)
                pl.gplan = make_gqa_plan_smclass(c.n_kv_heads, (cls_tiles[0] + (int64_t)bnd * n) * c.n_kv_heads,
                                                 3 * (pool->n_sm - pool->n_slow_sms), 3 * pool->n_slow_sms, pool->slow_ratio, bnd);
            else
            pl.gplan = make_gqa_plan(c.n_kv_heads, (cls_tiles[0] + (int64_t)bnd * n) * c.n_kv_heads, ctas, dynamic, bnd);
            GqaPlan& g = pl.gplan;
            pl.gqa_ctas = g.sm_mode ? g.n_total : g.n_static;     // (SM-class ranges: one CTA per range, long and short)
            if (g.n_total <= kMaxRangeItems) {
                int32_t* range_item = reinterpret_cast<int32_t*>(items + n_items);    // after ALL items
                int32_t ii = 0;
                for (int32_t r = 0; r < g.n_total; ++r) {
                    const int64_t lo = g.range_lo(r);
                    while (ii + 1 < n && ((int64_t)its[ii + 1].tile_off + (int64_t)bnd * (ii + 1)) * c.n_kv_heads <= lo) ++ii;
                    range_item[r] = ii;
                }
                pl.n_range_items = g.n_total;
            }
            for (int i = 0; i < n; ++i) {
                const int32_t pieces = g.max_pieces(its[i].n_tiles);
                its[i].n_splits = pieces;      // upper bound on the pieces of one (item, head) pair
                if (pieces > pl.max_splits) pl.max_splits = pieces;
            }
            // The fused decode step (step_gqa.cuh): one contiguous range per WARP of a single wave (CTA 0 of
            // that kernel does the bookkeeping), at least 8 tiles each; the work list in 16 bytes per item.
            if (step_items && n_cls[1] == 0 && n <= kStepMaxItems && c.n_kv_heads <= 255 && pool->tune_fused_step == 2 && !pool->fp8) {
                // One contiguous range per warp of a single wave (minus the bookkeeping CTA), at least 8 tiles each:
                // long ranges for the warps on fast SMs, ranges shorter by the measured speed ratio for those on slow SMs.
                const int32_t wps = step_workers_per_sm(pool->G * pl.cls_max_q[0]);
                const int64_t workers_max = (int64_t)pool->n_sm * wps - StepCfg<128, 1>::NWARP;
                GqaPlan& sg = pl.step_plan;
                sg = GqaPlan{};
                sg.n_kv_heads = c.n_kv_heads;
                sg.total_tiles = total_tiles;
                const int64_t share = (total_tiles + workers_max - 1) / workers_max;
                if (pool->tune_split_tokens > 0 || share < 16 || pool->n_slow_sms == 0) {
                    sg.q1 = sg.q2 = pool->tune_split_tokens > 0 ? min_tiles : std::max<int64_t>(8, share);
                    sg.n_static = sg.n_total = (int32_t)((total_tiles + sg.q1 - 1) / sg.q1);
                    sg.g1 = total_tiles;
                } else {
                    const int64_t n_short = (int64_t)pool->n_slow_sms * wps;
                    const int64_t n_long = workers_max - n_short;
                    sg.q1 = (int64_t)std::ceil((double)total_tiles / ((double)n_long + pool->slow_ratio * (double)n_short));
                    sg.q2 = std::max<int64_t>(1, (int64_t)std::ceil(pool->slow_ratio * (double)sg.q1));
                    sg.n_static = (int32_t)std::min<int64_t>(n_long, (total_tiles + sg.q1 - 1) / sg.q1);
                    sg.g1 = std::min<int64_t>(sg.q1 * sg.n_static, total_tiles);
                    sg.n_total = sg.n_static + (int32_t)((total_tiles - sg.g1 + sg.q2 - 1) / sg.q2);
                }
                const int64_t ctas = std::min<int64_t>(workers_max / StepCfg<128, 1>::NWARP,
                                                       ((int64_t)sg.n_total + StepCfg<128, 1>::NWARP - 1) / StepCfg<128, 1>::NWARP);
                pl.step_workers = (int32_t)(ctas * StepCfg<128, 1>::NWARP);
                step_items->resize(n);
                for (int i = 0; i < n; ++i) {
                    (*step_items)[i] = StepItem{its[i].sid | (its[i].q_len << 16), its[i].len, its[i].q_row_off, its[i].tile_off};
                    const int32_t pieces = (int32_t)((its[i].n_tiles + sg.q2 - 1) / sg.q2) + 2;
                    if (pieces > pl.max_splits) pl.max_splits = pieces;
                }
                pl.step_ok = true;
            }
            continue;
        }
        // segments sized for >= 2 waves of CTAs, each with a useful run of tiles
        const bool umma_cls = family == 2;
        const int64_t target_ctas = (int64_t)pool->n_sm * (umma_cls ? 4 : 16);
        int32_t tps = pool->tune_split_tokens > 0 ? (pool->tune_split_tokens + kBlockTokens - 1) / kBlockTokens
                                                  : (int32_t)((units + target_ctas - 1) / target_ctas);
        if (pool->tune_split_tokens <= 0 && tps < 8) tps = 8;
        if (umma_cls && pool->tune_split_tokens <= 0) {
            // tcgen05 chunk kernel, one CTA per SM: whole (item, head) pairs when they alone give
            // >= 3 CTAs per SM (no partials to merge), else whole 128-key stages, >= 4 per segment
            if ((int64_t)n * c.n_kv_heads >= 3 * (int64_t)pool->n_sm) tps = INT32_MAX / 2;
            else tps = std::max(32, (tps + 7) / 8 * 8);
        }
        if (tps < 1) tps = 1;
        for (int i = 0; i < n; ++i) {
            AttendItem& it = its[i];
            int32_t ns = (it.n_tiles + tps - 1) / tps;
            if (ns > kMaxSplits) ns = kMaxSplits;
            if (ns < 1) ns = 1;
            it.tiles_per_split = (it.n_tiles + ns - 1) / ns;
            it.n_splits = (it.n_tiles + it.tiles_per_split - 1) / it.tiles_per_split;
            it.split_off = pl.total_splits[cls];
            pl.total_splits[cls] += it.n_splits;
            if (it.n_splits > pl.max_splits) pl.max_splits = it.n_splits;
            if (it.n_splits > 1) pl.merge_cls[cls] = true;
        }
    }
    if (pl.max_splits > 1) {
        const int rc = ensure_workspace(pool, (size_t)pl.total_rows * c.n_q_heads * pl.max_splits);
        if (rc) return rc;
    }
    if (pool->inject_fault == 1) { pool->inject_fault = 0; return METRONOME_ERR_OUT_OF_MEMORY; }   // (as if the growth had failed)
    pl.valid = true;
    return METRONOME_OK;
}

__global__ void init_stamps_kernel(unsigned long long* stamps, int n) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        stamps[2 * i] = ~0ull;
        stamps[2 * i + 1] = 0ull;
    }
}

// profiling mode 2: the stamp slot of the next attention launch (null when off or the ring is full)
unsigned long long* next_stamp(metronome_pool* pool, int32_t kind) {
    if (!pool->stamping || !pool->d_stamps || pool->stamp_kind.size() >= (size_t)kStampSlots) return nullptr;
    pool->stamp_kind.push_back(kind);
    return pool->d_stamps + 2 * (pool->stamp_kind.size() - 1);
}

// Launches the attention kernels (rows a5 / a7) and the split merge (a6) of one attend_frame call.
// `pdl`: the work list was written by the append kernel that precedes this launch on the stream
// (cached plan): launch programmatically so the prologue overlaps that kernel's tail.
AttendParams make_attend_params(metronome_pool* pool, int32_t layer, const AttendPlan& pl, const void* q, void* out) {
    const metronome_pool_config_t& c = pool->cfg;
    AttendParams p{};
    p.table = pool->d_table;
    p.tbl_width = pool->tbl_width; p.n_sink = pool->n_sink; p.ring = pool->ring;
    p.q = (const __nv_bfloat16*)q;
    p.out = (__nv_bfloat16*)out;
    p.kv_layer = pool->d_kv + (int64_t)layer * pool->L.layer_bytes;
    p.L = pool->L;
    p.S = pool->unbounded ? 0 : c.n_sinks; p.W = pool->W_eff;
    p.scale_log2 = pool->scale * 1.4426950408889634f;
    p.Hq = c.n_q_heads; p.G = pool->G;
    p.ws_acc = pool->d_ws_acc; p.ws_ml = pool->d_ws_ml;
    p.max_splits = pl.max_splits;
    p.tickets = pool->d_tickets;
    p.gqa_ctr = pool->d_bk_flag + 2;              // same 16-byte allocation: [flag, -, claims, exits]
    p.sm_class = pool->d_sm_class;                // (null: off) its claim counters are gqa_ctr[4], [5] = d_bk_flag[6], [7]
    // measured on B200 (configs 2-4): letting the next append kernel launch early hides its host-memory
    // reads behind the attention kernel (-4..6 % per frame)
    p.pdl_early = 1;
    p.items_flag = pool->d_bk_flag + 1;
    p.items_epoch = -1;
    p.pastwait_flag = nullptr;
    return p;
}

int launch_attend(metronome_pool* pool, int32_t layer, const AttendPlan& pl, const AttendItem* d_items, const void* q,
                  void* out, cudaStream_t st, bool pdl) {
    const metronome_pool_config_t& c = pool->cfg;
    AttendParams p = make_attend_params(pool, layer, pl, q, out);
    p.range_item = pl.n_range_items ? reinterpret_cast<const int32_t*>(d_items + pl.n_items) : nullptr;
    // behind the fused append kernel of the same step the attention kernels may start early (they wait for
    // their work list, stream the untouched blocks, and wait for the append before the fresh ones); with the
    // poison fill or the profiling brackets in between, and on the general path, they wait at the top
    p.items_epoch = (pdl && pl.early && !pool->profiling) ? (int32_t)pl.epoch : -1;

    if (pool->profiling) {
        if (pool->prof_used + 2 > pool->prof_ev.size()) {
            cudaEvent_t a, b;
            CU(cudaEventCreate(&a));
            CU(cudaEventCreate(&b));
            pool->prof_ev.push_back(a);
            pool->prof_ev.push_back(b);
        }
        CU(cudaEventRecord(pool->prof_ev[pool->prof_used], st));
        pdl = false;
    }
    const bool publish = pl.family == 2 && pdl && !pool->profiling && !pool->poison;
    if (publish) { p.pastwait_flag = pool->d_bk_flag + 12; p.pastwait_epoch = (int32_t)pool->epoch; }
    if (pl.family == 2) {
        if (pl.n_cls[0] > 0) {
            p.items = d_items; p.n_items = pl.n_cls[0];
            p.stamp = next_stamp(pool, 2);
            CU(launch_attend_gqa(p, pl.gplan, c.head_dim, pl.gqa_ctas, st, pdl));
            ++pool->n_launch;
        }
        if (pl.n_cls[1] > 0) {
            p.items = d_items + pl.n_cls[0]; p.n_items = pl.n_cls[1];
            p.stamp = next_stamp(pool, 3);
            if (pool->fp8) CU(launch_attend_umma_fp8(p, c.head_dim, c.n_kv_heads, pl.total_splits[1], st, pdl));
            else {
                const int32_t R_max = pool->G * pl.cls_max_q[1];
                const bool half = pool->tune_umma_half >= 2 || (pool->tune_umma_half == 1 && R_max <= 128);
                CU(launch_attend_umma(p, c.head_dim, c.n_kv_heads, pl.total_splits[1], st, pdl, half, (R_max + 127) / 128));
            }
            ++pool->n_launch;
        }
    } else {
        p.items = d_items; p.n_items = pl.n_items;
        dim3 grid(c.n_q_heads, pl.total_splits[0], pl.cls_max_q[0]);
        p.stamp = next_stamp(pool, 1);
        if (pool->fp8) {
            if (c.head_dim == 128) CU(launch_kernel(attend_rows_kernel<128, true>, grid, dim3(128), 0, st, pdl, p));
            else CU(launch_kernel(attend_rows_kernel<64, true>, grid, dim3(128), 0, st, pdl, p));
        } else {
            if (c.head_dim == 128) CU(launch_kernel(attend_rows_kernel<128, false>, grid, dim3(128), 0, st, pdl, p));
            else CU(launch_kernel(attend_rows_kernel<64, false>, grid, dim3(128), 0, st, pdl, p));
        }
        ++pool->n_launch;
    }
    if (pool->profiling) {
        CU(cudaEventRecord(pool->prof_ev[pool->prof_used + 1], st));
        pool->prof_used += 2;
    }
    // ---- row a6: combine the split-KV partials (the GQA decode kernel merges its own pieces) ----
    for (int cls = (pl.family == 2 ? 1 : 0); cls < 2; ++cls) {
        if (!pl.merge_cls[cls] || (pl.family != 2 && cls == 1)) continue;
        p.items = d_items + (cls == 0 ? 0 : pl.n_cls[0]); p.n_items = pl.n_cls[cls];
        dim3 grid((unsigned)pl.cls_rows[cls], c.n_q_heads);
        if (c.head_dim == 128) CU(launch_kernel(merge_kernel<128>, grid, dim3(32), 0, st, !pool->profiling, p));
        else CU(launch_kernel(merge_kernel<64>, grid, dim3(16), 0, st, !pool->profiling, p));
        ++pool->n_launch;
    }
    if (publish) { pool->pastwait_launches = pool->n_launch; pool->pastwait_epoch = (int32_t)pool->epoch; }
    return METRONOME_OK;
}

// Device address of g_static_scratch on the CURRENT device (looked up on the first call made with that device
// current; cudaGetSymbolAddress allocates nothing).  Returns null and sets *err on failure.
constexpr int kMaxDevices = 64;
void* static_scratch_ptr(cudaError_t* err) {
    static void* ptr[kMaxDevices] = {};
    int dev = 0;
    *err = cudaGetDevice(&dev);
    if (*err != cudaSuccess) return nullptr;
    if (dev < 0 || dev >= kMaxDevices) { *err = cudaErrorInvalidDevice; return nullptr; }
    void* p = __atomic_load_n(&ptr[dev], __ATOMIC_ACQUIRE);
    if (!p) {
        *err = cudaGetSymbolAddress(&p, g_static_scratch);
        if (*err != cudaSuccess) return nullptr;
        __atomic_store_n(&ptr[dev], p, __ATOMIC_RELEASE);      // (two racing first calls store the same address)
    }
    return p;
}

// Row a8 for metronome_attend_frame_static: the work list of the split-KV row kernel (one class, every item),
// with the same item fields and the same segment rule as plan_attend's row-kernel branch (segments of >= 8 tiles,
// sized for >= 16 CTAs per SM, at most kMaxSplits per item) -- but no workspace growth: the caller checks the
// plan against the fixed scratch.  Writes items[0 .. n_items) (the pool's pinned staging slot: no host allocation).
void plan_rows_static(metronome_pool* pool, int32_t n_batch, const int32_t* sids, const int32_t* q_lens, AttendItem* items,
                      AttendPlan& pl) {
    const metronome_pool_config_t& c = pool->cfg;
    pl = AttendPlan();
    pl.family = 1;
    const int32_t W = pool->W_eff;
    int32_t row = 0, n_items = 0;
    int64_t units = 0, tiles = 0;
    for (int i = 0; i < n_batch; ++i) {
        if (q_lens[i] == 0) continue;
        const Session& s = pool->sessions[sids[i]];
        AttendItem& it = items[n_items++];
        memset(&it, 0, sizeof(it));
        it.sid = sids[i];
        it.len = (int32_t)s.len;
        it.q_len = q_lens[i];
        it.q_row_off = row;
        it.class_row_off = row;
        row += q_lens[i];
        const int32_t n_blk = (int32_t)((s.len + kBlockTokens - 1) / kBlockTokens);
        const int64_t t0 = s.len - q_lens[i];                      // oldest query of this call
        const int64_t wfirst = t0 - W + 1 > 0 ? t0 - W + 1 : 0;    // its oldest window key
        int32_t first_blk = (int32_t)(wfirst / kBlockTokens);
        if (first_blk < pool->n_sink) first_blk = pool->n_sink;
        it.n_sink_tiles = n_blk < pool->n_sink ? n_blk : pool->n_sink;
        it.first_blk = first_blk;
        it.n_tiles = it.n_sink_tiles + (n_blk > first_blk ? n_blk - first_blk : 0);
        it.fresh_blk = 0;                                          // (plain launch: the kernel waits at the top)
        it.tile_off = (int32_t)tiles;
        tiles += it.n_tiles;
        units += (int64_t)it.n_tiles * c.n_q_heads * it.q_len;
        if (it.q_len > pl.cls_max_q[0]) pl.cls_max_q[0] = it.q_len;
    }
    pl.n_items = n_items;
    pl.n_cls[0] = n_items;
    pl.total_rows = row;
    pl.cls_rows[0] = row;
    const int64_t target_ctas = (int64_t)pool->n_sm * 16;
    int32_t tps = pool->tune_split_tokens > 0 ? (pool->tune_split_tokens + kBlockTokens - 1) / kBlockTokens
                                              : (int32_t)((units + target_ctas - 1) / target_ctas);
    if (pool->tune_split_tokens <= 0 && tps < 8) tps = 8;
    if (tps < 1) tps = 1;
    for (int i = 0; i < n_items; ++i) {
        AttendItem& it = items[i];
        int32_t ns = (it.n_tiles + tps - 1) / tps;
        if (ns > kMaxSplits) ns = kMaxSplits;
        if (ns < 1) ns = 1;
        it.tiles_per_split = (it.n_tiles + ns - 1) / ns;
        it.n_splits = (it.n_tiles + it.tiles_per_split - 1) / it.tiles_per_split;
        if (it.n_splits < 1) it.n_splits = 1;
        it.split_off = pl.total_splits[0];
        pl.total_splits[0] += it.n_splits;
        if (it.n_splits > pl.max_splits) pl.max_splits = it.n_splits;
        if (it.n_splits > 1) pl.merge_cls[0] = true;
    }
    if (pl.max_splits < 1) pl.max_splits = 1;
    pl.valid = true;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
extern "C" {

int metronome_abi_version(void) { return METRONOME_ABI_VERSION; }

const char* metronome_strerror(int status) {
    switch (status) {
        case METRONOME_OK: return "OK";
        case METRONOME_ERR_INVALID_ARG: return "INVALID_ARG";
        case METRONOME_ERR_INVALID_SESSION: return "INVALID_SESSION";
        case METRONOME_ERR_DUPLICATE_SESSION: return "DUPLICATE_SESSION";
        case METRONOME_ERR_SESSIONS_FULL: return "SESSIONS_FULL";
        case METRONOME_ERR_POOL_EXHAUSTED: return "POOL_EXHAUSTED";
        case METRONOME_ERR_CHUNK_TOO_LARGE: return "CHUNK_TOO_LARGE";
        case METRONOME_ERR_QLEN_EXCEEDS_LAST_APPEND: return "QLEN_EXCEEDS_LAST_APPEND";
        case METRONOME_ERR_LAYER_SEQUENCE: return "LAYER_SEQUENCE";
        case METRONOME_ERR_LEN_OVERFLOW: return "LEN_OVERFLOW";
        case METRONOME_ERR_CUDA: return "CUDA";
        case METRONOME_ERR_UNSUPPORTED: return "UNSUPPORTED";
        case METRONOME_ERR_OUT_OF_MEMORY: return "OUT_OF_MEMORY";
        case METRONOME_ERR_SCRATCH_EXCEEDED: return "SCRATCH_EXCEEDED";
        default: return "UNKNOWN";
    }
}

const char* metronome_last_cuda_error(metronome_pool_t* pool) { return pool ? pool->cuda_err.c_str() : ""; }

size_t metronome_kv_storage_bytes(const metronome_pool_config_t* c) {
    if (!valid_cfg(c) || (c->flags & METRONOME_FLAG_BOOKKEEPING_ONLY)) return 0;
    return (size_t)c->n_layers * make_layout(c->head_dim, c->n_kv_heads, c->n_blocks, c->flags & METRONOME_FLAG_KV_FP8).layer_bytes;
}

int32_t metronome_max_blocks_per_session(int32_t S, int32_t W, int32_t B, int32_t max_new_tokens) {
    if (S < 0 || W < 1 || B < 1 || max_new_tokens < 1) return -1;
    const int64_t v = (int64_t)((S + B - 1) / B) + ((int64_t)W + max_new_tokens - 1) / B + 2;
    return v > INT32_MAX ? -1 : (int32_t)v;
}

int metronome_pool_create(const metronome_pool_config_t* cfg, metronome_pool_t** out) {
    if (!out) return METRONOME_ERR_INVALID_ARG;
    *out = nullptr;
    if (!valid_cfg(cfg)) return METRONOME_ERR_INVALID_ARG;
    metronome_pool* pool = new (std::nothrow) metronome_pool();
    if (!pool) return METRONOME_ERR_OUT_OF_MEMORY;
    pool->cfg = *cfg;
    const metronome_pool_config_t& c = pool->cfg;
    pool->bookkeeping_only = c.flags & METRONOME_FLAG_BOOKKEEPING_ONLY;
    pool->poison = c.flags & METRONOME_FLAG_POISON_ON_FREE;
    pool->unbounded = c.flags & METRONOME_FLAG_UNBOUNDED;
    if (pool->cfg.max_session_len == 0) pool->cfg.max_session_len = (int64_t)INT32_MAX - c.max_new_tokens;
    const int32_t B = c.block_size;
    pool->n_sink = (c.n_sinks + B - 1) / B;
    if (pool->unbounded) {
        const int64_t blocks = (pool->cfg.max_session_len + B - 1) / B + 1;
        if (blocks > (1 << 24)) { delete pool; return METRONOME_ERR_INVALID_ARG; }
        pool->tbl_width = (int32_t)blocks;
        pool->ring = pool->tbl_width;        // never wraps: slots are linear
        pool->n_sink = 0;                    // nothing is pinned because nothing is freed
        pool->W_eff = INT32_MAX / 2;
    } else {
        pool->tbl_width = metronome_max_blocks_per_session(c.n_sinks, c.window, B, c.max_new_tokens);
        if (pool->tbl_width < 0) { delete pool; return METRONOME_ERR_INVALID_ARG; }
        pool->ring = pool->tbl_width - pool->n_sink;
        pool->W_eff = c.window;
    }
    pool->G = c.n_q_heads / c.n_kv_heads;
    pool->scale = c.softmax_scale > 0.f ? c.softmax_scale : 1.0f / sqrtf((float)(c.head_dim > 0 ? c.head_dim : 1));
    pool->sessions.assign(c.max_sessions, Session());
    pool->stamp.assign(c.max_sessions, 0);
    pool->layer_epoch.assign(c.n_layers, 0);
    pool->n_free = c.n_blocks;

    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&pool->n_sm, cudaDevAttrMultiProcessorCount, dev);
    auto fail = [&](int code, cudaError_t ce, const char* what) {
        if (code == METRONOME_ERR_CUDA) cuda_fail(pool, ce, what);
        metronome_pool_destroy(pool);
        return code;
    };
    if (e != cudaSuccess) return fail(METRONOME_ERR_CUDA, e, "cudaGetDevice");
    e = cudaMalloc(&pool->d_table, (size_t)c.max_sessions * pool->tbl_width * sizeof(int32_t));
    if (e != cudaSuccess) return fail(METRONOME_ERR_OUT_OF_MEMORY, e, "cudaMalloc table");
    e = cudaMalloc(&pool->d_free, (size_t)c.n_blocks * sizeof(int32_t));
    if (e != cudaSuccess) return fail(METRONOME_ERR_OUT_OF_MEMORY, e, "cudaMalloc free stack");
    cudaMemset(pool->d_table, 0xFF, (size_t)c.max_sessions * pool->tbl_width * sizeof(int32_t));
    if (!pool->bookkeeping_only) {
        pool->fp8 = c.flags & METRONOME_FLAG_KV_FP8;
        pool->L = make_layout(c.head_dim, c.n_kv_heads, c.n_blocks, pool->fp8);
        const size_t need = metronome_kv_storage_bytes(&pool->cfg);
        if (c.kv_storage) {
            if (c.kv_storage_bytes < need || ((uintptr_t)c.kv_storage & 127)) return fail(METRONOME_ERR_INVALID_ARG, e, "");
            pool->d_kv = (uint8_t*)c.kv_storage;
        } else {
            e = cudaMalloc(&pool->d_kv, need);
            if (e != cudaSuccess) return fail(METRONOME_ERR_OUT_OF_MEMORY, e, "cudaMalloc kv storage");
            pool->own_kv = true;
        }
        if (pool->poison) fill_nan_kernel<<<1184, 256>>>((uint4*)pool->d_kv, (int64_t)(need / 16));
    }
    pool->slot_bytes = (size_t)c.max_sessions * (sizeof(AppendItem) + sizeof(AttendItem)) + kMaxRangeItems * sizeof(int32_t) + 16;
    { const char* ev = getenv("METRONOME_HOST_STEP_EVENTS"); pool->tune_host_direct = !(ev && ev[0] == '1'); }
    { const char* ev = getenv("METRONOME_UMMA_HALF"); pool->tune_umma_half = ev ? atoi(ev) : kUmmaHalfDefault; }
    { const char* ev = getenv("METRONOME_GQA_SMCLASS"); pool->tune_gqa_smclass = ev ? atoi(ev) : kGqaSmClassDefault; }
    e = cudaMalloc(&pool->d_tickets, (size_t)c.max_sessions * c.n_kv_heads * sizeof(int32_t));
    if (e != cudaSuccess) return fail(METRONOME_ERR_OUT_OF_MEMORY, e, "cudaMalloc tickets");
    cudaMemset(pool->d_tickets, 0, (size_t)c.max_sessions * c.n_kv_heads * sizeof(int32_t));
    e = cudaMalloc(&pool->d_bk_flag, 64);
    if (e != cudaSuccess) return fail(METRONOME_ERR_OUT_OF_MEMORY, e, "cudaMalloc flag");
    cudaMemset(pool->d_bk_flag, 0, 64);
    pool->attend_buf_bytes = (((size_t)c.max_sessions * sizeof(AttendItem) + kMaxRangeItems * sizeof(int32_t) + 16) + 255) & ~(size_t)255;
    e = cudaMalloc(&pool->d_attend_items, 2 * pool->attend_buf_bytes);      // two buffers, by epoch parity
    if (e != cudaSuccess) return fail(METRONOME_ERR_OUT_OF_MEMORY, e, "cudaMalloc attend items");
    e = cudaMallocHost(&pool->h_stage, pool->slot_bytes * kStagingSlots);
    if (e != cudaSuccess) return fail(METRONOME_ERR_OUT_OF_MEMORY, e, "cudaMallocHost staging");
    e = cudaMalloc(&pool->d_stage, pool->slot_bytes * kStagingSlots);
    if (e != cudaSuccess) return fail(METRONOME_ERR_OUT_OF_MEMORY, e, "cudaMalloc staging");
    for (int i = 0; i < kStagingSlots / kStagingGroup; ++i) {
        e = cudaEventCreateWithFlags(&pool->ev[i], cudaEventDisableTiming);
        if (e != cudaSuccess) return fail(METRONOME_ERR_CUDA, e, "cudaEventCreate");
    }
    init_free_stack_kernel<<<(c.n_blocks + 255) / 256, 256>>>(pool->d_free, c.n_blocks);
    e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return fail(METRONOME_ERR_CUDA, e, "pool init kernels");
    e = configure_attend_mma_kernels();
    if (e == cudaSuccess) e = configure_attend_umma_kernels();
    if (e == cudaSuccess) e = configure_attend_umma_fp8_kernels();
    if (e == cudaSuccess) e = configure_step_kernels();
    if (e != cudaSuccess) return fail(METRONOME_ERR_CUDA, e, "cudaFuncSetAttribute");

    // GQA decode ranges sized by the SMs' streaming speeds: classify the SMs once (a few ms), keep the table on the device
    if (pool->tune_gqa_smclass && !pool->bookkeeping_only && pool->G > 1) {
        calibrate_sm_speeds(pool);
        if (pool->n_slow_sms > 0) {
            e = cudaMalloc(&pool->d_sm_class, sizeof(pool->sm_class));
            if (e == cudaSuccess) e = cudaMemcpy(pool->d_sm_class, pool->sm_class, sizeof(pool->sm_class), cudaMemcpyHostToDevice);
            if (e != cudaSuccess) return fail(METRONOME_ERR_CUDA, e, "SM class table");
        }
    }

    *out = pool;
    return METRONOME_OK;
}

int metronome_pool_destroy(metronome_pool_t* pool) {
    if (!pool) return METRONOME_OK;
    cudaDeviceSynchronize();
    if (pool->d_table) cudaFree(pool->d_table);
    if (pool->d_tickets) cudaFree(pool->d_tickets);
    if (pool->d_bk_flag) cudaFree(pool->d_bk_flag);
    if (pool->d_stamps) cudaFree(pool->d_stamps);
    if (pool->d_attend_items) cudaFree(pool->d_attend_items);
    if (pool->d_free) cudaFree(pool->d_free);
    if (pool->own_kv && pool->d_kv) cudaFree(pool->d_kv);
    if (pool->d_ws_acc) cudaFree(pool->d_ws_acc);
    if (pool->d_ws_ml) cudaFree(pool->d_ws_ml);
    if (pool->d_io) cudaFree(pool->d_io);
    if (pool->d_io2[2]) cudaFree(pool->d_io2[2]);
    for (int b = 0; b < 2; ++b) {
        if (pool->d_io2[b]) cudaFree(pool->d_io2[b]);
        if (pool->ev_h2d[b]) cudaEventDestroy(pool->ev_h2d[b]);
        if (pool->ev_comp[b]) cudaEventDestroy(pool->ev_comp[b]);
        if (pool->ev_d2h[b]) cudaEventDestroy(pool->ev_d2h[b]);
    }
    if (pool->d_sm_class) cudaFree(pool->d_sm_class);
    if (pool->d_h2d_flag) cudaFree(pool->d_h2d_flag);
    if (pool->h_done) cudaFreeHost(pool->h_done);
    if (pool->h_seq_ring) cudaFreeHost(pool->h_seq_ring);
    if (pool->s_h2d) cudaStreamDestroy(pool->s_h2d);
    if (pool->s_d2h) cudaStreamDestroy(pool->s_d2h);
    if (pool->h_stage) cudaFreeHost(pool->h_stage);
    if (pool->d_stage) cudaFree(pool->d_stage);
    for (int i = 0; i < kStagingSlots / kStagingGroup; ++i)
        if (pool->ev[i]) cudaEventDestroy(pool->ev[i]);
    for (cudaEvent_t e : pool->prof_ev) cudaEventDestroy(e);
    delete pool;
    return METRONOME_OK;
}

int metronome_session_open(metronome_pool_t* pool, int32_t* sid_out) {
    if (!pool || !sid_out) return METRONOME_ERR_INVALID_ARG;
    if (pool->n_open >= pool->cfg.max_sessions) return METRONOME_ERR_SESSIONS_FULL;
    for (int32_t s = 0; s < pool->cfg.max_sessions; ++s) {
        if (!pool->sessions[s].open) {           // lowest free slot (reading R6)
            Session& ss = pool->sessions[s];
            ss.open = true; ss.len = 0; ss.first_live = pool->n_sink; ss.last_n = 0;
            ++pool->n_open;
            *sid_out = s;
            return METRONOME_OK;
        }
    }
    return METRONOME_ERR_SESSIONS_FULL;
}

int metronome_session_close(metronome_pool_t* pool, int32_t sid, void* cuda_stream) {
    if (!pool) return METRONOME_ERR_INVALID_ARG;
    if (sid < 0 || sid >= pool->cfg.max_sessions || !pool->sessions[sid].open) return METRONOME_ERR_INVALID_SESSION;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Session& s = pool->sessions[sid];
    const int32_t B = pool->cfg.block_size;
    const int32_t n_blk = (int32_t)((s.len + B - 1) / B);
    const int32_t n_sink_res = n_blk < pool->n_sink ? n_blk : pool->n_sink;
    const int32_t n_win = n_blk > s.first_live ? n_blk - s.first_live : 0;
    const int32_t cnt = n_sink_res + n_win;
    if (cnt > 0) {
        close_session_kernel<<<1, 256, 0, st>>>(pool->d_table + (int64_t)sid * pool->tbl_width, pool->n_sink, pool->ring,
                                                n_sink_res, s.first_live, n_blk, pool->d_free, pool->n_free);
        ++pool->n_launch;
        CU(cudaGetLastError());
        if (pool->poison && !pool->bookkeeping_only) {
            poison_blocks_kernel<<<dim3(cnt, pool->cfg.n_layers), 256, 0, st>>>(pool->d_free, pool->n_free, pool->d_kv,
                                                                               pool->L.block_bytes, pool->L.layer_bytes);
            ++pool->n_launch;
            CU(cudaGetLastError());
        }
    }
    pool->n_free += cnt;
    s = Session();
    --pool->n_open;
    // a closed session can no longer be part of a layer > 0 replay
    pool->last_sids.clear(); pool->last_n_new.clear();
    return METRONOME_OK;
}

}  // extern "C"

namespace {

// metronome_append_kv, and the append half of metronome_append_attend.  `q` / `out` non-null: the caller
// will attend exactly this batch next (q_lens = n_new); when the step can run as ONE launch
// (step_gqa.cuh) it is launched here and *fused is set, else only the append is done.
int append_impl(metronome_pool_t* pool, int32_t layer, int32_t n_batch, const int32_t* sids, const int32_t* n_new,
                const void* k_new, const void* v_new, void* cuda_stream, const void* q, void* out, bool* fused) {
    if (!pool || layer < 0 || layer >= pool->cfg.n_layers) return METRONOME_ERR_INVALID_ARG;
    int rc = check_batch(pool, n_batch, sids, n_new);
    if (rc) return rc;
    const metronome_pool_config_t& c = pool->cfg;
    const int32_t B = c.block_size;
    int64_t total_new = 0;
    int32_t max_n = 0;
    for (int i = 0; i < n_batch; ++i) {
        if (n_new[i] > c.max_new_tokens) return METRONOME_ERR_CHUNK_TOO_LARGE;
        if (pool->sessions[sids[i]].len + n_new[i] > c.max_session_len) return METRONOME_ERR_LEN_OVERFLOW;
        total_new += n_new[i];
        if (n_new[i] > max_n) max_n = n_new[i];
    }
    if (pool->bookkeeping_only ? (k_new || v_new) : (total_new > 0 && (!k_new || !v_new)))
        return METRONOME_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    if (layer > 0) {
        // must repeat layer 0's batch of this step, once (reading R16)
        if (pool->epoch == 0 || pool->layer_epoch[layer] >= pool->epoch || (int32_t)pool->last_sids.size() != n_batch ||
            (n_batch && (memcmp(pool->last_sids.data(), sids, n_batch * sizeof(int32_t)) ||
                         memcmp(pool->last_n_new.data(), n_new, n_batch * sizeof(int32_t)))))
            return METRONOME_ERR_LAYER_SEQUENCE;
    }

    uint8_t *h = nullptr, *d = nullptr;
    int slot = 0;
    AppendItem* items = nullptr;
    int32_t total_freed = 0, total_alloc = 0;
    if (n_batch > 0) {
        rc = acquire_stage(pool, &h, &d, &slot);
        if (rc) return rc;
        items = reinterpret_cast<AppendItem*>(h);
        int32_t row = 0;
        for (int i = 0; i < n_batch; ++i) {
            const Session& s = pool->sessions[sids[i]];
            AppendItem& it = items[i];
            memset(&it, 0, sizeof(it));
            it.sid = sids[i];
            it.n_new = n_new[i];
            it.row_off = row;
            row += n_new[i];
            if (layer == 0) {
                const int64_t L0 = s.len, L1 = s.len + n_new[i];
                it.len0 = (int32_t)L0;
                int64_t new_first = s.first_live;
                if (!pool->unbounded) {
                    // block b is entirely behind the window of position L0 iff (b+1)*B <= L0-W+1 (L256);
                    // the first ceil(S/B) blocks are pinned (L258)
                    const int64_t behind = L0 - c.window + 1 > 0 ? (L0 - c.window + 1) / B : 0;
                    if (behind > new_first) new_first = behind;
                    if (pool->n_sink > new_first) new_first = pool->n_sink;
                }
                it.free_lo = s.first_live;
                it.n_freed = (int32_t)(new_first - s.first_live);
                it.free_off = total_freed;
                it.alloc_lo = (int32_t)((L0 + B - 1) / B);
                it.n_alloc = (int32_t)((L1 + B - 1) / B) - it.alloc_lo;
                it.alloc_off = total_alloc;
                total_freed += it.n_freed;
                total_alloc += it.n_alloc;
            } else {
                it.len0 = (int32_t)(s.len - n_new[i]);
            }
        }
    }
    const AppendItem* h_items = reinterpret_cast<const AppendItem*>(h);     // pinned host memory, read by the kernels
    AttendItem* h_attend = reinterpret_cast<AttendItem*>(h + (size_t)n_batch * sizeof(AppendItem));
    bool fused_bookkeeping = false, unfused_bookkeeping = false, have_plan = false;
    const int32_t n_free0 = pool->n_free;
    // Everything that can fail comes BEFORE the shadow counts are final ("no state change on error"):
    // the counts are committed tentatively (the work list of this step is planned from the lengths
    // AFTER the append), and rolled back if the plan, the workspace growth or the first launch fails.
    std::vector<Session>& undo_sessions = pool->undo_sessions;
    undo_sessions.clear();
    const int64_t undo_epoch = pool->epoch, undo_layer_epoch = pool->layer_epoch[layer];
    const int32_t undo_last_early = pool->last_early_epoch;
    std::vector<int32_t>&undo_sids = pool->undo_sids, &undo_n_new = pool->undo_n_new;
    const AttendPlan undo_plan = pool->cached_plan;
    auto rollback = [&]() {
        if (layer == 0) {
            for (int i = 0; i < n_batch; ++i) pool->sessions[sids[i]] = undo_sessions[i];
            pool->n_free = n_free0;
            pool->last_sids.swap(undo_sids);
            pool->last_n_new.swap(undo_n_new);
        }
        pool->epoch = undo_epoch;
        pool->layer_epoch[layer] = undo_layer_epoch;
        pool->last_early_epoch = undo_last_early;
        pool->cached_plan = undo_plan;
    };
    if (layer == 0) {
        if (pool->n_free + total_freed < total_alloc) return METRONOME_ERR_POOL_EXHAUSTED;  // nothing changed
        if (n_batch > 0 && total_freed + total_alloc > 0) {
            // unfused in poison / bookkeeping-only mode: the poison fill has to sit between the frees and
            // the K/V writes
            if (pool->poison || pool->bookkeeping_only) unfused_bookkeeping = true;
            else fused_bookkeeping = true;
        }
        // tentative commit of the shadow counts
        undo_sessions.reserve(n_batch);
        for (int i = 0; i < n_batch; ++i) undo_sessions.push_back(pool->sessions[sids[i]]);
        undo_sids = pool->last_sids;
        undo_n_new = pool->last_n_new;
        ++pool->epoch;
        for (int i = 0; i < n_batch; ++i) {
            Session& s = pool->sessions[sids[i]];
            s.first_live += items[i].n_freed;
            s.len += n_new[i];
            s.prev_n = s.last_n; s.prev_epoch = s.last_epoch;
            s.last_n = n_new[i]; s.last_epoch = pool->epoch;
        }
        pool->n_free += total_freed - total_alloc;
        pool->layer_epoch[0] = pool->epoch;
        pool->last_sids.assign(sids, sids + n_batch);
        pool->last_n_new.assign(n_new, n_new + n_batch);
        // row a8 ahead of time: the work list of attend_frame(q_lens = n_new) for this step; the
        // append kernel carries it to the device
        pool->cached_plan.valid = false;
        if (!pool->bookkeeping_only && total_new > 0) {
            rc = plan_attend(pool, n_batch, sids, n_new, h_attend, pool->cached_plan, &pool->step_items);
            if (rc) { rollback(); return rc; }
            pool->cached_plan.epoch = pool->epoch;
            have_plan = true;
        }
        if (unfused_bookkeeping) {
            bookkeeping_kernel<<<1, 512, 0, st>>>(h_items, n_batch, pool->d_table, pool->tbl_width, pool->n_sink,
                                                  pool->ring, pool->d_free, n_free0, total_freed);
            const cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) { rollback(); return cuda_fail(pool, e, "bookkeeping_kernel"); }
            ++pool->n_launch;
            // (a failure from here on follows a kernel that is already enqueued: it is reported, and the
            // CUDA context is in a sticky error state anyway)
            if (pool->poison && !pool->bookkeeping_only && total_freed > 0) {
                poison_blocks_kernel<<<dim3(total_freed, c.n_layers), 256, 0, st>>>(pool->d_free, n_free0, pool->d_kv,
                                                                                   pool->L.block_bytes, pool->L.layer_bytes);
                ++pool->n_launch;
                CU(cudaGetLastError());
            }
        }
    } else {
        pool->layer_epoch[layer] = pool->epoch;
    }
    if (n_batch > 0 && (fused_bookkeeping || (!pool->bookkeeping_only && total_new > 0))) {
        AppendParams a{};
        a.items = h_items;
        a.n_items = n_batch;
        a.table = pool->d_table;
        a.tbl_width = pool->tbl_width; a.n_sink = pool->n_sink; a.ring = pool->ring;
        a.free_stack = pool->d_free;
        a.n_free0 = n_free0; a.total_freed = total_freed;
        a.do_bookkeeping = fused_bookkeeping ? 1 : 0;
        a.bk_flag = pool->d_bk_flag;
        a.epoch = (int32_t)pool->epoch;
        // early mode (measured on B200): only for the row kernel (pure multi-head decode, config 2: -5 %);
        // with the GQA decode / chunk kernels resident next to the append kernel configs 4 and 5 lose 20 %
        const bool early = have_plan && pool->cached_plan.family == 1 && !pool->poison && !pool->profiling;
        pool->cached_plan.early = early;
        a.pdl_early = early ? 1 : 0;
        a.items_flag = pool->d_bk_flag + 1;
        a.gate_epoch = pool->last_early_epoch;
        pool->last_early_epoch = early ? (int32_t)pool->epoch : 0;
        // Early bookkeeping (tensor-core family): when the kernel right before this one on the stream is the previous
        // step's attention kernel (nothing launched since, and it publishes when it is past its wait), rows a2 / a3
        // run under its tail.  Not when a block allocated now would take the table slot of a block that kernel may
        // still look up (a block freed in THIS call can hold the oldest key of the previous step's window).
        bool early_bk = layer == 0 && have_plan && !early && pool->cached_plan.family == 2 && !pool->poison && !pool->profiling &&
                        pool->pastwait_launches == pool->n_launch && pool->pastwait_epoch == (int32_t)pool->epoch - 1;
        for (int i = 0; early_bk && i < n_batch; ++i)
            if (items[i].n_alloc > 0 && items[i].alloc_lo + items[i].n_alloc - 1 - pool->ring >= undo_sessions[i].first_live) early_bk = false;
        a.early_bk = early_bk ? 1 : 0;
        a.pastwait_flag = pool->d_bk_flag + 12;
        a.pastwait_gate = pool->pastwait_epoch;
        if (have_plan) {
            a.attend_src = reinterpret_cast<const uint4*>(h_attend);
            a.attend_dst = reinterpret_cast<uint4*>(reinterpret_cast<uint8_t*>(pool->d_attend_items) + (pool->epoch & 1) * pool->attend_buf_bytes);
            a.attend_n16 = (int32_t)((pool->cached_plan.n_items * sizeof(AttendItem) + pool->cached_plan.n_range_items * sizeof(int32_t) + 15) / 16);
        }
        a.k_new = (const uint4*)k_new; a.v_new = (const uint4*)v_new;
        a.kv_layer = pool->bookkeeping_only ? nullptr : pool->d_kv + (int64_t)layer * pool->L.layer_bytes;
        a.L = pool->L;
        a.h2d_flag = pool->cur_h2d_flag; a.h2d_seq = pool->cur_h2d_seq;
        const int32_t chunks = max_n * c.n_kv_heads * (c.head_dim / 8);
        dim3 grid(std::max(1, (chunks + 255) / 256), n_batch + 1);      // (n_batch <= max_sessions <= 65534)
        const size_t smem = (fused_bookkeeping && n_batch <= kAppendSmemItems) ? (size_t)n_batch * sizeof(AppendItem) : 0;
        cudaError_t e = cudaSuccess;
        const AttendPlan& cp = pool->cached_plan;
        const bool fuse = q && out && fused && cp.valid && cp.epoch == pool->epoch && cp.step_ok && !unfused_bookkeeping &&
                          !pool->poison && !pool->profiling && n_batch <= kAppendSmemItems;
        if (pool->inject_fault == 2) { pool->inject_fault = 0; e = cudaErrorLaunchFailure; }
        else if (fuse) {
            // rows a2-a6 of this step in ONE launch: CTA 0 does the bookkeeping, every other warp streams
            // its share of the (item, head, tile) list and writes the new rows on the way
            StepParams* sp = &pool->step_params;
            sp->p = make_attend_params(pool, layer, cp, q, out);
            sp->p.stamp = next_stamp(pool, 2);
            sp->a = a;
            sp->a.pdl_early = 0;
            sp->a.attend_src = nullptr; sp->a.attend_n16 = 0;
            sp->plan = cp.step_plan;
            sp->n_workers = cp.step_workers;
            sp->claim_ctr = pool->d_bk_flag + 8;
            memcpy(sp->sm_class, pool->sm_class, sizeof(sp->sm_class));
            sp->n_items = (int32_t)pool->step_items.size();
            memcpy(sp->items, pool->step_items.data(), pool->step_items.size() * sizeof(StepItem));
            e = launch_step_gqa(*sp, c.head_dim, pool->G * cp.cls_max_q[0], st, true);
            if (e == cudaSuccess) { *fused = true; ++pool->n_attend; }
        } else {
            e = launch_kernel(append_fused_kernel, grid, dim3(256), smem, st, true, a);
        }
        if (e != cudaSuccess) {
            if (!unfused_bookkeeping) rollback();      // nothing was enqueued: the call never happened
            return cuda_fail(pool, e, fuse ? "step_gqa_kernel" : "append_fused_kernel");
        }
        ++pool->n_launch;
    }
    ++pool->n_append;
    if (n_batch > 0) return release_stage(pool, slot, st);
    return METRONOME_OK;
}

}  // namespace

extern "C" {

int metronome_append_kv(metronome_pool_t* pool, int32_t layer, int32_t n_batch, const int32_t* sids,
                        const int32_t* n_new, const void* k_new, const void* v_new, void* cuda_stream) {
    return append_impl(pool, layer, n_batch, sids, n_new, k_new, v_new, cuda_stream, nullptr, nullptr, nullptr);
}

int metronome_append_attend(metronome_pool_t* pool, int32_t layer, int32_t n_batch, const int32_t* sids,
                            const int32_t* n_new, const void* k_new, const void* v_new, const void* q, void* out,
                            void* cuda_stream) {
    if (!pool) return METRONOME_ERR_INVALID_ARG;
    if (pool->bookkeeping_only) return METRONOME_ERR_UNSUPPORTED;
    // (the attention half can only fail on arguments: check them before the append changes anything)
    int64_t rows = 0;
    if (n_batch > 0 && n_new)
        for (int i = 0; i < n_batch; ++i) rows += n_new[i] > 0 ? n_new[i] : 0;
    if (rows > 0 && (!q || !out)) return METRONOME_ERR_INVALID_ARG;
    bool fused = false;
    int rc = append_impl(pool, layer, n_batch, sids, n_new, k_new, v_new, cuda_stream, q, out, &fused);
    if (rc || fused) return rc;
    return metronome_attend_frame(pool, layer, n_batch, sids, n_new, q, out, cuda_stream);
}

int metronome_attend_frame(metronome_pool_t* pool, int32_t layer, int32_t n_batch, const int32_t* sids,
                           const int32_t* q_lens, const void* q, void* out, void* cuda_stream) {
    if (!pool || layer < 0 || layer >= pool->cfg.n_layers) return METRONOME_ERR_INVALID_ARG;
    if (pool->bookkeeping_only) return METRONOME_ERR_UNSUPPORTED;
    int rc = check_batch(pool, n_batch, sids, q_lens);
    if (rc) return rc;
    int64_t total_rows = 0;
    for (int i = 0; i < n_batch; ++i) {
        if (q_lens[i] > pool->sessions[sids[i]].last_n) return METRONOME_ERR_QLEN_EXCEEDS_LAST_APPEND;
        total_rows += q_lens[i];
    }
    if (total_rows > 0 && (!q || !out)) return METRONOME_ERR_INVALID_ARG;
    ++pool->n_attend;
    if (total_rows == 0) return METRONOME_OK;
    if (pool->epoch == 0 || pool->layer_epoch[layer] != pool->epoch) return METRONOME_ERR_LAYER_SEQUENCE;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    // Fast path: the queries are exactly the rows of this step's append (decode: 1, chunk: n), whose
    // work list append_kv(layer 0) already planned and its kernel already copied to the device.
    const AttendPlan& cp = pool->cached_plan;
    if (cp.valid && cp.epoch == pool->epoch && (int32_t)pool->last_sids.size() == n_batch &&
        !memcmp(pool->last_sids.data(), sids, n_batch * sizeof(int32_t)) &&
        !memcmp(pool->last_n_new.data(), q_lens, n_batch * sizeof(int32_t)))
        return launch_attend(pool, layer, cp,
                             reinterpret_cast<const AttendItem*>(reinterpret_cast<const uint8_t*>(pool->d_attend_items) +
                                                                 (cp.epoch & 1) * pool->attend_buf_bytes),
                             q, out, st, /*after_append=*/true);

    uint8_t *h = nullptr, *d = nullptr;
    int slot = 0;
    rc = acquire_stage(pool, &h, &d, &slot);
    if (rc) return rc;
    AttendPlan plan;
    rc = plan_attend(pool, n_batch, sids, q_lens, reinterpret_cast<AttendItem*>(h), plan);
    if (rc) return rc;
    rc = commit_stage(pool, slot, (size_t)plan.n_items * sizeof(AttendItem) + (size_t)plan.n_range_items * sizeof(int32_t), st);
    if (rc) return rc;
    return launch_attend(pool, layer, plan, reinterpret_cast<const AttendItem*>(d), q, out, st, false);
}

// metronome_attend_frame without any allocation (include/metronome.h): the split-KV row kernel + the merge kernel,
// their partials in the library's fixed scratch array instead of the pool's grow-on-demand workspace.  Calls no
// cudaMalloc / cudaFree (nor plan_attend -> ensure_workspace, which does); the work list goes through the pool's
// staging ring like the general path of attend_frame.
int metronome_attend_frame_static(metronome_pool_t* pool, int32_t layer, int32_t n_batch, const int32_t* sids,
                                  const int32_t* q_lens, const void* q, void* out, void* cuda_stream) {
    if (!pool || layer < 0 || layer >= pool->cfg.n_layers) return METRONOME_ERR_INVALID_ARG;
    if (pool->bookkeeping_only) return METRONOME_ERR_UNSUPPORTED;
    int rc = check_batch(pool, n_batch, sids, q_lens);
    if (rc) return rc;
    int64_t total_rows = 0;
    for (int i = 0; i < n_batch; ++i) {
        if (q_lens[i] > pool->sessions[sids[i]].last_n) return METRONOME_ERR_QLEN_EXCEEDS_LAST_APPEND;
        total_rows += q_lens[i];
    }
    if (total_rows > 0 && (!q || !out)) return METRONOME_ERR_INVALID_ARG;
    if (total_rows == 0) { ++pool->n_attend; return METRONOME_OK; }
    if (pool->epoch == 0 || pool->layer_epoch[layer] != pool->epoch) return METRONOME_ERR_LAYER_SEQUENCE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const metronome_pool_config_t& c = pool->cfg;

    cudaError_t ce = cudaSuccess;
    uint8_t* scratch = static_cast<uint8_t*>(static_scratch_ptr(&ce));
    if (!scratch) return cuda_fail(pool, ce, "cudaGetSymbolAddress(g_static_scratch)");

    uint8_t *h = nullptr, *d = nullptr;
    int slot = 0;
    rc = acquire_stage(pool, &h, &d, &slot);
    if (rc) return rc;
    AttendPlan plan;
    plan_rows_static(pool, n_batch, sids, q_lens, reinterpret_cast<AttendItem*>(h), plan);
    // [row][Hq][max_splits][D] floats of partial outputs, then [row][Hq][max_splits][2] floats of (m, l)
    const size_t slots = (size_t)plan.total_rows * c.n_q_heads * plan.max_splits;
    const size_t need = plan.max_splits > 1 ? slots * (size_t)(c.head_dim + 2) * sizeof(float) : 0;
    if (need > (size_t)METRONOME_STATIC_SCRATCH_BYTES) {
        char msg[192];
        snprintf(msg, sizeof(msg), "attend_frame_static: %lld rows x %d heads x %d segments x (%d + 2) floats = %zu bytes of "
                 "split-KV partials, the static scratch holds %u", (long long)plan.total_rows, c.n_q_heads, plan.max_splits,
                 c.head_dim, need, (unsigned)METRONOME_STATIC_SCRATCH_BYTES);
        pool->cuda_err = msg;
        return METRONOME_ERR_SCRATCH_EXCEEDED;
    }
    ++pool->n_attend;
    rc = commit_stage(pool, slot, (size_t)plan.n_items * sizeof(AttendItem), st);
    if (rc) return rc;

    AttendParams p = make_attend_params(pool, layer, plan, q, out);
    p.ws_acc = reinterpret_cast<float*>(scratch);                                    // (256-byte aligned; slots * D * 4
    p.ws_ml = reinterpret_cast<float*>(scratch + slots * (size_t)c.head_dim * sizeof(float));   //  is a multiple of 16)
    p.max_splits = plan.max_splits;
    p.items = reinterpret_cast<const AttendItem*>(d);
    p.n_items = plan.n_items;
    p.range_item = nullptr;
    p.items_epoch = -1;                       // the list came by a copy: the kernel waits for its predecessor at the top
    p.stamp = nullptr;
    dim3 grid(c.n_q_heads, plan.total_splits[0], plan.cls_max_q[0]);
    if (pool->fp8) {
        if (c.head_dim == 128) CU(launch_kernel(attend_rows_kernel<128, true>, grid, dim3(128), 0, st, false, p));
        else CU(launch_kernel(attend_rows_kernel<64, true>, grid, dim3(128), 0, st, false, p));
    } else {
        if (c.head_dim == 128) CU(launch_kernel(attend_rows_kernel<128, false>, grid, dim3(128), 0, st, false, p));
        else CU(launch_kernel(attend_rows_kernel<64, false>, grid, dim3(128), 0, st, false, p));
    }
    ++pool->n_launch;
    if (plan.merge_cls[0]) {                  // row a6: every slot the merge reads was written by the launch above
        dim3 mgrid((unsigned)plan.cls_rows[0], c.n_q_heads);
        if (c.head_dim == 128) CU(launch_kernel(merge_kernel<128>, mgrid, dim3(32), 0, st, true, p));
        else CU(launch_kernel(merge_kernel<64>, mgrid, dim3(16), 0, st, true, p));
        ++pool->n_launch;
    }
    return release_stage(pool, slot, st);
}

int metronome_step_host(metronome_pool_t* pool, int32_t layer, int32_t n_batch, const int32_t* sids,
                        const int32_t* n_new, const void* k_new_host, const void* v_new_host,
                        const void* q_host, void* out_host, void* cuda_stream) {
    if (!pool || n_batch < 0 || (n_batch > 0 && (!sids || !n_new))) return METRONOME_ERR_INVALID_ARG;
    if (pool->bookkeeping_only) return METRONOME_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const metronome_pool_config_t& c = pool->cfg;
    int64_t rows = 0;
    for (int i = 0; i < n_batch; ++i) {
        if (n_new[i] < 0) return METRONOME_ERR_INVALID_ARG;
        if (n_new[i] > c.max_new_tokens) return METRONOME_ERR_CHUNK_TOO_LARGE;
        rows += n_new[i];
    }
    if (rows > 0 && (!k_new_host || !v_new_host || !q_host || !out_host)) return METRONOME_ERR_INVALID_ARG;
    const size_t kv_b = (size_t)rows * c.n_kv_heads * c.head_dim * 2, q_b = (size_t)rows * c.n_q_heads * c.head_dim * 2;
    const size_t kv_al = (kv_b + 255) & ~(size_t)255, q_al = (q_b + 255) & ~(size_t)255;
    const size_t need = 2 * kv_al + 2 * q_al;
    if (need > pool->io_bytes) {
        if (pool->d_io) cudaFree(pool->d_io);
        pool->d_io = nullptr; pool->io_bytes = 0;
        CU(cudaMalloc(&pool->d_io, need + need / 2));
        pool->io_bytes = need + need / 2;
    }
    uint8_t* dk = pool->d_io; uint8_t* dv = dk + kv_al; uint8_t* dq = dv + kv_al; uint8_t* dout = dq + q_al;
    if (rows > 0) {
        CU(cudaMemcpyAsync(dk, k_new_host, kv_b, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(dv, v_new_host, kv_b, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(dq, q_host, q_b, cudaMemcpyHostToDevice, st));
    }
    int rc = metronome_append_attend(pool, layer, n_batch, sids, n_new, rows ? dk : nullptr, rows ? dv : nullptr, dq, dout,
                                     cuda_stream);
    if (rc) return rc;
    if (rows > 0) CU(cudaMemcpyAsync(out_host, dout, q_b, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return METRONOME_OK;
}

// Event-free host steps: the host's side of step_done_kernel.  Polls the pinned flag; looks at the stream now and then so
// that a faulted GPU comes back as an error, not as a hang.
static int wait_step_done(metronome_pool* pool, int32_t seq) {
    if (!pool->h_done || seq <= 0) return METRONOME_OK;
    volatile int32_t* flag = pool->h_done;
    for (uint64_t spin = 1; *flag - seq < 0; ++spin) {
        if ((spin & 0x3fff) == 0 && pool->have_stream) {
            const cudaError_t e = cudaStreamQuery(pool->last_stream);
            if (e != cudaSuccess && e != cudaErrorNotReady) return cuda_fail(pool, e, "cudaStreamQuery (waiting for a host step)");
        }
#if defined(__x86_64__)
        __builtin_ia32_pause();
#endif
    }
    __atomic_thread_fence(__ATOMIC_ACQUIRE);     // the kernels' writes into out_host are behind the flag
    return METRONOME_OK;
}

int metronome_step_host_wait(metronome_pool_t* pool, int32_t keep) {
    if (!pool || keep < 0) return METRONOME_ERR_INVALID_ARG;
    if (pool->direct_mode) return wait_step_done(pool, pool->direct_seq - keep);
    // steps host_seq-1 (newest) and host_seq-2 may be outstanding; wait for all but the newest `keep`
    for (int64_t k = pool->host_seq - 2; k <= pool->host_seq - 1 - keep; ++k) {
        if (k < 0) continue;
        const int b = (int)(k & 1);
        if (!pool->slot_busy[b]) continue;
        CU(cudaEventSynchronize(pool->ev_d2h[b]));
        pool->slot_busy[b] = false;
    }
    return METRONOME_OK;
}

int metronome_step_host_async(metronome_pool_t* pool, int32_t layer, int32_t n_batch, const int32_t* sids,
                              const int32_t* n_new, const void* k_new_host, const void* v_new_host,
                              const void* q_host, void* out_host, void* cuda_stream) {
    if (!pool || n_batch < 0 || (n_batch > 0 && (!sids || !n_new))) return METRONOME_ERR_INVALID_ARG;
    if (pool->bookkeeping_only) return METRONOME_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const metronome_pool_config_t& c = pool->cfg;
    int64_t rows = 0;
    for (int i = 0; i < n_batch; ++i) {
        if (n_new[i] < 0) return METRONOME_ERR_INVALID_ARG;
        if (n_new[i] > c.max_new_tokens) return METRONOME_ERR_CHUNK_TOO_LARGE;
        rows += n_new[i];
    }
    if (rows > 0 && (!k_new_host || !v_new_host || !q_host || !out_host)) return METRONOME_ERR_INVALID_ARG;
    if (!pool->s_h2d) {
        CU(cudaStreamCreateWithFlags(&pool->s_h2d, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&pool->s_d2h, cudaStreamNonBlocking));
        for (int b = 0; b < 2; ++b) {
            CU(cudaEventCreateWithFlags(&pool->ev_h2d[b], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&pool->ev_comp[b], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&pool->ev_d2h[b], cudaEventDisableTiming));
        }
    }
    // Event-free mode when the copies are truly asynchronous (out_host pinned) and the driver's stream wait-value /
    // write-value operations are there.  Pageable buffers, the profiling brackets and the poison fill (more launches per
    // step) keep the event-chained path below.
    if (pool->memops_state == 0) {
        void *fw = nullptr, *fs = nullptr;
        cudaDriverEntryPointQueryResult qa, qb;
        const bool ok = cudaGetDriverEntryPoint("cuStreamWaitValue32", &fw, cudaEnableDefault, &qa) == cudaSuccess &&
                        cudaGetDriverEntryPoint("cuStreamWriteValue32", &fs, cudaEnableDefault, &qb) == cudaSuccess &&
                        qa == cudaDriverEntryPointSuccess && qb == cudaDriverEntryPointSuccess && fw && fs;
        if (!ok) cudaGetLastError();
        pool->fn_wait32 = reinterpret_cast<metronome_pool::memop32_fn>(fw);
        pool->fn_write32 = reinterpret_cast<metronome_pool::memop32_fn>(fs);
        pool->memops_state = ok ? 1 : -1;
    }
    bool direct = false;
    if (rows > 0 && !pool->profiling && !pool->poison && pool->tune_host_direct && pool->memops_state == 1) {
        cudaPointerAttributes at{};
        if (cudaPointerGetAttributes(&at, out_host) == cudaSuccess) direct = at.type == cudaMemoryTypeHost;
        else cudaGetLastError();
    }
    if (direct != pool->direct_mode) {              // drain the other mode's steps before switching
        const int rcw = metronome_step_host_wait(pool, 0);
        if (rcw) return rcw;
        pool->direct_mode = direct;
    }
    if (direct) {
        if (!pool->d_h2d_flag) {
            CU(cudaMalloc(&pool->d_h2d_flag, 256));
            CU(cudaMemset(pool->d_h2d_flag, 0, 256));
            CU(cudaHostAlloc(&pool->h_done, 256, cudaHostAllocMapped));
            CU(cudaHostAlloc(&pool->h_seq_ring, 64 * sizeof(int32_t), cudaHostAllocDefault));
            pool->h_done[0] = 0;
            void* dp = nullptr;
            CU(cudaHostGetDevicePointer(&dp, pool->h_done, 0));
            pool->h_done_dev = (unsigned long long)(uintptr_t)dp;
        }
        int32_t* d_done = pool->d_h2d_flag + 32;    // (its own 128-byte line)
        const int32_t seq = pool->direct_seq + 1;
        const int b = seq % kDirectSlots;
        const size_t kv_b = (size_t)rows * c.n_kv_heads * c.head_dim * 2, q_b = (size_t)rows * c.n_q_heads * c.head_dim * 2;
        const size_t kv_al = (kv_b + 255) & ~(size_t)255, q_al = (q_b + 255) & ~(size_t)255;
        const size_t need = 2 * kv_al + 2 * q_al;
        // the slot's previous step (three steps back) must be through -- kernels and read-back -- before it is reused:
        // the host may run two steps ahead of the GPU (metronome_step_host_wait(2))
        int rc = wait_step_done(pool, seq - kDirectSlots);
        if (rc) return rc;
        if (need > pool->io2_bytes[b]) {
            if (pool->d_io2[b]) cudaFree(pool->d_io2[b]);
            pool->d_io2[b] = nullptr; pool->io2_bytes[b] = 0;
            CU(cudaMalloc(&pool->d_io2[b], need + need / 2));
            pool->io2_bytes[b] = need + need / 2;
        }
        uint8_t* dk = pool->d_io2[b]; uint8_t* dv = dk + kv_al; uint8_t* dq = dv + kv_al; uint8_t* dout = dq + q_al;
        CU(cudaMemcpyAsync(dk, k_new_host, kv_b, cudaMemcpyHostToDevice, pool->s_h2d));
        CU(cudaMemcpyAsync(dv, v_new_host, kv_b, cudaMemcpyHostToDevice, pool->s_h2d));
        CU(cudaMemcpyAsync(dq, q_host, q_b, cudaMemcpyHostToDevice, pool->s_h2d));
        pool->h_seq_ring[seq & 63] = seq;
        CU(cudaMemcpyAsync(pool->d_h2d_flag, pool->h_seq_ring + (seq & 63), sizeof(int32_t), cudaMemcpyHostToDevice, pool->s_h2d));
        pool->direct_seq = seq;                     // (from here on the step exists: an error still publishes its number)
        pool->cur_h2d_flag = pool->d_h2d_flag; pool->cur_h2d_seq = seq;
        rc = metronome_append_attend(pool, layer, n_batch, sids, n_new, dk, dv, dq, dout, cuda_stream);
        pool->cur_h2d_flag = nullptr;
        // "the kernels of step seq are complete", behind the step's last kernel, programmatic on both sides; transparent
        // for the early bookkeeping of the next append kernel (it touches nothing that kernel or the attention kernels use)
        const bool adjacent = pool->pastwait_launches == pool->n_launch;
        CU(launch_kernel(step_done_kernel, dim3(1), dim3(32), 0, st, rc == METRONOME_OK, d_done, seq));
        ++pool->n_launch;
        if (adjacent) pool->pastwait_launches = pool->n_launch;
        pool->last_stream = st; pool->have_stream = true;
        // read-back on its own stream: wait for that value, copy, publish to the host
        if (pool->fn_wait32(pool->s_d2h, (unsigned long long)(uintptr_t)d_done, (unsigned int)seq, 0u /* GEQ, wrap-safe */) != 0)
            return cuda_fail(pool, cudaErrorUnknown, "cuStreamWaitValue32");
        if (rc == METRONOME_OK) CU(cudaMemcpyAsync(out_host, dout, q_b, cudaMemcpyDeviceToHost, pool->s_d2h));
        if (pool->fn_write32(pool->s_d2h, pool->h_done_dev, (unsigned int)seq, 0u) != 0)
            return cuda_fail(pool, cudaErrorUnknown, "cuStreamWriteValue32");
        if (rc) return rc;
        ++pool->host_seq;
        return METRONOME_OK;
    }
    const int b = (int)(pool->host_seq & 1);
    const size_t kv_b = (size_t)rows * c.n_kv_heads * c.head_dim * 2, q_b = (size_t)rows * c.n_q_heads * c.head_dim * 2;
    const size_t kv_al = (kv_b + 255) & ~(size_t)255, q_al = (q_b + 255) & ~(size_t)255;
    const size_t need = 2 * kv_al + 2 * q_al;
    if (need > pool->io2_bytes[b]) {
        // (the slot's previous step must be through before its buffer goes away)
        if (pool->slot_busy[b]) { CU(cudaEventSynchronize(pool->ev_d2h[b])); pool->slot_busy[b] = false; }
        if (pool->d_io2[b]) cudaFree(pool->d_io2[b]);
        pool->d_io2[b] = nullptr; pool->io2_bytes[b] = 0;
        CU(cudaMalloc(&pool->d_io2[b], need + need / 2));
        pool->io2_bytes[b] = need + need / 2;
    }
    uint8_t* dk = pool->d_io2[b]; uint8_t* dv = dk + kv_al; uint8_t* dq = dv + kv_al; uint8_t* dout = dq + q_al;
    // H2D of this step: once the slot's previous step (two steps back) has been read out.  The host waits for that here, so
    // that metronome_step_host_wait(keep >= 2) holds as well: whatever is older than the two newest steps is complete
    if (pool->slot_busy[b]) { CU(cudaEventSynchronize(pool->ev_d2h[b])); pool->slot_busy[b] = false; }
    if (rows > 0) {
        CU(cudaMemcpyAsync(dk, k_new_host, kv_b, cudaMemcpyHostToDevice, pool->s_h2d));
        CU(cudaMemcpyAsync(dv, v_new_host, kv_b, cudaMemcpyHostToDevice, pool->s_h2d));
        CU(cudaMemcpyAsync(dq, q_host, q_b, cudaMemcpyHostToDevice, pool->s_h2d));
    }
    CU(cudaEventRecord(pool->ev_h2d[b], pool->s_h2d));
    CU(cudaStreamWaitEvent(st, pool->ev_h2d[b], 0));
    int rc = metronome_append_attend(pool, layer, n_batch, sids, n_new, rows ? dk : nullptr, rows ? dv : nullptr, dq, dout,
                                     cuda_stream);
    if (rc) return rc;          // (nothing of this step was enqueued but its input copies)
    CU(cudaEventRecord(pool->ev_comp[b], st));
    CU(cudaStreamWaitEvent(pool->s_d2h, pool->ev_comp[b], 0));
    if (rows > 0) CU(cudaMemcpyAsync(out_host, dout, q_b, cudaMemcpyDeviceToHost, pool->s_d2h));
    CU(cudaEventRecord(pool->ev_d2h[b], pool->s_d2h));
    pool->slot_busy[b] = true;
    ++pool->host_seq;
    return METRONOME_OK;
}

int metronome_session_query(metronome_pool_t* pool, int32_t sid, void* cuda_stream, int64_t* len,
                            int32_t* first_live_block, int32_t* n_blocks, int32_t* block_ids) {
    if (!pool) return METRONOME_ERR_INVALID_ARG;
    if (sid < 0 || sid >= pool->cfg.max_sessions || !pool->sessions[sid].open) return METRONOME_ERR_INVALID_SESSION;
    const Session& s = pool->sessions[sid];
    const int32_t B = pool->cfg.block_size;
    const int32_t n_blk = (int32_t)((s.len + B - 1) / B);
    const int32_t n_sink_res = n_blk < pool->n_sink ? n_blk : pool->n_sink;
    const int32_t n_win = n_blk > s.first_live ? n_blk - s.first_live : 0;
    if (len) *len = s.len;
    // the unbounded arm pins nothing internally (nothing is ever freed), but reports the same
    // "first non-sink block" = ceil(S / block) as the bounded rule of session_open (SURVEY 8(c) rule 2)
    if (first_live_block)
        *first_live_block = pool->unbounded ? (pool->cfg.n_sinks + pool->cfg.block_size - 1) / pool->cfg.block_size
                                            : s.first_live;
    if (n_blocks) *n_blocks = n_sink_res + n_win;
    if (block_ids && n_sink_res + n_win > 0) {
        std::vector<int32_t> rowbuf(pool->tbl_width);
        cudaStream_t st = (cudaStream_t)cuda_stream;
        CU(cudaMemcpyAsync(rowbuf.data(), pool->d_table + (int64_t)sid * pool->tbl_width,
                           (size_t)pool->tbl_width * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        int k = 0;
        for (int b = 0; b < n_sink_res; ++b) block_ids[k++] = rowbuf[table_slot(b, pool->n_sink, pool->ring)];
        for (int b = s.first_live; b < n_blk; ++b) block_ids[k++] = rowbuf[table_slot(b, pool->n_sink, pool->ring)];
    }
    return METRONOME_OK;
}

int metronome_pool_query(metronome_pool_t* pool, void* cuda_stream, int32_t* n_free, int32_t* free_ids) {
    if (!pool) return METRONOME_ERR_INVALID_ARG;
    if (n_free) *n_free = pool->n_free;
    if (free_ids && pool->n_free > 0) {
        std::vector<int32_t> buf(pool->n_free);
        cudaStream_t st = (cudaStream_t)cuda_stream;
        CU(cudaMemcpyAsync(buf.data(), pool->d_free, (size_t)pool->n_free * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        for (int i = 0; i < pool->n_free; ++i) free_ids[i] = buf[pool->n_free - 1 - i];   // pop order
    }
    return METRONOME_OK;
}

int metronome_read_kv(metronome_pool_t* pool, int32_t layer, int32_t sid, int64_t pos0, int32_t n, void* k_out,
                      void* v_out, void* cuda_stream) {
    if (!pool || layer < 0 || layer >= pool->cfg.n_layers || n < 0 || pos0 < 0) return METRONOME_ERR_INVALID_ARG;
    if (pool->bookkeeping_only) return METRONOME_ERR_UNSUPPORTED;
    if (sid < 0 || sid >= pool->cfg.max_sessions || !pool->sessions[sid].open) return METRONOME_ERR_INVALID_SESSION;
    if (n == 0) return METRONOME_OK;
    if (!k_out || !v_out || pos0 + n > INT32_MAX) return METRONOME_ERR_INVALID_ARG;
    const Session& s = pool->sessions[sid];
    const int32_t n_blk = (int32_t)((s.len + kBlockTokens - 1) / kBlockTokens);
    const int32_t n_sink_res = n_blk < pool->n_sink ? n_blk : pool->n_sink;
    const int64_t chunks = (int64_t)n * pool->cfg.n_kv_heads * (pool->cfg.head_dim / 8);
    if (pool->fp8)
        kv_read_fp8_kernel<<<(unsigned)((chunks + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(
            pool->d_table + (int64_t)sid * pool->tbl_width, pool->n_sink, pool->ring, n_sink_res, s.first_live, n_blk,
            (int32_t)pos0, n, pool->d_kv + (int64_t)layer * pool->L.layer_bytes, pool->L, (float*)k_out, (float*)v_out);
    else
        kv_read_kernel<<<(unsigned)((chunks + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(
            pool->d_table + (int64_t)sid * pool->tbl_width, pool->n_sink, pool->ring, n_sink_res, s.first_live, n_blk,
            (int32_t)pos0, n, pool->d_kv + (int64_t)layer * pool->L.layer_bytes, pool->L, (uint4*)k_out, (uint4*)v_out);
    ++pool->n_launch;
    CU(cudaGetLastError());
    return METRONOME_OK;
}

int metronome_pool_stats(metronome_pool_t* pool, int64_t* kernel_launches, int64_t* append_calls, int64_t* attend_calls) {
    if (!pool) return METRONOME_ERR_INVALID_ARG;
    if (kernel_launches) *kernel_launches = pool->n_launch;
    if (append_calls) *append_calls = pool->n_append;
    if (attend_calls) *attend_calls = pool->n_attend;
    return METRONOME_OK;
}

int metronome_pool_sm_speeds(metronome_pool_t* pool, int32_t* n_sms, int32_t* n_slow_sms, double* slow_ratio) {
    if (!pool) return METRONOME_ERR_INVALID_ARG;
    if (n_sms) *n_sms = pool->n_sm;
    if (n_slow_sms) *n_slow_sms = pool->n_slow_sms;
    if (slow_ratio) *slow_ratio = pool->slow_ratio;
    return METRONOME_OK;
}

int metronome_pool_set_profiling(metronome_pool_t* pool, int32_t mode) {
    if (!pool || mode < 0 || mode > 2) return METRONOME_ERR_INVALID_ARG;
    pool->profiling = mode == 1;
    pool->stamping = mode == 2;
    if (mode == 2) {
        if (!pool->d_stamps) CU(cudaMalloc(&pool->d_stamps, (size_t)kStampSlots * 2 * sizeof(unsigned long long)));
        CU(cudaDeviceSynchronize());
        init_stamps_kernel<<<64, 256>>>(pool->d_stamps, kStampSlots);
        CU(cudaDeviceSynchronize());
        pool->stamp_kind.clear();
    }
    return METRONOME_OK;
}

int metronome_pool_read_stamps(metronome_pool_t* pool, int32_t max_launches, int32_t* kinds, double* span_ms,
                               double* start_ms, int32_t* n_out) {
    if (!pool || max_launches < 0 || !n_out) return METRONOME_ERR_INVALID_ARG;
    CU(cudaDeviceSynchronize());
    const int32_t n = (int32_t)std::min<size_t>(pool->stamp_kind.size(), (size_t)max_launches);
    std::vector<unsigned long long> h(2 * (size_t)n);
    if (n > 0) CU(cudaMemcpy(h.data(), pool->d_stamps, h.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    for (int32_t i = 0; i < n; ++i) {
        if (kinds) kinds[i] = pool->stamp_kind[i];
        const bool ok = h[2 * i] != ~0ull && h[2 * i + 1] >= h[2 * i];
        if (span_ms) span_ms[i] = ok ? (double)(h[2 * i + 1] - h[2 * i]) * 1e-6 : -1.0;
        if (start_ms) start_ms[i] = ok ? (double)(h[2 * i] - h[0]) * 1e-6 : -1.0;
    }
    *n_out = n;
    if (pool->d_stamps) {
        init_stamps_kernel<<<64, 256>>>(pool->d_stamps, kStampSlots);
        CU(cudaDeviceSynchronize());
    }
    pool->stamp_kind.clear();
    return METRONOME_OK;
}

int metronome_pool_read_profile(metronome_pool_t* pool, double* attend_kernel_ms, int64_t* attend_kernel_launches,
                                int32_t reset) {
    if (!pool) return METRONOME_ERR_INVALID_ARG;
    double ms = 0.0;
    for (size_t i = 0; i + 1 < pool->prof_used; i += 2) {
        CU(cudaEventSynchronize(pool->prof_ev[i + 1]));
        float t = 0.f;
        CU(cudaEventElapsedTime(&t, pool->prof_ev[i], pool->prof_ev[i + 1]));
        ms += t;
    }
    if (attend_kernel_ms) *attend_kernel_ms = ms;
    if (attend_kernel_launches) *attend_kernel_launches = (int64_t)(pool->prof_used / 2);
    if (reset) pool->prof_used = 0;
    return METRONOME_OK;
}

// ---- measurement aid: read-only HBM stream ----
int metronome_stream_read_gbs(size_t bytes, int32_t reps, void* cuda_stream, double* gbs_out) {
    if (bytes < (1u << 20) || reps < 1 || !gbs_out) return METRONOME_ERR_INVALID_ARG;
    metronome_pool* pool = nullptr;                      // (CU() reports through a pool; none here)
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint4* buf = nullptr;
    unsigned int* sink = nullptr;
    const int64_t n16 = (int64_t)(bytes / 16);
    if (cudaMalloc(&buf, (size_t)n16 * 16) != cudaSuccess) return METRONOME_ERR_OUT_OF_MEMORY;
    if (cudaMalloc(&sink, 4) != cudaSuccess) { cudaFree(buf); return METRONOME_ERR_OUT_OF_MEMORY; }
    int dev = 0, n_sm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    cudaMemsetAsync(buf, 1, (size_t)n16 * 16, st);
    cudaMemsetAsync(sink, 0, 4, st);
    double best = 0.0;
    cudaError_t err = cudaSuccess;
    for (int r = 0; r < reps + 1 && err == cudaSuccess; ++r) {          // first pass is a warm-up
        cudaEventRecord(e0, st);
        stream_read_kernel<<<n_sm * 8, 512, 0, st>>>(buf, n16, sink);
        cudaEventRecord(e1, st);
        err = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms > 0.f) best = std::max(best, (double)n16 * 16.0 / (ms * 1e-3) / 1e9);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    cudaFree(sink);
    if (err != cudaSuccess) return cuda_fail(pool, err, "stream_read");
    *gbs_out = best;
    return METRONOME_OK;
}

// ---- NEXT f3: AIMD admission gate, host-only ----
struct metronome_gate {
    metronome_gate_config_t cfg;
    float cap;
};

int metronome_gate_create(const metronome_gate_config_t* c, metronome_gate_t** out) {
    if (!c || !out) return METRONOME_ERR_INVALID_ARG;
    *out = nullptr;
    if (!(c->budget_ms > 0.f) || !(c->target_frac > 0.f && c->target_frac <= 1.f) || !(c->add_step > 0.f) ||
        !(c->mult_factor > 0.f && c->mult_factor < 1.f) || !(c->cap_min >= 1.f) || !(c->cap_max >= c->cap_min) ||
        !(c->cap_init >= c->cap_min && c->cap_init <= c->cap_max))
        return METRONOME_ERR_INVALID_ARG;
    metronome_gate* g = new (std::nothrow) metronome_gate();
    if (!g) return METRONOME_ERR_OUT_OF_MEMORY;
    g->cfg = *c;
    g->cap = c->cap_init;
    *out = g;
    return METRONOME_OK;
}

int metronome_gate_destroy(metronome_gate_t* gate) {
    delete gate;
    return METRONOME_OK;
}

int metronome_gate_observe(metronome_gate_t* g, float latency_ms, float* cap_out) {
    if (!g || !(latency_ms >= 0.f)) return METRONOME_ERR_INVALID_ARG;
    if (latency_ms >= g->cfg.target_frac * g->cfg.budget_ms) g->cap = std::max(g->cfg.cap_min, g->cap * g->cfg.mult_factor);
    else g->cap = std::min(g->cfg.cap_max, g->cap + g->cfg.add_step);
    if (cap_out) *cap_out = g->cap;
    return METRONOME_OK;
}

int metronome_gate_admit(metronome_gate_t* g, int32_t n_live, int32_t* admitted_out) {
    if (!g || !admitted_out || n_live < 0) return METRONOME_ERR_INVALID_ARG;
    *admitted_out = n_live < (int32_t)floorf(g->cap) ? 1 : 0;
    return METRONOME_OK;
}

int metronome_pool_debug_fail_next(metronome_pool_t* pool, int32_t stage) {
    if (!pool || stage < 0 || stage > 2) return METRONOME_ERR_INVALID_ARG;
    pool->inject_fault = stage;
    return METRONOME_OK;
}

int metronome_pool_debug_read_flags(metronome_pool_t* pool, void* cuda_stream, int32_t* flags16) {
    if (!pool || !flags16) return METRONOME_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaMemcpyAsync(flags16, pool->d_bk_flag, 64, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return METRONOME_OK;
}

int metronome_pool_set_tuning(metronome_pool_t* pool, int32_t split_tokens, int32_t kernel_family, int32_t gqa_dynamic,
                              int32_t fused_step) {
    if (!pool || split_tokens < 0 || kernel_family < 0 || kernel_family > 2 || gqa_dynamic < 0 || gqa_dynamic > 2 ||
        fused_step < 0 || fused_step > 2)
        return METRONOME_ERR_INVALID_ARG;
    if (fused_step == 2 && pool->tune_fused_step != 2 && !pool->bookkeeping_only) {
        cudaDeviceSynchronize();
        calibrate_sm_speeds(pool);
    }
    pool->tune_split_tokens = split_tokens;
    pool->tune_family = kernel_family;
    pool->tune_gqa_dynamic = gqa_dynamic;
    pool->tune_fused_step = fused_step;
    pool->cached_plan.valid = false;
    return METRONOME_OK;
}

}  // extern "C"
