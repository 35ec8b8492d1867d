/*
 * metronome_measure.h -- measurement and test aids of libmetronome.so.  NOT part of the product
 * boundary (include/metronome.h): nothing here is needed to serve a frame.
 * bench.py, the sweeps next to it and tests/ use these; a serving engine would not.
 */
#ifndef METRONOME_MEASURE_H_
#define METRONOME_MEASURE_H_

#include "metronome.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Counters since pool_create: kernels launched by the library, append / attend calls.  host. */
int metronome_pool_stats(metronome_pool_t* pool, int64_t* kernel_launches, int64_t* append_calls,
                         int64_t* attend_calls);

/* Tuning knobs (0 = automatic): keys per split-KV segment target; the kernel family (1 CUDA-core row
 * kernel, 2 tensor-core kernels: mma.sync GQA decode + tcgen05 chunk prefill); the GQA decode kernel's
 * dynamically claimed tail ranges (1 forced on, 2 forced off; automatic = on for shares >= 512 tiles);
 * fused_step 2 = metronome_append_attend runs a decode step of a grouped-query pool as ONE launch (step_gqa.cuh;
 * built and verified, but measured 0.4-4.5 % slower per frame than the two launches on B200, so it is off unless
 * asked for: DESIGN.md sec. 5.2); setting it measures the SMs' streaming speeds once (metronome_pool_sm_speeds).
 * For benchmarks and tests of "both launch modes" (L258).  Errors: INVALID_ARG.
 * Three more switches are read from the environment at pool creation (measurement aids):
 * METRONOME_UMMA_HALF=0 | 1 | 2 picks the chunk-prefill kernel: full-size (one CTA per SM) only, half-size (two CTAs per SM) for
 * launches whose items have at most 128 query rows, or half-size always (default 2);
 * METRONOME_GQA_SMCLASS=1 sizes the GQA decode kernel's ranges by the SMs' measured streaming speeds (a calibration pass per
 * pool; off by default), METRONOME_HOST_STEP_EVENTS=1 makes metronome_step_host_async chain events even for pinned buffers. */
int metronome_pool_set_tuning(metronome_pool_t* pool, int32_t split_tokens, int32_t kernel_family,
                              int32_t gqa_dynamic, int32_t fused_step);

/* What set_tuning(fused_step = 2) measured (otherwise 0 slow SMs, ratio 1): the SMs of one GPU do not
 * stream at the same speed when all of them stream, and the fused decode step gives the warps that run on the slow
 * ones shorter ranges.  n_sms = SMs of the device, n_slow_sms = those whose mean time was > 4 % above the median
 * SM's, slow_ratio = their speed relative to the others (0.75 .. 1).  All pointers host, optional. */
int metronome_pool_sm_speeds(metronome_pool_t* pool, int32_t* n_sms, int32_t* n_slow_sms, double* slow_ratio);

/* Test aid for the "no state change on error" contract: the NEXT append_kv(layer 0) fails as if
 * (stage 1) growing the split-KV workspace had run out of memory, or (stage 2) the launch of the append
 * kernel had failed -- both sit after the point where the shadow counts are tentatively committed.
 * One-shot; stage 0 disarms.  Errors: INVALID_ARG. */
int metronome_pool_debug_fail_next(metronome_pool_t* pool, int32_t stage);

/* Test aid: copies the pool's 16 internal device flag words to flags16 (host) after cuda_stream has
 * drained: [0] bookkeeping epoch, [1] work-list epoch, [2] / [3] claim and exit counters of the GQA decode
 * kernel's dynamic ranges (must be 0 between launches), [5] past-wait epoch of the early-mode append kernel, [8] / [9] / [10] range
 * claims and exits of the fused step kernel (0 between launches), [12] epoch of the last tensor-core attention kernel that got
 * past its wait (early bookkeeping).  Errors: INVALID_ARG, CUDA. */
int metronome_pool_debug_read_flags(metronome_pool_t* pool, void* cuda_stream, int32_t* flags16);

/* Measurement aids for the time of the attention kernels (the dominant kernels; not the append kernel, not the merge).
 *   mode 1  attend_frame brackets its attention kernel with CUDA events on the caller's stream.  Events between the
 *           launches break their programmatic (PDL) edges, so in this mode every launch is plain and early mode is off:
 *           the kernel is timed ALONE, not as it runs inside a normal step.  read_profile waits for the events, returns
 *           the summed kernel time in milliseconds and the number of bracketed launches, and (reset != 0) clears them.
 *   mode 2  the attention kernels stamp %globaltimer themselves (first CTA in, last CTA out; two atomics per CTA), the
 *           launches stay exactly as in a normal step.  read_stamps synchronises the device, returns per attention launch
 *           since the mode was set / the last read (at most max_launches, at most 32768 are kept) its kind (1 row kernel,
 *           2 GQA decode kernel, 3 chunk-prefill kernel), its span and its start relative to the first launch, both in
 *           milliseconds (-1: the kernel never stamped), and clears them.  All pointers host; kinds / span_ms / start_ms
 *           may be NULL.
 *   mode 0  off.  Errors: INVALID_ARG, CUDA. */
int metronome_pool_set_profiling(metronome_pool_t* pool, int32_t mode);
int metronome_pool_read_profile(metronome_pool_t* pool, double* attend_kernel_ms, int64_t* attend_kernel_launches,
                                int32_t reset);
int metronome_pool_read_stamps(metronome_pool_t* pool, int32_t max_launches, int32_t* kinds, double* span_ms,
                               double* start_ms, int32_t* n_out);


/* Measurement aid ("plus a read-only stream microbenchmark run in the same job").
 * Streams `bytes` of a scratch device buffer (allocated and freed inside) `reps` times with 16-byte
 * loads from every SM and returns the best read-only bandwidth in GB/s in *gbs_out: the ceiling a pure
 * KV stream can reach on this GPU, next to the read+write copy figure of MEASURED_PEAKS.json.
 * Blocking; uses the current device and `cuda_stream`.  Errors: INVALID_ARG (bytes < 1 MiB, reps < 1,
 * null), OUT_OF_MEMORY, CUDA. */
int metronome_stream_read_gbs(size_t bytes, int32_t reps, void* cuda_stream, double* gbs_out);

#ifdef __cplusplus
}
#endif
#endif /* METRONOME_MEASURE_H_ */
