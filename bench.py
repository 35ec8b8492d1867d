#!/usr/bin/env python
"""bench.py -- session-frames/s and windowed-attention HBM GB/s on synthetic Metronome sessions.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl reference]

A "step" is one frame of the whole hot path for every due session on one layer:
append_kv (evict + allocate + KV write) then attend_frame (work list, attention, merge).
At N=1 the workload is BASELINE.json configs[1] (Moshi-shaped: 128 sessions, 32Q/32KV, D=128,
S=4, W=750, ages U{1..3750}); histories are built through the library first (untimed).
Prints ONE JSON line (contract in the task statement): `value` = whole-job session-frames/s with
inputs resident in HBM, `e2e` = the same through metronome_step_host with pinned HOST buffers,
`roofline` for the dominant kernel (attention), `cpu_baseline` = the oracle on the host cores.

N > 1 (launched by torch.distributed.run): replicas only -- one pool per GPU, sessions never
cross GPUs, no data-path collective; max-over-ranks time, `"scaling": "weak"`.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

RANK = int(os.environ.get("RANK", "0"))
LOCAL_RANK = int(os.environ.get("LOCAL_RANK", "0"))
WORLD = int(os.environ.get("WORLD_SIZE", "1"))

METRIC = "session_frames_per_sec"
UNIT = "session-frames/s (per layer)"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0,
                    help="timed frames (default: 400 for config 2; 20 for configs 3-5, whose sessions would otherwise age "
                         "past the config's own age range during the run)")
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="metronome", choices=["metronome", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index 1..5 (2 = the metric's)")
    ap.add_argument("--history-scale", type=float, default=1.0)
    ap.add_argument("--sessions", type=int, default=0, help="override the session count (0 = the config's)")
    ap.add_argument("--family", type=int, default=0, help="0 auto, 1 CUDA-core rows, 2 tensor-core tiles")
    ap.add_argument("--split-tokens", type=int, default=0)
    ap.add_argument("--two-calls", action="store_true",
                    help="issue every sub-step as metronome_append_kv + metronome_attend_frame instead of the one-call "
                         "metronome_append_attend (A/B of the fused decode step)")
    ap.add_argument("--kv-fp8", action="store_true",
                    help="store K / V as fp8 (E4M3 codes + a float32 scale per (token, KV head): METRONOME_FLAG_KV_FP8, NEXT row "
                         "f4); algorithmic bytes per key drop from 4 D to 2 D + 8 per KV head")
    ap.add_argument("--fused-step", action="store_true",
                    help="run GQA decode steps as one launch (step_gqa.cuh; measured slower than the two launches, off by default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--layers", type=int, default=1,
                    help="KV pools cycled per sub-step (a model runs its 30-50 layers one after the other: with >= 4 "
                         "layers consecutive passes over one layer's pool cannot hit in the 126 MB L2, SURVEY 8(d))")
    ap.add_argument("--sweep", default="", choices=["", "age", "sessions", "sw", "occupancy", "admission"],
                    help="shape checks of SURVEY sec. 8(d)/(f) instead of the bench line: one JSON line per point")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region (NVML, a polling thread)."""

    def __init__(self, gpu_index: int, period_s: float = 0.01):
        import threading
        self.sm, self.reasons, self.max_mhz, self.err = [], set(), None, None
        self._stop = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(gpu_index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:          # noqa: BLE001
            self.err = f"nvml unavailable: {e}"
            self.nv = None
        self.period = period_s
        self.t = threading.Thread(target=self._loop, daemon=True)
        if self.nv:
            self.t.start()

    def _loop(self):
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        while not self._stop.is_set():
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:       # noqa: BLE001
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception as e:      # noqa: BLE001
                self.err = str(e)
                break
            self._stop.wait(self.period)

    def stop(self):
        self._stop.set()
        if self.nv:
            self.t.join(timeout=2)
        sm = sorted(self.sm)
        out = {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": self.max_mhz, "samples": len(sm),
               "reasons": sorted(self.reasons)}
        if self.err:
            out["note"] = self.err
        return out


E2E_DEPTH = 2       # host steps kept in flight by the e2e leg (the library stages three: metronome_step_host_async)
KV_FP8 = False      # --kv-fp8: a key costs 2 D + 8 bytes per KV head (codes + two scales) instead of 4 D


def item_bytes(w, L, n):
    """per session keys_read x Hkv x 4D (K+V bf16) + q and out rows.
    keys_read = min(len, S+W) for decode; for a chunk the union over its rows min(L1, S+W+n-1)."""
    keys = min(L, w.S + w.W + n - 1)
    per_key = (2 * w.head_dim + 8) if KV_FP8 else 4 * w.head_dim
    return keys * w.n_kv_heads * per_key + n * w.n_q_heads * 4 * w.head_dim


def item_flops(w, L, n):
    """4 D flop per (query row, q head, admitted key); the query at t admits
    |[0,S) U (t-W, t]| = min(t+1, W) + max(0, min(S, t-W+1)) keys."""
    total = 0
    for t in range(L - n, L):
        total += min(t + 1, w.W) + max(0, min(w.S, t - w.W + 1))
    return 4 * w.head_dim * w.n_q_heads * total


def algorithmic_bytes(w, lengths, n_new):
    return sum(item_bytes(w, int(L), int(n)) for L, n in zip(lengths, n_new))


def launch_classes(w, n_new, family):
    """The attention launches one attend_frame(q_lens = n_new) makes, in launch order, as
    (kind, item mask): kind 1 row kernel, 2 GQA decode kernel, 3 chunk-prefill kernel -- the library's rule
    (metronome.cu plan_attend): tensor-core family when G x max(q_len) >= 4 (and <= 256), then per item
    chunk class iff G x q_len > 16."""
    import numpy as np
    n_new = np.asarray(n_new)
    G = w.n_q_heads // w.n_kv_heads
    fam = family or (2 if G * int(n_new.max()) >= 4 else 1)
    if fam == 2 and G * int(n_new.max()) > 256:
        fam = 1
    if fam == 1:
        return [(1, n_new > 0)]
    out = []
    dec = (n_new > 0) & (G * n_new <= 16)
    chk = G * n_new > 16
    if dec.any():
        out.append((2, dec))
    if chk.any():
        out.append((3, chk))
    return out


KIND_NAME = {1: "attend_rows_kernel", 2: "attend_gqa_kernel", 3: "attend_umma_kernel"}


def host_info():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model}


def config_dict(w, args, world):
    """The `config` object of the JSON line -- the same for both arms (--impl metronome / reference)."""
    return {"workload": f"BASELINE.json configs[{w.index - 1}] {w.name}: {w.n_sessions} sessions, "
                        f"{w.n_q_heads}Q/{w.n_kv_heads}KV, D={w.head_dim}, S={w.S}, W={w.W}, block 16",
            "sessions_per_gpu": w.n_sessions, "n_layers": max(1, args.layers), "parallelism": f"replicas x{world}",
            "kv_storage": "fp8 e4m3 + f32 scale per (token, kv head)" if getattr(args, "kv_fp8", False) else "bf16",
            "history_scale": args.history_scale,
            "l2": "inputs larger than L2: every step streams each session's whole window (GBs per step vs 126 MB "
                  "L2), no flush needed"}


def oracle_sample(w, history_scale):
    """The bounded sample both arms time the oracle on: a seeded subset of the workload's sessions (32 of
    config 2's 128, 8 of the others'), at the ages the workload's own schedule gives them, attending their
    FIRST timed frame (all its sub-steps: chunk prefill + decode steps).  Pure function of (config,
    history_scale): `cpu_baseline` of the GPU arm and `--impl reference` get the same sessions, the same
    rows, the same frames.  Inputs are regenerated on the CPU from their coordinates (synth.rows)."""
    import numpy as np
    import torch
    from dataclasses import replace
    from paper_2607_02640_b200 import synth
    from paper_2607_02640_b200 import workloads as wl
    events, _ = wl.build_schedule(replace(w, n_timed_frames=1), history_scale=history_scale)
    length, uid, nxt, first = {}, {}, 0, {}
    for ev in events:
        if ev[0] == "open":
            uid[ev[1]] = nxt; nxt += 1; length[ev[1]] = 0
        elif ev[0] == "close":
            del uid[ev[1]], length[ev[1]]
        elif ev[3]:
            for i, n in zip(ev[1], ev[2]):
                first.setdefault(int(i), []).append(int(n))
        else:
            for i, n in zip(ev[1], ev[2]):
                length[int(i)] += int(n)
    rng = np.random.default_rng(w.seed + 99)
    due = sorted(first)
    n_pick = min(32 if w.index <= 2 else 8, len(due))
    pick = sorted(int(x) for x in rng.permutation(due)[:n_pick])
    oc = w.outlier_channels()
    oc_t = torch.from_numpy(oc) if oc.size else None

    def rows(tag, u, pos, heads):
        return synth.to_u16(synth.rows(w.seed, tag, 0, torch.full((len(pos),), u, dtype=torch.int64), torch.from_numpy(pos),
                                       heads, w.head_dim, oc_t if tag != synth.STREAM_Q else None, w.outlier_scale))
    sample = []
    for i in pick:
        L0, subs = length[i], first[i]
        L1 = L0 + sum(subs)
        lo = max(0, L0 - w.W + 1)                       # oldest key the frame's oldest query can see
        pos = np.concatenate([np.arange(0, min(w.S, lo)), np.arange(lo, L1)]).astype(np.int64)
        qpos = np.arange(L0, L1, dtype=np.int64)
        sample.append({"L0": L0, "subs": subs, "pos": pos, "k": rows(synth.STREAM_K, uid[i], pos, w.n_kv_heads),
                       "v": rows(synth.STREAM_V, uid[i], pos, w.n_kv_heads), "qpos": qpos,
                       "q": rows(synth.STREAM_Q, uid[i], qpos, w.n_q_heads)})
    what = (f"{len(sample)} seeded sessions of the {len(due)} due in config {w.index}'s first timed frame, at the "
            f"schedule's own ages, every sub-step of that frame (attention only: oracle_attend_f32, OpenMP over rows x heads)")
    return sample, what


def oracle_frame(w, sample, n_threads):
    """One pass of the oracle over the sample = len(sample) session-frames."""
    from oracle import bounded_kv as O
    for s in sample:
        off = 0
        for n in s["subs"]:
            L = s["L0"] + off + n
            nk = int((s["pos"] < L).sum())              # keys appended so far (positions ascending)
            O.attend(s["q"][off:off + n], s["qpos"][off:off + n], s["k"][:nk], s["v"][:nk], s["pos"][:nk],
                     w.S, w.W, None, "f32", False, n_threads)
            off += n
    return len(sample)


def cpu_baseline(w, sample, what, budget_s=12.0, n_threads=None):
    """The oracle as it stands, on this box's host cores, repeated over the sample until the budget."""
    from oracle import bounded_kv as O
    n_threads = n_threads or O.max_threads()
    t0 = time.perf_counter()
    frames = 0
    while True:
        frames += oracle_frame(w, sample, n_threads)
        el = time.perf_counter() - t0
        if el >= budget_s or frames >= 100000:
            break
    return {"value": frames / el, "unit": UNIT, "cores": int(n_threads), "kind": "oracle",
            "sample": f"{what}; repeated for {el:.1f} s = {frames} session-frames", **host_info()}


def run_reference(args):
    """--impl reference: the oracle (there is no reference implementation to install), on the
    SAME bounded sample as the GPU arm's cpu_baseline leg; one step = one pass over the sample.  Rank 0 only."""
    if RANK != 0:
        return
    from oracle import bounded_kv as O
    from paper_2607_02640_b200 import workloads as wl
    w = wl.make_workload(args.config, n_sessions=args.sessions or None)
    n_threads = O.max_threads()
    sample, what = oracle_sample(w, args.history_scale)
    for _ in range(args.warmup):
        oracle_frame(w, sample, n_threads)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_frame(w, sample, n_threads)
    el = time.perf_counter() - t0
    value = len(sample) * args.steps / el
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": config_dict(w, args, WORLD),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(n_threads), "kind": "oracle",
                             "sample": what + "; one step = one pass over the sample", **host_info()},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    args = parse()
    if args.steps <= 0:
        args.steps = 400 if args.config == 2 else 20
    if args.impl == "reference":
        return run_reference(args)

    # one process per GPU: make this rank's GPU the only visible one BEFORE CUDA initialises, so the
    # library (static cudart) and torch agree on "device 0"
    if WORLD > 1 and "CUDA_VISIBLE_DEVICES" not in os.environ:
        os.environ["CUDA_VISIBLE_DEVICES"] = str(LOCAL_RANK)
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2607_02640_b200 import build as _build
    _build.build_library()
    from paper_2607_02640_b200 import replicas, synth
    from paper_2607_02640_b200 import workloads as wl
    from paper_2607_02640_b200.runner import Runner

    assert torch.cuda.is_available(), "bench.py needs a GPU (there is no CPU fallback for the product path)"
    torch.cuda.set_device(0)
    if WORLD > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", 0))

    if args.sweep:
        import bench_sweeps as sweeps
        if args.sweep == "age":
            rows = sweeps.age_sweep(args.config, n_sessions=args.sessions or None)
        elif args.sweep == "sessions":
            rows = sweeps.sessions_sweep(history_scale=args.history_scale)
        elif args.sweep == "admission":
            rows = sweeps.admission_run()
        elif args.sweep == "occupancy":
            rows = sweeps.occupancy_trace(n_sessions=args.sessions or 128)
        else:
            rows = sweeps.sw_sweep(n_sessions=args.sessions or 128)
        for row in rows:
            print(json.dumps(row), flush=True)
        return

    K, W = args.steps, max(args.warmup, 3)
    # a bench "step" = one FRAME (all its sub-steps: chunk prefill + decode steps) for every due
    # session.  The timed region is EXACTLY K frames; it is repeated REPS times on fresh frames (each
    # repeat bracketed on its own) so that at least 200 frames are timed whatever --steps says (SURVEY
    # sec. 8(d) ">= 200 timed frames"; a single 20-frame region of config 2 is 4 ms and moved by +-12 %
    # from run to run), and `value` is the MEDIAN repeat.  Every phase needs fresh frames: warm-up +
    # REPS x timed + stamped + bracketed + e2e warm-up + e2e timed.
    w0 = wl.make_workload(args.config, n_sessions=args.sessions or None)
    churn0 = w0.index == 5
    REPS = max(1, -(-200 // K)) if w0.index == 2 else 1     # (configs 3-5: 200 extra frames would age the sessions
    #                                                          past the config's age range; their frames are 9-17 launches)
    need = 2 * W + (REPS + 3) * K
    w = wl.make_workload(args.config, n_sessions=args.sessions or None, n_timed_frames=need)
    events, info = wl.build_schedule(w, history_scale=args.history_scale)
    NL = max(1, args.layers)
    global KV_FP8
    KV_FP8 = bool(args.kv_fp8)
    from paper_2607_02640_b200 import binding as _bind
    r = Runner(w, n_layers=NL, uid_base=replicas.uid_base(RANK), flags=_bind.FLAG_KV_FP8 if args.kv_fp8 else 0)
    r.pool.set_tuning(args.split_tokens, args.family, 0, 2 if args.fused_step else 0)
    t_hist = time.perf_counter()
    rest = r.run_history(events)
    torch.cuda.synchronize()
    t_hist = time.perf_counter() - t_hist
    frames, cur, cur_fid = [], [], None       # a frame = its opens/closes, then its steps
    for ev in rest:
        fid = ev[4] if ev[0] == "step" else None
        if cur and cur_fid is not None and fid != cur_fid:
            frames.append(cur)
            cur, cur_fid = [], None
        cur.append(ev)
        if fid is not None:
            cur_fid = fid
    if cur and cur_fid is not None:
        frames.append(cur)
    assert len(frames) >= need, (len(frames), need)

    # Sessions that open and close inside the timed frames (config 5, pool churn) need the frames
    # prepared one at a time (an open needs the slot an earlier frame's close frees): the GPU time of
    # the K frames is then the sum of K event brackets instead of one.
    churn = any(ev[0] != "step" for fr in frames for ev in fr)

    def prepare(frs):
        """Resolve the frames' steps and generate their inputs in HBM before the timed region."""
        out = []
        for fr in frs:
            for ev in fr:
                if ev[0] == "open":
                    r.open(ev[1]); continue
                if ev[0] == "close":
                    if churn:
                        r.close(ev[1]); continue       # frees the slot a later open of this frame needs
                    out.append(("close", r.sid[ev[1]], ev[1])); continue
                st = r.make_step(ev)
                k = r.rows(synth.STREAM_K, 0, st.uid_rows, st.pos_rows)
                v = r.rows(synth.STREAM_V, 0, st.uid_rows, st.pos_rows)
                q = r.rows(synth.STREAM_Q, 0, st.uid_rows, st.pos_rows)
                lens_after = [r.length[int(i)] for i in st.local]
                out.append((st, k, v, q, torch.empty_like(q), lens_after))
        return out

    def run(prepped):
        for item in prepped:
            if item[0] == "close":
                r.pool.session_close(item[1]); continue
            st, k, v, q, o, _ = item
            for layer in range(NL):                   # the same rows stand in for every layer's K/V/Q
                if args.two_calls:
                    r.pool.append_kv(layer, st.sids, st.n_new, k, v)
                    r.pool.attend_frame(layer, st.sids, st.n_new, q, o)
                else:
                    r.pool.append_attend(layer, st.sids, st.n_new, k, v, q, o)

    def finish_closes(prepped):
        for item in prepped:
            if item[0] == "close":
                i = item[2]
                r.sid.pop(i, None); r.uid.pop(i, None); r.length.pop(i, None)

    def session_frames(frs):
        return sum(len({int(i) for ev in fr if ev[0] == "step" for i in ev[1]}) for fr in frs)

    def barrier():
        torch.cuda.synchronize()
        if WORLD > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cursor = 0

    def take(n):
        nonlocal cursor
        frs = frames[cursor:cursor + n]
        cursor += n
        return frs

    def run_frames(frs, nvtx=None):
        """-> (prepared items, GPU milliseconds).  `nvtx` names the range around the library calls
        only (input generation stays outside), so `ncu --nvtx --nvtx-include` lists just our kernels."""
        total, allp = 0.0, []
        for group in ([[fr] for fr in frs] if churn else [frs]):
            prepped = prepare(group)
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            if nvtx:
                torch.cuda.nvtx.range_push(nvtx)
            e0.record()
            run(prepped)
            e1.record()
            if nvtx:
                torch.cuda.nvtx.range_pop()
            barrier()
            total += e0.elapsed_time(e1)
            if churn:
                finish_closes(prepped)
                # (one frame's K/V/Q at a time: keep the step records, drop the tensors)
                prepped = [it if it[0] == "close" else (it[0], None, None, None, None, it[5]) for it in prepped]
            allp += prepped
        if not churn:
            finish_closes(allp)
        return allp, total

    # ---- device-resident timing: W warm-up steps, then EXACTLY K timed steps (x REPS, median) ----
    run_frames(take(W))
    gpu_index = int(os.environ.get("CUDA_VISIBLE_DEVICES", str(LOCAL_RANK)).split(",")[0] or 0)
    sampler = ClockSampler(gpu_index) if RANK == 0 else None
    launches0 = r.pool.stats()["kernel_launches"]
    reps = []
    for _ in range(REPS):
        tf = take(K)
        _, ms_i = run_frames(tf, nvtx="metronome_timed")
        v_i, ms_i = replicas.aggregate(ms_i, session_frames(tf) * NL, device="cuda")   # max over ranks; per layer
        reps.append((ms_i, v_i))
    clocks = sampler.stop() if sampler else None
    launches = (r.pool.stats()["kernel_launches"] - launches0) // REPS
    ms, value = sorted(reps)[len(reps) // 2]

    # ---- roofline of the dominant kernel, measured two ways on K fresh frames each ----
    # (1) "in step": the attention kernels stamp %globaltimer themselves (first CTA in, last CTA out);
    #     launches exactly as in the timed region (programmatic edges, early mode): the kernel's span
    #     INSIDE a normal step, which is what the contract's `achieved` is.
    # (2) "alone": CUDA-event brackets around each attention launch; events break the programmatic
    #     edges, so the kernel runs alone, after its predecessor has drained (labelled as such).
    r.pool.set_profiling(2)
    st_items, st_ms = run_frames(take(K))
    kinds, spans, starts = r.pool.read_stamps()
    # A kernel launched programmatically starts while its predecessor's tail is still running, so raw spans
    # overlap and their sum can exceed the wall time.  The time a launch has the GPU to itself is its span
    # minus the part overlapped by the previous attention launch: that is what `achieved` divides by.
    import numpy as _np
    ends = starts + spans
    prev_end = _np.concatenate([[0.0], _np.maximum.accumulate(ends)[:-1]]) if len(ends) else ends
    excl = _np.where(spans >= 0, ends - _np.maximum(starts, prev_end), -1.0)
    r.pool.set_profiling(1)
    br_items, br_ms = run_frames(take(K))
    torch.cuda.synchronize()
    k_ms, k_n = r.pool.read_profile()
    r.pool.set_profiling(0)

    # per stamped launch: kind, algorithmic bytes and flops, in launch order
    exp = []
    for it in st_items:
        if it[0] == "close":
            continue
        st, lens_after = it[0], it[5]
        per_step = []
        for kind, mask in launch_classes(w, st.n_new, args.family):
            byt = sum(item_bytes(w, int(L), int(n)) for L, n, m in zip(lens_after, st.n_new, mask) if m)
            flo = sum(item_flops(w, int(L), int(n)) for L, n, m in zip(lens_after, st.n_new, mask) if m) if kind == 3 else 0
            per_step.append((kind, byt, flo))
        exp += per_step * NL
    peak, peak_src = peaks()
    pk = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
    per_kind = {}
    stamps_ok = len(exp) == len(kinds) and all(int(k) == e[0] for k, e in zip(kinds, exp)) and bool((spans >= 0).all())
    if stamps_ok:
        for (kind, byt, flo), sp, ex in zip(exp, spans, excl):
            d = per_kind.setdefault(kind, {"launches": 0, "ms": 0.0, "span_ms": 0.0, "bytes": 0, "flops": 0})
            d["launches"] += 1; d["ms"] += float(ex); d["span_ms"] += float(sp); d["bytes"] += byt; d["flops"] += flo
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    tj = json.load(open(tpath)) if os.path.exists(tpath) else {}

    def kind_obj(kind):
        d = per_kind[kind]
        gbs = d["bytes"] / (d["ms"] * 1e-3) / 1e9
        o = {"kernel": "attend_umma_fp8_kernel" if (KV_FP8 and kind == 3) else KIND_NAME[kind], "bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
             "launches": d["launches"], "kernel_ms_avg": d["ms"] / d["launches"],
             "raw_span_ms_avg": d["span_ms"] / d["launches"],
             "algorithmic_bytes_per_launch": d["bytes"] / d["launches"], "share_of_step": d["ms"] / st_ms,
             "frac_of_nominal_8TBs": gbs / 8000.0, "traffic": tj.get(f"config{w.index}{'_fp8' if KV_FP8 else ''}_{KIND_NAME[kind]}")}
        if kind == 3:
            tf_s = d["flops"] / (d["ms"] * 1e-3) / 1e12
            sustained = pk.get("bf16_tflops_sustained", 1423.1)
            o["tensor"] = {"bound": "tensor", "achieved": tf_s, "peak": sustained, "unit": "TFLOP/s", "frac": tf_s / sustained,
                           "peak_source": "MEASURED_PEAKS.json bf16_tflops_sustained (a kernel timed inside a long step)",
                           "frac_of_burst": tf_s / pk.get("bf16_tflops", 1694.4),
                           "algorithmic_gflop_per_launch": d["flops"] / d["launches"] / 1e9}
        return o

    if per_kind:
        dom = max(per_kind, key=lambda k_: per_kind[k_]["ms"])
        roofline = kind_obj(dom)
        roofline["pass"] = ("in step: %globaltimer stamps written by the kernel (first CTA in, last CTA out), launches exactly "
                            "as in the timed region (programmatic edges / early mode kept); kernel_ms_avg = span not "
                            "overlapped by the previous attention launch, raw_span_ms_avg = first CTA in to last CTA out")
        roofline["pass_ms_per_step"] = st_ms / K
        roofline["peak_source"] = peak_src
        roofline["other_kernels"] = [kind_obj(k_) for k_ in sorted(per_kind) if k_ != dom]
    else:
        roofline = {"bound": "hbm", "achieved": None, "peak": peak, "unit": "GB/s", "frac": None, "traffic": None,
                    "note": f"stamp pass unusable: expected {len(exp)} launches, got {len(kinds)}"}
    alg_bytes = NL * sum(algorithmic_bytes(w, it[5], it[0].n_new) for it in br_items if it[0] != "close")
    alone = alg_bytes / (k_ms * 1e-3) / 1e9 if k_ms > 0 else 0.0
    roofline["alone"] = {"pass": "brackets_on_no_pdl: CUDA events around every attention launch, plain launches, kernel "
                                 "runs after its predecessor has drained (all attention kernels of the step together)",
                         "achieved": alone, "frac": alone / peak, "kernel_ms_avg": k_ms / max(k_n, 1),
                         "pass_ms_per_step": br_ms / K, "share_of_its_pass": k_ms / br_ms if br_ms > 0 else None}
    achieved = roofline.get("achieved") or alone
    if RANK == 0:
        # read-only stream microbenchmark in the same job: a second, read-only denominator
        from paper_2607_02640_b200 import binding as _b
        rs = _b.stream_read_gbs(4 << 30, 5)
        roofline["read_stream_gbs"] = rs
        roofline["frac_of_read_stream"] = achieved / rs if rs > 0 else None
        roofline["note"] = ("peak is the driver's copy figure (read + write); a read-only stream on the same GPU reaches "
                            "read_stream_gbs, so frac can exceed 1: frac_of_read_stream is the tighter bound for a kernel "
                            "that only reads")

    # ---- end to end: HOST buffers through metronome_step_host, copies inside the timed region ----
    e2e = None
    if not args.no_e2e and not churn and NL == 1:       # (config 5 is a latency sweep workload: no host arm)
        def to_host(prepped):
            out = []
            for item in prepped:
                if item[0] == "close":
                    out.append(item); continue
                st, k, v, q, o, _ = item
                out.append((st, k.cpu().pin_memory(), v.cpu().pin_memory(), q.cpu().pin_memory(),
                            torch.empty(q.shape, dtype=q.dtype).pin_memory()))
            return out

        def run_host(hp):
            """Pipelined: step k's uploads are enqueued while step k-1 computes; the result of step k-1 is read on the
            host (so its D2H copy is inside the timed region) once at most one step is still in flight."""
            chk, inflight = 0.0, []
            for item in hp:
                if item[0] == "close":
                    r.pool.session_close(item[1]); continue
                st, k, v, q, o = item
                r.pool.step_host_async(0, st.sids, st.n_new, k, v, q, o)
                inflight.append(o)
                r.pool.step_host_wait(E2E_DEPTH)           # all but the newest E2E_DEPTH steps are complete:
                while len(inflight) > E2E_DEPTH:           # their results are read on the host while those run
                    chk += float(inflight.pop(0)[0, 0, 0])
            r.pool.step_host_wait(0)
            for o in inflight:
                chk += float(o[0, 0, 0])
            return chk
        hw_f, ht_f = take(W), take(K)
        hw = to_host(prepare(hw_f))
        run_host(hw)
        finish_closes(hw)
        ht = to_host(prepare(ht_f))
        barrier()
        t0 = time.perf_counter()
        run_host(ht)
        el = time.perf_counter() - t0
        e2e_value, el_ms = replicas.aggregate(el * 1e3, session_frames(ht_f), device="cuda")
        el = el_ms * 1e-3
        hsteps = [it for it in ht if it[0] != "close"]
        h2d = sum(k.numel() * 2 + v.numel() * 2 + q.numel() * 2 for _, k, v, q, _ in hsteps) / K
        d2h = sum(o.numel() * 2 for *_, o in hsteps) / K
        e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * el / K,
               "api": "metronome_step_host_async + metronome_step_host_wait(2) (pinned host buffers; event-free pipeline, three "
                      "staging slots: the uploads of the next steps and the read-back of the previous ones overlap the kernels "
                      "of step k; the result of step k-2 is read on the host inside the timed region)"}

    if RANK != 0:
        if WORLD > 1:
            dist.destroy_process_group()
        return
    cpu = None
    if not args.no_cpu_baseline and WORLD == 1:
        sample, what = oracle_sample(w0, args.history_scale)
        cpu = cpu_baseline(w0, sample, what, budget_s=12.0)
        one = cpu_baseline(w0, sample, what, budget_s=6.0, n_threads=1)      # 1 core and all cores
        cpu["single_core_value"] = one["value"]
        print(f"host: nproc={cpu['nproc']} cpu_model={cpu['cpu_model']}", file=sys.stderr)
    cfg = config_dict(w0, args, WORLD)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": WORLD, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16 in, f32 accumulate", "data": "synthetic", "config": cfg,
        "timed_repeats": {"n": REPS, "rule": "EXACTLY `steps` frames per repeat, each on fresh frames and bracketed on its "
                                             "own; value / ms_per_step are the median repeat",
                          "ms_per_step_each_in_time_order": [m_ / K for m_, _ in reps]},
        "history_build_s": round(t_hist, 2),
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
        "attention_gbs": achieved,
    }
    print(json.dumps(line), flush=True)
    if WORLD > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
