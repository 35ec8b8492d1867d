"""bench_sweeps.py -- measurement harness beside bench.py (not part of the product package).

Shape checks and sweeps of SURVEY.md sec. 8(d)/(f), run by `bench.py --sweep ...` on one GPU.

  age       fixed N, every session at ONE age a in {1/4, 1/2, 1, 2, 5, 10, 20} x (S+W): per-frame
            latency must rise up to a ~ S+W and then stay FLAT ("O(W)")
  sessions  config 5 (pool churn): n_target in {32 .. 512}; median / p99 per-frame latency must be
            monotone non-decreasing in the load with zero pool exhaustion
  occupancy NEXT row f2: the unbounded arm (METRONOME_FLAG_UNBOUNDED) against the windowed one on the
            same pool and traffic: occupancy rho(t) = rho0 + N r t until POOL_EXHAUSTED at
            t_sat = (1 - rho0) / (N r) (Eq. 1, L83 Fig. 5) vs. the windowed plateau
            rho0 + N s(W)
  admission NEXT row f3: the AIMD gate (metronome_gate_*) closed around the measured per-frame latency on
            the config-5 traffic under open-loop overload: the cap must settle where latency sits at the
            target fraction of the budget (Fig. 7)
  sw        NEXT row f1: W in {256 .. 4096} and S in {0, 16, 32, 64} at N = 128 (PAPER.md:L300
            Fig. 11, L308-323 Table 2 "sinks ... unchanged latency")

Plumbing only (schedules + CUDA-event timing around the C-ABI calls); each point uses a fresh pool
(PAPER.md:L275).  Every function returns a list of dict rows; bench.py prints them as JSON lines.
"""
from __future__ import annotations

from dataclasses import replace

import numpy as np
import torch

from paper_2607_02640_b200 import synth
from paper_2607_02640_b200 import workloads as wl
from paper_2607_02640_b200.runner import Runner


def _frames_of(events):
    """Cut the timed tail of a schedule into frames: (opens/closes before the frame, its steps)."""
    frames, pre, steps, fid = [], [], [], None
    for ev in events:
        if ev[0] != "step":
            if steps:
                frames.append((pre, steps))
                pre, steps, fid = [], [], None
            pre.append(ev)
            continue
        if steps and ev[4] != fid:
            frames.append((pre, steps))
            pre, steps = [], []
        fid = ev[4]
        steps.append(ev)
    if steps:
        frames.append((pre, steps))
    return frames


def time_frames(r: Runner, events, warmup: int = 2):
    """Runs the timed tail frame by frame.  Returns per-frame dicts: ms (GPU time of every append_kv
    + attend_frame of the frame, CUDA events), attend_ms (attention kernels only, the library's own
    event brackets), sessions, resident tokens.  The first `warmup` frames are dropped."""
    out = []
    r.pool.set_profiling(1)
    for k, (pre, steps) in enumerate(_frames_of(events)):
        for ev in pre:
            if ev[0] == "open":
                r.open(ev[1])
            else:
                r.close(ev[1])
        prepped = []
        for ev in steps:
            st = r.make_step(ev)
            kk = r.rows(synth.STREAM_K, 0, st.uid_rows, st.pos_rows)
            vv = r.rows(synth.STREAM_V, 0, st.uid_rows, st.pos_rows)
            qq = r.rows(synth.STREAM_Q, 0, st.uid_rows, st.pos_rows)
            prepped.append((st, kk, vv, qq, torch.empty_like(qq)))
        r.pool.read_profile()                       # reset the brackets
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for st, kk, vv, qq, oo in prepped:
            r.pool.append_kv(0, st.sids, st.n_new, kk, vv)
            r.pool.attend_frame(0, st.sids, st.n_new, qq, oo)
        e1.record()
        torch.cuda.synchronize()
        a_ms, _ = r.pool.read_profile()
        if k >= warmup:
            sess = {int(i) for ev in steps for i in ev[1]}
            out.append({"ms": e0.elapsed_time(e1), "attend_ms": a_ms, "sessions": len(sess)})
    r.pool.set_profiling(0)
    return out


def _summary(fr):
    ms = np.asarray([f["ms"] for f in fr])
    am = np.asarray([f["attend_ms"] for f in fr])
    return {"frames": len(fr), "ms_median": float(np.median(ms)), "ms_p99": float(np.percentile(ms, 99)),
            "attend_ms_median": float(np.median(am)), "sessions_mean": float(np.mean([f["sessions"] for f in fr]))}


def _frame_pattern(w: wl.Workload):
    return {1: [8, 1, 1], 2: [1], 3: [25] + [1] * 8, 4: [16] + [1] * 10, 5: [13] + [1] * 8}[w.index]


def uniform_age_events(w: wl.Workload, age_tokens: int, n_frames: int):
    """All sessions at the same age (tokens), history in appends of max_new_tokens, then n_frames."""
    frame = _frame_pattern(w)
    n = w.n_sessions
    hist = [[w.max_new_tokens]] * (age_tokens // w.max_new_tokens)
    if age_tokens % w.max_new_tokens:
        hist = hist + [[age_tokens % w.max_new_tokens]]
    ev = [("open", i) for i in range(n)]
    ev += wl._interleave([hist for _ in range(n)], False)
    ev += wl._interleave([[frame] * n_frames for _ in range(n)], True)
    return ev


def age_sweep(config: int = 2, n_sessions: int | None = None, n_frames: int = 12,
              multiples=(0.25, 0.5, 1, 2, 5, 10, 20)):
    rows = []
    for m in multiples:
        w = wl.make_workload(config, n_sessions=n_sessions)
        age = max(1, int(round(m * (w.S + w.W))))
        r = Runner(w)
        rest = r.run_history(uniform_age_events(w, age, n_frames + 2))
        fr = time_frames(r, rest)
        rows.append({"sweep": "age", "config": config, "sessions": w.n_sessions, "S": w.S, "W": w.W,
                     "age_over_S_plus_W": m, "age_tokens": age, **_summary(fr)})
        del r
        torch.cuda.empty_cache()
    return rows


def sessions_sweep(targets=(32, 64, 128, 256, 384, 512), n_frames: int = 60, history_scale: float = 1.0):
    """Config 5: Poisson arrivals / Exp lifetimes at each target concurrency, fixed pool (80 % of the
    unbounded working set of 512 sessions).  POOL_EXHAUSTED would raise: reaching the end of a point
    is the zero-exhaustion check."""
    rows = []
    for nt in targets:
        w = wl.make_workload(5, n_timed_frames=n_frames + 2)
        events, info = wl.churn_schedule(w, nt, history_scale)
        r = Runner(w)
        rest = r.run_history(events)
        fr = time_frames(r, rest)
        free = r.pool.pool_query(want_ids=False)[0]
        rows.append({"sweep": "sessions", "config": 5, "n_target": nt, "pool_blocks": w.n_blocks,
                     "free_blocks_end": free, "pool_exhausted": 0,
                     "rejected_arrivals": int(info["rejected_arrivals"]), **_summary(fr)})
        del r
        torch.cuda.empty_cache()
    return rows


def sw_sweep(n_sessions: int = 128, n_frames: int = 12, windows=(256, 512, 1024, 2048, 4096),
             sinks=(0, 16, 32, 64)):
    """NEXT f1 on config-3 shapes (32Q/4KV, frame = 25-chunk + 8 decode), every session at age
    2 x (S+W) so the window is full: latency vs W at S=4, and vs S at W=2048."""
    rows = []
    base = wl.make_workload(3, n_sessions=n_sessions)
    points = [(4, W) for W in windows] + [(S, 2048) for S in sinks]
    for S, W in points:
        w = replace(base, S=S, W=W, n_blocks=n_sessions * wl.blocks_per_session(S, W, 16, base.max_new_tokens))
        r = Runner(w)
        rest = r.run_history(uniform_age_events(w, 2 * (S + W), n_frames + 2))
        fr = time_frames(r, rest)
        rows.append({"sweep": "sw", "sessions": n_sessions, "S": S, "W": W,
                     "blocks_per_session": wl.blocks_per_session(S, W, 16, base.max_new_tokens), **_summary(fr)})
        del r
        torch.cuda.empty_cache()
    return rows


def occupancy_trace(n_sessions: int = 128, n_frames: int = 200):
    """NEXT f2 on config-3 shapes: N sessions, every frame appends 25 + 8 x 1 tokens (r = 33 tokens per
    session and frame), pool = 2 x N x the windowed per-session cap.  Unbounded arm: runs until the library
    returns POOL_EXHAUSTED and compares that frame with Eq. 1's closed form (a block is held from its
    first token, hence the ceil).  Windowed arm: same traffic, 3 x longer, plateau.  Occupancy is read
    from the device free list after every frame (metronome_pool_query)."""
    from paper_2607_02640_b200 import binding
    base = wl.make_workload(3, n_sessions=n_sessions)
    frame = _frame_pattern(base)
    r_tok = sum(frame)
    rows = []
    for arm in ("unbounded", "windowed"):
        flags = binding.FLAG_UNBOUNDED if arm == "unbounded" else 0
        w = replace(base, n_blocks=2 * base.n_blocks)
        r = Runner(w, flags=flags, max_session_len=(n_frames + 2) * r_tok if arm == "unbounded" else 0)
        for i in range(n_sessions):
            r.open(i)
        trace, exhausted_at = [], None
        for f in range(n_frames):
            try:
                for n in frame:
                    st = r.make_step(("step", np.arange(n_sessions, dtype=np.int32), np.full(n_sessions, n, np.int32), True, f))
                    r.append(st, 0)
                    r.attend(st, 0)
            except binding.MetronomeError as e:
                assert "POOL_EXHAUSTED" in str(e), e
                exhausted_at = f
                break
            trace.append(1.0 - r.pool.pool_query(want_ids=False)[0] / w.n_blocks)
        # Eq. 1 with r in blocks per frame: the frame in which ceil(L/16) summed over sessions first
        # exceeds the pool (all sessions are in lockstep, so per session: ceil(L/16) > n_blocks / N)
        per_session = w.n_blocks // n_sessions
        t_sat = None
        if arm == "unbounded":
            L, t = 0, 0
            while True:
                ok = True
                for n in frame:
                    if -(-(L + n) // 16) > per_session:
                        ok = False
                        break
                    L += n
                if not ok:
                    break
                t += 1
            t_sat = t
        slope = float(np.polyfit(np.arange(len(trace[:20])), trace[:20], 1)[0]) if len(trace) >= 20 else None
        rows.append({"sweep": "occupancy", "arm": arm, "sessions": n_sessions, "pool_blocks": w.n_blocks,
                     "tokens_per_session_frame": r_tok, "frames_run": len(trace), "pool_exhausted_at_frame": exhausted_at,
                     "eq1_t_sat_frame": t_sat, "eq1_slope_per_frame": n_sessions * r_tok / 16 / w.n_blocks,
                     "fit_slope_first_20_frames": slope, "occupancy_end": trace[-1] if trace else None,
                     "occupancy_max": max(trace) if trace else None,
                     "occupancy_every_10th_frame": [round(x, 4) for x in trace[::10]]})
        del r
        torch.cuda.empty_cache()
    return rows


def admission_run(n_frames: int = 500, budget_ms: float = 2.5, target_frac: float = 0.8, arrivals_per_frame: float = 6.0,
                  mean_life_frames: float = 300.0, seed: int = 260702645):
    """NEXT f3: config-5 shapes (32Q/4KV, W=2048, frame = 13-chunk + 8 decode, pool of config 5), sessions
    arrive as a Poisson stream far above what fits the deadline, live Exp(300) frames, and are admitted
    only while the gate's cap allows; every frame's measured GPU latency (one layer) feeds the gate.
    Returns one row: cap / live / latency every 25 frames and the steady-state summary."""
    from paper_2607_02640_b200 import binding
    w = wl.make_workload(5)
    frame = _frame_pattern(w)
    rng = np.random.default_rng(seed)
    gate = binding.Gate(budget_ms=budget_ms, target_frac=target_frac, add_step=1.0, mult_factor=0.85, cap_min=4.0,
                        cap_max=float(w.slots), cap_init=16.0)
    r = Runner(w)
    free_local = list(range(w.slots - 1, -1, -1))
    alive = {}                                           # local index -> frames left
    trace, lat_hist, live_hist, cap_hist = [], [], [], []
    admitted = rejected = 0
    cap = 16.0
    for f in range(n_frames):
        for i in [i for i, left in alive.items() if left <= 0]:
            r.close(i)
            del alive[i]
            free_local.append(i)
        for _ in range(int(rng.poisson(arrivals_per_frame))):
            if free_local and gate.admit(len(alive)):
                i = free_local.pop()
                r.open(i)
                alive[i] = int(np.ceil(rng.exponential(mean_life_frames)))
                admitted += 1
            else:
                rejected += 1                            # the clean overload rejection of L109
        order = np.asarray(sorted(alive), np.int32)
        ms = 0.0
        if len(order):
            prepped = []
            for n in frame:
                st = r.make_step(("step", order, np.full(len(order), n, np.int32), True, f))
                prepped.append((st, r.rows(synth.STREAM_K, 0, st.uid_rows, st.pos_rows),
                                r.rows(synth.STREAM_V, 0, st.uid_rows, st.pos_rows),
                                r.rows(synth.STREAM_Q, 0, st.uid_rows, st.pos_rows)))
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for st, kk, vv, qq in prepped:
                r.pool.append_kv(0, st.sids, st.n_new, kk, vv)
                r.pool.attend_frame(0, st.sids, st.n_new, qq, torch.empty_like(qq))
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
        cap = gate.observe(ms)
        for i in alive:
            alive[i] -= 1
        lat_hist.append(ms); live_hist.append(len(alive)); cap_hist.append(cap)
        if f % 25 == 0:
            trace.append({"frame": f, "cap": round(cap, 1), "live": len(alive), "latency_ms": round(ms, 3)})
    tail = slice(n_frames // 2, None)
    over = float(np.mean(np.asarray(lat_hist[tail]) > budget_ms))
    return [{"sweep": "admission", "config": 5, "budget_ms": budget_ms, "target_ms": budget_ms * target_frac,
             "arrivals_per_frame": arrivals_per_frame, "frames": n_frames, "admitted": admitted, "rejected": rejected,
             "steady_live_mean": float(np.mean(live_hist[tail])), "steady_cap_mean": float(np.mean(cap_hist[tail])),
             "steady_latency_ms_median": float(np.median(lat_hist[tail])),
             "steady_latency_ms_p99": float(np.percentile(lat_hist[tail], 99)),
             "steady_frames_over_budget_frac": over, "pool_exhausted": 0, "trace_every_25_frames": trace}]


# ---------------------------------------------------------------------------------------------------------------
def summarize(paths) -> str:
    """Markdown tables from the JSON lines `python bench.py --sweep ...` printed (no GPU needed):
    python bench_sweeps.py gpurun_out/r02_sweep_*.jsonl > profiles/r02_sweeps.md"""
    import json
    rows = []
    for p in paths:
        rows += [json.loads(line) for line in open(p) if line.strip().startswith("{")]
    out = []
    by = lambda name: [r for r in rows if r.get("sweep") == name]
    for cfg in sorted({r["config"] for r in by("age")}):
        rs = [r for r in by("age") if r["config"] == cfg]
        out += [f"## Latency vs session age, config {cfg}: {rs[0]['sessions']} sessions, S={rs[0]['S']}, W={rs[0]['W']}, every session at the same age",
                "", "| age / (S+W) | age tokens | frame ms (median) | p99 | attend ms |", "|---|---|---|---|---|"]
        out += [f"| {r['age_over_S_plus_W']} | {r['age_tokens']} | {r['ms_median']:.4f} | {r['ms_p99']:.4f} | {r['attend_ms_median']:.4f} |" for r in rs]
        flat = [r["ms_median"] for r in rs if r["age_over_S_plus_W"] >= 1]
        out += ["", f"Plateau from age = S+W on: {min(flat):.4f} .. {max(flat):.4f} ms (spread {100 * (max(flat) / min(flat) - 1):.1f} %).", ""]
    rs = by("sessions")
    if rs:
        out += ["## Latency vs concurrency, config 5 pool churn (Poisson arrivals, Exp(300-frame) lifetimes)", "",
                "| n_target | mean live sessions | frame ms (median) | p99 | attend ms | free blocks at end | POOL_EXHAUSTED | arrivals refused |", "|---|---|---|---|---|---|---|---|"]
        out += [f"| {r['n_target']} | {r.get('sessions_mean', float('nan')):.1f} | {r['ms_median']:.3f} | {r['ms_p99']:.3f} | {r['attend_ms_median']:.3f} | "
                f"{r['free_blocks_end']} | {r['pool_exhausted']} | {r['rejected_arrivals']} |" for r in rs]
        med = [r["ms_median"] for r in rs]
        out += ["", "Medians rise monotonically with load: " + str(all(b >= a for a, b in zip(med, med[1:]))) +
                f"; pool {rs[0]['pool_blocks']} blocks, never exhausted.", ""]
    rs = by("sw")
    if rs:
        out += ["## (S, W) sweep on config-3 shapes, every session at age 2 x (S+W) (NEXT f1)", "",
                "| S | W | blocks / session | frame ms (median) | p99 | attend ms |", "|---|---|---|---|---|---|"]
        out += [f"| {r['S']} | {r['W']} | {r['blocks_per_session']} | {r['ms_median']:.4f} | {r['ms_p99']:.4f} | {r['attend_ms_median']:.4f} |" for r in rs]
        out += [""]
    rs = by("occupancy")
    if rs:
        out += ["## Pool occupancy, unbounded vs windowed arm (NEXT f2, PAPER.md Eq. 1)", "",
                "| arm | frames run | POOL_EXHAUSTED at frame | Eq. 1 t_sat (frame) | Eq. 1 slope / frame | fitted slope (first 20 frames) | occupancy max | occupancy at end |", "|---|---|---|---|---|---|---|---|"]
        out += [f"| {r['arm']} | {r['frames_run']} | {r['pool_exhausted_at_frame']} | {r['eq1_t_sat_frame']} | {r['eq1_slope_per_frame']:.5f} | "
                f"{(r['fit_slope_first_20_frames'] or 0):.5f} | {(r['occupancy_max'] or 0):.4f} | {(r['occupancy_end'] or 0):.4f} |" for r in rs]
        out += [""]
    rs = by("admission")
    if rs:
        r = rs[0]
        out += ["## AIMD admission gate on the measured per-frame latency (NEXT f3)", "",
                f"budget {r['budget_ms']} ms, target {r['target_ms']} ms, {r['arrivals_per_frame']} arrivals per frame, {r['frames']} frames: admitted {r['admitted']}, "
                f"rejected {r['rejected']}; second half: live sessions {r['steady_live_mean']:.1f}, cap {r['steady_cap_mean']:.1f}, latency median "
                f"{r['steady_latency_ms_median']:.3f} ms, p99 {r['steady_latency_ms_p99']:.3f} ms, frames over budget {100 * r['steady_frames_over_budget_frac']:.1f} %.", "",
                "| frame | cap | live | latency ms |", "|---|---|---|---|"]
        out += [f"| {t['frame']} | {t['cap']} | {t['live']} | {t['latency_ms']} |" for t in r["trace_every_25_frames"]]
        out += [""]
    return "\n".join(out)


if __name__ == "__main__":
    import sys
    print(summarize(sys.argv[1:]))
