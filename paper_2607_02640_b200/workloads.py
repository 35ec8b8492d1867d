"""Seeded shape recipes for BASELINE.json's five configs.

Shapes only: session counts, head layout, (S, W), ages, chunk / decode lengths, arrival process.
No method arithmetic.  Used by tests/, bench.py and __graft_entry__.smoke(); values come from
synth.rows().  The paper's real-audio workloads and model weights are not
available; these synthetic sessions stand in for them.

A schedule is a list of events in issue order:
    ("open",  i)                          open workload-local session i
    ("close", i)                          close it
    ("step",  idx, n_new, timed, frame)   append n_new[j] tokens to session idx[j] and attend the
                                          same rows (decode: 1; chunk prefill: n);
                                          timed=False for history building, frame = frame number
Histories are built THROUGH the library, frame by frame, all sessions interleaved, so physical
blocks end up scattered as in a long-running server.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np

BASE_SEED = 260702640


@dataclass(frozen=True)
class Workload:
    index: int
    name: str
    n_sessions: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    S: int
    W: int
    max_new_tokens: int
    n_blocks: int
    block_size: int = 16
    n_timed_frames: int = 3
    max_sessions: int = 0            # 0 -> n_sessions
    outlier_frac: float = 0.0        # config 4
    outlier_scale: float = 1.0
    note: str = ""

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index

    @property
    def slots(self) -> int:
        return self.max_sessions or self.n_sessions

    def outlier_channels(self) -> np.ndarray:
        """round(frac * Hkv * D) channels of the flattened (KV head, dim) axis, seeded shuffle."""
        n = int(round(self.outlier_frac * self.n_kv_heads * self.head_dim))
        if n == 0:
            return np.zeros(0, dtype=np.int64)
        rng = np.random.default_rng(self.seed + 7)
        return np.sort(rng.permutation(self.n_kv_heads * self.head_dim)[:n]).astype(np.int64)


def blocks_per_session(S: int, W: int, B: int, n_max: int) -> int:
    """Sizing rule for the synthetic pools (same closed form the library exports)."""
    return -(-S // B) + (W + n_max - 1) // B + 2


def make_workload(index: int, n_sessions: int | None = None, n_timed_frames: int | None = None) -> Workload:
    """index 1..5 = BASELINE.json configs[0..4].  n_sessions shrinks a config for parity tests."""
    if index == 1:
        n = n_sessions or 4
        w = Workload(1, "tiny", n, 8, 2, 64, 4, 128, 8, n * blocks_per_session(4, 128, 16, 8),
                     n_timed_frames=3)
    elif index == 2:
        n = n_sessions or 128
        w = Workload(2, "moshi_shaped", n, 32, 32, 128, 4, 750, 1,
                     n * blocks_per_session(4, 750, 16, 1), n_timed_frames=200)
    elif index == 3:
        n = n_sessions or 128
        w = Workload(3, "qwen3_omni_shaped", n, 32, 4, 128, 4, 2048, 25,
                     n * blocks_per_session(4, 2048, 16, 25), n_timed_frames=8)
    elif index == 4:
        n = n_sessions or 256
        w = Workload(4, "minicpm_o_shaped", n, 32, 8, 128, 4, 1024, 25,
                     n * blocks_per_session(4, 1024, 16, 25), n_timed_frames=4,
                     outlier_frac=0.01, outlier_scale=20.0)
    elif index == 5:
        n = n_sessions or 512
        # pool = 80% of the UNBOUNDED working set of max_sessions sessions of mean lifetime 300
        # frames x 21 tokens (BASELINE.json config 5)
        per_session_unbounded = -(-300 * 21 // 16)
        w = Workload(5, "pool_churn", n, 32, 4, 128, 4, 2048, 13,
                     int(0.8 * n * per_session_unbounded), n_timed_frames=300, max_sessions=n)
    else:
        raise ValueError("config index must be 1..5")
    if n_timed_frames is not None:
        w = replace(w, n_timed_frames=n_timed_frames)
    return w


# ----------------------------------------------------------------------------- schedules


def _interleave(per_session_frames: list[list[list[int]]], timed: bool, frame0: int = 0):
    """per_session_frames[i] = list of frames, each a list of sub-step sizes.  Frames are aligned at
    the END (every session's last frame is the global last frame); inside a frame, sub-step j of
    every session that has one goes into one batched step."""
    events = []
    n_frames = max((len(f) for f in per_session_frames), default=0)
    for f in range(n_frames):
        active = []
        for i, frames in enumerate(per_session_frames):
            k = f - (n_frames - len(frames))
            if k >= 0:
                active.append((i, frames[k]))
        n_sub = max((len(fr) for _, fr in active), default=0)
        for j in range(n_sub):
            idx = [i for i, fr in active if j < len(fr) and fr[j] > 0]
            nn = [fr[j] for i, fr in active if j < len(fr) and fr[j] > 0]
            if idx:
                events.append(("step", np.asarray(idx, np.int32), np.asarray(nn, np.int32), timed, frame0 + f))
    return events


def _split_tokens(total: int, frame: list[int]) -> list[list[int]]:
    """Cut a history of `total` tokens into copies of `frame`, the LAST one truncated."""
    per = sum(frame)
    frames = [list(frame) for _ in range(total // per)]
    rem = total % per
    if rem:
        last = []
        for n in frame:
            take = min(n, rem)
            if take:
                last.append(take)
            rem -= take
        frames.append(last)
    return frames


def build_schedule(w: Workload, history_scale: float = 1.0):
    """Returns (events, info).  history_scale < 1 shortens the ages (parity tests at small cost)."""
    rng = np.random.default_rng(w.seed)
    n = w.n_sessions
    info = {}
    events = []
    if w.index == 1:
        frame = [8, 1, 1]
        ages = rng.integers(50, 401, size=n)
        ages = np.maximum(1, (ages * history_scale).astype(np.int64))
        events += [("open", i) for i in range(n)]
        events += _interleave([_split_tokens(int(a), frame) for a in ages], False)
        events += _interleave([[frame] * w.n_timed_frames for _ in range(n)], True)
        info["ages_tokens"] = ages
    elif w.index == 2:
        ages = rng.integers(1, 3751, size=n)
        ages = np.maximum(1, (ages * history_scale).astype(np.int64))
        events += [("open", i) for i in range(n)]
        events += _interleave([[[1]] * int(a) for a in ages], False)
        events += _interleave([[[1]] * w.n_timed_frames for _ in range(n)], True)
        info["ages_tokens"] = ages
    elif w.index == 3:
        frame = [25] + [1] * 8
        ages = rng.integers(0, 151, size=n)
        ages = (ages * history_scale).astype(np.int64)
        events += [("open", i) for i in range(n)]
        events += _interleave([[frame] * int(a) for a in ages], False)
        events += _interleave([[frame] * w.n_timed_frames for _ in range(n)], True)
        info["ages_frames"] = ages
    elif w.index == 4:
        ages = rng.integers(0, 601, size=n)
        ages = (ages * history_scale).astype(np.int64)

        def frames_for(k):
            out = []
            for _ in range(k):
                chunk = int(rng.integers(6, 26))
                dec = int(rng.integers(4, 17))
                out.append([chunk] + [1] * dec)
            return out
        events += [("open", i) for i in range(n)]
        events += _interleave([frames_for(int(a)) for a in ages], False)
        events += _interleave([frames_for(w.n_timed_frames) for _ in range(n)], True)
        info["ages_frames"] = ages
    elif w.index == 5:
        events, info = _churn_schedule(w, rng, n_target=n, history_scale=history_scale)
    return events, info


def _churn_schedule(w: Workload, rng, n_target: int, history_scale: float):
    """Config 5: Poisson arrivals at n_target/300 per frame, Exp(300-frame) lifetimes, 1 s frames,
    frame = 13-token chunk + 8 decode steps; starts from steady state (residual ages Exp(300))."""
    mean_life = 300.0 * history_scale
    frame = [13] + [1] * 8
    slots = w.slots
    events = []
    # steady-state population: n_target sessions whose elapsed age and remaining life are Exp(mean)
    n0 = min(n_target, slots)
    ages = np.floor(rng.exponential(mean_life, size=n0)).astype(np.int64)
    remaining = np.ceil(rng.exponential(mean_life, size=n0)).astype(np.int64)
    events += [("open", i) for i in range(n0)]
    events += _interleave([[frame] * int(a) for a in ages], False)
    alive = {i: int(remaining[i]) for i in range(n0)}        # local index -> frames left
    free_local = [i for i in range(slots - 1, n0 - 1, -1)]   # local indices not in use
    rejected = 0
    for f in range(w.n_timed_frames):
        for i in [i for i, r in alive.items() if r <= 0]:
            events.append(("close", i))
            del alive[i]
            free_local.append(i)
        free_local.sort(reverse=True)
        for _ in range(int(rng.poisson(n_target / mean_life))):
            if not free_local:
                rejected += 1
                continue
            i = free_local.pop()
            events.append(("open", i))
            alive[i] = int(np.ceil(rng.exponential(mean_life)))
        order = sorted(alive)
        if order:
            events += [("step", np.asarray(order, np.int32), np.full(len(order), n, np.int32), True, f)
                       for n in frame]
        for i in alive:
            alive[i] -= 1
    return events, {"initial_ages_frames": ages, "rejected_arrivals": rejected}


def churn_schedule(w: Workload, n_target: int, history_scale: float = 1.0):
    """Config 5 at one point of its concurrency sweep (n_target in {32..512})."""
    rng = np.random.default_rng(w.seed + 1000 * n_target)
    return _churn_schedule(w, rng, n_target, history_scale)
