"""Full-size GPU parity (`-m gpu`): BASELINE.json's configs at their real sizes, in the launch
configuration bench.py times (automatic kernel family and split), checked on

  * sampled outputs the oracle computes one by one: for sampled sessions, every query row of a timed
    step against oracle.attend() on K/V rows regenerated on the CPU (only sinks and the union window
    can be admitted, so only those rows are regenerated);
  * bookkeeping at full size: every session's block table, first live block, length, and the whole
    free list, bit-exact against a bookkeeping-only replay in the oracle;
  * properties that hold at any size: all outputs finite, free + resident = n_blocks.
"""
import numpy as np
import pytest
import torch

from oracle import bounded_kv as O
from oracle import kv_fp8 as F
from paper_2607_02640_b200 import binding, synth
from paper_2607_02640_b200 import workloads as wl
from paper_2607_02640_b200.runner import Runner
from parity_helpers import assert_parity, oracle_cfg

pytestmark = pytest.mark.gpu


def _reference_rows(r, w, local, n, layer=0, kv_fp8=False):
    """oracle output for the last n rows of workload-local session `local` (definition layer on the
    rows that can be admitted; kv_fp8: on what their stored fp8 form decodes to, oracle/kv_fp8.py)."""
    L = r.length[local]
    lo = max(0, L - n - w.W + 1)
    pos = np.concatenate([np.arange(0, min(w.S, lo)), np.arange(lo, L)]).astype(np.int64)
    uid = np.full(len(pos), r.uid[local], np.int64)
    k = synth.to_u16(r.rows(synth.STREAM_K, layer, uid, pos, device="cpu"))
    v = synth.to_u16(r.rows(synth.STREAM_V, layer, uid, pos, device="cpu"))
    qpos = np.arange(L - n, L, dtype=np.int64)
    q = synth.to_u16(r.rows(synth.STREAM_Q, layer, np.full(n, r.uid[local], np.int64), qpos, device="cpu"))
    if kv_fp8:
        k, v = F.roundtrip(k), F.roundtrip(v)
    return O.attend(q, qpos, k, v, pos, w.S, w.W, None, "f32", False, O.max_threads())


def _run_fullsize(index, n_frames, n_sample, history_scale=1.0, n_sessions=None, kv_fp8=False):
    w = wl.make_workload(index, n_sessions=n_sessions, n_timed_frames=n_frames)
    events, _ = wl.build_schedule(w, history_scale=history_scale)
    r = Runner(w, flags=binding.FLAG_KV_FP8 if kv_fp8 else 0)
    book = O.PagedOracle(oracle_cfg(w), store_kv=False)          # bookkeeping-only replay
    osid = {}
    rng = np.random.default_rng(w.seed + 5)
    # history through the library (batched generation), mirrored into the bookkeeping oracle
    k = 0
    while k < len(events) and not (events[k][0] == "step" and events[k][3]):
        ev = events[k]
        if ev[0] == "open":
            osid[ev[1]] = book.session_open()
        elif ev[0] == "close":
            book.session_close(osid.pop(ev[1]))
        else:
            book.append_kv(0, [osid[int(i)] for i in ev[1]], [int(n) for n in ev[2]])
        k += 1
    rest = r.run_history(events)
    assert len(rest) == len(events) - k
    worst = {"max_abs": 0.0, "max_rel": 0.0, "row_l2": 0.0}
    checked_rows = 0
    for ev in rest:
        if ev[0] == "open":
            r.open(ev[1]); osid[ev[1]] = book.session_open(); continue
        if ev[0] == "close":
            r.close(ev[1]); book.session_close(osid.pop(ev[1])); continue
        st = r.make_step(ev)
        r.append(st, 0)
        book.append_kv(0, [osid[int(i)] for i in st.local], [int(n) for n in st.n_new])
        rows = int(st.n_new.sum())
        out = torch.full((rows, w.n_q_heads, w.head_dim), float("nan"), dtype=torch.bfloat16, device="cuda")
        out = r.attend(st, 0, out=out)                 # (NaN first: a row no CTA wrote cannot pass as finite)
        assert torch.isfinite(out.float()).all()
        # sampled sessions of this step: always include the youngest and the oldest due session
        lens = np.array([r.length[int(i)] for i in st.local])
        pick = set(int(x) for x in rng.permutation(len(st.local))[:n_sample])
        pick |= {int(lens.argmin()), int(lens.argmax())}
        offs = np.concatenate([[0], np.cumsum(st.n_new)])
        for j in sorted(pick):
            n = int(st.n_new[j])
            ref = _reference_rows(r, w, int(st.local[j]), n, kv_fp8=kv_fp8)
            rep = assert_parity(out[offs[j]:offs[j] + n], ref, f"{w.name} frame {st.frame} session {st.local[j]} len {lens[j]}",
                                unit_scale=w.outlier_frac == 0)
            checked_rows += n
            for key in worst:
                worst[key] = max(worst[key], rep[key])
    # bookkeeping, full size, bit-exact
    n_free, free_ids = r.pool.pool_query()
    assert free_ids == book.pool_query()
    resident = 0
    for i, s in osid.items():
        got, want = r.pool.session_query(r.sid[i]), book.session_query(s)
        assert (got[0], got[1], got[2]) == (want[0], want[1], want[2]), i
        resident += len(got[2])
    assert n_free + resident == w.n_blocks
    print(f"config {index}{' fp8 KV' if kv_fp8 else ''}: {checked_rows} sampled rows x {w.n_q_heads} heads, worst {worst}")
    return worst


def test_config2_full_size_sampled():
    """configs[1], exactly what bench.py times: 128 sessions, ages U{1..3750}, decode frames."""
    _run_fullsize(2, n_frames=3, n_sample=6)


def test_config3_full_size_sampled():
    """configs[2]: 128 sessions, GQA 8, W=2048, 25-token chunk + 8 decode steps per frame."""
    _run_fullsize(3, n_frames=1, n_sample=3)


def test_config4_full_size_sampled():
    """configs[3] at its stated size: 256 sessions, GQA 4, W=1024, ages U{0..600} frames, ragged chunks /
    decode counts, x20 outlier channels."""
    _run_fullsize(4, n_frames=1, n_sample=2)


def test_config5_churn_sampled():
    """configs[4] at its stated size: 512 sessions, Exp(300-frame) lifetimes, Poisson opens / closes inside
    the timed frames.  A CTA's share of the GQA decode kernel is >= 512 tiles here, so this is also the
    launch configuration that takes the dynamically claimed tail ranges by itself."""
    _run_fullsize(5, n_frames=3, n_sample=2)


def test_config3_fp8_full_size_sampled():
    """configs[2] on an fp8 (E4M3) KV pool (NEXT row f4, "the two compose"): the 8 decode steps of the
    frame run on the GQA decode kernel's fp8 tile, the 25-token chunk on the row kernel."""
    _run_fullsize(3, n_frames=1, n_sample=3, kv_fp8=True)


def test_config4_fp8_full_size_sampled():
    """configs[3] on an fp8 KV pool: the x20 outlier channels give rows whose scales differ by 20x inside one tile
    (the V scale is folded into the softmax weight relative to a running reference)."""
    _run_fullsize(4, n_frames=1, n_sample=2, kv_fp8=True)


def test_config5_fp8_churn_sampled():
    """configs[4] on an fp8 KV pool: the dynamically claimed tail ranges of the GQA decode kernel with fp8 tiles."""
    _run_fullsize(5, n_frames=2, n_sample=2, kv_fp8=True)
