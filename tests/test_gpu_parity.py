"""GPU parity tests (`-m gpu`): the CUDA path, through the C ABI, against the oracle.

Bookkeeping (block tables, free list, eviction order) must match bit-exactly after every call;
attention within north_star's tolerance (helpers.assert_parity).  Every input is seeded
(synth.rows) and regenerated on the CPU for the oracle; nothing here reads /root/reference.
"""
import os

import numpy as np
import pytest
import torch

from oracle import bounded_kv as O
from paper_2607_02640_b200 import binding, synth
from paper_2607_02640_b200 import workloads as wl
from paper_2607_02640_b200.runner import Runner
from parity_helpers import OracleMirror, assert_parity, parity_report
from test_oracle_bookkeeping import GOLDEN, parse_trace, run_trace

pytestmark = pytest.mark.gpu


def _loaded_native():
    """The driver checks that the in-tree .so is what ran: fail loudly if it is not loaded."""
    with open("/proc/self/maps") as f:
        assert "libmetronome.so" in f.read(), "native library not loaded"


# ------------------------------------------------------------------------------ bookkeeping


def test_hand_trace_on_device():
    def make(B, S, W, n_blocks):
        return binding.Pool(n_q_heads=1, n_kv_heads=1, head_dim=64, n_sinks=S, window=W, n_blocks=n_blocks,
                            max_sessions=4, max_new_tokens=8, block_size=B, flags=binding.FLAG_BOOKKEEPING_ONLY)

    run_trace(parse_trace(os.path.join(GOLDEN, "bookkeeping_hand_trace.txt")), make,
              lambda p, sids, n: p.append_kv(0, sids, n, None, None),
              lambda p, sid: p.session_close(sid), lambda p: p.session_open(),
              lambda p, sid: p.session_query(sid), lambda p: p.pool_query()[1])
    _loaded_native()


@pytest.mark.parametrize("S,W,B,n_blocks,seed", [(4, 32, 16, 20, 0), (0, 20, 16, 12, 1), (17, 40, 16, 64, 2),
                                                 (3, 7, 4, 30, 3), (40, 5, 8, 60, 4), (4, 2048, 16, 700, 5)])
def test_bookkeeping_fuzz_bit_exact(S, W, B, n_blocks, seed):
    """Random open / append / close traffic incl. pool exhaustion: tables and free list after EVERY call."""
    rng = np.random.default_rng(seed)
    n_max, slots = 25, 6
    pool = binding.Pool(n_q_heads=1, n_kv_heads=1, head_dim=64, n_sinks=S, window=W, n_blocks=n_blocks,
                        max_sessions=slots, max_new_tokens=n_max, block_size=B, flags=binding.FLAG_BOOKKEEPING_ONLY)
    ora = O.PagedOracle(O.PoolConfig(n_q_heads=1, n_kv_heads=1, head_dim=64, S=S, W=W, n_blocks=n_blocks,
                                     block_size=B, max_sessions=slots, max_new_tokens=n_max), store_kv=False)
    live, exhausted = [], 0
    for step in range(400):
        r = rng.random()
        if (r < 0.1 and len(live) < slots) or not live:
            a, b = pool.session_open(), ora.session_open()
            assert a == b
            live.append(a)
        elif r < 0.15:
            sid = live.pop(int(rng.integers(len(live))))
            pool.session_close(sid); ora.session_close(sid)
        else:
            k = int(rng.integers(1, len(live) + 1))
            sids = [int(x) for x in rng.permutation(live)[:k]]
            n_new = [int(rng.integers(1, n_max + 1)) if rng.random() < 0.5 else 1 for _ in sids]
            err = None
            try:
                ora.append_kv(0, sids, n_new)
            except O.OracleError as e:
                err = e.code
            if err:
                exhausted += 1
                with pytest.raises(binding.MetronomeError, match=err):
                    pool.append_kv(0, sids, n_new, None, None)
            else:
                pool.append_kv(0, sids, n_new, None, None)
        for sid in live:
            got, want = pool.session_query(sid), ora.session_query(sid)
            assert (got[0], got[1], got[2]) == (want[0], want[1], want[2]), (step, sid)
        assert pool.pool_query()[1] == ora.pool_query(), step
    if n_blocks <= 20:
        assert exhausted > 0, "the fuzz never reached pool exhaustion"


def test_error_codes_and_no_state_change():
    pool = binding.Pool(n_q_heads=4, n_kv_heads=2, head_dim=64, n_sinks=4, window=32, n_blocks=7,
                        max_sessions=2, max_new_tokens=16)
    a = pool.session_open(); b = pool.session_open()
    with pytest.raises(binding.MetronomeError, match="SESSIONS_FULL"):
        pool.session_open()
    k = torch.zeros(64, 2, 64, dtype=torch.bfloat16, device="cuda")
    q = torch.zeros(64, 4, 64, dtype=torch.bfloat16, device="cuda")
    for sids, n, code in [([a, a], [1, 1], "DUPLICATE_SESSION"), ([5], [1], "INVALID_SESSION"),
                          ([a], [17], "CHUNK_TOO_LARGE"), ([a], [-1], "INVALID_ARG")]:
        with pytest.raises(binding.MetronomeError, match=code):
            pool.append_kv(0, sids, n, k, k)
    with pytest.raises(binding.MetronomeError, match="QLEN_EXCEEDS_LAST_APPEND"):
        pool.attend_frame(0, [a], [1], q, q)            # nothing appended yet
    pool.append_kv(0, [a, b], [16, 16], k, k)
    pool.append_kv(0, [a, b], [16, 16], k, k)
    pool.append_kv(0, [a, b], [16, 16], k, k)           # 6 of 7 blocks in use
    before = (pool.session_query(a), pool.session_query(b), pool.pool_query())
    with pytest.raises(binding.MetronomeError, match="POOL_EXHAUSTED"):
        pool.append_kv(0, [a, b], [16, 16], k, k)       # L0=48, W=32: nothing is behind the window yet; needs 2
    assert (pool.session_query(a), pool.session_query(b), pool.pool_query()) == before
    with pytest.raises(binding.MetronomeError, match="QLEN_EXCEEDS_LAST_APPEND"):
        pool.attend_frame(0, [a], [17], q, q)
    pool.session_close(a)
    with pytest.raises(binding.MetronomeError, match="INVALID_SESSION"):
        pool.session_close(a)
    assert pool.session_open() == a
    # layers: layer 1 must repeat layer 0's batch, once; attend needs this step's append on that layer
    p2 = binding.Pool(n_q_heads=4, n_kv_heads=2, head_dim=64, n_sinks=4, window=32, n_blocks=8,
                      max_sessions=2, max_new_tokens=16, n_layers=2)
    s0 = p2.session_open()
    with pytest.raises(binding.MetronomeError, match="LAYER_SEQUENCE"):
        p2.append_kv(1, [s0], [3], k, k)
    p2.append_kv(0, [s0], [3], k, k)
    with pytest.raises(binding.MetronomeError, match="LAYER_SEQUENCE"):
        p2.attend_frame(1, [s0], [3], q, q)
    with pytest.raises(binding.MetronomeError, match="LAYER_SEQUENCE"):
        p2.append_kv(1, [s0], [2], k, k)
    p2.append_kv(1, [s0], [3], k, k)
    p2.attend_frame(1, [s0], [3], q, q)
    with pytest.raises(binding.MetronomeError, match="LAYER_SEQUENCE"):
        p2.append_kv(1, [s0], [3], k, k)
    torch.cuda.synchronize()


# ------------------------------------------------------------------------------ KV write


def test_kv_write_reads_back_through_the_table():
    w = wl.make_workload(1)
    r = Runner(w)
    events, _ = wl.build_schedule(w)
    rest = r.run_history(events)
    for i in range(w.n_sessions):
        L = r.length[i]
        k = torch.empty(L, w.n_kv_heads, w.head_dim, dtype=torch.bfloat16, device="cuda")
        v = torch.empty_like(k)
        r.pool.read_kv(0, r.sid[i], 0, L, k, v)
        pos = np.arange(L)
        want_k = r.rows(synth.STREAM_K, 0, np.full(L, r.uid[i]), pos, device="cpu")
        want_v = r.rows(synth.STREAM_V, 0, np.full(L, r.uid[i]), pos, device="cpu")
        ln, first_live, blocks = r.pool.session_query(r.sid[i])
        resident = np.array([(p // 16 < 1) or (p // 16 >= first_live) for p in pos])   # n_sink = 1
        kc, vc = k.cpu(), v.cpu()
        assert torch.equal(kc[resident].view(torch.int16), want_k[resident].view(torch.int16))
        assert torch.equal(vc[resident].view(torch.int16), want_v[resident].view(torch.int16))
        assert torch.isnan(kc[~resident].float()).all()      # evicted rows are reported as NaN


# ------------------------------------------------------------------------------ attention parity


def _run_parity(w, history_scale=1.0, n_layers=1, flags=0, family=0, split_tokens=0, max_timed=None,
                check_tables=True, check_history_attend_every=0, one_call=False):
    """one_call: every attended step goes through metronome_append_attend, with the fused decode step switched on
    (one launch for a GQA decode step)."""
    r = Runner(w, n_layers=n_layers, flags=flags)
    r.pool.set_tuning(split_tokens, family, 0, 2 if one_call else 0)
    m = OracleMirror(r)
    events, _ = wl.build_schedule(w, history_scale=history_scale)
    worst = {"max_abs": 0.0, "max_rel": 0.0, "row_l2": 0.0}
    n_timed = 0
    hist_i = 0
    for ev in events:
        if ev[0] == "open":
            r.open(ev[1]); m.open(ev[1])
        elif ev[0] == "close":
            r.close(ev[1]); m.close(ev[1])
            if check_tables:
                m.check_tables(r.pool)
        else:
            st = r.make_step(ev)
            do_attend = st.timed
            if not st.timed and check_history_attend_every:
                hist_i += 1
                do_attend = hist_i % check_history_attend_every == 0
            for layer in range(n_layers):
                m.append(st, layer)
                if do_attend and one_call:
                    out = r.step(st, layer)
                else:
                    r.append(st, layer)
                if do_attend:
                    out = out if one_call else r.attend(st, layer)
                    ref = m.attend(st, layer)
                    rep = assert_parity(out, ref, f"{w.name} frame {st.frame} layer {layer} n={st.n_new[:4]}",
                                        unit_scale=w.outlier_frac == 0)
                    for k_ in worst:
                        worst[k_] = max(worst[k_], rep[k_])
            if check_tables and (st.timed or hist_i % 7 == 0):
                m.check_tables(r.pool)
            if st.timed:
                n_timed += 1
                if max_timed and n_timed >= max_timed:
                    break
    _loaded_native()
    return worst


@pytest.mark.parametrize("family", [0, 1, 2])
def test_config1_tiny_full(family):
    """BASELINE.json configs[0] exactly as specified, every frame, tables after every call."""
    worst = _run_parity(wl.make_workload(1), family=family, check_history_attend_every=5)
    print("config 1 worst", family, worst)


@pytest.mark.parametrize("split_tokens", [16, 48, 4096])
def test_config1_both_launch_modes(split_tokens):
    """PAPER.md:L258 'both launch modes': plain (one segment) and segmented (split-KV) decode."""
    for family in (1, 2):
        _run_parity(wl.make_workload(1), family=family, split_tokens=split_tokens, check_tables=False)


def test_config1_poisoned_frees_two_layers():
    """freed blocks NaN-poisoned: nothing outside sinks U window is ever read."""
    _run_parity(wl.make_workload(1), n_layers=2, flags=binding.FLAG_POISON_ON_FREE, check_history_attend_every=3)


@pytest.mark.parametrize("index,n_sessions,scale,timed", [(2, 6, 0.3, 12), (3, 5, 0.6, 2), (4, 6, 0.12, 2), (5, 12, 0.05, 6)])
def test_configs_2_to_5_reduced(index, n_sessions, scale, timed):
    """Configs 2-5 at their true head shapes and (S, W), with fewer sessions / shorter ages so the
    oracle finishes in seconds; several tiles, ragged tails, mixed chunk+decode, outliers, churn."""
    w = wl.make_workload(index, n_sessions=n_sessions, n_timed_frames=timed)
    worst = _run_parity(w, history_scale=scale, flags=binding.FLAG_POISON_ON_FREE)
    print("config", index, "worst", worst)


def test_mixed_prefill_and_decode_in_one_call():
    """PAPER.md:L258 'mixed prefill/decode': one attend_frame call with q_len 1 and q_len n items."""
    w = wl.make_workload(3, n_sessions=4)
    for family in (1, 2):
        r = Runner(w)
        r.pool.set_tuning(0, family)
        m = OracleMirror(r, paged=False)
        for i in range(4):
            r.open(i); m.open(i)
        rng = np.random.default_rng(0)
        for step in range(40):
            n_new = np.array([int(rng.integers(1, 26)) if rng.random() < 0.5 else 1 for _ in range(4)], np.int32)
            st = r.make_step(("step", np.arange(4, dtype=np.int32), n_new, True, step))
            r.append(st, 0); m.append(st, 0)
            assert_parity(r.attend(st, 0), m.attend(st, 0), f"mixed step {step} {n_new}")


@pytest.mark.parametrize("family", [1, 2])
def test_spike_keys_at_every_mask_boundary_on_device(family):
    S, W, L = 4, 128, 300
    t = L - 1
    kw = dict(n_sinks=S, window=W, n_blocks=64)

    def run(j):
        D = 64
        pool = binding.Pool(n_q_heads=1, n_kv_heads=1, head_dim=D, max_sessions=1, max_new_tokens=16, **kw)
        pool.set_tuning(0, family)
        sid = pool.session_open()
        k = torch.zeros(L, 1, D); v = torch.zeros(L, 1, D)
        k[j, 0, 0] = 10.0
        v[:, 0, 1] = 1.0
        v[j, 0, 0] = 1000.0; v[j, 0, 1] = 0.0
        k = k.to(torch.bfloat16).cuda(); v = v.to(torch.bfloat16).cuda()
        for a in range(0, L, 16):
            n = min(16, L - a)
            pool.append_kv(0, [sid], [n], k[a:a + n].contiguous(), v[a:a + n].contiguous())
        q = torch.zeros(1, 1, D); q[0, 0, 0] = 32.0
        q = q.to(torch.bfloat16).cuda()
        out = torch.empty_like(q)
        pool.attend_frame(0, [sid], [1], q, out)
        torch.cuda.synchronize()
        return out[0, 0].float().cpu().numpy()

    assert run(t - W)[0] == 0.0 and abs(run(t - W)[1] - 1.0) < 1e-2      # just behind the window: OUT
    assert run(t - W + 1)[0] > 990.0                                       # oldest window key: IN
    assert run(S - 1)[0] > 990.0                                           # last sink: IN
    assert run(S)[0] == 0.0                                                # first non-sink, far behind: OUT
    assert run(t)[0] > 990.0                                               # the query's own key: IN


def test_attend_on_a_reordered_subset_with_shorter_queries():
    """attend_frame need not repeat the append's batch: a reordered subset of the sessions, with
    q_len <= the rows just appended (reading R15), takes the library's general path (work list built
    and uploaded by attend_frame itself instead of the one planned at append time)."""
    from paper_2607_02640_b200.runner import Step
    w = wl.make_workload(3, n_sessions=5)
    for family in (1, 2):
        r = Runner(w)
        r.pool.set_tuning(0, family)
        m = OracleMirror(r, paged=False)
        for i in range(5):
            r.open(i); m.open(i)
        rng = np.random.default_rng(3)
        for step in range(30):
            n_new = np.array([int(rng.integers(2, 26)) for _ in range(5)], np.int32)
            st = r.make_step(("step", np.arange(5, dtype=np.int32), n_new, True, step))
            r.append(st, 0); m.append(st, 0)
            keep = rng.permutation(5)[: int(rng.integers(1, 5))]
            q_lens = np.array([int(rng.integers(1, n_new[i] + 1)) for i in keep], np.int32)
            uid = np.repeat(np.asarray([r.uid[int(i)] for i in keep], np.int64), q_lens)
            pos = np.concatenate([np.arange(r.length[int(i)] - int(n), r.length[int(i)], dtype=np.int64)
                                  for i, n in zip(keep, q_lens)])
            sub = Step(keep.astype(np.int32), np.asarray([r.sid[int(i)] for i in keep], np.int32), q_lens, uid, pos,
                       True, step)
            assert_parity(r.attend(sub, 0), m.attend(sub, 0), f"subset step {step} keep={keep} q={q_lens}")
    _loaded_native()


def test_bookkeeping_with_more_sessions_than_the_kernel_stages():
    """> 1024 sessions in one append call: the fused append kernel's bookkeeping CTA reads the batch
    from memory instead of its shared-memory copy; tables and free list stay bit-exact."""
    n = 1500
    pool = binding.Pool(n_q_heads=2, n_kv_heads=1, head_dim=64, n_sinks=4, window=32, n_blocks=n * 5, max_sessions=n,
                        max_new_tokens=16)
    cfg = O.PoolConfig(n_q_heads=2, n_kv_heads=1, head_dim=64, S=4, W=32, n_blocks=n * 5, block_size=16,
                       max_sessions=n, max_new_tokens=16)
    ora = O.PagedOracle(cfg)
    sids = [pool.session_open() for _ in range(n)]
    assert sids == [ora.session_open() for _ in range(n)]
    rng = np.random.default_rng(5)
    for step in range(8):
        n_new = rng.integers(0, 17, size=n).astype(np.int32)
        rows = int(n_new.sum())
        k = torch.zeros(rows, 1, 64, dtype=torch.bfloat16, device="cuda")
        pool.append_kv(0, sids, n_new, k, k)
        kz = np.zeros((rows, 1, 64), np.uint16)
        ora.append_kv(0, sids, [int(x) for x in n_new], kz, kz)
    n_free, ids = pool.pool_query()
    assert ids == ora.pool_query()
    for s in sids[::37]:
        got, want = pool.session_query(s), ora.session_query(s)
        assert (got[0], got[1], list(got[2])) == (want[0], want[1], list(want[2]))
    _loaded_native()


def test_unbounded_arm_matches_the_oracle_until_the_pool_is_exhausted():
    """NEXT f2 (Eq. 1): METRONOME_FLAG_UNBOUNDED keeps every block (W = infinity, nothing
    pinned, nothing freed): attention = plain causal attention over the whole history, occupancy grows
    linearly, and the append that does not fit returns POOL_EXHAUSTED with nothing changed."""
    from dataclasses import replace
    w = replace(wl.make_workload(1), n_blocks=4 * 9)
    for family in (1, 2):
        r = Runner(w, flags=binding.FLAG_UNBOUNDED, max_session_len=4096)
        r.pool.set_tuning(0, family)
        m = OracleMirror(r, unbounded=True)
        for i in range(4):
            r.open(i); m.open(i)
        exhausted = False
        for step in range(40):
            n_new = np.array([8, 1, 5, 3], np.int32)
            ev = ("step", np.arange(4, dtype=np.int32), n_new, True, step)
            lengths = dict(r.length)
            st = r.make_step(ev)
            try:
                r.append(st, 0)
            except binding.MetronomeError as e:
                assert e.code == "POOL_EXHAUSTED"
                with pytest.raises(O.OracleError):
                    m.append(st, 0)
                r.length.update(lengths)
                exhausted = True
                break
            m.append(st, 0)
            assert_parity(r.attend(st, 0), m.attend(st, 0), f"unbounded step {step}")
            m.check_tables(r.pool)
        assert exhausted
        m.check_tables(r.pool)
    _loaded_native()


@pytest.mark.parametrize("q_len", [4, 25])
def test_chunk_kernel_with_score_jumps_between_half_stages(q_len):
    """Chunk-prefill kernel (tcgen05 path: R = 8 x q_len = 32 rows, one row tile, and 200 rows, two row
    tiles) on keys whose scores jump by far more than 2^8 from one 64-key half-stage to a later one: the
    lazy rescale of the TMEM accumulator (after the previous P V has completed) and the -inf handling of
    rows that admit nothing in a half-stage must hold.  Seeded inputs built here; the oracle gets the
    same bf16 bits."""
    S, W, D, G = 4, 256, 128, 8
    rng = np.random.default_rng(11 + q_len)
    pool = binding.Pool(n_q_heads=G, n_kv_heads=1, head_dim=D, n_sinks=S, window=W, n_blocks=64, max_sessions=2,
                        max_new_tokens=25)
    pool.set_tuning(0, 2)
    cfg = O.PoolConfig(n_q_heads=G, n_kv_heads=1, head_dim=D, S=S, W=W, n_blocks=64, block_size=16, max_sessions=2,
                       max_new_tokens=25)
    ora = O.DefinitionOracle(cfg)
    sid = pool.session_open()
    assert sid == ora.session_open()
    direction = rng.standard_normal(D).astype(np.float32)
    direction /= np.linalg.norm(direction)
    total, worst = 0, 0.0
    for step in range(40):
        n = q_len if step % 3 else min(25, q_len + 5)
        k = 0.3 * rng.standard_normal((n, 1, D)).astype(np.float32)
        v = rng.standard_normal((n, 1, D)).astype(np.float32)
        for j in range(n):                       # every ~37th key is a spike, each taller than the last
            if (total + j) % 37 == 36:
                k[j, 0] = direction * (4.0 + 0.5 * ((total + j) // 37))
                v[j, 0] = 50.0 * np.sign(rng.standard_normal(D))
        q = (0.3 * rng.standard_normal((n, G, D)) + 30.0 * direction).astype(np.float32)
        kb, vb, qb = (torch.from_numpy(a).to(torch.bfloat16).cuda() for a in (k, v, q))
        pool.append_kv(0, [sid], [n], kb, vb)
        ora.append_kv(0, [sid], [n], synth.to_u16(kb), synth.to_u16(vb))
        out = torch.empty_like(qb)
        pool.attend_frame(0, [sid], [n], qb, out)
        ref = ora.attend_frame(0, [sid], [n], synth.to_u16(qb))
        rep = assert_parity(out, ref, f"spiky chunk step {step} n={n}", unit_scale=False)
        worst = max(worst, rep["row_l2"])
        total += n
    print("spiky chunk worst row l2", worst)
    _loaded_native()


def test_empty_batches_and_zero_length_items():
    """Degenerate calls: an empty batch, and a batch in which some sessions append 0 tokens / ask for 0
    query rows, must be accepted, leave those sessions untouched and give the other sessions' rows
    exactly what they get alone (parity with the oracle)."""
    from paper_2607_02640_b200.runner import Step
    w = wl.make_workload(3, n_sessions=4)
    for family in (1, 2):
        r = Runner(w)
        r.pool.set_tuning(0, family)
        m = OracleMirror(r)
        for i in range(4):
            r.open(i); m.open(i)
        empty = np.zeros(0, np.int32)
        z = torch.zeros(0, w.n_kv_heads, w.head_dim, dtype=torch.bfloat16, device="cuda")
        zq = torch.zeros(0, w.n_q_heads, w.head_dim, dtype=torch.bfloat16, device="cuda")
        r.pool.append_kv(0, empty, empty, z, z)
        r.pool.attend_frame(0, empty, empty, zq, zq)
        rng = np.random.default_rng(9)
        for step in range(24):
            n_new = np.array([int(rng.integers(0, 26)) if rng.random() < 0.7 else 0 for _ in range(4)], np.int32)
            st = r.make_step(("step", np.arange(4, dtype=np.int32), n_new, True, step))
            r.append(st, 0); m.append(st, 0)
            if n_new.sum() == 0:
                r.pool.attend_frame(0, st.sids, st.n_new, zq, zq)
            else:
                assert_parity(r.attend(st, 0), m.attend(st, 0), f"zero-length items step {step} {n_new}")
            m.check_tables(r.pool)
    _loaded_native()


@pytest.mark.parametrize("side_stream", [False, True])
def test_early_mode_decode_with_constant_eviction_and_reuse(side_stream):
    """Multi-head decode runs in 'early mode': the row kernel of step k streams the blocks the append of
    step k does not touch while that append (and the tail of step k-1's attention) is still running.
    A small window makes every session free a block every 16 steps, and the freed blocks are reused at
    once by other sessions, so a read of a stale or reassigned block would show.  300 back-to-back
    steps, every output and every table against the oracle."""
    from dataclasses import replace
    w = replace(wl.make_workload(2, n_sessions=24), W=40, n_blocks=24 * 5 + 3, max_new_tokens=4)
    r = Runner(w, flags=0)
    m = OracleMirror(r)
    for i in range(24):
        r.open(i); m.open(i)
    rng = np.random.default_rng(21)
    steps = []
    for step in range(300):
        idx = np.sort(rng.permutation(24)[: int(rng.integers(12, 25))]).astype(np.int32)
        n_new = rng.integers(1, 4, size=len(idx)).astype(np.int32)
        steps.append(r.make_step(("step", idx, n_new, True, step)))
    # inputs first, so that nothing but the library's own kernels sits on the stream in the loop below
    kvq = [(r.rows(synth.STREAM_K, 0, st.uid_rows, st.pos_rows), r.rows(synth.STREAM_V, 0, st.uid_rows, st.pos_rows),
            r.rows(synth.STREAM_Q, 0, st.uid_rows, st.pos_rows)) for st in steps]
    outs = [torch.empty_like(q) for _, _, q in kvq]
    torch.cuda.synchronize()
    stream = torch.cuda.Stream() if side_stream else None      # the caller's own stream, or the default one
    handle = stream.cuda_stream if side_stream else 0
    for st, (k, v, q), o in zip(steps, kvq, outs):     # no host sync inside: the kernels run back to back
        r.pool.append_kv(0, st.sids, st.n_new, k, v, handle)
        r.pool.attend_frame(0, st.sids, st.n_new, q, o, handle)
    torch.cuda.synchronize()
    for st, out in zip(steps, outs):
        m.append(st, 0)
        assert_parity(out, m.attend(st, 0), f"early-mode step {st.frame}")
    m.check_tables(r.pool)
    _loaded_native()


@pytest.mark.parametrize("family", [1, 2])
def test_two_layers_on_the_fused_path(family):
    """Layers > 0 repeat layer 0's batch (reading R16): their append kernels only scatter K/V and the
    work list planned at layer 0's append is reused by every layer's attend_frame (no poison flag here,
    so this is the fused one-kernel-per-append path, in early mode for family 1)."""
    _run_parity(wl.make_workload(1), n_layers=2, family=family, check_history_attend_every=4)


def test_read_only_stream_microbenchmark_reports_a_plausible_bandwidth():
    gbs = binding.stream_read_gbs(1 << 30, 3)
    assert 1000.0 < gbs < 20000.0, gbs
    with pytest.raises(binding.MetronomeError):
        binding.stream_read_gbs(1024, 1)
    _loaded_native()


def test_chunk_kernel_on_a_segment_longer_than_256_tiles():
    """A window of 4400 tokens gives a chunk-prefill segment of 276 tiles: beyond the 256 block ids the
    producer warp keeps in registers, it looks the table up per entry.  Two row tiles (200 rows) and one."""
    S, W, D, G = 4, 4400, 128, 8
    rng = np.random.default_rng(31)
    kw = dict(n_q_heads=G, n_kv_heads=1, head_dim=D, max_sessions=1, max_new_tokens=25)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=300, **kw)
    pool.set_tuning(0, 2)
    ora = O.DefinitionOracle(O.PoolConfig(S=S, W=W, n_blocks=300, block_size=16, **kw))
    sid = pool.session_open()
    assert sid == ora.session_open()
    total = 0
    for step in range(255):
        n = 25 if step % 2 == 0 else 11
        k, v = rng.standard_normal((2, n, 1, D)).astype(np.float32)
        q = rng.standard_normal((n, G, D)).astype(np.float32)
        kb, vb, qb = (torch.from_numpy(a).to(torch.bfloat16).cuda() for a in (k, v, q))
        pool.append_kv(0, [sid], [n], kb, vb)
        ora.append_kv(0, [sid], [n], synth.to_u16(kb), synth.to_u16(vb))
        total += n
        if total > 4100:                     # attend only once the segment is long (keeps the oracle cheap)
            out = torch.empty_like(qb)
            pool.attend_frame(0, [sid], [n], qb, out)
            assert_parity(out, ora.attend_frame(0, [sid], [n], synth.to_u16(qb)), f"long segment step {step} len {total}")
    assert total > 16 * 256 + 25
    _loaded_native()
