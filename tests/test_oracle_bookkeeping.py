"""Pins for the oracle's pool / block-table / free-list rules (CPU only).

What the paper and arithmetic fix:
  * hand-derived trace (tests/golden/bookkeeping_hand_trace.txt, re-derived in DESIGN.md)
  * resident tokens reachable by the newest query = min(len, S+W)            (north_star)
  * sinks never evicted: physical ids of logical blocks < ceil(S/B) are constant
  * only blocks ENTIRELY behind the window are freed: residency >= admitted set,
    proven by layer 1 (whole history) == layer 2 (paged, NaN-poisoned) bit for bit (L258's own test idea)
  * conservation: free + resident = n_blocks, no id twice, after every call
  * worst-case blocks per session, brute force vs closed form: 11 / 49 / 132 / 68 / 131
  * pool-occupancy numbers the paper prints (Table 2 pool column, 0.2%/session, 0.1%/sink block)
  * Eq. 1: unbounded occupancy is linear, exhaustion at t_sat = (1-rho0)/(N r)
  * pool exhaustion is all-or-nothing (the clean version of the stall at PAPER.md:L60)
"""
import os

import numpy as np
import pytest
import torch

from oracle import bounded_kv as O
from paper_2607_02640_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _cfg(**kw):
    base = dict(n_q_heads=4, n_kv_heads=2, head_dim=16, S=4, W=32, n_blocks=64, block_size=16,
                max_sessions=8, max_new_tokens=16)
    base.update(kw)
    return O.PoolConfig(**base)


def check_conservation(p: O.PagedOracle):
    used = []
    for s in p.sessions.values():
        used += list(s.table.values())
    allb = used + p.free
    assert len(allb) == p.cfg.n_blocks, "free + resident != n_blocks"
    assert sorted(allb) == list(range(p.cfg.n_blocks)), "a block id is duplicated or lost"


def parse_trace(path):
    ops = []
    for line in open(path):
        line = line.split("#")[0].strip()
        if line:
            ops.append(line)
    return ops


def run_trace(ops, make_pool, append, close, open_, query, pop_order, attends=None):
    """Replays a golden trace against any implementation exposing the five callbacks."""
    names = {}
    pool = None
    for op in ops:
        head, _, rest = op.partition(" ")
        if head == "config":
            kv = dict(x.split("=") for x in rest.split())
            pool = make_pool(B=int(kv["B"]), S=int(kv["S"]), W=int(kv["W"]), n_blocks=int(kv["n_blocks"]))
        elif head == "open":
            names[rest] = open_(pool)
        elif head == "close":
            close(pool, names.pop(rest))
        elif head == "append":
            items = [x.split("+") for x in rest.split()]
            append(pool, [names[a] for a, _ in items], [int(n) for _, n in items])
        elif head == "expect":
            name, ids = rest.split(":")
            assert query(pool, names[name.strip()])[2] == [int(x) for x in ids.split()], op
        elif head == "len":
            name, n = rest.split()
            assert query(pool, names[name])[0] == int(n), op
        elif head == "pop:":
            assert pop_order(pool) == [int(x) for x in rest.split()], op
        elif head == "attends":
            if attends is not None:
                name, ids = rest.split(":")
                assert attends(pool, names[name.strip()]) == [int(x) for x in ids.split()], op
        else:
            raise ValueError(op)


def test_hand_trace():
    def make(B, S, W, n_blocks):
        return O.PagedOracle(_cfg(block_size=B, S=S, W=W, n_blocks=n_blocks, max_new_tokens=8), store_kv=False)

    def attends(p, sid):
        s = p.sessions[sid]
        t = s.length - 1
        res = p.resident_positions(sid)
        return [int(j) for j in res if O.admit(int(j), t, p.cfg.S, p.cfg.W)]

    run_trace(parse_trace(os.path.join(GOLDEN, "bookkeeping_hand_trace.txt")), make,
              lambda p, sids, n: (p.append_kv(0, sids, n), check_conservation(p)),
              lambda p, sid: (p.session_close(sid), check_conservation(p)),
              lambda p: p.session_open(), lambda p, sid: p.session_query(sid),
              lambda p: p.pool_query(), attends)


@pytest.mark.parametrize("S,W,n_max,want", [(4, 128, 8, 11), (4, 750, 1, 49), (4, 2048, 25, 132),
                                            (4, 1024, 25, 68), (4, 2048, 13, 131)])
def test_max_blocks_brute_force_equals_closed_form(S, W, n_max, want):
    B = 16
    assert O.max_blocks_per_session(S, W, B, n_max) == want
    assert -(-S // B) + (W + n_max - 1) // B + 2 == want


@pytest.mark.parametrize("S,W,B", [(4, 32, 16), (0, 20, 16), (16, 16, 16), (17, 40, 16), (3, 7, 4), (40, 5, 8)])
def test_residency_invariants_over_a_long_session(S, W, B):
    """Every step: sinks keep their ids; resident set contains the admitted set of the oldest
    pending query; keys attended by the newest query = min(len, S+W); only whole blocks behind
    the window are gone and none of the first ceil(S/B)."""
    rng = np.random.default_rng(1)
    p = O.PagedOracle(_cfg(S=S, W=W, block_size=B, n_blocks=64, max_new_tokens=9), store_kv=False)
    sid = p.session_open()
    n_sink = -(-S // B)
    sink_ids = {}
    for step in range(200):
        n = int(rng.integers(1, 10))
        p.append_kv(0, [sid], [n])
        check_conservation(p)
        L, first_live, blocks = p.session_query(sid)
        s = p.sessions[sid]
        for b in range(min(n_sink, -(-L // B))):
            sink_ids.setdefault(b, s.table[b])
            assert s.table[b] == sink_ids[b], "a sink block moved or was evicted"
        res = set(int(x) for x in p.resident_positions(sid))
        for t in range(L - n, L):                       # every query of this frame
            need = {j for j in range(L) if O.admit(j, t, S, W)}
            assert need <= res
        newest = {j for j in res if O.admit(j, L - 1, S, W)}
        assert len(newest) == min(L, S + W)
        # nothing needed was freed, and nothing whole-block-droppable for the oldest query is kept
        L0 = L - n
        for b in range(-(-L // B)):
            droppable = b >= n_sink and (b + 1) * B <= L0 - W + 1
            assert (b in s.table) == (not droppable)
        assert len(blocks) <= O.max_blocks_per_session(S, W, B, 9)
        assert len(blocks) == min(n_sink, -(-L // B)) + max(0, -(-L // B) - first_live)


def _random_run(seed, cfg, steps, check):
    """Random open / append / attend / close traffic through both layers."""
    rng = np.random.default_rng(seed)
    d1, d2 = O.DefinitionOracle(cfg), O.PagedOracle(cfg, poison_on_free=True)
    live = []
    row_seed = 0
    for step in range(steps):
        r = rng.random()
        if (r < 0.15 and len(live) < cfg.max_sessions) or not live:
            a, b = d1.session_open(), d2.session_open()
            assert a == b
            live.append(a)
            continue
        if r < 0.22:
            sid = live.pop(int(rng.integers(len(live))))
            d1.session_close(sid); d2.session_close(sid)
            check_conservation(d2)
            continue
        k = int(rng.integers(1, len(live) + 1))
        sids = [int(x) for x in rng.permutation(live)[:k]]
        n_new = [int(rng.integers(1, cfg.max_new_tokens + 1)) if rng.random() < 0.4 else 1 for _ in sids]
        T = sum(n_new)
        row_seed += 1
        g = torch.Generator().manual_seed(seed * 100003 + row_seed)
        kn = synth.to_u16(torch.randn(T, cfg.n_kv_heads, cfg.head_dim, generator=g).to(torch.bfloat16))
        vn = synth.to_u16(torch.randn(T, cfg.n_kv_heads, cfg.head_dim, generator=g).to(torch.bfloat16))
        qn = synth.to_u16(torch.randn(T, cfg.n_q_heads, cfg.head_dim, generator=g).to(torch.bfloat16))
        try:
            d2.append_kv(0, sids, n_new, kn, vn)
        except O.OracleError as e:
            assert e.code == "POOL_EXHAUSTED"
            continue
        d1.append_kv(0, sids, n_new, kn, vn)
        check_conservation(d2)
        check(d1, d2, sids, n_new, qn)


def test_layer1_equals_layer2_under_nan_poison():
    """'freed blocks NaN-poisoned to prove nothing outside sinks U window is ever read'.
    Whole-history attention and table-only attention must agree BIT FOR BIT (same summation order),
    with mixed prefill/decode batches and GQA."""
    cfg = _cfg(S=4, W=24, n_blocks=40, max_sessions=5, max_new_tokens=7, n_q_heads=4, n_kv_heads=2)

    def check(d1, d2, sids, n_new, q):
        a = d1.attend_frame(0, sids, n_new, q)
        b = d2.attend_frame(0, sids, n_new, q)
        assert np.isfinite(b).all(), "a poisoned (freed or never-written) slot was read"
        np.testing.assert_array_equal(a, b)

    _random_run(3, cfg, 300, check)


def test_qlen_may_not_exceed_last_append():
    p = O.PagedOracle(_cfg(), store_kv=False)
    sid = p.session_open()
    p.append_kv(0, [sid], [5]); p.append_kv(0, [sid], [2])
    with pytest.raises(O.OracleError, match="QLEN_EXCEEDS_LAST_APPEND"):
        p.attend_frame(0, [sid], [3], np.zeros((3, 4, 16), np.uint16))


def test_pool_exhaustion_is_all_or_nothing():
    """the engine stalls when it cannot allocate; here the call fails and NOTHING changes."""
    p = O.PagedOracle(_cfg(n_blocks=5, W=1000, max_new_tokens=64), store_kv=False)
    a, b = p.session_open(), p.session_open()
    p.append_kv(0, [a, b], [30, 30])                    # 2 + 2 blocks, 1 free
    before = (p.session_query(a), p.session_query(b), p.pool_query())
    with pytest.raises(O.OracleError, match="POOL_EXHAUSTED"):
        p.append_kv(0, [a, b], [10, 10])                # needs 1 + 1
    assert (p.session_query(a), p.session_query(b), p.pool_query()) == before
    p.append_kv(0, [a], [10])                           # 1 block still fits
    check_conservation(p)


def test_frees_in_the_same_call_count_toward_the_check():
    """Two-phase rule (reading R6): all frees of the batch happen before any allocation."""
    p = O.PagedOracle(_cfg(S=0, W=16, n_blocks=3, max_new_tokens=16), store_kv=False)
    a = p.session_open()
    for _ in range(10):                                 # steady state: frees 1, allocates 1 per call
        p.append_kv(0, [a], [16])
        check_conservation(p)
    assert len(p.session_query(a)[2]) <= 3


def test_duplicate_and_invalid_sessions():
    p = O.PagedOracle(_cfg(), store_kv=False)
    a = p.session_open()
    with pytest.raises(O.OracleError, match="DUPLICATE_SESSION"):
        p.append_kv(0, [a, a], [1, 1])
    with pytest.raises(O.OracleError, match="INVALID_SESSION"):
        p.append_kv(0, [a + 1], [1])
    with pytest.raises(O.OracleError, match="CHUNK_TOO_LARGE"):
        p.append_kv(0, [a], [17])
    assert p.session_query(a)[0] == 0
    p.session_close(a)
    assert p.session_open() == a                        # lowest free slot is reused


def _paper_numbers():
    out = {}
    for line in open(os.path.join(GOLDEN, "paper_pool_numbers.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def _plateau_blocks(S, W, n_sessions=4, frame=(25, 1, 1, 1, 1, 1, 1, 1, 1)):
    """Mean resident blocks per session after the window has slid (time average over frames)."""
    p = O.PagedOracle(_cfg(S=S, W=W, n_blocks=n_sessions * 200, max_sessions=n_sessions, max_new_tokens=32),
                      store_kv=False)
    sids = [p.session_open() for _ in range(n_sessions)]
    for i, s in enumerate(sids):                        # de-phase the sessions
        p.append_kv(0, [s], [1 + 3 * i])
    samples = []
    frames = 2 * (S + W) // sum(frame) + 60
    for f in range(frames):
        for n in frame:
            p.append_kv(0, sids, [n] * n_sessions)
        if f * sum(frame) > 2 * (S + W):
            samples.append(np.mean([len(p.session_query(s)[2]) for s in sids]))
    return float(np.mean(samples))


def test_paper_table2_pool_column_and_per_session_plateau():
    """Table 2 'pool' column is block arithmetic: plateau ~ W, + ~0.1% per pinned
    sink block at N=32; ~0.2% of pool per session at W=1024 (L87).  The pool size is not printed;
    it follows from 0.1% = 32 sessions x 1 block / pool  =>  pool ~ 32000 blocks."""
    num = _paper_numbers()
    N = int(num["table2_N"])
    pool = N * 1 / (num["sink_block_cost_pct"] / 100.0)
    assert num["block_tokens"] == 16
    tol = 0.35                                           # percentage points: the paper rounds to 0.1 and pool is inferred
    for key, (W, S) in {"table2_pool_W512_S0": (512, 0), "table2_pool_W1024_S0": (1024, 0),
                        "table2_pool_W2048_S0": (2048, 0), "table2_pool_W1024_S16": (1024, 16),
                        "table2_pool_W1024_S32": (1024, 32), "table2_pool_W512_S32": (512, 32),
                        "table2_pool_W2048_S32": (2048, 32)}.items():
        pct = 100.0 * N * _plateau_blocks(S, W) / pool
        assert abs(pct - num[key]) < tol, (key, pct, num[key])
    per_session = 100.0 * _plateau_blocks(0, 1024) / pool
    assert abs(per_session - num["plateau_pct_per_session_W1024"]) < 0.03
    # each pinned sink block costs exactly one block per session
    assert abs((_plateau_blocks(32, 1024) - _plateau_blocks(0, 1024)) - 2.0) < 0.2


def test_eq1_unbounded_fill_is_linear_and_saturates_at_t_sat():
    """PAPER.md:L74-79 Eq. 1: rho(t) = rho0 + N r t, t_sat = (1 - rho0)/(N r); windowed plateaus (L87)."""
    N, n_per_frame, B, n_blocks = 8, 32, 16, 400
    cfg = _cfg(S=4, W=64, n_blocks=n_blocks, max_sessions=N, max_new_tokens=32, unbounded=True)
    p = O.PagedOracle(cfg, store_kv=False)
    sids = [p.session_open() for _ in range(N)]
    r = (n_per_frame / B) / n_blocks                    # pool fraction per session per frame
    t_sat = (1.0 - 0.0) / (N * r)
    frames = 0
    rho = []
    while True:
        try:
            p.append_kv(0, sids, [n_per_frame] * N)
        except O.OracleError as e:
            assert e.code == "POOL_EXHAUSTED"
            break
        frames += 1
        rho.append(p.occupancy())
        assert abs(rho[-1] - N * r * frames) < 1e-12     # exactly linear
    assert frames == int(t_sat)                          # saturates on schedule
    # the windowed arm under the same load never approaches saturation
    pw = O.PagedOracle(_cfg(S=4, W=64, n_blocks=n_blocks, max_sessions=N, max_new_tokens=32), store_kv=False)
    sw = [pw.session_open() for _ in range(N)]
    for _ in range(4 * frames):
        pw.append_kv(0, sw, [n_per_frame] * N)
    per = O.max_blocks_per_session(4, 64, B, 32)
    assert pw.occupancy() <= N * per / n_blocks < 0.2


def test_layer_sequence_rule():
    cfg = _cfg(n_layers=2)
    p = O.PagedOracle(cfg, store_kv=False)
    a = p.session_open()
    with pytest.raises(O.OracleError, match="LAYER_SEQUENCE"):
        p.append_kv(1, [a], [1])
    p.append_kv(0, [a], [3])
    with pytest.raises(O.OracleError, match="LAYER_SEQUENCE"):
        p.append_kv(1, [a], [2])                        # must repeat layer 0's batch
    p.append_kv(1, [a], [3])
    with pytest.raises(O.OracleError, match="LAYER_SEQUENCE"):
        p.append_kv(1, [a], [3])                        # once per layer per step
