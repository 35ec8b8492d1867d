"""GPU parity of metronome_append_attend (`-m gpu`): one call per sub-step, which -- with the fused decode step switched
on (set_tuning fused_step = 2) -- runs a decode step of a grouped-query model as ONE launch (csrc/step_gqa.cuh: bookkeeping CTA + warp-granular stream over the
(item, head, tile) list, this step's rows taken from k_new / v_new and written to their paged slots on the
way).  PAPER.md:L46 ("prefill the new chunk, then decode up to tau output tokens"), L258 (union mask, sink
blocks pinned, segments merged exactly once).

Every case is compared with the oracle exactly as the two-call path is: outputs within the contract
tolerance (parity_helpers), block tables / free list bit-exact, and the K/V rows read back through the
table bit-exact (the scatter now happens inside the attention warps).  Inputs are seeded; nothing reads
/root/reference.
"""
import numpy as np
import pytest
import torch

from oracle import bounded_kv as O
from paper_2607_02640_b200 import binding, synth
from paper_2607_02640_b200 import workloads as wl
from paper_2607_02640_b200.runner import Runner
from parity_helpers import OracleMirror, assert_parity
from test_gpu_parity import _run_parity
from test_gpu_parity_sinks import SINKS, _bf16_rows, _pools

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("split_tokens", [0, 16, 48])
@pytest.mark.parametrize("family", [0, 2])
def test_config1_one_call(family, split_tokens):
    """configs[0] as specified, every attended step through the one-call entry, tables after every call;
    split_tokens forces ranges of 1 and 3 tiles per warp (every (item, head) pair in several pieces)."""
    worst = _run_parity(wl.make_workload(1), family=family, split_tokens=split_tokens, check_history_attend_every=5,
                        one_call=True)
    print("config 1 one call", family, split_tokens, worst)


@pytest.mark.parametrize("index,n_sessions,scale,timed", [(2, 6, 0.3, 12), (3, 5, 0.6, 2), (4, 6, 0.12, 2), (5, 12, 0.05, 6)])
def test_configs_2_to_5_reduced_one_call(index, n_sessions, scale, timed):
    w = wl.make_workload(index, n_sessions=n_sessions, n_timed_frames=timed)
    worst = _run_parity(w, history_scale=scale, one_call=True)
    print("config", index, "one call worst", worst)


def test_two_layers_one_call():
    _run_parity(wl.make_workload(1), n_layers=2, family=2, check_history_attend_every=3, one_call=True)


def test_decode_step_is_one_launch_and_falls_back_otherwise():
    """A pure decode step of a GQA pool is ONE kernel launch; a chunk step, a multi-head (G = 1) pool, the poison
    mode and fused_step = 1 take the two-launch path (same results either way)."""
    def launches(Hq, Hkv, n_new, flags=0, fused_step=2):
        per = 1 + (64 + 24) // 16 + 2
        pool = binding.Pool(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=128, n_sinks=4, window=64, n_blocks=4 * per,
                            max_sessions=4, max_new_tokens=25, flags=flags)
        pool.set_tuning(0, 0, 0, fused_step)
        sids = [pool.session_open() for _ in range(3)]
        rng = np.random.default_rng(0)
        rows = 3 * n_new
        k, v, q = _bf16_rows(rng, rows, Hkv, 128).cuda(), _bf16_rows(rng, rows, Hkv, 128).cuda(), _bf16_rows(rng, rows, Hq, 128).cuda()
        out = torch.empty_like(q)
        pool.append_attend(0, sids, [n_new] * 3, k, v, q, out)      # (first step: block allocation)
        before = pool.stats()["kernel_launches"]
        pool.append_attend(0, sids, [n_new] * 3, k, v, q, out)
        torch.cuda.synchronize()
        assert torch.isfinite(out.float()).all()
        return pool.stats()["kernel_launches"] - before
    assert launches(8, 2, 1) == 1
    assert launches(8, 2, 4) == 1                      # G x q_len = 16: still decode class
    assert launches(8, 2, 1, fused_step=1) == 2
    assert launches(8, 2, 1, fused_step=0) == 2        # (off unless asked for: measured slower)
    assert launches(8, 2, 5) == 2                      # chunk class
    assert launches(8, 8, 1) == 2                      # multi-head decode: row kernel, early mode
    assert launches(8, 2, 1, flags=binding.FLAG_POISON_ON_FREE) >= 2


@pytest.mark.parametrize("G", [4, 8])
@pytest.mark.parametrize("S", SINKS)
def test_decode_over_sink_counts_one_call(S, G):
    """S in {0, 16, 17, 32, 64}: sessions grow from empty far past S + W through one-call decode steps of 1..16/G
    tokens (rows crossing block boundaries: a step then holds a patched old block AND a freshly allocated one),
    outputs, tables and the K/V rows read back through the table checked at every step."""
    Hkv, D, W, N = 2, 128, 72, 3
    Hq = Hkv * G
    n_max = 16 // G
    per = -(-S // 16) + (W + n_max - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N, max_new_tokens=n_max)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=N * per, **kw)
    pool.set_tuning(0, 0, 0, 2)
    cfg = O.PoolConfig(S=S, W=W, n_blocks=N * per, block_size=16, **kw)
    defn, paged = O.DefinitionOracle(cfg), O.PagedOracle(cfg)
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)] == [paged.session_open() for _ in range(N)]
    rng = np.random.default_rng(77 + S + G)
    launches0 = pool.stats()["kernel_launches"]
    n_steps = 0
    worst = 0.0
    while min(defn.length[s] for s in sids) <= S + W + 40:
        n_new = rng.integers(1, n_max + 1, size=N).astype(np.int32)
        rows = int(n_new.sum())
        k, v, q = _bf16_rows(rng, rows, Hkv, D), _bf16_rows(rng, rows, Hkv, D), _bf16_rows(rng, rows, Hq, D)
        out = torch.empty_like(q, device="cuda")
        pool.append_attend(0, sids, n_new, k.cuda(), v.cuda(), q.cuda(), out)
        n_steps += 1
        for o in (defn, paged):
            o.append_kv(0, sids, [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        ref = defn.attend_frame(0, sids, [int(x) for x in n_new], synth.to_u16(q))
        rep = assert_parity(out, ref, f"S={S} G={G} step {n_steps} n={n_new} len={[defn.length[s] for s in sids]}")
        worst = max(worst, rep["max_abs"])
        off = 0
        for s, n in zip(sids, n_new):
            got, want = pool.session_query(int(s)), paged.session_query(int(s))
            assert (got[0], got[1], list(got[2])) == (want[0], want[1], list(want[2])), (n_steps, s)
            # the rows this step appended, read back through the table
            L = defn.length[s]
            kb, vb = torch.empty(int(n), Hkv, D, dtype=torch.bfloat16, device="cuda"), torch.empty(int(n), Hkv, D, dtype=torch.bfloat16, device="cuda")
            pool.read_kv(0, int(s), L - int(n), int(n), kb, vb)
            assert torch.equal(kb.cpu().view(torch.int16), k[off:off + int(n)].view(torch.int16)), (n_steps, s)
            assert torch.equal(vb.cpu().view(torch.int16), v[off:off + int(n)].view(torch.int16)), (n_steps, s)
            off += int(n)
    assert pool.stats()["kernel_launches"] - launches0 == n_steps * (1 + N), "one launch per step (+ one read_kv per session)"
    assert pool.pool_query()[1] == paged.pool_query()
    print(f"S={S} G={G}: {n_steps} one-launch steps, worst max_abs {worst:.2e}")


def test_whole_window_read_back_after_one_call_steps():
    """After many one-call decode steps every resident row (sinks + window), read back through the table, is the row
    that was appended: the scatter done by the attention warps lands where the bookkeeping CTA's table says."""
    Hq, Hkv, D, S, W, N = 16, 2, 64, 20, 100, 5
    per = 2 + (W + 1 - 1) // 16 + 2
    pool = binding.Pool(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, n_sinks=S, window=W, n_blocks=N * per, max_sessions=N,
                        max_new_tokens=2)
    pool.set_tuning(0, 0, 0, 2)
    sids = [pool.session_open() for _ in range(N)]
    rng = np.random.default_rng(5)
    hist_k = {s: [] for s in sids}
    hist_v = {s: [] for s in sids}
    for step in range(260):
        due = [s for s in sids if rng.random() < 0.8] or sids[:1]
        n_new = rng.integers(1, 3, size=len(due)).astype(np.int32)
        rows = int(n_new.sum())
        k, v, q = _bf16_rows(rng, rows, Hkv, D), _bf16_rows(rng, rows, Hkv, D), _bf16_rows(rng, rows, Hq, D)
        out = torch.empty_like(q, device="cuda")
        pool.append_attend(0, due, n_new, k.cuda(), v.cuda(), q.cuda(), out)
        off = 0
        for s, n in zip(due, n_new):
            hist_k[s].append(k[off:off + int(n)]); hist_v[s].append(v[off:off + int(n)])
            off += int(n)
    for s in sids:
        K, V = torch.cat(hist_k[s]), torch.cat(hist_v[s])
        L = K.shape[0]
        assert pool.session_query(s)[0] == L
        first_live = pool.session_query(s)[1]
        for lo, hi in ((0, min(L, 32)), (first_live * 16, L)):           # two pinned sink blocks, then the live window blocks
            if hi <= lo:
                continue
            kb = torch.empty(hi - lo, Hkv, D, dtype=torch.bfloat16, device="cuda")
            vb = torch.empty_like(kb)
            pool.read_kv(0, s, lo, hi - lo, kb, vb)
            assert torch.equal(kb.cpu().view(torch.int16), K[lo:hi].view(torch.int16)), (s, lo, hi)
            assert torch.equal(vb.cpu().view(torch.int16), V[lo:hi].view(torch.int16)), (s, lo, hi)


def test_back_to_back_one_call_steps_without_host_sync():
    """300 decode steps enqueued back to back on a side stream (programmatic launches: the next step's CTAs start while
    the previous kernel drains), constant eviction and block reuse, every output compared afterwards."""
    from dataclasses import replace
    w = replace(wl.make_workload(3, n_sessions=6, n_timed_frames=1), W=40, n_blocks=6 * 5 + 2, max_new_tokens=2)
    r = Runner(w)
    r.pool.set_tuning(0, 0, 0, 2)
    m = OracleMirror(r, paged=True)
    for i in range(6):
        r.open(i); m.open(i)
    stream = torch.cuda.Stream()
    steps, outs = [], []
    rng = np.random.default_rng(3)
    with torch.cuda.stream(stream):
        for e in range(300):
            idx = np.array(sorted(rng.permutation(6)[:int(rng.integers(3, 7))]), np.int32)
            st = r.make_step(("step", idx, np.ones(len(idx), np.int32), True, e))
            steps.append(st)
            k, v, q = (r.rows(t, 0, st.uid_rows, st.pos_rows) for t in (synth.STREAM_K, synth.STREAM_V, synth.STREAM_Q))
            outs.append(r.step(st, 0, k, v, q, stream=stream.cuda_stream))
    stream.synchronize()
    for st, out in zip(steps, outs):
        m.append(st, 0)
        assert_parity(out, m.attend(st, 0), f"step {st.frame}")
    m.check_tables(r.pool)


def test_one_call_errors_change_nothing():
    """The one-call entry validates both halves before anything changes: a null q with rows to attend, a duplicate
    session, pool exhaustion -- tables, lengths and the free list stay as they were."""
    pool = binding.Pool(n_q_heads=8, n_kv_heads=2, head_dim=128, n_sinks=4, window=32, n_blocks=6, max_sessions=4, max_new_tokens=8)
    pool.set_tuning(0, 0, 0, 2)
    a, b = pool.session_open(), pool.session_open()
    rng = np.random.default_rng(1)
    k, v, q = _bf16_rows(rng, 2, 2, 128).cuda(), _bf16_rows(rng, 2, 2, 128).cuda(), _bf16_rows(rng, 2, 8, 128).cuda()
    out = torch.empty_like(q)
    pool.append_attend(0, [a, b], [1, 1], k, v, q, out)
    before = (pool.session_query(a), pool.session_query(b), pool.pool_query())
    with pytest.raises(binding.MetronomeError) as e:
        pool.append_attend(0, [a, b], [1, 1], k, v, None, out)
    assert e.value.code == "INVALID_ARG"
    with pytest.raises(binding.MetronomeError) as e:
        pool.append_attend(0, [a, a], [1, 1], k, v, q, out)
    assert e.value.code == "DUPLICATE_SESSION"
    k8, q8 = _bf16_rows(rng, 16, 2, 128).cuda(), _bf16_rows(rng, 16, 8, 128).cuda()
    for _ in range(10):                                        # fill the 6-block pool
        try:
            pool.append_attend(0, [a, b], [8, 8], k8, k8, q8, torch.empty_like(q8))
        except binding.MetronomeError as err:
            assert err.code == "POOL_EXHAUSTED"
            break
        before = (pool.session_query(a), pool.session_query(b), pool.pool_query())
    else:
        pytest.fail("the pool never filled up")
    assert (pool.session_query(a), pool.session_query(b), pool.pool_query()) == before
