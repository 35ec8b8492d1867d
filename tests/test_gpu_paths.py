"""GPU tests (`-m gpu`) of launch paths that the workload-shaped parity tests do not reach on their own:
the dynamically claimed tail ranges of the GQA decode kernel, early mode on grids that fit one wave, and
append_kv's "no state change on error" contract past the point where the shadow counts are committed.
Seeded inputs; the oracle gets the same bf16 bits.
"""
import numpy as np
import pytest
import torch

from oracle import bounded_kv as O
from paper_2607_02640_b200 import binding, synth
from parity_helpers import assert_parity

pytestmark = pytest.mark.gpu


def _rows(rng, n, H, D):
    return torch.from_numpy(rng.standard_normal((n, H, D)).astype(np.float32)).to(torch.bfloat16)


@pytest.mark.parametrize("kv_fp8", [False, True])
@pytest.mark.parametrize("split_tokens", [0, 1024, 4096])
def test_gqa_decode_with_dynamic_ranges_forced(split_tokens, kv_fp8):
    """attend_gqa_kernel's dynamic regime (the last ~10 % of the flattened tile list is cut into small
    ranges that CTAs claim with an atomic counter; the last CTA out resets the counters) is enabled by
    itself only when a CTA's share is >= 512 tiles, i.e. on full config 5.  Here it is FORCED on a small
    GQA-8 workload (split_tokens sets the static share: 64 / 256 tiles; 0 = the automatic one-wave cut),
    for 12 consecutive launches with no host sync in between: every output against the oracle, and the
    claim / exit counters back to zero after the launches (a stale counter would make the next launch skip
    or repeat ranges).  kv_fp8: the same through the kernel's fp8 tile (four private stages per warp instead of two)."""
    Hq, Hkv, D, S, W, N, n_max = 32, 4, 128, 4, 2048, 6, 25
    per = 1 + (W + n_max - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N, max_new_tokens=n_max)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=N * per, flags=binding.FLAG_KV_FP8 if kv_fp8 else 0, **kw)
    pool.set_tuning(split_tokens, 2, 1)
    ora = O.DefinitionOracle(O.PoolConfig(S=S, W=W, n_blocks=N * per, block_size=16, kv_fp8=kv_fp8, **kw))
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [ora.session_open() for _ in range(N)]
    rng = np.random.default_rng(4242 + split_tokens)
    # ragged histories of 300 .. 2600 tokens, appended in 25-token chunks (no attention)
    target = rng.integers(300, 2600, size=N)
    done = np.zeros(N, np.int64)
    while (done < target).any():
        idx = [i for i in range(N) if done[i] < target[i]]
        n_new = np.array([min(n_max, target[i] - done[i]) for i in idx], np.int32)
        rows = int(n_new.sum())
        k, v = _rows(rng, rows, Hkv, D), _rows(rng, rows, Hkv, D)
        pool.append_kv(0, [sids[i] for i in idx], n_new, k.cuda(), v.cuda())
        ora.append_kv(0, [sids[i] for i in idx], [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        done[idx] += n_new
    # 12 decode steps back to back
    ones = np.ones(N, np.int32)
    ins = [(_rows(rng, N, Hkv, D), _rows(rng, N, Hkv, D), _rows(rng, N, Hq, D)) for _ in range(12)]
    dev = [(k.cuda(), v.cuda(), q.cuda()) for k, v, q in ins]
    outs = [torch.empty_like(q) for _, _, q in dev]
    torch.cuda.synchronize()
    for (k, v, q), o in zip(dev, outs):
        pool.append_kv(0, sids, ones, k, v)
        pool.attend_frame(0, sids, ones, q, o)
    flags = pool.debug_read_flags()
    assert flags[2] == 0 and flags[3] == 0, f"dynamic-range counters not reset: {flags[:6]}"
    for step, ((k, v, q), o) in enumerate(zip(ins, outs)):
        ora.append_kv(0, sids, [1] * N, synth.to_u16(k), synth.to_u16(v))
        assert_parity(o, ora.attend_frame(0, sids, [1] * N, synth.to_u16(q)), f"dynamic ranges, split {split_tokens}, step {step}")
    # the general path (a reordered subset: work list uploaded by attend_frame itself) under the same knob
    k, v, q = _rows(rng, N, Hkv, D), _rows(rng, N, Hkv, D), _rows(rng, 3, Hq, D)
    pool.append_kv(0, sids, ones, k.cuda(), v.cuda())
    ora.append_kv(0, sids, [1] * N, synth.to_u16(k), synth.to_u16(v))
    sub = [sids[4], sids[0], sids[2]]
    o = torch.empty_like(q, device="cuda")
    pool.attend_frame(0, sub, [1, 1, 1], q.cuda(), o)
    assert_parity(o, ora.attend_frame(0, sub, [1, 1, 1], synth.to_u16(q)), "dynamic ranges, subset")
    flags = pool.debug_read_flags()
    assert flags[2] == 0 and flags[3] == 0


@pytest.mark.parametrize("n_sessions,heads", [(1, 8), (2, 8), (4, 4), (3, 32)])
def test_early_mode_on_grids_that_fit_one_wave(n_sessions, heads):
    """Multi-head decode in early mode with FEW CTAs per launch (1-4 sessions x 4-32 heads x a few
    segments: every launch fits one resident wave), so the append and row kernels of consecutive steps
    can be co-resident: A(e-1), R(e-1), A(e), R(e).  R(e) may then read rows A(e-1) is still writing
    unless it waits before the block that holds them (AttendItem::fresh_blk covers the previous step's
    rows).  Session lengths cross multiples of 16 all the time (1-3 tokens per step); 600 steps with no
    host sync; every output and every table against the oracle."""
    D, S, W, n_max = 128, 4, 100, 3
    per = 1 + (W + n_max - 1) // 16 + 2
    kw = dict(n_q_heads=heads, n_kv_heads=heads, head_dim=D, max_sessions=n_sessions, max_new_tokens=n_max)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=n_sessions * per + 1, **kw)
    cfg = O.PoolConfig(S=S, W=W, n_blocks=n_sessions * per + 1, block_size=16, **kw)
    defn, paged = O.DefinitionOracle(cfg), O.PagedOracle(cfg)
    sids = [pool.session_open() for _ in range(n_sessions)]
    assert sids == [defn.session_open() for _ in sids] == [paged.session_open() for _ in sids]
    rng = np.random.default_rng(99 + n_sessions * 100 + heads)
    steps = []
    for step in range(600):
        idx = np.sort(rng.permutation(n_sessions)[: int(rng.integers(1, n_sessions + 1))])
        n_new = rng.integers(1, n_max + 1, size=len(idx)).astype(np.int32)
        # every third step asks for fewer query rows than it appended (general path, plain launch order)
        q_lens = np.maximum(1, n_new - 1).astype(np.int32) if step % 3 == 2 else n_new
        rows, qrows = int(n_new.sum()), int(q_lens.sum())
        steps.append(([sids[i] for i in idx], n_new, q_lens, _rows(rng, rows, heads, D), _rows(rng, rows, heads, D),
                      _rows(rng, qrows, heads, D)))
    dev = [(k.cuda(), v.cuda(), q.cuda()) for *_, k, v, q in steps]
    outs = [torch.empty_like(q) for _, _, q in dev]
    torch.cuda.synchronize()
    for (ss, n_new, q_lens, *_), (k, v, q), o in zip(steps, dev, outs):
        pool.append_kv(0, ss, n_new, k, v)
        pool.attend_frame(0, ss, q_lens, q, o)
    torch.cuda.synchronize()
    for step, ((ss, n_new, q_lens, k, v, q), o) in enumerate(zip(steps, outs)):
        defn.append_kv(0, ss, [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        paged.append_kv(0, ss, [int(x) for x in n_new])
        assert_parity(o, defn.attend_frame(0, ss, [int(x) for x in q_lens], synth.to_u16(q)),
                      f"one-wave early mode, {n_sessions} x {heads}, step {step}")
    for s in sids:
        got, want = pool.session_query(s), paged.session_query(s)
        assert (got[0], got[1], list(got[2])) == (want[0], want[1], list(want[2]))
    assert pool.pool_query()[1] == paged.pool_query()


@pytest.mark.parametrize("stage", [1, 2])
@pytest.mark.parametrize("family", [1, 2])
def test_append_failure_after_the_tentative_commit_changes_nothing(stage, family):
    """metronome_append_kv plans the step's attention (and may grow the split-KV workspace) and launches
    its kernel AFTER the shadow counts are committed tentatively; a failure there (injected:
    metronome_pool_debug_fail_next) must roll everything back: lengths, first live blocks, block tables,
    the free list, the layer sequence -- and the same call must then succeed and match the oracle."""
    Hq, Hkv, D, S, W, N, n_max = 8, 2, 64, 4, 40, 3, 16
    per = 1 + (W + n_max - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N, max_new_tokens=n_max)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=N * per, **kw)
    pool.set_tuning(16, family)                       # 16-token segments: the plan needs the split workspace
    cfg = O.PoolConfig(S=S, W=W, n_blocks=N * per, block_size=16, **kw)
    defn, paged = O.DefinitionOracle(cfg), O.PagedOracle(cfg)
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in sids] == [paged.session_open() for _ in sids]
    rng = np.random.default_rng(5 + stage)

    def state():
        return [pool.session_query(s) for s in sids], pool.pool_query()

    for step in range(30):
        n_new = rng.integers(1, n_max + 1, size=N).astype(np.int32)
        rows = int(n_new.sum())
        k, v, q = _rows(rng, rows, Hkv, D), _rows(rng, rows, Hkv, D), _rows(rng, rows, Hq, D)
        if step % 4 == 1:
            before = state()
            pool.debug_fail_next(stage)
            with pytest.raises(binding.MetronomeError, match="OUT_OF_MEMORY" if stage == 1 else "CUDA"):
                pool.append_kv(0, sids, n_new, k.cuda(), v.cuda())
            assert state() == before, f"step {step}: a failed append_kv changed the pool"
        pool.append_kv(0, sids, n_new, k.cuda(), v.cuda())
        defn.append_kv(0, sids, [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        paged.append_kv(0, sids, [int(x) for x in n_new])
        o = torch.empty(rows, Hq, D, dtype=torch.bfloat16, device="cuda")
        pool.attend_frame(0, sids, n_new, q.cuda(), o)
        assert_parity(o, defn.attend_frame(0, sids, [int(x) for x in n_new], synth.to_u16(q)), f"after rollback, step {step}")
        for s in sids:
            got, want = pool.session_query(s), paged.session_query(s)
            assert (got[0], got[1], list(got[2])) == (want[0], want[1], list(want[2]))
        assert pool.pool_query()[1] == paged.pool_query()


def test_max_sessions_is_capped_where_the_append_grid_ends():
    """n_batch + 1 is a gridDim.y of the append kernel (<= 65535): a pool may have at most 65534 slots."""
    kw = dict(n_q_heads=1, n_kv_heads=1, head_dim=64, n_sinks=0, window=16, n_blocks=8, max_new_tokens=1,
              flags=binding.FLAG_BOOKKEEPING_ONLY)
    with pytest.raises(binding.MetronomeError, match="INVALID_ARG"):
        binding.Pool(max_sessions=65535, **kw)
    binding.Pool(max_sessions=65534, **kw).destroy()


@pytest.mark.parametrize("buffers", ["pinned", "pageable", "alternating"])
@pytest.mark.parametrize("Hkv", [8, 2])
def test_pipelined_host_steps_match_the_blocking_ones(Hkv, buffers):
    """metronome_step_host_async / _wait (two staging slots, copies on the pool's own streams) give what the oracle
    gives, step by step, with up to two steps in flight and host buffers reused only after their wait.
    buffers: pinned = the event-free mode (kernels wait for the input copies' flag, write the result straight into the
    pinned buffer, step_done_kernel publishes completion); pageable = the event-chained mode (a kernel cannot write
    pageable memory); alternating = the library has to drain one mode before it switches to the other."""
    Hq, D, S, W, N = 8, 128, 4, 48, 3
    per = 1 + (W + 8 - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N, max_new_tokens=8)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=N * per, **kw)
    defn = O.DefinitionOracle(O.PoolConfig(S=S, W=W, n_blocks=N * per, block_size=16, **kw))
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)]
    rng = np.random.default_rng(3 + Hkv)
    pending = []                                       # (out_host, reference, label) of steps not yet waited for
    for step in range(60):
        n_new = rng.integers(1, 9, size=N).astype(np.int32) if step % 5 == 0 else np.ones(N, np.int32)
        rows = int(n_new.sum())
        pin = buffers == "pinned" or (buffers == "alternating" and (step // 7) % 2 == 0)
        k, v, q = (_rows(rng, rows, H, D) for H in (Hkv, Hkv, Hq))
        out = torch.full((rows, Hq, D), float("nan"), dtype=torch.bfloat16)
        if pin:
            k, v, q, out = k.pin_memory(), v.pin_memory(), q.pin_memory(), out.pin_memory()
        pool.step_host_async(0, sids, n_new, k, v, q, out)
        defn.append_kv(0, sids, [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        pending.append((out, defn.attend_frame(0, sids, [int(x) for x in n_new], synth.to_u16(q)), f"step {step}", k, v, q))
        pool.step_host_wait(1)
        while len(pending) > 1:
            o, ref, what, *_ = pending.pop(0)
            assert_parity(o, ref, what)
    pool.step_host_wait(0)
    for o, ref, what, *_ in pending:
        assert_parity(o, ref, what)


def test_event_free_host_step_that_fails_does_not_stall_the_pipeline():
    """metronome_step_host_async, event-free mode: a step that fails validation inside the library (here: a session named
    twice, a session that is not open) has already had its input copies enqueued and its step number taken; the library
    still publishes that number, so the waits of the surrounding good steps return, the pool is as it was before the bad
    step (no state change on error), and the good steps' results match the oracle."""
    Hq, Hkv, D, S, W, N = 8, 8, 128, 4, 48, 3
    per = 1 + (W + 8 - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N + 1, max_new_tokens=8)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=(N + 1) * per, **kw)
    defn = O.DefinitionOracle(O.PoolConfig(S=S, W=W, n_blocks=(N + 1) * per, block_size=16, **kw))
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)]
    rng = np.random.default_rng(77)
    ones = np.ones(N, np.int32)
    pending = []
    for step in range(40):
        k, v, q = (_rows(rng, N, H, D).pin_memory() for H in (Hkv, Hkv, Hq))
        out = torch.full((N, Hq, D), float("nan"), dtype=torch.bfloat16).pin_memory()
        if step % 4 == 2:                                 # a bad step between good ones: nothing may change, nothing may hang
            bad = [sids[0], sids[0], sids[1]] if step % 8 == 2 else [sids[0], N, sids[1]]      # (slot N was never opened)
            with pytest.raises(binding.MetronomeError) as ei:
                pool.step_host_async(0, bad, ones, k, v, q, out)
            assert ei.value.code in ("DUPLICATE_SESSION", "INVALID_SESSION"), ei.value.code
            continue
        pool.step_host_async(0, sids, ones, k, v, q, out)
        defn.append_kv(0, sids, [1] * N, synth.to_u16(k), synth.to_u16(v))
        pending.append((out, defn.attend_frame(0, sids, [1] * N, synth.to_u16(q)), f"step {step}", k, v, q))
        pool.step_host_wait(1)
        while len(pending) > 1:
            o, ref, what, *_ = pending.pop(0)
            assert_parity(o, ref, what)
    pool.step_host_wait(0)
    for o, ref, what, *_ in pending:
        assert_parity(o, ref, what)
    for s_ in sids:
        assert pool.session_query(s_)[0] == defn.length[s_]


@pytest.mark.parametrize("G", [1, 8])
def test_event_free_host_steps_under_load(G):
    """The event-free mode on shapes where everything it touches is live: 24 sessions x 32 query heads, W = 750 (split-KV
    + merge kernel for G = 1, early mode: the row kernel reads q before any griddepcontrol.wait and so waits for the input
    copies' flag itself; stream-K GQA decode for G = 8, early bookkeeping behind step_done_kernel), 150 decode steps with
    at most two in flight and THREE sets of pinned host buffers reused round-robin -- a result that lands late, a flag
    seen early or a buffer overwritten too soon all show up as a mismatch with the oracle."""
    Hq, D, S, W, N = 32, 128, 4, 750, 24
    Hkv = Hq // G
    per = 1 + (W + 25 - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N, max_new_tokens=25)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=N * per, **kw)
    defn = O.DefinitionOracle(O.PoolConfig(S=S, W=W, n_blocks=N * per, block_size=16, **kw))
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)]
    rng = np.random.default_rng(900 + G)
    target = rng.integers(30, 1500, size=N)
    done = np.zeros(N, np.int64)
    while (done < target).any():                        # ragged histories, device buffers, no attention
        idx = [i for i in range(N) if done[i] < target[i]]
        n_new = np.array([min(25, target[i] - done[i]) for i in idx], np.int32)
        rows = int(n_new.sum())
        k, v = _rows(rng, rows, Hkv, D), _rows(rng, rows, Hkv, D)
        pool.append_kv(0, [sids[i] for i in idx], n_new, k.cuda(), v.cuda())
        defn.append_kv(0, [sids[i] for i in idx], [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        done[idx] += n_new
    ones = np.ones(N, np.int32)
    bufs = [tuple(torch.empty(N, H, D, dtype=torch.bfloat16).pin_memory() for H in (Hkv, Hkv, Hq, Hq)) for _ in range(3)]
    launches0 = pool.stats()["kernel_launches"]
    pending = []
    for step in range(150):
        k, v, q, out = bufs[step % 3]                    # (its previous use, step - 3, has been waited for)
        for t, H in ((k, Hkv), (v, Hkv), (q, Hq)):
            t.copy_(_rows(rng, N, H, D))
        out.fill_(float("nan"))
        pool.step_host_async(0, sids, ones, k, v, q, out)
        defn.append_kv(0, sids, [1] * N, synth.to_u16(k), synth.to_u16(v))
        pending.append((out, defn.attend_frame(0, sids, [1] * N, synth.to_u16(q)), f"G={G} step {step}"))
        pool.step_host_wait(1)
        while len(pending) > 1:
            o, ref, what = pending.pop(0)
            assert_parity(o.clone(), ref, what)
    pool.step_host_wait(0)
    assert_parity(pending[0][0], pending[0][1], pending[0][2])
    # append + attention (+ merge) + step_done_kernel per step: the extra launch proves the event-free mode ran
    per_step = (pool.stats()["kernel_launches"] - launches0) / 150
    assert per_step >= 3, per_step


@pytest.mark.parametrize("mode", ["0", "1", "2"])
def test_chunk_kernel_variants(monkeypatch, mode):
    """METRONOME_UMMA_HALF (read at pool creation): 0 = the full-size chunk kernel only (one CTA per SM, two row tiles),
    1 = the half-size variant (two CTAs per SM, one row tile) when every chunk item of a launch has R <= 128 rows, 2 (the
    default) = always, items of more than 128 rows as two CTAs of 128 rows each.  GQA 8: launches of 25-token chunks
    (R = 200: two row tiles / two CTAs), of 9-token chunks (R = 72), mixed ones (25, 5, 13 tokens + decode rows, so CTAs whose
    row offset lies past a small item's rows exit at once), S = 17 (a partly filled second sink block), windows that
    slide; outputs pre-filled with NaN and compared with the oracle on every row."""
    monkeypatch.setenv("METRONOME_UMMA_HALF", mode)
    Hq, Hkv, D, S, W, N, n_max = 16, 2, 128, 17, 300, 4, 25
    per = 2 + (W + n_max - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N, max_new_tokens=n_max)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=N * per, **kw)
    defn = O.DefinitionOracle(O.PoolConfig(S=S, W=W, n_blocks=N * per, block_size=16, **kw))
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)]
    rng = np.random.default_rng(2607 + int(mode))
    plans = [[25] * N, [9] * N, [25, 5, 13, 1], [1] * N, [25, 25, 1, 9], [3, 25, 25, 25]]
    for step in range(36):
        n_new = np.asarray(plans[step % len(plans)], np.int32)
        rows = int(n_new.sum())
        k, v, q = _rows(rng, rows, Hkv, D), _rows(rng, rows, Hkv, D), _rows(rng, rows, Hq, D)
        out = torch.full((rows, Hq, D), float("nan"), dtype=torch.bfloat16, device="cuda")
        pool.append_attend(0, sids, n_new, k.cuda(), v.cuda(), q.cuda(), out)
        defn.append_kv(0, sids, [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        ref = defn.attend_frame(0, sids, [int(x) for x in n_new], synth.to_u16(q))
        assert torch.isfinite(out.float()).all(), f"mode {mode} step {step}: rows no CTA wrote"
        assert_parity(out, ref, f"chunk kernel mode {mode}, step {step}, n_new {n_new}")
    assert min(defn.length.values()) > S + W


def test_gqa_ranges_by_sm_class(monkeypatch):
    """GqaPlan::sm_mode (METRONOME_GQA_SMCLASS=1 at pool creation; off by default): the GQA decode kernel's CTAs read %smid
    and claim a long range (fast SMs) or a shorter one (the SMs that a calibration pass found to stream slower) from two
    lists.  Every range must be processed exactly once whatever the placement: outputs are pre-filled with NaN (a range
    nobody claimed leaves NaN rows -- the first version of this mode launched one CTA per LONG range only, skipped a sixth
    of the work and still passed every sampled check), compared with the oracle on every row, over 8 launches back to
    back, and the claim counters must be back to zero."""
    monkeypatch.setenv("METRONOME_GQA_SMCLASS", "1")
    Hq, Hkv, D, S, W, N = 32, 4, 128, 4, 750, 24
    per = 1 + (W + 25 - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N, max_new_tokens=25)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=N * per, **kw)
    n_sm, n_slow, ratio = pool.sm_speeds()
    if n_slow == 0:
        pytest.skip("the calibration found no slow SMs on this GPU: the mode stays off")
    assert 0.75 <= ratio <= 1.0
    defn = O.DefinitionOracle(O.PoolConfig(S=S, W=W, n_blocks=N * per, block_size=16, **kw))
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)]
    rng = np.random.default_rng(1234)
    target = rng.integers(500, 1500, size=N)
    done = np.zeros(N, np.int64)
    while (done < target).any():
        idx = [i for i in range(N) if done[i] < target[i]]
        n_new = np.array([min(25, target[i] - done[i]) for i in idx], np.int32)
        rows = int(n_new.sum())
        k, v = _rows(rng, rows, Hkv, D), _rows(rng, rows, Hkv, D)
        pool.append_kv(0, [sids[i] for i in idx], n_new, k.cuda(), v.cuda())
        defn.append_kv(0, [sids[i] for i in idx], [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        done[idx] += n_new
    ones = np.ones(N, np.int32)
    ins = [(_rows(rng, N, Hkv, D), _rows(rng, N, Hkv, D), _rows(rng, N, Hq, D)) for _ in range(8)]
    dev = [(k.cuda(), v.cuda(), q.cuda()) for k, v, q in ins]
    outs = [torch.full_like(q, float("nan")) for _, _, q in dev]
    torch.cuda.synchronize()
    for (k, v, q), o in zip(dev, outs):
        pool.append_attend(0, sids, ones, k, v, q, o)
    flags = pool.debug_read_flags()
    assert flags[3] == 0 and flags[6] == 0 and flags[7] == 0, f"SM-class claim counters not reset: {flags[:8]}"
    for step, ((k, v, q), o) in enumerate(zip(ins, outs)):
        assert torch.isfinite(o.float()).all(), f"step {step}: rows no CTA wrote"
        defn.append_kv(0, sids, [1] * N, synth.to_u16(k), synth.to_u16(v))
        assert_parity(o, defn.attend_frame(0, sids, [1] * N, synth.to_u16(q)), f"SM-class ranges, step {step}")


@pytest.mark.parametrize("n_max", [2, 25])
def test_early_bookkeeping_under_the_previous_attention_kernel(n_max):
    """Tensor-core family, two launches per step, 300 steps back to back with NOTHING else on the stream: the append
    kernel of step e does rows a2 / a3 while the attention kernel of step e-1 is still running (early bookkeeping).  A
    small window frees a block per session every few steps and the freed blocks are reallocated at once (LIFO); with
    n_max = 25 the chunk steps fill the ring, so the host has to fall back whenever a new block would take the table slot
    of a block freed in the same call.  Every output and the final tables against the oracle."""
    Hq, Hkv, D, S, W, N = 16, 2, 128, 4, 40, 6
    per = 1 + (W + n_max - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N, max_new_tokens=n_max)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=N * per, **kw)
    cfg = O.PoolConfig(S=S, W=W, n_blocks=N * per, block_size=16, **kw)
    defn, paged = O.DefinitionOracle(cfg), O.PagedOracle(cfg, store_kv=False)
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)] == [paged.session_open() for _ in range(N)]
    rng = np.random.default_rng(40 + n_max)
    steps = []
    for e in range(300):
        due = sorted(rng.permutation(N)[:int(rng.integers(3, N + 1))].tolist())
        n_new = np.where(rng.random(len(due)) < 0.15, rng.integers(1, n_max + 1, size=len(due)), 1).astype(np.int32)
        rows = int(n_new.sum())
        steps.append(([sids[i] for i in due], n_new, _rows(rng, rows, Hkv, D), _rows(rng, rows, Hkv, D), _rows(rng, rows, Hq, D)))
    dev = [(k.cuda(), v.cuda(), q.cuda(), torch.empty(q.shape, dtype=torch.bfloat16, device="cuda")) for _, _, k, v, q in steps]
    torch.cuda.synchronize()
    stream = torch.cuda.Stream()
    for (ss, n_new, *_), (k, v, q, o) in zip(steps, dev):       # no host sync, no foreign kernel in between
        pool.append_kv(0, ss, n_new, k, v, stream.cuda_stream)
        pool.attend_frame(0, ss, n_new, q, o, stream.cuda_stream)
    stream.synchronize()
    for e, ((ss, n_new, k, v, q), (*_, o)) in enumerate(zip(steps, dev)):
        for orc in (defn, paged):
            orc.append_kv(0, ss, [int(x) for x in n_new], *((synth.to_u16(k), synth.to_u16(v)) if orc is defn else ()))
        assert_parity(o, defn.attend_frame(0, ss, [int(x) for x in n_new], synth.to_u16(q)), f"step {e} n={n_new}")
    for s in sids:
        got, want = pool.session_query(s), paged.session_query(s)
        assert (got[0], got[1], list(got[2])) == (want[0], want[1], list(want[2])), s
    assert pool.pool_query()[1] == paged.pool_query()
