"""GPU parity of the fp8 KV arm (`-m gpu`): METRONOME_FLAG_KV_FP8 pools (PAPER.md:L101
"we bound which tokens stay resident, and the two compose"; quantiser = DESIGN.md reading R18, stated in
oracle/kv_fp8.py and pinned in tests/test_oracle_kv_fp8.py).

  * the stored rows: what metronome_read_kv decodes (float32) equals the oracle's round trip BIT FOR BIT -- both
    sides take the rounding decision in float32 (scale = max|x| / 448, x / scale, nearest-even E4M3);
  * attention over sinks + window of the decoded rows: same contract tolerance as the bf16 arm, against the oracle's
    fp8 arm (which attends over the identical float32 rows), for decode / chunk / mixed steps, G = 1 and G = 4,
    D = 64 and 128, several sink counts, split-KV on and off; block tables and free list bit-exact.
Seeded inputs; nothing reads /root/reference.
"""
import numpy as np
import pytest
import torch

from oracle import bounded_kv as O
from oracle import kv_fp8 as F
from paper_2607_02640_b200 import binding, synth
from parity_helpers import assert_parity

pytestmark = pytest.mark.gpu


def _bf16(rng, n, H, D, scale=1.0):
    return torch.from_numpy((rng.standard_normal((n, H, D)) * scale).astype(np.float32)).to(torch.bfloat16)


def _make(S, W, Hq, Hkv, D, N, n_max, split_tokens=0, extra_flags=0, scale=None):
    per = -(-S // 16) + (W + n_max - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N, max_new_tokens=n_max)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=N * per, flags=binding.FLAG_KV_FP8 | extra_flags,
                        softmax_scale=scale or 0.0, **kw)
    pool.set_tuning(split_tokens, 0)
    cfg = O.PoolConfig(S=S, W=W, n_blocks=N * per, block_size=16, kv_fp8=True, scale=scale, **kw)
    return pool, O.DefinitionOracle(cfg), O.PagedOracle(cfg, store_kv=False)


@pytest.mark.parametrize("D,Hkv", [(128, 4), (64, 2)])
def test_stored_rows_decode_to_the_oracle_round_trip_bit_for_bit(D, Hkv):
    pool, defn, book = _make(4, 64, Hkv * 2, Hkv, D, 3, 25)
    assert pool.kv_storage_bytes() == pool.cfg.n_blocks * Hkv * (2 * 16 * D + 128)
    sids = [pool.session_open() for _ in range(3)]
    rng = np.random.default_rng(D)
    hist = {s: ([], []) for s in sids}
    for step in range(12):
        n_new = rng.integers(0, 26, size=3).astype(np.int32) if step % 3 == 0 else np.ones(3, np.int32)
        rows = int(n_new.sum())
        scale = rng.choice([1e-3, 1.0, 30.0])
        k, v = _bf16(rng, rows, Hkv, D, scale), _bf16(rng, rows, Hkv, D, 1.0)
        if rows:
            k[0] = 0                                                   # an all-zero row: scale 1, codes 0
            v[-1, :, 1:] = 0                                           # a single non-zero element: it is the row's 448
        pool.append_kv(0, sids, n_new, k.cuda(), v.cuda())
        off = 0
        for s, n in zip(sids, n_new):
            hist[s][0].append(synth.to_u16(k[off:off + int(n)])); hist[s][1].append(synth.to_u16(v[off:off + int(n)]))
            off += int(n)
    for s in sids:
        K, V = np.concatenate(hist[s][0]), np.concatenate(hist[s][1])
        L = K.shape[0]
        first_live = pool.session_query(s)[1]
        for lo, hi in ((0, min(L, 16)), (first_live * 16, L)):           # the pinned sink block, the live window blocks
            kb = torch.empty(hi - lo, Hkv, D, dtype=torch.float32, device="cuda")
            vb = torch.empty_like(kb)
            pool.read_kv(0, s, lo, hi - lo, kb, vb)
            assert np.array_equal(kb.cpu().numpy().view(np.uint32), F.roundtrip(K[lo:hi]).view(np.uint32)), (s, lo, hi)
            assert np.array_equal(vb.cpu().numpy().view(np.uint32), F.roundtrip(V[lo:hi]).view(np.uint32)), (s, lo, hi)


@pytest.mark.parametrize("mode", ["decode", "chunk", "mixed"])
@pytest.mark.parametrize("G,D", [(1, 128), (4, 128), (4, 64)])
@pytest.mark.parametrize("S,split_tokens", [(4, 0), (0, 0), (17, 48)])
def test_fp8_attention_parity(S, split_tokens, G, D, mode):
    Hkv, W, n_max, N = 2, 72, 25, 3
    Hq = Hkv * G
    pool, defn, book = _make(S, W, Hq, Hkv, D, N, n_max, split_tokens)
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)] == [book.session_open() for _ in range(N)]
    rng = np.random.default_rng(500 + 7 * S + G + D)
    worst = 0.0
    for step in range(120 if mode == "decode" else 30):
        if mode == "decode" and step > 0:
            n_new = np.ones(N, np.int64)
        elif mode == "chunk" or step == 0:
            n_new = rng.integers(5, n_max + 1, size=N)
        else:
            n_new = np.where(rng.random(N) < 0.5, 1, rng.integers(2, n_max + 1, size=N))
        n_new = n_new.astype(np.int32)
        rows = int(n_new.sum())
        k, v, q = _bf16(rng, rows, Hkv, D), _bf16(rng, rows, Hkv, D), _bf16(rng, rows, Hq, D)
        out = torch.empty_like(q, device="cuda")
        pool.append_attend(0, sids, n_new, k.cuda(), v.cuda(), q.cuda(), out)
        defn.append_kv(0, sids, [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        book.append_kv(0, sids, [int(x) for x in n_new])
        ref = defn.attend_frame(0, sids, [int(x) for x in n_new], synth.to_u16(q))
        rep = assert_parity(out, ref, f"fp8 S={S} G={G} D={D} {mode} step {step} n={n_new}")
        worst = max(worst, rep["max_abs"])
        for s in sids:
            got, want = pool.session_query(int(s)), book.session_query(int(s))
            assert (got[0], got[1], list(got[2])) == (want[0], want[1], list(want[2])), (step, s)
    assert min(defn.length.values()) > S + W, "the sessions never left the full-causal regime"
    assert pool.pool_query()[1] == book.pool_query()
    print(f"fp8 S={S} G={G} D={D} {mode}: worst max_abs {worst:.2e}")


def test_fp8_with_poisoned_frees_and_two_layers():
    """Freed blocks are filled with NaN bytes ("freed blocks NaN-poisoned"): nothing outside sinks U
    window may be read in the fp8 layout either; layer 1 repeats layer 0's batch with its own rows."""
    S, W, Hq, Hkv, D, N = 4, 40, 8, 8, 128, 4
    per = 1 + (W + 4 - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=N, max_new_tokens=4)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=N * per, n_layers=2, flags=binding.FLAG_KV_FP8 | binding.FLAG_POISON_ON_FREE, **kw)
    defn = O.DefinitionOracle(O.PoolConfig(S=S, W=W, n_blocks=N * per, block_size=16, n_layers=2, kv_fp8=True, **kw))
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)]
    rng = np.random.default_rng(9)
    for step in range(120):
        due = sorted(rng.permutation(N)[:int(rng.integers(2, N + 1))].tolist())
        n_new = rng.integers(1, 4, size=len(due)).astype(np.int32)
        rows = int(n_new.sum())
        for layer in range(2):
            k, v, q = _bf16(rng, rows, Hkv, D), _bf16(rng, rows, Hkv, D), _bf16(rng, rows, Hq, D)
            out = torch.empty_like(q, device="cuda")
            pool.append_kv(layer, [sids[i] for i in due], n_new, k.cuda(), v.cuda())
            pool.attend_frame(layer, [sids[i] for i in due], n_new, q.cuda(), out)
            defn.append_kv(layer, [sids[i] for i in due], [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
            ref = defn.attend_frame(layer, [sids[i] for i in due], [int(x) for x in n_new], synth.to_u16(q))
            assert_parity(out, ref, f"fp8 poison step {step} layer {layer}")


@pytest.mark.parametrize("qmag", ["mixed", "huge"])
@pytest.mark.parametrize("G,D", [(4, 128), (8, 128), (4, 64)])
def test_fp8_gqa_decode_with_rows_of_very_different_magnitude(G, D, qmag):
    """The GQA decode kernel's fp8 tile never applies a scale to a tensor-core operand: K scales multiply the finished
    dot products, V scales are folded into the softmax weights relative to a running reference that is raised (and
    the accumulator rescaled) when a larger scale arrives, and the query row is brought into fp16 range by a power of
    two.  Here the rows' magnitudes span 1e-3 .. 1e2 for V (log-uniform per row, so the reference is raised many times,
    also across split pieces) and {1e-3, 3e-2, 1} for K; Q rows are x {1e-2, 1, 300} ("mixed": flat to one-hot softmax
    rows) or x {2.5e5, 1e6} with a softmax scale of 1e-6 / sqrt(D) ("huge": far outside fp16 range).  Freed blocks are
    NaN-poisoned, S = 17 gives a partly filled second sink block, split-KV pieces of 64 tokens."""
    Hkv, S, W, N = 2, 17, 150, 3
    Hq = Hkv * G
    scale = 1e-6 / np.sqrt(D) if qmag == "huge" else None
    pool, defn, book = _make(S, W, Hq, Hkv, D, N, 4, split_tokens=64, extra_flags=binding.FLAG_POISON_ON_FREE, scale=scale)
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)] == [book.session_open() for _ in range(N)]
    rng = np.random.default_rng(77 + G + D)

    def mag(choices, shape):
        return torch.from_numpy(np.asarray(choices, np.float32)[rng.integers(0, len(choices), size=shape)]).to(torch.bfloat16)

    for step in range(260):
        n_new = np.ones(N, np.int32) if step % 7 else rng.integers(1, 3, size=N).astype(np.int32)
        rows = int(n_new.sum())
        k = _bf16(rng, rows, Hkv, D) * mag([1e-3, 3e-2, 1.0], (rows, Hkv, 1))
        v = _bf16(rng, rows, Hkv, D) * torch.from_numpy((10.0 ** rng.uniform(-3, 2, size=(rows, Hkv, 1))).astype(np.float32)).to(torch.bfloat16)
        q = _bf16(rng, rows, Hq, D) * mag([2.5e5, 1e6] if qmag == "huge" else [1e-2, 1.0, 300.0], (rows, Hq, 1))
        out = torch.empty_like(q, device="cuda")
        pool.append_attend(0, sids, n_new, k.cuda(), v.cuda(), q.cuda(), out)
        defn.append_kv(0, sids, [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        book.append_kv(0, sids, [int(x) for x in n_new])
        ref = defn.attend_frame(0, sids, [int(x) for x in n_new], synth.to_u16(q))
        assert_parity(out, ref, f"fp8 magnitudes G={G} D={D} {qmag} step {step}", unit_scale=False)
    assert min(defn.length.values()) > S + W
    assert pool.pool_query()[1] == book.pool_query()


@pytest.mark.parametrize("mode", ["decode", "chunk"])
def test_fp8_weights_stay_inside_fp16_when_the_row_maximum_lags(mode):
    """Both fp8 tensor-core kernels round softmax weight x V scale to fp16 relative to a LAZILY updated row maximum (the
    accumulators are rescaled only when the true maximum has moved by more than 2^6 (GQA decode tile) / 2^8 (chunk
    kernel)) and to a V reference that is raised only when a scale exceeds it.  Worst case for the fp16 range: scores
    that rise key after key (0.12 per key in the log2 domain: the stale maximum lags by almost the whole bound) while the
    keys' V scales sit just under the reference (first 64 keys x 1, the rest x 3.9 with a reference of 4 x the first
    maximum).  A weight factor that forgets either effect overflows to inf (this did happen: the decode tile at 2^11, and
    2^9 in the chunk kernel was only safe by luck); outputs must be finite and match the oracle."""
    G, Hkv, D, S, W, N = 4, 2, 128, 4, 640, 2
    Hq = G * Hkv
    n_max = 20
    pool, defn, book = _make(S, W, Hq, Hkv, D, N, n_max)
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)] == [book.session_open() for _ in range(N)]
    rng = np.random.default_rng(321)
    length = np.zeros(N, np.int64)
    beta, delta = 8.0, 0.12 / (1.4426950408889634 / np.sqrt(D)) / 8.0          # score rises 0.12 per key (log2 domain)

    def rows_for(n_new):
        ks, vs, qs = [], [], []
        for i, n in enumerate(n_new):
            pos = length[i] + np.arange(n)
            k = rng.standard_normal((n, Hkv, D)).astype(np.float32) * 0.05
            k[:, :, 0] = (delta * pos)[:, None]
            v = rng.standard_normal((n, Hkv, D)).astype(np.float32) * np.where(pos < 64, 1.0, 3.9)[:, None, None]
            q = rng.standard_normal((n, Hq, D)).astype(np.float32) * 0.05
            q[:, :, 0] = beta
            ks.append(k); vs.append(v); qs.append(q)
            length[i] += n
        t = lambda xs: torch.from_numpy(np.concatenate(xs)).to(torch.bfloat16)
        return t(ks), t(vs), t(qs)

    for step in range(60):
        if mode == "chunk" or step < 12:
            n_new = np.full(N, n_max, np.int32)                 # (R = 80 rows: chunk class; also builds the decode history)
        else:
            n_new = np.ones(N, np.int32)
        k, v, q = rows_for(n_new)
        out = torch.empty_like(q, device="cuda")
        pool.append_attend(0, sids, n_new, k.cuda(), v.cuda(), q.cuda(), out)
        assert torch.isfinite(out.float()).all(), f"{mode} step {step}: non-finite output (fp16 weight overflow)"
        defn.append_kv(0, sids, [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
        book.append_kv(0, sids, [int(x) for x in n_new])
        ref = defn.attend_frame(0, sids, [int(x) for x in n_new], synth.to_u16(q))
        assert_parity(out, ref, f"fp8 lagging maximum, {mode} step {step}", unit_scale=False)
    assert pool.pool_query()[1] == book.pool_query()
