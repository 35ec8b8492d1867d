"""GPU parity over the sink count (`-m gpu`): S in {0, 16, 17, 32, 64} x both kernel families x
{decode, chunk, mixed} ("with S=0 every touched path is
byte-identical to stock", Table 2 L308-323 rows S in {0, 16, 32, 42, 58, 64}, L145 "two KV blocks").

n_sink = ceil(S/16) covers 0 blocks, exactly one full block, one full + one partly filled, two, four:
the sink-tile paths of the three attention kernels (leading sink tiles, the full-tile shortcut, the
half-stage that mixes sink and window tiles).  Every input is seeded here and handed bit-identically to
the library and to the oracle; nothing reads /root/reference.
"""
import numpy as np
import pytest
import torch

from oracle import bounded_kv as O
from paper_2607_02640_b200 import binding, synth
from parity_helpers import assert_parity

pytestmark = pytest.mark.gpu

SINKS = [0, 16, 17, 32, 64]


def _pools(S, W, Hq, Hkv, D, n_sessions, n_max, family, split_tokens=0):
    per = -(-S // 16) + (W + n_max - 1) // 16 + 2
    kw = dict(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, max_sessions=n_sessions, max_new_tokens=n_max)
    pool = binding.Pool(n_sinks=S, window=W, n_blocks=n_sessions * per, flags=binding.FLAG_POISON_ON_FREE, **kw)
    pool.set_tuning(split_tokens, family)
    cfg = O.PoolConfig(S=S, W=W, n_blocks=n_sessions * per, block_size=16, **kw)
    return pool, O.DefinitionOracle(cfg), O.PagedOracle(cfg)


def _bf16_rows(rng, n, H, D):
    return torch.from_numpy(rng.standard_normal((n, H, D)).astype(np.float32)).to(torch.bfloat16)


def _step(pool, defn, paged, sids, n_new, rng, Hq, Hkv, D, what, q_lens=None):
    rows = int(np.sum(n_new))
    k, v = _bf16_rows(rng, rows, Hkv, D), _bf16_rows(rng, rows, Hkv, D)
    pool.append_kv(0, sids, n_new, k.cuda(), v.cuda())
    defn.append_kv(0, sids, [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
    paged.append_kv(0, sids, [int(x) for x in n_new], synth.to_u16(k), synth.to_u16(v))
    q_lens = n_new if q_lens is None else q_lens
    q = _bf16_rows(rng, int(np.sum(q_lens)), Hq, D)
    out = torch.empty_like(q, device="cuda")
    pool.attend_frame(0, sids, q_lens, q.cuda(), out)
    ref = defn.attend_frame(0, sids, [int(x) for x in q_lens], synth.to_u16(q))
    rep = assert_parity(out, ref, what)
    # bookkeeping: pinned sink blocks and the ring, bit-exact
    for s in sids:
        got, want = pool.session_query(int(s)), paged.session_query(int(s))
        assert (got[0], got[1], list(got[2])) == (want[0], want[1], list(want[2])), (what, s)
    return out, rep


@pytest.mark.parametrize("mode", ["decode", "chunk", "mixed"])
@pytest.mark.parametrize("family", [1, 2])
@pytest.mark.parametrize("S", SINKS)
def test_attention_parity_over_sink_counts(S, family, mode):
    """Sessions grow from empty (full causal while len <= S + W) far past S + W (the window leaves the
    sinks behind, blocks are freed and reused); W = 72 is not a block multiple, so window edges fall
    inside blocks.  GQA 4 at D = 128: decode items go to the GQA decode kernel, chunks (R = 4 n > 16)
    to the tcgen05 kernel in family 2, everything to the row kernel in family 1."""
    Hq, Hkv, D, W, n_max, N = 8, 2, 128, 72, 25, 3
    pool, defn, paged = _pools(S, W, Hq, Hkv, D, N, n_max, family)
    sids = [pool.session_open() for _ in range(N)]
    assert sids == [defn.session_open() for _ in range(N)] == [paged.session_open() for _ in range(N)]
    rng = np.random.default_rng(1000 + 10 * S + family)
    worst = 0.0
    # history without attention up to ~30 tokens short of S + W (ragged: the sessions sit at different
    # phases of the 16-token block), so the checked steps cross from full causal into the sliding regime
    target = np.array([S + W - 30 + int(rng.integers(0, 16)) for _ in sids])
    while True:
        idx = [i for i in range(N) if defn.length[sids[i]] < target[i]]
        if not idx:
            break
        take = np.array([min(n_max, target[i] - defn.length[sids[i]]) for i in idx], np.int32)
        rows = int(take.sum())
        k, v = _bf16_rows(rng, rows, Hkv, D), _bf16_rows(rng, rows, Hkv, D)
        pool.append_kv(0, [sids[i] for i in idx], take, k.cuda(), v.cuda())
        defn.append_kv(0, [sids[i] for i in idx], [int(x) for x in take], synth.to_u16(k), synth.to_u16(v))
        paged.append_kv(0, [sids[i] for i in idx], [int(x) for x in take], synth.to_u16(k), synth.to_u16(v))
    for step in range(90 if mode == "decode" else 36):
        if mode == "decode":
            n_new = np.ones(N, np.int64)
        elif mode == "chunk":
            n_new = rng.integers(5, n_max + 1, size=N)
        else:
            n_new = np.where(rng.random(N) < 0.5, 1, rng.integers(2, n_max + 1, size=N))
        _, rep = _step(pool, defn, paged, sids, n_new.astype(np.int32), rng, Hq, Hkv, D,
                       f"S={S} family={family} {mode} step {step} n={n_new}")
        worst = max(worst, rep["max_abs"])
    assert min(defn.length.values()) > S + W + 32, "the sessions never left the full-causal regime"
    assert pool.pool_query()[1] == paged.pool_query()
    print(f"S={S} family={family} {mode}: worst max_abs {worst:.2e}")


@pytest.mark.parametrize("family", [1, 2])
@pytest.mark.parametrize("G", [1, 8])
def test_no_sinks_is_the_stock_sliding_window(family, G):
    """PAPER.md:L258 "with S=0 every touched path is byte-identical to stock": with S = 0 the library must
    give the textbook sliding window.  Checked against a LIBRARY routine (torch SDPA on the CPU with a band
    mask from tril / triu), not against this repo's oracle."""
    Hkv, D, W, n_max = 2, 128, 50, 20
    Hq = Hkv * G
    pool, defn, paged = _pools(0, W, Hq, Hkv, D, 1, n_max, family)
    sid = pool.session_open()
    rng = np.random.default_rng(77 + G)
    K, V = [], []
    for step in range(14):
        n = int(rng.integers(1, n_max + 1)) if step % 2 == 0 else 1
        k, v, q = _bf16_rows(rng, n, Hkv, D), _bf16_rows(rng, n, Hkv, D), _bf16_rows(rng, n, Hq, D)
        K.append(k); V.append(v)
        pool.append_kv(0, [sid], [n], k.cuda(), v.cuda())
        out = torch.empty_like(q, device="cuda")
        pool.attend_frame(0, [sid], [n], q.cuda(), out)
        kk, vv = torch.cat(K), torch.cat(V)
        L = kk.shape[0]
        t = torch.arange(L - n, L)[:, None]
        j = torch.arange(L)[None, :]
        band = (j <= t) & (t - j < W)                                   # the W most recent keys, own included
        qq = q.double().permute(1, 0, 2)[None]
        kx = kk.double().repeat_interleave(G, dim=1).permute(1, 0, 2)[None]
        vx = vv.double().repeat_interleave(G, dim=1).permute(1, 0, 2)[None]
        ref = torch.nn.functional.scaled_dot_product_attention(qq, kx, vx, attn_mask=band)[0].permute(1, 0, 2).numpy()
        assert_parity(out, ref, f"S=0 stock window, G={G} family={family} step {step} n={n} len={L}")


@pytest.mark.parametrize("q_len", [1, 20])
@pytest.mark.parametrize("family", [1, 2])
@pytest.mark.parametrize("S", [17, 32, 64])
def test_spike_keys_at_the_sink_boundary_with_several_sink_blocks(S, family, q_len):
    """n_sink >= 2: a key with a dominating score and a distinctive V at S-1 must be attended by every
    query row, the one at S by none once it is out of the row's window (and by the rows whose window
    still reaches it).  An off-by-one in the sink term moves the output by ~1/W only, far inside the
    tolerance, without a spike.  q_len = 20 at G = 1 is R = 20 > 16 rows: the tcgen05 chunk kernel in
    family 2; q_len = 1 is the GQA decode kernel (family 2) / the row kernel (family 1)."""
    W, D = 40, 64
    L = S + W + 30

    def run(j):
        pool = binding.Pool(n_q_heads=1, n_kv_heads=1, head_dim=D, max_sessions=1, max_new_tokens=25, n_sinks=S,
                            window=W, n_blocks=32)
        pool.set_tuning(0, family)
        sid = pool.session_open()
        k = torch.zeros(L, 1, D); v = torch.zeros(L, 1, D)
        k[j, 0, 0] = 10.0
        v[:, 0, 1] = 1.0
        v[j, 0, 0] = 1000.0; v[j, 0, 1] = 0.0
        k = k.to(torch.bfloat16).cuda(); v = v.to(torch.bfloat16).cuda()
        cuts = list(range(0, L - q_len, 16)) + [L - q_len, L]
        for a, b in zip(cuts[:-1], cuts[1:]):
            if b > a:
                pool.append_kv(0, [sid], [b - a], k[a:b].contiguous(), v[a:b].contiguous())
        q = torch.zeros(q_len, 1, D); q[:, 0, 0] = 32.0
        q = q.to(torch.bfloat16).cuda()
        out = torch.empty_like(q)
        pool.attend_frame(0, [sid], [q_len], q, out)
        torch.cuda.synchronize()
        return out[:, 0].float().cpu().numpy()

    t = np.arange(L - q_len, L)
    for j in (S - 1, S, S + 1, 15, 16, L - q_len - W, L - q_len - W + 1, L - W, L - W + 1):
        o = run(j)
        want = (j <= t) & ((j < S) | (t - j < W))          # the paper's literal union mask
        for r in range(q_len):
            if want[r]:
                assert o[r, 0] > 990.0, (S, family, q_len, j, r, o[r, :2])
            else:
                assert o[r, 0] == 0.0 and abs(o[r, 1] - 1.0) < 1e-2, (S, family, q_len, j, r, o[r, :2])
