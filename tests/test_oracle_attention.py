"""Pins for the oracle's attention arithmetic (CPU only, `-m "not gpu"`).

The oracle (oracle/attention_ref.c) is pinned to things OTHER than itself:
  * library routine: torch SDPA (is_causal) when W >= len and S = 0            (special case)
  * library routine: torch SDPA with a band mask from torch.tril/triu when S = 0 (textbook SWA)
  * the paper's literal interval set [0,S) U (t-W, t] (reading R1) with zero keys
    -> the output must be the plain mean of V over that set (closed form)
  * spike keys at t-W / t-W+1 / S-1 / S / t+1: exactly which boundary keys are admitted
  * invariants: weights sum to 1, number of attended keys = min(t+1, S+W) (north_star)
  * GQA head map h -> h // G, scale factor, fp64 twin
A dropped term, wrong sign, off-by-one boundary, transposed operand or wrong head map fails
at least one of these.
"""
import math

import numpy as np
import pytest
import torch

from oracle import bounded_kv as O
from paper_2607_02640_b200 import synth


def _bf16(x: torch.Tensor) -> np.ndarray:
    return synth.to_u16(x.to(torch.bfloat16))


def _rand(seed, n, H, D):
    g = torch.Generator().manual_seed(seed)
    return torch.randn(n, H, D, generator=g).to(torch.bfloat16)


def _sdpa(q, k, v, mask=None, causal=False, scale=None):
    """torch library attention in fp64; q [nq,Hq,D], k/v [nk,Hkv,D] bf16 tensors."""
    Hq, Hkv = q.shape[1], k.shape[1]
    G = Hq // Hkv
    qq = q.double().permute(1, 0, 2)[None]
    kk = k.double().repeat_interleave(G, dim=1).permute(1, 0, 2)[None]
    vv = v.double().repeat_interleave(G, dim=1).permute(1, 0, 2)[None]
    o = torch.nn.functional.scaled_dot_product_attention(qq, kk, vv, attn_mask=mask, is_causal=causal, scale=scale)
    return o[0].permute(1, 0, 2).numpy()


@pytest.mark.parametrize("Hq,Hkv,D", [(4, 4, 32), (8, 2, 64), (8, 1, 16)])
def test_full_causal_equals_sdpa_when_window_covers_everything(Hq, Hkv, D):
    """north_star: 'window attention equals full attention when len <= S+W'; S=0, W>=len -> SDPA is_causal."""
    L = 37
    q, k, v = _rand(1, L, Hq, D), _rand(2, L, Hkv, D), _rand(3, L, Hkv, D)
    pos = np.arange(L)
    got = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=0, W=L)
    ref = _sdpa(q, k, v, causal=True)
    np.testing.assert_allclose(got, ref, rtol=0, atol=2e-5)
    # and with sinks: len <= S + W is still full causal attention (sets overlap, each key once)
    got2 = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=5, W=L - 5)
    np.testing.assert_allclose(got2, ref, rtol=0, atol=2e-5)


@pytest.mark.parametrize("W", [1, 2, 7, 16])
def test_sliding_window_equals_sdpa_band_mask(W):
    """S = 0 is the textbook sliding window; band from torch.tril/triu."""
    L, Hq, Hkv, D = 41, 4, 2, 32
    q, k, v = _rand(4, L, Hq, D), _rand(5, L, Hkv, D), _rand(6, L, Hkv, D)
    band = torch.ones(L, L, dtype=torch.bool).tril(0).triu(-(W - 1))  # W diagonals incl. the main one
    ref = _sdpa(q, k, v, mask=band)
    pos = np.arange(L)
    got = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=0, W=W)
    np.testing.assert_allclose(got, ref, rtol=0, atol=2e-5)


@pytest.mark.parametrize("S,W", [(1, 3), (4, 8), (5, 1), (16, 16), (3, 100)])
def test_union_mask_equals_sdpa_with_band_or_first_columns(S, W):
    """[0,S) U window: band (library tril/triu) OR the first S columns, under the causal triangle."""
    L, Hq, Hkv, D = 45, 6, 3, 16
    q, k, v = _rand(7, L, Hq, D), _rand(8, L, Hkv, D), _rand(9, L, Hkv, D)
    causal = torch.ones(L, L, dtype=torch.bool).tril(0)
    band = causal.clone().triu(-(W - 1))
    first = torch.zeros(L, L, dtype=torch.bool)
    first[:, :S] = True
    ref = _sdpa(q, k, v, mask=(band | first) & causal)
    pos = np.arange(L)
    got = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=S, W=W)
    np.testing.assert_allclose(got, ref, rtol=0, atol=2e-5)


def test_zero_keys_give_mean_of_v_over_the_papers_interval_set():
    """With K = 0 every admitted weight is equal, so o = mean of V over [0,S) U (t-W, t] -- the set
    written out from PAPER.md:L103 with reading R1, not from the oracle's predicate."""
    L, H, D, S, W = 60, 2, 8, 3, 10
    q, v = _rand(10, L, H, D), _rand(11, L, H, D)
    k = torch.zeros(L, H, D, dtype=torch.bfloat16)
    pos = np.arange(L)
    got = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=S, W=W)
    vd = v.double().numpy()
    for t in range(L):
        members = sorted((set(range(0, S)) | set(range(t - W + 1, t + 1))) & set(range(0, t + 1)))
        assert len(members) == min(t + 1, S + W)            # north_star: resident = min(len, S+W)
        np.testing.assert_allclose(got[t], vd[members].mean(axis=0), rtol=0, atol=1e-5)


def test_weights_sum_to_one_and_count_is_min_len_S_plus_W():
    L, Hq, Hkv, D, S, W = 80, 4, 2, 16, 4, 21
    q, k, v = _rand(12, L, Hq, D), _rand(13, L, Hkv, D), _rand(14, L, Hkv, D)
    pos = np.arange(L)
    out, w = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=S, W=W, want_weights=True)
    np.testing.assert_allclose(w.sum(axis=-1), 1.0, rtol=0, atol=1e-6)
    nz = (w > 0).sum(axis=-1)
    for t in range(L):
        assert np.all(nz[t] == min(t + 1, S + W))


def _spike_case(L, S, W, j_spike, t):
    """One query at t whose score with key j_spike dominates (+40 in logit); V marks that key."""
    D = 16
    qv = torch.zeros(1, 1, D)
    qv[0, 0, 0] = 16.0
    k = torch.zeros(L, 1, D)
    k[j_spike, 0, 0] = 10.0            # logit = 16*10/sqrt(16) = 40 above every other key
    v = torch.zeros(L, 1, D)
    v[:, 0, 1] = 1.0                   # background marker
    v[j_spike, 0, 0] = 1000.0
    v[j_spike, 0, 1] = 0.0
    out = O.attend(_bf16(qv), np.array([t]), _bf16(k), _bf16(v), np.arange(L), S=S, W=W)
    return out[0, 0]


def test_spike_keys_pin_every_mask_boundary():
    """An off-by-one at W >= 128 moves the output by ~1/W, far inside 1e-2: spikes make it O(1000)."""
    L, S, W, t = 300, 4, 128, 299
    # window edge: t-W is OUT, t-W+1 is IN  (window = W keys including t)
    assert _spike_case(L, S, W, t - W, t)[0] == 0.0
    assert _spike_case(L, S, W, t - W + 1, t)[0] > 999.0
    # sink edge: S-1 is IN although far behind the window, S is OUT  ("k < S")
    assert _spike_case(L, S, W, S - 1, t)[0] > 999.0
    assert _spike_case(L, S, W, S, t)[0] == 0.0
    # the query's own key is IN; a key after the query is OUT (causal inside a chunk)
    assert _spike_case(L, S, W, t, t)[0] > 999.0
    assert _spike_case(L, S, W, 200, 199)[0] == 0.0
    assert _spike_case(L, S, W, 199, 199)[0] > 999.0
    # young session: everything causal is in
    assert _spike_case(100, S, W, 50, 99)[0] > 999.0
    # when spike is out, the output is the background marker exactly (weights still sum to 1)
    assert abs(_spike_case(L, S, W, t - W, t)[1] - 1.0) < 1e-6


def test_gqa_head_map_and_operand_roles():
    """q head h reads KV head h // G (PAPER.md:L258 'grouped-query attention'); V marks its head."""
    L, Hq, Hkv, D = 9, 8, 2, 4
    q, k = _rand(15, L, Hq, D), _rand(16, L, Hkv, D)
    v = torch.zeros(L, Hkv, D)
    for hk in range(Hkv):
        v[:, hk, :] = float(hk + 1)
    pos = np.arange(L)
    out = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=2, W=4)
    for h in range(Hq):
        np.testing.assert_allclose(out[:, h, :], float(h // (Hq // Hkv) + 1), atol=1e-6)
    # transposed operands would break this: with one key the output is exactly that key's V row
    out1 = O.attend(_bf16(q[:1]), np.array([0]), _bf16(k[:1]), _bf16(_rand(17, 1, Hkv, D)), np.array([0]), S=0, W=1)
    np.testing.assert_array_equal(out1[0, 0], _rand(17, 1, Hkv, D)[0, 0].float().numpy())


def test_scale_default_is_inverse_sqrt_d_and_is_applied_to_logits():
    L, H, D = 12, 1, 64
    q, k, v = _rand(18, L, H, D), _rand(19, L, H, D), _rand(20, L, H, D)
    pos = np.arange(L)
    a = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=0, W=L)
    b = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=0, W=L, scale=1.0 / math.sqrt(D))
    np.testing.assert_array_equal(a, b)
    c = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=0, W=L, scale=0.3)
    np.testing.assert_allclose(c, _sdpa(q, k, v, causal=True, scale=0.3), atol=2e-5)


def test_f32_oracle_rounding_is_bounded_by_its_f64_twin():
    """The fp32 oracle's own error must be far below the 1e-2 contract tolerance."""
    L, Hq, Hkv, D = 700, 4, 2, 128
    q, k, v = _rand(21, 3, Hq, D), _rand(22, L, Hkv, D), _rand(23, L, Hkv, D)
    qp = np.array([L - 3, L - 2, L - 1])
    a = O.attend(_bf16(q), qp, _bf16(k), _bf16(v), np.arange(L), S=4, W=512, precision="f32")
    b = O.attend(_bf16(q), qp, _bf16(k), _bf16(v), np.arange(L), S=4, W=512, precision="f64")
    assert np.abs(a - b).max() < 5e-6


def test_tiny_brute_force_python_loops():
    """Brute force in pure Python floats on a tiny case, keys listed from the interval set."""
    L, D, S, W = 11, 3, 2, 4
    q, k, v = _rand(24, L, 1, D), _rand(25, L, 1, D), _rand(26, L, 1, D)
    pos = np.arange(L)
    got = O.attend(_bf16(q), pos, _bf16(k), _bf16(v), pos, S=S, W=W, precision="f64")
    qf, kf, vf = q.double().tolist(), k.double().tolist(), v.double().tolist()
    for t in range(L):
        keys = [j for j in range(t + 1) if j in range(0, S) or j in range(t - W + 1, t + 1)]
        logit = [sum(qf[t][0][d] * kf[j][0][d] for d in range(D)) / math.sqrt(D) for j in keys]
        mx = max(logit)
        e = [math.exp(x - mx) for x in logit]
        z = sum(e)
        for d in range(D):
            want = sum(e[i] / z * vf[j][0][d] for i, j in enumerate(keys))
            assert abs(got[t, 0, d] - want) < 1e-6


def test_synth_generator_is_deterministic_and_unit_variance():
    a = synth.rows(5, synth.STREAM_K, 0, torch.arange(64) % 5, torch.arange(64) * 3, 4, 64)
    b = synth.rows(5, synth.STREAM_K, 0, torch.arange(64) % 5, torch.arange(64) * 3, 4, 64)
    c = synth.rows(5, synth.STREAM_V, 0, torch.arange(64) % 5, torch.arange(64) * 3, 4, 64)
    assert torch.equal(a, b) and not torch.equal(a, c)
    # a row is a pure function of its coordinates, not of its place in the batch
    one = synth.rows(5, synth.STREAM_K, 0, torch.tensor([13 % 5]), torch.tensor([13 * 3]), 4, 64)
    assert torch.equal(a[13], one[0])
    x = a.float()
    assert abs(x.mean().item()) < 0.03 and abs(x.std().item() - 1.0) < 0.03
    ch = torch.tensor([1, 70])
    o = synth.rows(5, synth.STREAM_K, 0, torch.arange(8), torch.arange(8), 4, 64, ch, 20.0).float().reshape(8, -1)
    base = synth.rows(5, synth.STREAM_K, 0, torch.arange(8), torch.arange(8), 4, 64).float().reshape(8, -1)
    ratio = o[:, ch] / base[:, ch]
    assert torch.allclose(ratio[base[:, ch] != 0], torch.tensor(20.0), rtol=1e-2)


@pytest.mark.parametrize("cls", ["definition", "paged"])
@pytest.mark.parametrize("S,W,L,ql", [(4, 6, 40, 5), (0, 9, 33, 8), (17, 5, 70, 3), (2, 100, 30, 7)])
def test_frame_queries_are_the_last_q_len_positions(cls, S, W, L, ql):
    """Pins the ONE line both oracle layers share that places a frame's queries (reading R15:
    the queries of attend_frame are the session's LAST q_len positions, row r at t = L - ql + r).
    With zero keys every admitted key gets the same weight, so row r of the chunk must be the plain
    mean of V over the paper's literal interval set [0,S) U (t-W, t] (reading R1) --
    computed here from the intervals, not from the oracle's mask.  A query placed one position off, in
    reverse order, or at the session's first positions moves that mean."""
    Hq, Hkv, D, B = 2, 1, 8, 4
    cfg = O.PoolConfig(n_q_heads=Hq, n_kv_heads=Hkv, head_dim=D, S=S, W=W, n_blocks=64, block_size=B,
                       max_sessions=2, max_new_tokens=16)
    ora = O.DefinitionOracle(cfg) if cls == "definition" else O.PagedOracle(cfg)
    sid = ora.session_open()
    g = torch.Generator().manual_seed(100 + L)
    v = torch.randn(L, Hkv, D, generator=g).to(torch.bfloat16)
    zeros = np.zeros((L, Hkv, D), np.uint16)
    # history in appends of <= 16 tokens, the last one exactly ql long
    cuts = list(range(0, L - ql, 11)) + [L - ql, L]
    for a, b in zip(cuts[:-1], cuts[1:]):
        if b > a:
            ora.append_kv(0, [sid], [b - a], zeros[a:b], _bf16(v[a:b]))
    q = _bf16(_rand(5, ql, Hq, D))
    out = ora.attend_frame(0, [sid], [ql], q)
    vf = v.double().numpy()
    for r in range(ql):
        t = L - ql + r
        keys = sorted(set(range(0, min(S, t + 1))) | set(range(max(0, t - W + 1), t + 1)))
        want = vf[keys, 0].mean(axis=0)
        for h in range(Hq):
            np.testing.assert_allclose(out[r, h], want, rtol=0, atol=1e-5)
