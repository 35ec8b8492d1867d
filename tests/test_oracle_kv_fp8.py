"""Pins of the fp8 KV quantiser of the oracle (oracle/kv_fp8.py, PAPER.md:L101
"we bound which tokens stay resident, and the two compose").  `-m "not gpu"`.

The format (E4M3, "e4m3fn") is fixed outside this repo: its value table has a closed form, torch ships a conversion
routine for it, and rounding to nearest can be checked by brute force over all 256 codes.  A wrong bias, a wrong
subnormal spacing, ties away from zero, a missing saturation or a transposed scale each fail one of these.
"""
import numpy as np
import pytest
import torch

from oracle import bounded_kv as O
from oracle import kv_fp8 as F


def test_code_table_is_the_e4m3fn_format():
    tab = F.decode_table()
    # the landmarks of the format
    assert tab[0x00] == 0.0 and np.signbit(tab[0x80]) and tab[0x80] == 0.0
    assert tab[0x7E] == 448.0 and tab[0xFE] == -448.0             # largest finite
    assert np.isnan(tab[0x7F]) and np.isnan(tab[0xFF])            # the only NaNs; no infinities
    assert tab[0x01] == 2.0 ** -9 and tab[0x07] == 7 * 2.0 ** -9  # subnormals
    assert tab[0x08] == 2.0 ** -6 and tab[0x38] == 1.0 and tab[0x3C] == 1.5
    # and all of it against the library's own decoding of the same bytes
    ref = torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).float().numpy()
    ok = ~np.isnan(ref)
    assert ok.sum() == 254 and np.array_equal(tab[ok], ref[ok]) and np.isnan(tab[~ok]).all()
    finite = tab[:0x7F]
    assert np.all(np.diff(finite) > 0), "positive codes are ordered like their values"


def test_encode_is_round_to_nearest_even_by_brute_force():
    tab = F.decode_table()
    vals = tab[:0x7F].astype(np.float64)                           # 0 .. 448, ascending
    rng = np.random.default_rng(0)
    # every value, every midpoint between neighbours, points just around the midpoints, random points, out of range
    mids = (vals[:-1] + vals[1:]) / 2
    pts = np.concatenate([vals, mids, np.nextafter(mids.astype(np.float32), np.float32(0)), np.nextafter(mids.astype(np.float32), np.float32(1e9)),
                          rng.uniform(0, 448, 20000), rng.uniform(0, 0.05, 5000), [448.0, 449.0, 464.0, 500.0, 1e9]]).astype(np.float32)
    pts = np.concatenate([pts, -pts])
    got = F.decode(F.encode(pts)).astype(np.float64)
    for x, g in zip(pts.astype(np.float64), got):
        a = min(abs(x), 448.0)
        d = np.abs(vals - a)
        best = d.min()
        cands = vals[d == best]
        if len(cands) == 2:                                        # a tie: the one with the even mantissa (even code)
            codes = [int(np.where(vals == c)[0][0]) for c in cands]
            want = cands[0] if codes[0] % 2 == 0 else cands[1]
        else:
            want = cands[0]
        assert abs(g) == want and (g == 0 or np.sign(g) == np.sign(x)), (x, g, want)


def test_encode_matches_the_library_conversion():
    rng = np.random.default_rng(1)
    x = np.concatenate([rng.standard_normal(200000) * 100, rng.standard_normal(50000) * 0.01, rng.uniform(-448, 448, 100000)]).astype(np.float32)
    x = x[np.abs(x) <= 448]
    ref = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    got = F.encode(x)
    same = got == ref
    # (+0 and -0 results may differ in sign for inputs that round to zero: compare values there)
    assert np.array_equal(F.decode(got[~same]), F.decode(ref[~same])) and (~same).mean() < 1e-3


def test_round_trip_error_bounds_and_the_row_scale():
    rng = np.random.default_rng(2)
    x = torch.from_numpy(rng.standard_normal((64, 3, 128)).astype(np.float32) * rng.uniform(0.01, 50, (64, 3, 1)).astype(np.float32)).to(torch.bfloat16)
    u16 = x.view(torch.int16).numpy().view(np.uint16)
    codes, scales = F.quantize_rows(u16)
    assert codes.shape == (64, 3, 128) and scales.shape == (64, 3) and scales.dtype == np.float32
    xf = x.float().numpy()
    amax = np.abs(xf).max(-1)
    assert np.array_equal(scales, (amax / np.float32(448)).astype(np.float32))            # one scale per (token, head) ROW
    xhat = F.dequantize(codes, scales)
    # the largest element of a row lands on +-448 and comes back within one float32 rounding
    idx = np.abs(xf).argmax(-1)
    top = np.take_along_axis(np.abs(F.decode(codes)), idx[..., None], -1)[..., 0]
    assert np.all(top == 448.0)
    back = np.take_along_axis(np.abs(xhat), idx[..., None], -1)[..., 0]
    assert np.all(np.abs(back - amax) <= amax * 2.0 ** -22)
    # half a unit in the last place: 2^-4 relative for normal codes, 2^-10 of the row maximum's scale below them
    err = np.abs(xhat - xf)
    bound = np.maximum(np.abs(xf) * 2.0 ** -4, scales[..., None] * 2.0 ** -10) * (1 + 1e-6)
    assert np.all(err <= bound)
    # an all-zero row keeps scale 1 and decodes to zeros
    z = np.zeros((1, 1, 16), np.uint16)
    c0, s0 = F.quantize_rows(z)
    assert s0[0, 0] == 1.0 and not F.dequantize(c0, s0).any()


def test_exactly_representable_rows_come_back_unchanged_and_the_fp8_arm_then_equals_the_bf16_arm():
    """Rows whose entries are (E4M3 values) x 2^k are stored without loss; the fp8 attention arm must then give
    exactly what the (pinned) bf16 arm gives: ties the new C entry point and the fp8 plumbing to the old one."""
    rng = np.random.default_rng(3)
    tab = F.decode_table()
    pool = tab[[0x00, 0x30, 0x38, 0x3C, 0x40, 0x44, 0x7E, 0xB8, 0xC0, 0xFE]]        # 0, .5, 1, 1.5, 2, 3, 448, -1, -2, -448
    def rows(n, H, D):
        x = rng.choice(pool, size=(n, H, D)).astype(np.float32)
        x[..., 0] = 448.0 * np.sign(rng.standard_normal((n, H)))                       # every row's maximum is 448 -> scale 1 ... x 2^-5
        x *= 2.0 ** -5
        return torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    cfgs = [O.PoolConfig(n_q_heads=4, n_kv_heads=2, head_dim=32, S=3, W=20, n_blocks=64, max_sessions=2, max_new_tokens=8, kv_fp8=f)
            for f in (False, True)]
    a, b = O.DefinitionOracle(cfgs[0]), O.DefinitionOracle(cfgs[1])
    sa, sb = a.session_open(), b.session_open()
    for step in range(12):
        n = int(rng.integers(1, 9))
        k, v = rows(n, 2, 32), rows(n, 2, 32)
        assert np.array_equal(F.roundtrip(k), F.bf16_to_f32(k))
        q = torch.from_numpy(rng.standard_normal((n, 4, 32)).astype(np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
        a.append_kv(0, [sa], [n], k, v); b.append_kv(0, [sb], [n], k, v)
        assert np.array_equal(a.attend_frame(0, [sa], [n], q), b.attend_frame(0, [sb], [n], q))


def test_fp8_attention_stays_close_to_the_unquantised_one():
    """Sanity on the composition itself: on N(0,1) rows the fp8 arm's outputs differ from the bf16 arm's by a few
    percent of the output scale (2^-4 per element, averaged down over the keys) -- not equal, not far."""
    rng = np.random.default_rng(4)
    mk = lambda n, H: torch.from_numpy(rng.standard_normal((n, H, 64)).astype(np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    cfgs = [O.PoolConfig(n_q_heads=4, n_kv_heads=2, head_dim=64, S=4, W=64, n_blocks=64, max_sessions=1, max_new_tokens=128, kv_fp8=f)
            for f in (False, True)]
    a, b = O.DefinitionOracle(cfgs[0]), O.DefinitionOracle(cfgs[1])
    sa, sb = a.session_open(), b.session_open()
    k, v, q = mk(100, 2), mk(100, 2), mk(100, 4)
    a.append_kv(0, [sa], [100], k, v); b.append_kv(0, [sb], [100], k, v)
    oa, ob = a.attend_frame(0, [sa], [100], q), b.attend_frame(0, [sb], [100], q)
    d = np.abs(oa - ob)
    assert 1e-4 < d.max() < 0.25 and np.sqrt((d ** 2).mean()) < 0.03
