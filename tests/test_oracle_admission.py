"""NEXT row f3: the AIMD admission gate.  CPU only.

Pins of the oracle (oracle/admission_ref.py) against what AIMD fixes mathematically, then the
library's host-only gate (metronome_gate_*) against the oracle, decision by decision.  The paper
prints no constants or traces for the controller, so there is no golden file: parity is pinned by
closed forms (linear ramp, geometric decay, the sawtooth band around N*) and by the paper's own
falsifiable claim (a flat signal makes the loop over-admit up to its ceiling, L111).
"""
import numpy as np
import pytest

from oracle.admission_ref import AimdGateRef

CFG = dict(budget_ms=80.0, target_frac=0.8, add_step=1.0, mult_factor=0.5, cap_min=1.0, cap_max=512.0, cap_init=8.0)


def test_headroom_gives_a_linear_ramp_clamped_at_cap_max():
    g = AimdGateRef(**CFG)
    caps = [g.observe(10.0) for _ in range(600)]
    assert caps[:5] == [9.0, 10.0, 11.0, 12.0, 13.0]
    assert caps[-1] == 512.0 and all(b - a in (0.0, 1.0) for a, b in zip(caps, caps[1:]))


def test_overload_gives_geometric_decay_clamped_at_cap_min():
    g = AimdGateRef(**{**CFG, "cap_init": 256.0})
    caps = [g.observe(79.0) for _ in range(12)]
    assert caps[:8] == [128.0, 64.0, 32.0, 16.0, 8.0, 4.0, 2.0, 1.0] and caps[-1] == 1.0


def test_threshold_is_inclusive_at_the_target_fraction_of_the_budget():
    g = AimdGateRef(**CFG)
    assert g.observe(63.9) == 9.0          # below 0.8 * 80 = 64: additive increase
    assert g.observe(64.0) == 4.5          # "nears a target fraction": at the target counts as overload


def test_monotone_signal_converges_to_a_sawtooth_around_n_star():
    """Latency = c * N with everyone admitted up to the cap (L111: 'works only if latency is a monotone
    signal of load'): the cap must end up oscillating in [mult * N*, N* + add] with N* = target / c."""
    c = 0.25                                # ms per session: N* = 64 / 0.25 = 256
    g = AimdGateRef(**CFG)
    n_live, caps = 0, []
    for _ in range(3000):
        while g.admit(n_live):              # open-loop overload: there is always another arrival
            n_live += 1
        n_live = min(n_live, int(np.floor(g.cap)))      # sessions above a lowered cap drain away
        caps.append(g.observe(c * n_live))
    tail = np.asarray(caps[-1000:])
    assert tail.max() <= 256.0 + 1.0 and tail.min() >= 0.5 * 256.0 - 1.0
    assert 0.7 * 256 <= tail.mean() <= 0.8 * 256        # AIMD sawtooth mean = (1 + mult) / 2 * N* = 0.75 N*


def test_flat_signal_over_admits_to_the_ceiling():
    """The unbounded arm's signal is flat until the pool is gone (L111): 'nothing but headroom'."""
    g = AimdGateRef(**CFG)
    for _ in range(1000):
        g.observe(20.0)
    assert g.cap == 512.0 and g.admit(511) and not g.admit(512)


def test_invalid_configs_and_inputs():
    for bad in (dict(budget_ms=0.0), dict(target_frac=1.5), dict(add_step=0.0), dict(mult_factor=1.0),
                dict(cap_min=0.0), dict(cap_max=0.5), dict(cap_init=1000.0)):
        with pytest.raises(ValueError):
            AimdGateRef(**{**CFG, **bad})
    g = AimdGateRef(**CFG)
    with pytest.raises(ValueError):
        g.observe(float("nan"))
    with pytest.raises(ValueError):
        g.admit(-1)


def test_library_gate_takes_the_same_decisions_as_the_oracle():
    """metronome_gate_* is host-only, so it runs here: every cap and every admit decision must equal
    the oracle's on a seeded latency trace that crosses the threshold both ways."""
    from paper_2607_02640_b200 import binding, build
    build.build_library()
    rng = np.random.default_rng(260702640)
    for cfg in (CFG, dict(budget_ms=12.5, target_frac=0.9, add_step=0.37, mult_factor=0.83, cap_min=2.0, cap_max=300.0,
                          cap_init=17.0)):
        lib_g, ref = binding.Gate(**cfg), AimdGateRef(**cfg)
        thr = cfg["budget_ms"] * cfg["target_frac"]
        for k in range(4000):
            lat = float(np.float32(thr * rng.uniform(0.2, 1.6) if k % 7 else thr))
            assert lib_g.observe(lat) == ref.observe(lat)
            n = int(rng.integers(0, 320))
            assert lib_g.admit(n) == ref.admit(n)
    for bad in (dict(budget_ms=0.0), dict(mult_factor=1.0), dict(cap_init=1000.0)):
        with pytest.raises(binding.MetronomeError):
            binding.Gate(**{**CFG, **bad})
    g = binding.Gate(**CFG)
    with pytest.raises(binding.MetronomeError):
        g.observe(float("nan"))
    with pytest.raises(binding.MetronomeError):
        g.admit(-1)
