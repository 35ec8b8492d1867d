"""Oracle for NEXT row f3: the AIMD admission loop of PAPER.md:L105-111 (sec. 4.2).

TEST INFRASTRUCTURE ONLY (imported by tests/ and nothing else); shares no code with the library.

The paper states the rule in words and gives no constants: "an AIMD loop [Chiu and Jain 1989,
Jacobson 1988] on the measured per-frame latency, which lowers the admission cap multiplicatively when
latency nears a target fraction of the budget and raises it additively to probe when there is
headroom.  Arrivals beyond the cap receive a clean overload rejection."  PARITY UNPINNED BY THE PAPER:
the recurrence below is this build's reading (R17); it is pinned against the textbook AIMD
closed forms in tests/test_oracle_admission.py.

All arithmetic in float32, one operation after the other, because the rule decides integers (admit or
shed) from floating point and both sides must take that decision in the same precision.
"""
import numpy as np

f32 = np.float32


class AimdGateRef:
    def __init__(self, budget_ms, target_frac, add_step, mult_factor, cap_min, cap_max, cap_init):
        ok = (budget_ms > 0 and 0 < target_frac <= 1 and add_step > 0 and 0 < mult_factor < 1 and cap_min >= 1
              and cap_max >= cap_min and cap_min <= cap_init <= cap_max)
        if not ok:
            raise ValueError("INVALID_ARG")
        self.budget, self.frac = f32(budget_ms), f32(target_frac)
        self.add, self.mult = f32(add_step), f32(mult_factor)
        self.lo, self.hi = f32(cap_min), f32(cap_max)
        self.cap = f32(cap_init)

    def observe(self, latency_ms):
        """One update per frame: multiplicative decrease at / above the target, else additive increase."""
        lat = f32(latency_ms)
        if not lat >= 0:
            raise ValueError("INVALID_ARG")
        if lat >= f32(self.frac * self.budget):
            self.cap = max(self.lo, f32(self.cap * self.mult))
        else:
            self.cap = min(self.hi, f32(self.cap + self.add))
        return float(self.cap)

    def admit(self, n_live):
        if n_live < 0:
            raise ValueError("INVALID_ARG")
        return n_live < int(np.floor(self.cap))
