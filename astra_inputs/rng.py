"""Counter-free splitmix64 stream used by the design-point sweeps (SURVEY.md 8(d) conventions).

One stream per design point, seed = 260610440*1000000 + config*100000 + point.
Uniform ints are `x mod range` on the raw 64-bit output; uniforms in [0,1) use the top
53 bits; normals use Box-Muller on two such uniforms.  The generator runs once in Python
and both simulators receive identical arrays, so its floating point cannot affect parity.
"""
from __future__ import annotations

import math

_M64 = (1 << 64) - 1


def config_seed(config: int, point: int) -> int:
    return 260610440 * 1000000 + config * 100000 + point


class SplitMix64:
    def __init__(self, seed: int):
        self.state = seed & _M64

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & _M64
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
        return z ^ (z >> 31)

    def randint(self, lo: int, hi: int) -> int:
        """Uniform integer in [lo, hi] (inclusive) by modulo."""
        return lo + self.next_u64() % (hi - lo + 1)

    def uniform(self) -> float:
        return (self.next_u64() >> 11) * (1.0 / (1 << 53))

    def normal(self) -> float:
        u1 = self.uniform()
        u2 = self.uniform()
        if u1 <= 0.0:
            u1 = 1.0 / (1 << 53)
        return math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2)
