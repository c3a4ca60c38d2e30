"""SplitMix64: the one PRNG every synthetic input is drawn from.

seed -> state; each draw: state += 0x9E3779B97F4A7C15, then the usual two
xor-shift-multiply rounds.  u01 = (x >> 11) * 2**-53.
Pure Python integers, so the stream is identical on every machine.
"""

_MASK = (1 << 64) - 1


class SplitMix64:
    def __init__(self, seed: int):
        self.state = seed & _MASK

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & _MASK
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
        return z ^ (z >> 31)

    def u01(self) -> float:
        return (self.next_u64() >> 11) * (2.0 ** -53)

    def uniform(self, lo: float, hi: float) -> float:
        return lo + (hi - lo) * self.u01()
