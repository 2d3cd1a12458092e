"""Second, independent statement of the clustering definition, for tiny modules only.

TEST INFRASTRUCTURE ONLY.  Pure Python with exact rationals (fractions.Fraction); shares no
code with oracle/sst_oracle.c or with the CUDA path.  It pins the C oracle by brute force:
enumerate EVERY interval [l, r] of one module and keep those that satisfy the definition
(BASELINE.json north_star; section 2):

  all strips of [l, r] active; strip l-1 and strip r+1 inactive or outside the module;
  at least one seed strip inside; (sum q)^2 >= t_cl^2 * sum noise^2.

Decisions are taken in exact rational arithmetic.  That equals the C oracle's float/double
forms whenever the double sum of noise^2 is exact (tests use short-mantissa noise values).
The float32 steps of the gain correction are reproduced by an explicit round-to-nearest-even
of the exact quotient to 24 significant bits (f32_round), not by a library division.
"""
from __future__ import annotations

from fractions import Fraction
from math import floor
from typing import List, Sequence, Tuple


def f32_round(x: Fraction) -> Fraction:
    """Round a positive rational to the nearest IEEE binary32 value (ties to even), normal
    range only."""
    if x == 0:
        return Fraction(0)
    assert x > 0
    e = 0
    # find e with 2^23 <= x / 2^e < 2^24
    while x / Fraction(2) ** e >= 2 ** 24:
        e += 1
    while x / Fraction(2) ** e < 2 ** 23:
        e -= 1
    m = x / Fraction(2) ** e
    lo = floor(m)
    rem = m - lo
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and lo % 2 == 1):
        lo += 1
    return Fraction(lo) * Fraction(2) ** e


def gain_correct(adc: int, gain: float) -> int:
    """min(254, floor(fl32(fl32(adc / gain) + 0.5))) with every float32 rounding explicit."""
    t = f32_round(Fraction(adc) / Fraction(gain))
    u = f32_round(t + Fraction(1, 2))
    return min(254, floor(u))


def strip_flags(adc: Sequence[int], noise: Sequence[float], bad: Sequence[int], t_ch: float,
                t_seed: float) -> Tuple[List[bool], List[bool]]:
    act, seed = [], []
    for a, n, b in zip(adc, noise, bad):
        is_a = (not b) and a > 0 and Fraction(a) >= Fraction(t_ch) * Fraction(n)
        act.append(bool(is_a))
        seed.append(bool(is_a and Fraction(a) >= Fraction(t_seed) * Fraction(n)))
    return act, seed


def clusters_of_module(adc: Sequence[int], gain: Sequence[float], noise: Sequence[float],
                       bad: Sequence[int], thresholds: Tuple[float, float, float]):
    """All clusters of ONE module by exhaustive interval enumeration, ascending first strip.
    Returns [(first, width, [q...], charge, barycenter Fraction, snr^2 Fraction)]."""
    t_ch, t_seed, t_cl = thresholds
    k = len(adc)
    act, seed = strip_flags(adc, noise, bad, t_ch, t_seed)
    out = []
    for l in range(k):
        for r in range(l, k):
            if not all(act[l:r + 1]):
                continue
            if l > 0 and act[l - 1]:
                continue
            if r < k - 1 and act[r + 1]:
                continue
            if not any(seed[l:r + 1]):
                continue
            q = [gain_correct(adc[i], gain[i]) for i in range(l, r + 1)]
            Q = sum(q)
            n2 = sum(Fraction(noise[i]) ** 2 for i in range(l, r + 1))
            if Fraction(Q) ** 2 < Fraction(t_cl) ** 2 * n2:
                continue
            bary = Fraction(l) + Fraction(sum(i * qi for i, qi in enumerate(q)), Q)
            out.append((l, r - l + 1, q, Q, bary, Fraction(Q) ** 2 / n2))
    return out
