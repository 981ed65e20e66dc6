"""Host check of the claim the metric kernels rest on (paper_2303_10785_b200/csrc/meg6_geom.cuh, `div12`): the
three-operation sequence  q = RN(x y), r = fma(-12, q, x), z = fma(r, y, q)  with y = RN(1/12)  equals the correctly
rounded quotient x / 12 -- the value the oracle's division of Eq. 16 produces -- for every operand away from
over/underflow.  The fused operations are evaluated exactly with rationals and rounded once (`float(Fraction)` rounds to
nearest even), so this restates the arithmetic, not the CUDA code."""
import random
from fractions import Fraction

import numpy as np


def fma(a, b, c):
    return float(Fraction(a) * Fraction(b) + Fraction(c))


def div12_sequence(x):
    y = 1.0 / 12.0
    q = x * y
    r = fma(-12.0, q, x)
    assert Fraction(r) == Fraction(x) - 12 * Fraction(q)      # the residual is exact
    return fma(r, y, q)


def test_sequence_equals_correctly_rounded_division():
    rng = random.Random(12)
    xs = [0.0, 1.0, 12.0, 3.0, 1.0 / 3.0, 2.0 / 3.0, np.nextafter(12.0, 0.0), np.nextafter(12.0, 24.0), 1e-30, -7.5e22]
    for _ in range(20000):
        m = rng.getrandbits(52) | (1 << 52)
        xs.append((-1.0) ** rng.getrandbits(1) * float(m) * 2.0 ** rng.randint(-120, 60))
    # operands whose quotient sits next to a rounding boundary: x = 12 (k + 1/2 +- tiny) ulp-wise is impossible (x/12
    # lies on thirds of an ulp), so probe the closest attainable neighbours: 3 q +- 1 in units of the last place
    for _ in range(20000):
        k = rng.getrandbits(52) | (1 << 52)
        for d in (-1, 1):
            xs.append(float(3 * k + d) * 2.0 ** rng.randint(-60, 10))
    for x in xs:
        x = float(x)
        assert div12_sequence(x) == x / 12.0, x.hex()
