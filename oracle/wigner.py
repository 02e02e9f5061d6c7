"""Wigner 6j and 9j symbols of the oracle (TEST INFRASTRUCTURE ONLY).

Textbook definitions written out; every argument is a DOUBLED spin (an integer 2j).

  6j  Racah's single-sum formula, evaluated in exact rational arithmetic (Python integers and
      Fractions): the four triangle coefficients Delta^2 are multiplied as one Fraction, the
      alternating sum is a Fraction, and only the final square root is floating point.
  9j  the standard contraction of three 6j symbols,
        {j1 j2 j3; j4 j5 j6; j7 j8 j9} = sum_x (-1)^{2x} (2x+1) {j1 j4 j7; j8 j9 x}
                                          {j2 j5 j8; j4 x j6} {j3 j6 j9; x j1 j2}.
  9j by definition (`wigner_9j_by_cg`): the recoupling coefficient
        <(j1 j2)j3, (j4 j5)j6; j9 | (j1 j4)j7, (j2 j5)j8; j9>
          = sqrt((2j3+1)(2j6+1)(2j7+1)(2j8+1)) {j1 j2 j3; j4 j5 j6; j7 j8 j9}
      summed over Clebsch-Gordan products; slow, used by the tests to pin `wigner_9j`.

Pins (tests/test_oracle_wigner.py): exact rational values, the closed form
{a b c; b a 0} = (-1)^{a+b+c}/sqrt((2a+1)(2b+1)), the 6j orthogonality sum, the 9j with one zero
argument reducing to a 6j, the 9j orthogonality sum, the definition by Clebsch-Gordan sums, and (when
sympy is importable) sympy.physics.wigner for every argument set with j <= 3.

Nothing here is shared with the CUDA library (which has its own lgamma-based routines).
"""
from fractions import Fraction
from functools import lru_cache
from math import factorial, sqrt


def triangle(a, b, c):
    """Doubled spins a, b, c can couple (|a-b| <= c <= a+b and a+b+c even)."""
    return abs(a - b) <= c <= a + b and (a + b + c) % 2 == 0


def _delta2(a, b, c):
    """Triangle coefficient squared: (a+b-c)! (a-b+c)! (-a+b+c)! / (a+b+c+1)!  (true spins)."""
    return Fraction(factorial((a + b - c) // 2) * factorial((a - b + c) // 2) * factorial((-a + b + c) // 2),
                    factorial((a + b + c) // 2 + 1))


@lru_cache(maxsize=None)
def wigner_6j(a, b, c, d, e, f):
    """{a b c; d e f}, doubled arguments (Racah 1942)."""
    if not (triangle(a, b, c) and triangle(a, e, f) and triangle(d, b, f) and triangle(d, e, c)):
        return 0.0
    pre2 = _delta2(a, b, c) * _delta2(a, e, f) * _delta2(d, b, f) * _delta2(d, e, c)
    t1, t2, t3, t4 = (a + b + c) // 2, (a + e + f) // 2, (d + b + f) // 2, (d + e + c) // 2
    u1, u2, u3 = (a + b + d + e) // 2, (b + c + e + f) // 2, (a + c + d + f) // 2
    s = Fraction(0)
    for t in range(max(t1, t2, t3, t4), min(u1, u2, u3) + 1):
        term = Fraction(factorial(t + 1),
                        factorial(t - t1) * factorial(t - t2) * factorial(t - t3) * factorial(t - t4)
                        * factorial(u1 - t) * factorial(u2 - t) * factorial(u3 - t))
        s += -term if t & 1 else term
    # sqrt of an exact rational: numerator and denominator separately
    v = sqrt(pre2.numerator) / sqrt(pre2.denominator) * float(abs(s))
    return v if s > 0 else -v


@lru_cache(maxsize=None)
def wigner_9j(j1, j2, j3, j4, j5, j6, j7, j8, j9):
    """{j1 j2 j3; j4 j5 j6; j7 j8 j9}, doubled arguments."""
    rows_cols = [(j1, j2, j3), (j4, j5, j6), (j7, j8, j9), (j1, j4, j7), (j2, j5, j8), (j3, j6, j9)]
    if not all(triangle(*t) for t in rows_cols):
        return 0.0
    lo = max(abs(j1 - j9), abs(j4 - j8), abs(j2 - j6))
    hi = min(j1 + j9, j4 + j8, j2 + j6)
    s = 0.0
    for x in range(lo, hi + 1, 2):
        v = (x + 1) * wigner_6j(j1, j4, j7, j8, j9, x) * wigner_6j(j2, j5, j8, j4, x, j6) * wigner_6j(j3, j6, j9, x, j1, j2)
        s += -v if x & 1 else v
    return s


def wigner_9j_by_cg(j1, j2, j3, j4, j5, j6, j7, j8, j9):
    """The 9j symbol from its definition as a recoupling coefficient of four angular momenta
    (sum over Clebsch-Gordan products at fixed total M = j9).  Slow; for the tests."""
    from .su2 import cg
    rows_cols = [(j1, j2, j3), (j4, j5, j6), (j7, j8, j9), (j1, j4, j7), (j2, j5, j8), (j3, j6, j9)]
    if not all(triangle(*t) for t in rows_cols):
        return 0.0
    M = j9
    s = 0.0
    for m1 in range(-j1, j1 + 1, 2):
        for m2 in range(-j2, j2 + 1, 2):
            m3 = m1 + m2
            if abs(m3) > j3:
                continue
            c12 = cg(j1, m1, j2, m2, j3, m3)
            if c12 == 0.0:
                continue
            for m4 in range(-j4, j4 + 1, 2):
                m5 = M - m3 - m4
                if abs(m5) > j5:
                    continue
                m6, m7, m8 = m4 + m5, m1 + m4, m2 + m5
                if abs(m6) > j6 or abs(m7) > j7 or abs(m8) > j8:
                    continue
                s += (c12 * cg(j4, m4, j5, m5, j6, m6) * cg(j3, m3, j6, m6, j9, M)
                      * cg(j1, m1, j4, m4, j7, m7) * cg(j2, m2, j5, m5, j8, m8) * cg(j7, m7, j8, m8, j9, M))
    return s / sqrt((j3 + 1) * (j6 + 1) * (j7 + 1) * (j8 + 1))
