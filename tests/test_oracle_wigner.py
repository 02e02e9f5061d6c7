"""Pins for oracle/wigner.py (SURVEY.md 8(c) "c4 SU(2)": Wigner symbols against orthogonality sums and
exact rational values for j <= 3).  Every argument is a doubled spin."""
from fractions import Fraction
from math import sqrt

import pytest

from oracle.wigner import triangle, wigner_6j, wigner_9j, wigner_9j_by_cg


def test_6j_exact_rational_values():
    # textbook values: {1 1 1; 1 1 1} = 1/6, {1 1 2; 1 1 2} = 1/30, {2 2 2; 2 2 2} = -3/70,
    # {1/2 1/2 1; 1/2 1/2 1} = 1/6, {1/2 1/2 1; 1/2 1/2 0} = 1/2, {1/2 1/2 0; 1/2 1/2 0} = -1/2
    assert wigner_6j(2, 2, 2, 2, 2, 2) == pytest.approx(1 / 6, abs=1e-15)
    assert wigner_6j(2, 2, 4, 2, 2, 4) == pytest.approx(1 / 30, abs=1e-15)
    assert wigner_6j(4, 4, 4, 4, 4, 4) == pytest.approx(-3 / 70, abs=1e-15)
    assert wigner_6j(1, 1, 2, 1, 1, 2) == pytest.approx(1 / 6, abs=1e-15)
    assert wigner_6j(1, 1, 2, 1, 1, 0) == pytest.approx(1 / 2, abs=1e-15)
    assert wigner_6j(1, 1, 0, 1, 1, 0) == pytest.approx(-1 / 2, abs=1e-15)
    assert wigner_6j(2, 2, 2, 2, 2, 0) == pytest.approx(-1 / 3, abs=1e-15)
    assert wigner_6j(2, 2, 2, 2, 2, 4) == pytest.approx(1 / 6, abs=1e-15)
    assert wigner_6j(6, 6, 6, 6, 6, 6) == pytest.approx(-1 / 14, abs=1e-15)


def test_6j_closed_form_with_a_zero_and_triangle_violations():
    # {a b c; b a 0} = (-1)^{a+b+c} / sqrt((2a+1)(2b+1))
    for a in range(0, 9):
        for b in range(0, 9):
            for c in range(abs(a - b), a + b + 1, 2):
                want = (-1) ** ((a + b + c) // 2) / sqrt((a + 1) * (b + 1))
                assert wigner_6j(a, b, c, b, a, 0) == pytest.approx(want, abs=1e-14)
    assert wigner_6j(1, 1, 4, 1, 1, 0) == 0.0          # 1/2, 1/2 cannot couple to 2
    assert wigner_6j(1, 2, 2, 1, 1, 1) == 0.0          # half-integer sum


def test_6j_orthogonality():
    # sum_x (2x+1)(2f+1) {a b x; c d f} {a b x; c d g} = delta_fg
    for (a, b, c, d) in [(1, 2, 3, 2), (2, 2, 2, 2), (3, 1, 2, 4), (4, 3, 5, 2), (6, 5, 3, 4), (7, 2, 6, 3)]:
        fs = [f for f in range(0, 14) if triangle(a, d, f) and triangle(c, b, f)]
        for f in fs:
            for g in fs:
                s = sum((x + 1) * (f + 1) * wigner_6j(a, b, x, c, d, f) * wigner_6j(a, b, x, c, d, g)
                        for x in range(0, 14) if triangle(a, b, x) and triangle(c, d, x))
                assert s == pytest.approx(1.0 if f == g else 0.0, abs=1e-13)


def test_9j_reduces_to_6j_when_an_argument_is_zero():
    # {a b c; d e f; g h 0} = delta_cf delta_gh (-1)^{b+c+d+g} / sqrt((2c+1)(2g+1)) {a b c; e d g}
    for a in range(0, 5):
        for b in range(0, 5):
            for c in range(abs(a - b), a + b + 1, 2):
                for d in range(0, 5):
                    for e in range(0, 5):
                        if not triangle(d, e, c):
                            continue
                        for g in range(abs(a - d), a + d + 1, 2):
                            if not triangle(b, e, g):
                                continue
                            want = (-1) ** ((b + c + d + g) // 2) / sqrt((c + 1) * (g + 1)) * wigner_6j(a, b, c, e, d, g)
                            assert wigner_9j(a, b, c, d, e, c, g, g, 0) == pytest.approx(want, abs=1e-13)


def test_9j_equals_its_definition_by_clebsch_gordan_sums():
    # the recoupling coefficient of four angular momenta, summed over six Clebsch-Gordan coefficients
    args = [(1, 1, 2, 1, 1, 0, 2, 2, 2), (1, 2, 3, 2, 1, 3, 1, 3, 2), (2, 1, 1, 1, 0, 1, 3, 1, 2), (2, 2, 2, 2, 2, 2, 2, 2, 2),
            (3, 1, 2, 2, 2, 2, 1, 1, 0), (4, 1, 3, 2, 1, 1, 2, 2, 2), (0, 1, 1, 1, 0, 1, 1, 1, 2), (3, 0, 3, 1, 1, 2, 2, 1, 1),
            (2, 1, 3, 0, 1, 1, 2, 2, 4), (5, 1, 4, 2, 1, 3, 3, 2, 1)]
    n = 0
    for a in args:
        d = wigner_9j_by_cg(*a)
        assert wigner_9j(*a) == pytest.approx(d, abs=1e-13)
        n += d != 0.0
    assert n >= 7                                      # the list is not made of trivially zero symbols


def test_9j_orthogonality():
    # sum_{c,f} (2c+1)(2f+1)(2g+1)(2h+1) {a b c; d e f; g h i} {a b c; d e f; g' h' i} = delta_gg' delta_hh'
    for (a, b, d, e, i) in [(1, 2, 1, 1, 1), (2, 1, 2, 1, 2), (3, 1, 2, 2, 2), (2, 2, 2, 2, 0), (4, 1, 1, 2, 2)]:
        gh = [(g, h) for g in range(0, 10) for h in range(0, 10)
              if triangle(a, d, g) and triangle(b, e, h) and triangle(g, h, i)]
        for (g, h) in gh:
            for (g2, h2) in gh:
                s = 0.0
                for c in range(abs(a - b), a + b + 1, 2):
                    for f in range(abs(d - e), d + e + 1, 2):
                        if triangle(c, f, i):
                            s += ((c + 1) * (f + 1) * (g + 1) * (h + 1) * wigner_9j(a, b, c, d, e, f, g, h, i)
                                  * wigner_9j(a, b, c, d, e, f, g2, h2, i))
                assert s == pytest.approx(1.0 if (g, h) == (g2, h2) else 0.0, abs=1e-12)


def test_against_sympy_for_all_small_arguments():
    """Exact rational/surd values for j <= 3 (SURVEY.md 8(c) pins); sympy is on the build machine, not required
    on the GPU box."""
    sw = pytest.importorskip("sympy.physics.wigner")
    import sympy
    half = lambda x: sympy.Rational(x, 2)
    n = 0
    for a in range(0, 7):
        for b in range(0, 7):
            for c in range(abs(a - b), min(a + b, 6) + 1, 2):
                for d in range(0, 5):
                    for e in range(0, 5):
                        for f in range(0, 5):
                            if triangle(a, e, f) and triangle(d, b, f) and triangle(d, e, c):
                                want = float(sw.wigner_6j(half(a), half(b), half(c), half(d), half(e), half(f)))
                                assert wigner_6j(a, b, c, d, e, f) == pytest.approx(want, abs=1e-14)
                                n += 1
    assert n > 500
    for args in [(1, 1, 2, 1, 1, 2, 2, 2, 4), (2, 1, 3, 1, 1, 2, 3, 2, 1), (2, 2, 2, 1, 1, 2, 1, 1, 0), (3, 1, 2, 1, 1, 2, 2, 2, 4),
                 (4, 2, 2, 1, 1, 2, 3, 1, 2), (2, 1, 1, 2, 1, 1, 2, 2, 2), (6, 1, 5, 2, 1, 3, 4, 2, 2)]:
        want = float(sw.wigner_9j(*[half(x) for x in args], prec=64))
        assert wigner_9j(*args) == pytest.approx(want, abs=1e-14)
