"""Pins of the oracle's performant-mode model (oracle/ozaki.py: emulated_gemm(keep=), class_exponents,
performant_keep, truncation_bound, emulated_sum) -- PAPER.md:53, 59 "performant mode ... dynamic mantissa bit
settings"; reading s21.  None of these call the CUDA path.

What fixes the functions from outside:
  * the exact product in Python integers (inputs on a dyadic grid), against which every error is measured;
  * the 2^-8-per-slice law: one kept slice less multiplies the error by about 2^8;
  * the a-priori bound derived in `truncation_bound`'s docstring (the error must be below it and not absurdly below);
  * the statement the rule is built for: no class's bound exceeds the reference class's bound at kappa slices.
"""
from fractions import Fraction

import numpy as np
import pytest

from oracle import ozaki as oz


def _dyadic(rng, shape, bits=30, scale=0):
    """Random values m 2^(scale - bits), m integer: products and sums are exact in Python ints."""
    m = rng.integers(-2 ** bits, 2 ** bits, size=shape)
    return np.ldexp(m.astype(np.float64), scale - bits), m


def _exact(mA, mB):
    """Integer matrix product with Python ints (no overflow)."""
    M, K = mA.shape
    N = mB.shape[1]
    return [[sum(int(mA[i, k]) * int(mB[k, j]) for k in range(K)) for j in range(N)] for i in range(M)]


def _err(C, ex, shift):
    """max |C - ex 2^shift| with ex a table of Python ints (exact rational arithmetic)."""
    worst = Fraction(0)
    for i, row in enumerate(ex):
        for j, v in enumerate(row):
            d = abs(Fraction(float(C[i, j])) - Fraction(v) * Fraction(2) ** shift)
            worst = max(worst, d)
    return float(worst)


def test_keep_kappa_is_the_whole_triangular_set():
    rng = np.random.default_rng(0)
    A, B = rng.standard_normal((9, 70)), rng.standard_normal((70, 6))
    for kappa in (4, 6, 7):
        assert np.array_equal(oz.emulated_gemm(A, B, kappa, keep=kappa), oz.emulated_gemm(A, B, kappa))


def test_two_to_the_minus_eight_per_kept_slice_and_the_bound():
    rng = np.random.default_rng(1)
    K = 96
    A, mA = _dyadic(rng, (7, K))
    B, mB = _dyadic(rng, (K, 5))
    ex = _exact(mA, mB)
    ea, eb = oz.exponents(A, 1), oz.exponents(B, 0)
    errs = []
    for keep in (2, 3, 4, 5, 6):
        C = oz.emulated_gemm(A, B, 6, keep=keep)
        e = _err(C, ex, -60)
        bound = oz.truncation_bound(ea, eb, K, 6, keep).max()
        assert e <= bound, (keep, e, bound)
        assert e >= bound * 2.0 ** -12, (keep, e, bound)       # the bound is not vacuous
        errs.append(e)
    for a, b in zip(errs, errs[1:]):
        assert 2.0 ** 6 <= a / b <= 2.0 ** 10, errs


def test_dropped_products_are_exactly_the_anti_diagonals_beyond_keep():
    """One-element lines whose digits are known: a = b = 1 + 2^-8 + 2^-16 (three digits 32, 32, 32 at exponent 1).
    The product keeps the anti-diagonals c = s + t <= keep + 1."""
    a = np.array([[1.0 + 2.0 ** -8 + 2.0 ** -16]])
    d, _ = oz.slice_lines(a, oz.exponents(a, 1), 3, 1)
    assert d[:, 0, 0].tolist() == [32, 32, 32]
    scale = 2.0 ** (2 * (1 - (8 * 3 - 2)))                      # 2^(ea + eb - 2 BASE)
    want = {3: 32 * 32 * (256 ** 4 + 2 * 256 ** 3 + 3 * 256 ** 2), 2: 32 * 32 * (256 ** 4 + 2 * 256 ** 3), 1: 32 * 32 * 256 ** 4}
    for keep, v in want.items():
        assert oz.emulated_gemm(a, a, 3, keep=keep)[0, 0] == v * scale


def test_class_exponents_bound_every_element_and_ignore_ambiguous_lines():
    rng = np.random.default_rng(2)
    A, B = rng.standard_normal((6, 100)) * 3.0, rng.standard_normal((100, 4)) * 0.01
    ea, eb = oz.exponents(A, 1), oz.exponents(B, 0)
    E_all, E_nz = oz.class_exponents(ea, eb, -0.3, 100)
    assert np.abs(-0.3 * A @ B).max() < 2.0 ** E_all
    assert E_all == ea.max() + eb.max() + (-1) + 2 and E_nz == E_all       # frexp(0.3) = 0.6 2^-1; 4 k steps -> 2
    # an all-zero line (exponent 0) among small lines must not raise the reference exponent
    B2 = B.copy(); B2[:, 1] = 0.0
    eb2 = oz.exponents(B2, 0)
    assert eb2[1] == 0 and eb2.max() == 0
    E_all2, E_nz2 = oz.class_exponents(ea, eb2, -0.3, 100)
    assert E_all2 > E_all - 1 and E_nz2 == ea.max() + np.delete(eb2, 1).max() - 1 + 2
    # no line with a non-zero exponent on one side: the class cannot serve as a reference
    assert oz.class_exponents(np.zeros(3, dtype=int), eb, 1.0, 32)[1] is None


def test_rule_drops_one_slice_per_eight_bits_of_spread():
    E = [40, 33, 32, 25, 24, 16, 8, 0, -50]
    assert oz.performant_keep(E, E, 6, 3) == [6, 6, 5, 5, 4, 3, 3, 3, 3]
    assert oz.performant_keep(E, E, 7, 2) == [7, 7, 6, 6, 5, 4, 3, 2, 2]
    assert oz.performant_keep([e + 123 for e in E], [e + 123 for e in E], 6, 3) == oz.performant_keep(E, E, 6, 3)
    assert oz.performant_keep(E, [None] * len(E), 6, 3) == [6] * len(E)
    # the reference is the largest E_nz, not the largest E_all
    assert oz.performant_keep([40, 20], [None, 20], 6, 3) == [6, 6]
    assert oz.performant_keep([40, 20], [28, 20], 6, 3) == [6, 5]
    rng = np.random.default_rng(3)
    for _ in range(50):
        E = rng.integers(-60, 60, size=12).tolist()
        k = oz.performant_keep(E, E, 6, 3)
        ref = max(E)
        for e, kp in zip(E, k):
            assert 3 <= kp <= 6
            d = 6 - kp
            assert ref - e >= 8 * d                                # a slice is dropped only per 8 whole bits of spread:
            assert e - 8 * kp <= ref - 48                          #   the class's bound exponent <= the reference's at kappa
            assert kp == 3 or ref - e < 8 * (d + 1)                # and none is kept that the rule lets go (above kmin)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_performant_sum_keeps_the_eager_error_level(seed):
    """Classes whose magnitudes are 2^0, 2^-9, 2^-17, 2^-30 relative to the first (none with a line exponent of 0): the rule keeps 6, 5, 4, 3 slices;
    the error of the sum stays below (number of classes) x (bound of the reference class at kappa slices), and the
    eager sum (6 slices everywhere) is not better than that level either by more than the bound allows."""
    rng = np.random.default_rng(seed)
    K, M, N = 64, 5, 4
    shifts = [5, -4, -12, -25]
    classes, exact = [], [[0] * N for _ in range(M)]
    for sft in shifts:
        A, mA = _dyadic(rng, (M, K), scale=3)
        B, mB = _dyadic(rng, (K, N), scale=sft)
        classes.append((1.0, A, B))
        ex = _exact(mA, mB)
        for i in range(M):
            for j in range(N):
                exact[i][j] += ex[i][j] * 2 ** (25 + sft)      # common scale 2^(3 - 30 - 30 - 25)
    C, keep = oz.emulated_sum(classes, 6, 3)
    assert keep == [6, 5, 4, 3]
    A0, B0 = classes[0][1], classes[0][2]
    ref_bound = oz.truncation_bound(oz.exponents(A0, 1), oz.exponents(B0, 0), K, 6, 6).max()
    err = _err(C, exact, 3 - 85)
    assert err <= len(classes) * ref_bound
    eager = sum(oz.emulated_gemm(A, B, 6) for _, A, B in classes)
    assert _err(eager, exact, 3 - 85) <= len(classes) * ref_bound
    # fewer products: 21 + 15 + 10 + 6 of 4 x 21
    assert sum(kp * (kp + 1) // 2 for kp in keep) == 52
