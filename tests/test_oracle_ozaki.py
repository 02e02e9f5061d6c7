"""Pins for oracle/ozaki.py (SURVEY.md 8(c) "Emulated mode", Appendix A6)."""
import numpy as np
import pytest

from oracle import ozaki


def _wide(shape, seed):
    rng = np.random.Generator(np.random.Philox(seed))
    return rng.standard_normal(shape) * 10.0 ** rng.uniform(-6, 0, shape)


@pytest.mark.parametrize("kappa", [3, 5, 6, 7])
def test_digit_identity_is_bit_exact(kappa):
    a = _wide((37, 211), 1)
    a[5] = 0.0                                  # an all-zero row
    a[7, 3] = 2.0 ** -40
    e = ozaki.exponents(a, 1)
    d, X = ozaki.slice_lines(a, e, kappa, 1)
    assert d.min() >= -128 and d.max() <= 127
    assert np.abs(d[0]).max() <= 65             # one bit of carry headroom in the top digit
    recon = sum(d[s].astype(object) * (256 ** (kappa - 1 - s)) for s in range(kappa))
    assert np.all(recon == X.astype(object))    # X = sum_s d_s 2^(8 (kappa - s)), exactly
    assert np.abs(X).max() <= 2 ** (8 * kappa - 2)
    # X is the correctly rounded fixed-point value of a
    assert np.abs(np.ldexp(X.astype(np.float64), (e - (8 * kappa - 2))[:, None]) - a).max() <= \
        np.ldexp(0.5, (e - (8 * kappa - 2))).max()
    assert np.all(d[:, 5] == 0)


def test_error_falls_with_kappa_and_meets_the_tolerance():
    rng = np.random.Generator(np.random.Philox(3))
    A, B = rng.standard_normal((48, 2048)), rng.standard_normal((2048, 40))
    ref = A @ B
    err = {k: np.linalg.norm(ozaki.emulated_gemm(A, B, k) - ref) / np.linalg.norm(ref) for k in (3, 4, 5, 6, 7)}
    for k in (3, 4, 5):
        assert err[k + 1] < err[k] / 50         # about 2^-8 per added slice until the FP64 floor
    assert err[6] < 1e-11 and err[7] < 1e-13    # kappa = 6 triangular (21 products): SURVEY Appendix A6 table
    Aw, Bw = _wide((48, 2048), 4), _wide((2048, 40), 5)
    refw = Aw @ Bw
    e6 = np.linalg.norm(ozaki.emulated_gemm(Aw, Bw, 6) - refw) / np.linalg.norm(refw)
    e6f = np.linalg.norm(ozaki.emulated_gemm(Aw, Bw, 6, full=True) - refw) / np.linalg.norm(refw)
    assert e6 < 1e-10 and e6f < e6              # BASELINE.json tolerance of the emulated mode; full set is tighter


def test_exact_cases_and_chunking():
    # small integers are represented exactly: the emulated product is the exact product
    rng = np.random.Generator(np.random.Philox(6))
    A = rng.integers(-1000, 1000, (17, 300)).astype(np.float64)
    B = rng.integers(-1000, 1000, (300, 9)).astype(np.float64)
    assert np.array_equal(ozaki.emulated_gemm(A, B, 6), A @ B)
    assert np.array_equal(ozaki.emulated_gemm(A, B, 6, kc=64), A @ B)
    # powers of two scale through the exponents only
    assert np.array_equal(ozaki.emulated_gemm(A * 2.0 ** -30, B * 2.0 ** 17, 6), (A @ B) * 2.0 ** -13)


@pytest.mark.parametrize("kappa", [3, 5, 6])
def test_recombination_is_the_exact_integer_sum_rounded_once(kappa):
    """DESIGN.md reading s12 (recombination by radix-2^24 super-digits): for kappa <= 6 the result equals the exact
    triangular product sum S = sum_c P_c 2^(8 (kappa + 1 - c)) (Python integers) converted to FP64 with ONE rounding."""
    A, B = _wide((9, 300), 21), _wide((300, 7), 22)
    ea, eb = ozaki.exponents(A, 1), ozaki.exponents(B, 0)
    da, _ = ozaki.slice_lines(A, ea, kappa, 1)
    db, _ = ozaki.slice_lines(B, eb, kappa, 0)
    got = ozaki.emulated_gemm(A, B, kappa)
    for i in range(A.shape[0]):
        for j in range(B.shape[1]):
            S = 0
            for s in range(1, kappa + 1):
                for t in range(1, kappa + 2 - s):                       # s + t <= kappa + 1
                    p = sum(int(x) * int(y) for x, y in zip(da[s - 1][i], db[t - 1][:, j]))
                    S += p * 256 ** (kappa + 1 - s - t)
            # scale of the smallest anti-diagonal (c = kappa + 1): 2^(16 kappa - 8 c), then the line exponents
            want = np.ldexp(float(S), int(16 * kappa - 8 * (kappa + 1) + ea[i] + eb[j] - 2 * (8 * kappa - 2)))
            assert got[i, j] == want


def test_tf32_split_properties_and_hand_values():
    """Reading s15.  hi and lo carry at most 11 significant bits; x - hi is below half a unit of hi's last place (plus the
    FP32 rounding of x), x - hi - lo below 2^-21 |x|; hand-computed values incl. a tie."""
    rng = np.random.default_rng(4)
    x = rng.standard_normal(20000) * 10.0 ** rng.uniform(-8, 8, 20000)
    hi, lo = ozaki.tf32_split(x)
    for part in (hi, lo):
        m, e = np.frexp(part.astype(np.float64))
        assert np.all(m * 2048 == np.rint(m * 2048))                     # 11 significant bits (1 implicit + 10)
    h64 = hi.astype(np.float64)
    assert np.all(np.abs(x - h64) <= np.abs(x) * (2.0 ** -11 + 2.0 ** -23))
    assert np.all(np.abs(x - h64 - lo.astype(np.float64)) <= np.abs(x) * 2.0 ** -21)
    assert np.all(np.abs(lo.astype(np.float64)) <= np.abs(h64) * 2.0 ** -10)
    # 1 + 2^-11 is a tie between 1 and 1 + 2^-10: away from zero; 1 + 2^-12 rounds down, its rest goes to lo exactly
    hi, lo = ozaki.tf32_split(np.array([1.0 + 2.0 ** -11, 1.0 + 2.0 ** -12, -(1.0 + 2.0 ** -11), 3.0, 0.0]))
    assert hi.tolist() == [1.0 + 2.0 ** -10, 1.0, -(1.0 + 2.0 ** -10), 3.0, 0.0]
    assert lo.tolist() == [-(2.0 ** -11), 2.0 ** -12, 2.0 ** -11, 0.0, 0.0]
