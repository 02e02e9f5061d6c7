"""Reference model of the Ozaki-emulated FP64 GEMM (test infrastructure).

PAPER.md:59,71 fix only "Ozaki scheme, fixed-point slices, 47-bit mantissa = kappa = 6 INT8 slices";
DESIGN.md reading s12 fixes the rest: per-row (A) and per-column (B) power-of-two exponents over the K
chunk, round to nearest, balanced signed digits in [-128, 127], slice products with s + t <= kappa + 1
(triangular) or all (full), INT32 partial sums per anti-diagonal; recombination: the sums are joined exactly,
three at a time from the smallest scale, into radix-2^24 super-digits (int64, < 2^48), which are added in FP64
from the smallest scale upward (one rounding at kappa <= 6).  Everything here is exact integer arithmetic in numpy int64 / Python ints.
"""
import numpy as np


def exponents(a, axis):
    """e = 1 + floor(log2 max|a|) along `axis` (0 for an all-zero line): max|a| = f 2^e, f in [1/2, 1)."""
    m = np.max(np.abs(a), axis=axis)
    _, e = np.frexp(m)
    return np.where(m > 0, e, 0).astype(np.int64)


def slice_lines(a, e, kappa, axis):
    """Digits d[s] (s = 0 is the top slice) of X = rint(a 2^(8 kappa - 2 - e)), e per line along `axis`
    (the K axis); returns (d, X) as int64."""
    sh = (8 * kappa - 2 - e).astype(np.int64)
    sh = np.expand_dims(sh, axis)
    X = np.rint(np.ldexp(a, sh)).astype(np.int64)
    r = X.copy()
    d = np.zeros((kappa,) + a.shape, dtype=np.int64)
    for s in range(kappa - 1, 0, -1):
        d[s] = ((r + 128) % 256) - 128
        r = (r - d[s]) // 256
    d[0] = r
    return d, X


def emulated_gemm(A, B, kappa=6, full=False, kc=None):
    """C = A B through the slice model; kc = K chunk length (exponents and INT32 sums are per chunk)."""
    M, K = A.shape
    N = B.shape[1]
    kc = K if kc is None else kc
    C = np.zeros((M, N))
    for k0 in range(0, K, kc):
        a, b = A[:, k0:k0 + kc], B[k0:k0 + kc]
        ea, eb = exponents(a, 1), exponents(b, 0)
        da, _ = slice_lines(a, ea, kappa, 1)
        db, _ = slice_lines(b, eb, kappa, 0)
        cmax = 2 * kappa if full else kappa + 1
        acc = np.zeros((M, N))
        G, n_in = None, 0
        for c in range(cmax, 1, -1):                      # smallest scale first
            P = np.zeros((M, N), dtype=np.int64)
            for s in range(1, kappa + 1):
                t = c - s
                if 1 <= t <= kappa:
                    P += da[s - 1] @ db[t - 1]
            assert np.abs(P).max() < 2 ** 31              # INT32 accumulators must not overflow
            # three neighbouring anti-diagonal sums join exactly into one radix-2^24 super-digit (|G| < 2^48, so
            # its conversion to FP64 is exact); the super-digits are added in FP64 from the smallest scale upward
            if n_in == 0:
                G, c_lo = P.copy(), c
            else:
                G += P * 256 ** n_in
            n_in += 1
            if n_in == 3 or c == 2:
                assert np.abs(G).max() < 2 ** 48
                acc = acc + G.astype(np.float64) * 2.0 ** (16 * kappa - 8 * c_lo)
                n_in = 0
        C += np.ldexp(acc, (ea[:, None] + eb[None, :] - 2 * (8 * kappa - 2)).astype(np.int64))
    return C
