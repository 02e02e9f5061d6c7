"""Reference model of the Ozaki-emulated FP64 GEMM (test infrastructure).

PAPER.md:59,71 fix only "Ozaki scheme, fixed-point slices, 47-bit mantissa = kappa = 6 INT8 slices";
DESIGN.md reading s12 fixes the rest: per-row (A) and per-column (B) power-of-two exponents over the K
chunk, round to nearest, balanced signed digits in [-128, 127], slice products with s + t <= kappa + 1
(triangular) or all (full), INT32 partial sums per anti-diagonal; recombination: the sums are joined exactly,
three at a time from the smallest scale, into radix-2^24 super-digits (int64, < 2^48), which are added in FP64
from the smallest scale upward (one rounding at kappa <= 6).  Everything here is exact integer arithmetic in numpy int64 / Python ints.

Performant mode (PAPER.md:53 "the library automatically calculates the bits required", :59 "dynamic mantissa bit
settings"; reading s21): per task class (one segment = one operator-pair class
meeting one psi block) the slice products kept are chosen from the spread of the class magnitudes' exponents inside the
output block's job: `class_exponents`, `performant_keep`, `truncation_bound`, `emulated_sum`.
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


def emulated_gemm(A, B, kappa=6, full=False, kc=None, keep=None):
    """C = A B through the slice model; kc = K chunk length (exponents and INT32 sums are per chunk).
    keep (performant mode, reading s21): the operands stay sliced into kappa digits, but only the
    products with s + t <= keep + 1 are formed (keep = kappa, or None: the whole triangular set)."""
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
                if 1 <= t <= kappa and (keep is None or c <= keep + 1):
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


def _ceil_log2(n):
    return int(n - 1).bit_length() if n > 1 else 0


def class_exponents(ea, eb, alpha, K):
    """Magnitude exponents of one task class  alpha * A B  (A lines with exponents ea, B lines with exponents eb, K the
    contraction length): every element of the product is below 2^E_all.  Returns (E_all, E_nz): E_all takes every line,
    E_nz only the lines whose exponent is not 0 (an all-zero line also carries exponent 0, see `exponents`, so a line
    with e = 0 cannot vouch for the class being large); E_nz is None when either side has no such line."""
    ea, eb = np.asarray(ea, dtype=np.int64), np.asarray(eb, dtype=np.int64)
    _, e_alpha = np.frexp(abs(float(alpha)))
    lk = _ceil_log2((K + 31) // 32)                     # k steps of 32, as the kernels count them
    E_all = int(ea.max()) + int(eb.max()) + int(e_alpha) + lk
    nza, nzb = ea[ea != 0], eb[eb != 0]
    E_nz = None if nza.size == 0 or nzb.size == 0 else int(nza.max()) + int(nzb.max()) + int(e_alpha) + lk
    return E_all, E_nz


def performant_keep(E_all, E_nz, kappa=6, kmin=3):
    """Slice count per class of one job (the classes accumulated into one output block): the reference exponent is
    E_ref = max E_nz; a class whose bound 2^E_all lies 8 d bits below it keeps kappa - d slices (not fewer than kmin),
    so that its truncation bound (`truncation_bound`) does not exceed that of the reference class at kappa slices."""
    ref = [e for e in E_nz if e is not None]
    if not ref:
        return [kappa] * len(E_all)
    E_ref = max(ref)
    return [kappa - min(kappa - kmin, max(0, E_ref - e) // 8) for e in E_all]


def truncation_bound(ea, eb, K, kappa, keep):
    """A-priori bound of |emulated - exact| per element of A B for lines with exponents ea (rows) and eb (columns).
    Dropped products: s + t = c >= keep + 2, at most c - 1 pairs each, |digit| <= 128, scale
    2^(ea + eb - 2 (8 kappa - 2)) 256^(2 kappa - c): sum_c (c - 1) 2^(18 - 8 c) <= 1.02 (keep + 1) 2^(2 - 8 keep);
    the rounding of the two operands to 8 kappa - 2 bits adds 2^(2 - 8 kappa) (1 + 2^(1 - 8 kappa)); the FP64
    recombination one rounding of the result."""
    ea, eb = np.asarray(ea, dtype=np.float64), np.asarray(eb, dtype=np.float64)
    scale = np.exp2(ea[:, None] + eb[None, :])
    rel = 1.02 * (keep + 1) * 2.0 ** (2 - 8 * keep) + 1.01 * 2.0 ** (2 - 8 * kappa) + 2.0 ** -52
    return K * scale * rel


def emulated_sum(classes, kappa=6, kmin=3):
    """C = sum_g alpha_g A_g B_g in performant mode: classes = [(alpha, A, B)], each class with its own exponents and
    its own slice count from `performant_keep`.  Returns (C, keep)."""
    E = [class_exponents(exponents(A, 1), exponents(B, 0), alpha, A.shape[1]) for alpha, A, B in classes]
    keep = performant_keep([e[0] for e in E], [e[1] for e in E], kappa, kmin)
    C = np.zeros((classes[0][1].shape[0], classes[0][2].shape[1]))
    for (alpha, A, B), kp in zip(classes, keep):
        C = C + alpha * emulated_gemm(A, B, kappa, keep=kp)
    return C, keep


# ---------------------------------------------------------------------------------------------------------------
# 3xTF32 mode (reading s15; SURVEY.md 8(a) a4 "TF32 hi/lo"): the operand split.  The three products
# hi*hi + hi*lo + lo*hi are accumulated in FP32 inside the tensor core in an order the hardware does not document, so
# only the split has a bit-exact model; the products are checked against FP64 at the mode's tolerance (1e-5).
def tf32_round(f):
    """Nearest TF32 number (8-bit exponent, 10 explicit mantissa bits) of FP32 values: the 13 low mantissa bits are
    dropped after adding half of their unit (ties away from zero)."""
    u = np.ascontiguousarray(f, dtype=np.float32).view(np.uint32)
    return ((u + np.uint32(0x1000)) & np.uint32(0xFFFFE000)).view(np.float32)


def tf32_split(x):
    """x = hi + lo + O(2^-22 |x|): hi = tf32(fp32(x)), lo = tf32(fp32(x - hi)), both exactly representable in TF32."""
    x = np.asarray(x, dtype=np.float64)
    hi = tf32_round(x.astype(np.float32))
    lo = tf32_round((x - hi.astype(np.float64)).astype(np.float32))
    return hi, lo
