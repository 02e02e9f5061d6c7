"""Pins for the parts of the oracle that round 1 left unpinned:
  * oracle/sweep.py::split under REAL truncation, against a dense SVD of the two-site wave function written as the
    matrix M[(l, s1), (s2, r)] (SURVEY.md Appendix A5 "Truncation"; PAPER.md:49 truncation error): discarded weight,
    kept counts per sector, kept subspace;
  * oracle/davidson.py: the iterate sequence -- one-step identities that a wrong preconditioner sign, a missing clamp or
    a one-pass Gram-Schmidt break -- and the sensitivity envelope that the GPU tests use as their derived tolerance."""
import numpy as np
import pytest

import fixtures as fx
from oracle import abelian as ab
from oracle.davidson import davidson
from oracle.sweep import split
from tests.helpers import davidson_envelope, make_case, oracle_two_site


def _dense_two_site(ts, psi, absorb_left):
    """M with rows = states of the block that grows, columns = the rest; also the (sector label, row slice) list."""
    tabL = list(zip(ts.A.X.basis.labels, ts.A.X.basis.dims))
    tabR = list(zip(ts.B.Y.basis.labels, ts.B.Y.basis.dims))
    offL = np.concatenate([[0], np.cumsum([d for _, d in tabL])])
    offR = np.concatenate([[0], np.cumsum([d for _, d in tabR])])
    DL, DR = int(offL[-1]), int(offR[-1])
    M = np.zeros((DL * 4, 4 * DR))                       # rows (l, s1), columns (s2, r)
    for (iL, s1, s2, iR, dL, dR, off) in ts.blocks:
        blk = psi[off:off + dL * dR].reshape(dL, dR)
        for a in range(dL):
            M[(offL[iL] + a) * 4 + s1, s2 * DR + offR[iR]: s2 * DR + offR[iR] + dR] = blk[a]
    if not absorb_left:
        M = M.T.copy()                                   # rows (s2, r)
    return M, DL, DR, offL, offR


@pytest.mark.parametrize("L,N,tw,D,bond,keep,left", [(4, 4, 0, 16, 1, 5, True), (4, 4, 0, 16, 1, 6, False), (5, 5, 1, 30, 2, 9, True),
                                                     (6, 6, 0, 40, 2, 17, False)])
def test_split_under_truncation_equals_the_dense_svd(L, N, tw, D, bond, keep, left):
    case = make_case(L, N, tw, D, bond)
    _, _, _, ts = oracle_two_site(case)
    psi = fx.random_psi(ts.n, 7)
    table, iso_blocks, iso_data, disc = split(ts, psi, keep, left)
    M, DL, DR, offL, offR = _dense_two_site(ts, psi, left)
    U, sv, _ = np.linalg.svd(M, full_matrices=False)
    w = sv ** 2
    assert w[keep - 1] - w[keep] > 1e-9                  # the cut is not inside a degenerate cluster on this input
    assert int(table[:, 2].sum()) == keep
    assert disc == pytest.approx(w[keep:].sum(), abs=1e-13)          # truncation error = sum of the dropped weights
    assert disc > 1e-4                                   # a real truncation, not a saturated bond
    # dense isometry from the packed blocks: rows in the (block state, site state) order used for M
    tab_prev = ts.A.X.basis if left else ts.B.Y.basis
    off_prev = offL if left else offR
    Dprev = DL if left else DR
    X = np.zeros((M.shape[0], keep))
    for (ip, s, inext, rows, cols, off) in iso_blocks:
        blk = iso_data[off:off + rows * cols].reshape(rows, cols)
        c0 = int(table[inext][3])
        for a in range(rows):
            row = (off_prev[ip] + a) * 4 + s if left else s * Dprev + off_prev[ip] + a
            X[row, c0:c0 + cols] = blk[a]
    assert np.abs(X.T @ X - np.eye(keep)).max() < 1e-12
    P_ref = U[:, :keep] @ U[:, :keep].T                  # the kept subspace is unique although its basis is not
    assert np.abs(X @ X.T - P_ref).max() < 1e-9
    # kept count per sector = number of the `keep` largest singular values whose vector lives in that sector
    counts = {}
    for j in range(keep):
        r = int(np.argmax(np.abs(U[:, j])))
        st, s = (divmod(r, 4) if left else tuple(reversed(divmod(r, Dprev))))
        ip = int(np.searchsorted(off_prev, st, side="right") - 1)
        q = tab_prev.labels[ip]
        key = (q[0] + ab.SITE_LABELS[s][0], q[1] + ab.SITE_LABELS[s][1])
        counts[key] = counts.get(key, 0) + 1
    assert {(int(r[0]), int(r[1])): int(r[2]) for r in table} == counts


def _dense_case():
    case = make_case(5, 5, 1, 9, 2)
    _, _, _, ts = oracle_two_site(case)
    H = np.stack([ts.apply(e) for e in np.eye(ts.n)], axis=1)
    H = 0.5 * (H + H.T)
    return H, np.diag(H).copy(), fx.random_psi(ts.n, 2)


def test_davidson_first_steps_equal_their_definition():
    """c6 step by step with dense linear algebra: theta_1 = <v0|H|v0>; the second basis vector is the normalised,
    V-orthogonal part of t = r / (theta - diag) with the 1e-12 clamp; theta_2 is the lowest eigenvalue of the 2 x 2
    projected matrix.  A flipped sign of the preconditioner leaves span(V) unchanged, so the test also checks the
    vector itself, not only theta."""
    H, dg, psi = _dense_case()
    seen = []
    x, th, rs = davidson(lambda v: (seen.append(v.copy()), H @ v)[1], dg, psi, 3)
    v0 = psi / np.linalg.norm(psi)
    assert np.allclose(seen[0], v0, atol=1e-15)
    t1 = v0 @ H @ v0
    assert th[0] == pytest.approx(t1, abs=1e-13)
    r = H @ v0 - t1 * v0
    assert rs[0] == pytest.approx(np.linalg.norm(r), abs=1e-13)
    den = t1 - dg
    den = np.where(np.abs(den) < 1e-12, np.where(den < 0, -1e-12, 1e-12), den)
    t = r / den
    t -= v0 * (v0 @ t)
    t -= v0 * (v0 @ t)
    v1 = t / np.linalg.norm(t)
    assert np.abs(seen[1] - v1).max() < 1e-12            # same vector, same sign
    V = np.stack([v0, v1], 1)
    assert th[1] == pytest.approx(np.linalg.eigvalsh(V.T @ H @ V)[0], abs=1e-12)
    # the basis stays orthonormal to rounding (two-pass Gram-Schmidt): one pass would leave ~1e-10 here
    Vall = np.stack(seen, 1)
    assert np.abs(Vall.T @ Vall - np.eye(Vall.shape[1])).max() < 1e-14


def test_davidson_clamp_and_breakdown():
    """|theta - diag_i| < 1e-12 is replaced by +-1e-12 (sign kept), and an exact eigenvector start ends the
    expansion instead of dividing by a vanishing norm (c6; the library mirrors both)."""
    H = np.diag([1.0, 2.0, 3.0, 4.0]) + 0.0
    H[0, 1] = H[1, 0] = 0.5
    dg = np.diag(H).copy()
    psi = np.array([0.0, 0.0, 1.0, 0.0])               # exact eigenvector: r = 0, t = 0
    x, th, rs = davidson(lambda v: H @ v, dg, psi, 4)
    assert len(th) == 1 and th[0] == 3.0 and rs[0] == 0.0
    # theta equal to a diagonal entry to rounding: the clamped component is r_i / (+-1e-12), finite
    H2 = np.array([[2.0, 1e-3, 0.0], [1e-3, 2.0, 1e-3], [0.0, 1e-3, 5.0]])
    psi2 = np.array([1.0, 1e-9, 1e-9])
    x, th, rs = davidson(lambda v: H2 @ v, np.diag(H2).copy(), psi2, 3)
    assert np.all(np.isfinite(th)) and np.all(np.isfinite(x)) and np.all(np.diff(th) <= 1e-12)


def test_davidson_sensitivity_envelope_grows_and_bounds_equivalent_implementations():
    """Derives the tolerance the GPU tests use.  Rounding-level noise in the matvec (4 ulp, componentwise) moves the
    Ritz values of later iterations by many orders of magnitude more than it moves the first: the preconditioner
    divides by theta - diag_i, which is nearly singular for some i when theta lies inside the range of the diagonal.
    A mathematically identical implementation that only sums in another order must stay inside the envelope."""
    H, dg, psi = _dense_case()
    nit = 8
    th0, rs0, env_t, env_r = davidson_envelope(lambda v: H @ v, dg, psi, nit)
    assert env_t[0] < 2e-12 * abs(th0[0])                 # iteration 1 is <psi|H|psi>: rounding level
    assert np.all(np.diff(env_t) >= -1e-18)               # the envelope is monotone by construction
    perm = np.random.default_rng(3).permutation(len(psi)) # same arithmetic, another summation order
    Hp = H[:, perm]
    _, th1, rs1 = davidson(lambda v: Hp @ v[perm], dg, psi, nit)
    assert np.all(np.abs(th1 - th0) <= env_t)
    assert np.all(np.abs(rs1 - rs0) <= env_r)
    assert env_t[-1] > 100 * env_t[0]                     # ... and later ones are not
    print("\ntheta envelope per iteration:", " ".join(f"{e:.1e}" for e in env_t))
