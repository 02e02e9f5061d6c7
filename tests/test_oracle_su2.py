"""Pins for oracle/su2.py (SURVEY.md 8(c) "c4 SU(2)": Wigner symbols against orthogonality sums and
exact values; the expansion is an isometry, preserves norms, and H stays inside the multiplet)."""
from fractions import Fraction
from math import sqrt

import numpy as np
import pytest

import fixtures as fx
from fixtures.configs import Config
from oracle import su2


def test_clebsch_gordan_exact_values_and_closed_forms():
    # textbook values (doubled arguments): <1/2 1/2; 1/2 -1/2 | 1 0> = 1/sqrt2, | 0 0> = 1/sqrt2
    assert su2.cg(1, 1, 1, -1, 2, 0) == pytest.approx(1 / sqrt(2), abs=1e-15)
    assert su2.cg(1, 1, 1, -1, 0, 0) == pytest.approx(1 / sqrt(2), abs=1e-15)
    assert su2.cg(1, -1, 1, 1, 0, 0) == pytest.approx(-1 / sqrt(2), abs=1e-15)
    # <1 0; 1 0 | 2 0> = sqrt(2/3), <1 0; 1 0 | 1 0> = 0, <1 0; 1 0 | 0 0> = -1/sqrt3
    assert su2.cg(2, 0, 2, 0, 4, 0) == pytest.approx(sqrt(2 / 3), abs=1e-15)
    assert su2.cg(2, 0, 2, 0, 2, 0) == 0.0 or abs(su2.cg(2, 0, 2, 0, 2, 0)) < 1e-15
    assert su2.cg(2, 0, 2, 0, 0, 0) == pytest.approx(-1 / sqrt(3), abs=1e-15)
    # <3/2 1/2; 1 -1 | 1/2 -1/2> = sqrt(1/6) ... sign by Condon-Shortley: +sqrt(1/6)
    assert su2.cg(3, 1, 2, -2, 1, -1) ** 2 == pytest.approx(1 / 6, abs=1e-15)
    # stretched state and j2 = 0
    for j in range(0, 7):
        assert su2.cg(j, j, 3, 3, j + 3, j + 3) == pytest.approx(1.0, abs=1e-14)
        for m in range(-j, j + 1, 2):
            assert su2.cg(j, m, 0, 0, j, m) == pytest.approx(1.0, abs=1e-14)
    # closed form <j m; 1/2 1/2 | j+1/2 m+1/2> = sqrt((j+m+1)/(2j+1))  (doubled: (j2+m2+2)/(2(j2+1)))
    for j2 in range(0, 8):
        for m2 in range(-j2, j2 + 1, 2):
            assert su2.cg(j2, m2, 1, 1, j2 + 1, m2 + 1) == pytest.approx(sqrt((j2 + m2 + 2) / (2 * (j2 + 1))), abs=1e-14)


def test_clebsch_gordan_orthogonality_and_symmetry():
    for j1 in range(0, 6):
        for j2 in range(0, 5):
            for J in range(abs(j1 - j2), j1 + j2 + 1, 2):
                for Jp in range(abs(j1 - j2), j1 + j2 + 1, 2):
                    for M in range(-min(J, Jp), min(J, Jp) + 1, 2):
                        s = sum(su2.cg(j1, m1, j2, M - m1, J, M) * su2.cg(j1, m1, j2, M - m1, Jp, M)
                                for m1 in range(-j1, j1 + 1, 2))
                        assert s == pytest.approx(1.0 if J == Jp else 0.0, abs=1e-13)
                # <j1 m1; j2 m2|J M> = (-1)^{j1+j2-J} <j2 m2; j1 m1|J M>
                for m1 in range(-j1, j1 + 1, 2):
                    for m2 in range(-j2, j2 + 1, 2):
                        a = su2.cg(j1, m1, j2, m2, J, m1 + m2)
                        b = su2.cg(j2, m2, j1, m1, J, m1 + m2)
                        assert a == pytest.approx((-1) ** ((j1 + j2 - J) // 2) * b, abs=1e-13)


def _case(L, N, S2, D, bond, seed=1):
    cfg = Config("t", L=L, N=N, twoS=S2, sym=1, D=D, n_chol=6, bond=bond)
    h, V, _ = fx.make_integrals(L, 6, 0)
    tabs = fx.block_tables(cfg)
    nl, nr = bond, L - bond - 2
    isoL = fx.random_isometries(cfg, tabs, nl, seed)
    isoR = fx.random_isometries(cfg, tabs, nr, seed + 1000)
    return cfg, h, V, tabs, nl, nr, isoL, isoR


@pytest.mark.parametrize("L,N,S2,D,bond", [(4, 4, 0, 6, 1), (5, 5, 1, 8, 2), (5, 4, 2, 8, 1), (6, 6, 0, 10, 2)])
def test_expansion_is_isometric_and_h_is_scalar(L, N, S2, D, bond):
    cfg, h, V, tabs, nl, nr, isoL, isoR = _case(L, N, S2, D, bond)
    # expanded isometries are isometries of the U(1)xU(1) blocks
    from oracle import abelian as ab
    for isos, n, right in ((isoL, nl, True), (isoR, nr, False)):
        for m in range(n):
            ta, tb, bl, dat = su2.expand_isometry(tabs[m], tabs[m + 1], isos[m][0], isos[m][1], right)
            for inext in range(len(tb)):
                rows = [dat[b[5]:b[5] + b[3] * b[4]].reshape(b[3], b[4]) for b in bl if b[2] == inext]
                Xf = np.concatenate(rows, axis=0)
                assert np.abs(Xf.T @ Xf - np.eye(Xf.shape[1])).max() < 1e-12
    results = []
    for M2 in range(-S2, S2 + 1, 2):
        ex = su2.ExpandedTwoSite(h, V, N, S2, bond, tabs[:nl + 1], isoL, tabs[:nr + 1], isoR, M2)
        psi = fx.random_psi(ex.n, 2)
        full = ex.expand(psi)
        assert np.linalg.norm(full) == pytest.approx(1.0, abs=1e-12)          # norm preserved
        assert np.abs(ex.project(full) - psi).max() < 1e-12                    # project o expand = 1
        assert ex.leakage(psi) < 1e-11                                         # H psi stays in the multiplet
        results.append(ex.apply(psi))
    for r in results[1:]:                                                      # independent of M
        assert np.abs(r - results[0]).max() < 1e-11
    # hermiticity of the reduced H_eff
    ex = su2.ExpandedTwoSite(h, V, N, S2, bond, tabs[:nl + 1], isoL, tabs[:nr + 1], isoR)
    u, w = fx.random_vector(ex.n, 11), fx.random_vector(ex.n, 12)
    assert abs(u @ ex.apply(w) - w @ ex.apply(u)) < 1e-11
