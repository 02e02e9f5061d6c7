"""Pins for oracle/fock.py (SURVEY.md 8(c) "What pins each part": c1 FCI)."""
import numpy as np
import pytest

import fixtures as fx
from oracle import fock


def test_hubbard_dimer_closed_form():
    # h12 = -t, V_iiii = U, N = 2: E0 = (U - sqrt(U^2 + 16 t^2)) / 2
    for t_, U in [(1.0, 4.0), (1.3, 2.7), (0.2, 9.0)]:
        h = np.array([[0.0, -t_], [-t_, 0.0]])
        V = np.zeros((2, 2, 2, 2))
        V[0, 0, 0, 0] = V[1, 1, 1, 1] = U
        H, _ = fock.fci_matrix(h, V, 1, 1)
        assert np.linalg.eigvalsh(H)[0] == pytest.approx((U - np.sqrt(U * U + 16 * t_ * t_)) / 2, abs=1e-13)


def test_noninteracting_spectrum():
    # V = 0: E = 2 * (sum of the N/2 lowest eigenvalues of h)
    h, V, _ = fx.make_integrals(5, 4, 3)
    H, _ = fock.fci_matrix(h, np.zeros_like(V), 2, 2)
    e = np.linalg.eigvalsh(h)
    assert np.linalg.eigvalsh(H)[0] == pytest.approx(2 * e[:2].sum(), abs=1e-12)
    H, _ = fock.fci_matrix(h, np.zeros_like(V), 3, 1)
    assert np.linalg.eigvalsh(H)[0] == pytest.approx(e[:3].sum() + e[0], abs=1e-12)


def test_sector_matrix_equals_jordan_wigner_definition():
    h, V, _ = fx.make_integrals(4, 6, 0)
    Hd = fock.hamiltonian_dense(h, V)
    assert abs(Hd - Hd.T).max() < 1e-14
    for nu, nd in [(2, 2), (3, 1), (1, 2)]:
        H, dets = fock.fci_matrix(h, V, nu, nd)
        idx = fock.dets_to_fock_index(dets, 4)
        assert abs(Hd[np.ix_(idx, idx)] - H).max() < 1e-13


def test_conservation_laws_and_spin():
    L = 3
    h, V, _ = fx.make_integrals(L, 5, 1)
    c = fock.jw_creators(L)
    H = fock.hamiltonian_dense(h, V, c)
    Nop = sum(m @ m.T for m in c)
    Sz = 0.5 * sum(c[2 * p] @ c[2 * p].T - c[2 * p + 1] @ c[2 * p + 1].T for p in range(L))
    Sp = sum(c[2 * p] @ c[2 * p + 1].T for p in range(L))
    S2 = Sz @ Sz + 0.5 * (Sp @ Sp.T + Sp.T @ Sp)
    for O in (Nop, Sz, S2):
        assert abs(H @ O - O @ H).max() < 1e-12
    # anticommutation of the Jordan-Wigner operators
    for i in range(2 * L):
        for j in range(2 * L):
            ac = c[i].T @ c[j] + c[j] @ c[i].T
            assert abs(ac - (i == j) * np.eye(4 ** L)).max() < 1e-14
            assert abs(c[i] @ c[j] + c[j] @ c[i]).max() < 1e-14
    # ground state in the N=2, Sz=0 sector is an S^2 eigenstate
    Hs, dets = fock.fci_matrix(h, V, 1, 1)
    w, U = np.linalg.eigh(Hs)
    idx = fock.dets_to_fock_index(dets, L)
    g = np.zeros(4 ** L)
    g[idx] = U[:, 0]
    s2 = g @ S2 @ g
    assert abs(S2 @ g - s2 * g).max() < 1e-10
    assert min(abs(s2 - s * (s + 1)) for s in (0, 1)) < 1e-10


def test_lanczos_jacobi_eigh_agree():
    h, V, _ = fx.make_integrals(4, 6, 0)
    H, dets = fock.fci_matrix(h, V, 2, 2)
    w_j, U_j = fock.jacobi_eigh(H)
    w_e = np.linalg.eigvalsh(H)
    assert abs(w_j - w_e).max() < 1e-12
    assert abs(H @ U_j - U_j * w_j).max() < 1e-11
    th, x, _ = fock.lanczos_lowest(lambda v: H @ v, len(dets), tol=1e-10)
    assert th == pytest.approx(w_e[0], abs=1e-10)
    assert np.linalg.norm(H @ x - th * x) < 1e-8


def test_cfg0_dimension():
    # BASELINE.json configs[0]: 4900 determinants
    assert len(fock.sector_dets(8, 4, 4)) == 4900
