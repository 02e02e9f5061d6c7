"""Pins for oracle/abelian.py, brute.py, davidson.py, sweep.py
(SURVEY.md 8(c) "What pins each part": A2/A3 identities, c3, c5, c6, DMRG as a whole)."""
import numpy as np
import pytest

import fixtures as fx
from fixtures.configs import Config
from oracle import abelian as ab
from oracle import brute, fock
from oracle.davidson import davidson
from oracle.sweep import two_site_sweeps


def _setup(L, N, tw, D, bond, seed=1, nchol=6):
    cfg = Config("t", L=L, N=N, twoS=tw, sym=0, D=D, n_chol=nchol, bond=bond)
    h, V, _ = fx.make_integrals(L, nchol, 0)
    tabs = fx.block_tables(cfg)
    nl, nr = bond, L - bond - 2
    isoL = fx.random_isometries(cfg, tabs, nl, seed)
    isoR = fx.random_isometries(cfg, tabs, nr, seed + 1000)
    ints = ab.Integrals(h, V)
    Lb = ab.build_block(ints, tabs, isoL, list(range(nl)), True)
    Rb = ab.build_block(ints, tabs, isoR, list(range(L - 1, bond + 1, -1)), False)
    ts = ab.TwoSite(Lb, ab.site_block(ints, bond), ab.site_block(ints, bond + 1), Rb, N, tw)
    vL = brute.block_vectors(tabs, isoL, nl, True)
    vR = brute.block_vectors(tabs, isoR, nr, False)
    P, _ = brute.projector(N, tw, tabs[nl], vL, tabs[nr], vR)
    # H restricted to the (N, Sz) sector (P has no support outside it)
    H, dets = fock.fci_matrix(h, V, (N + tw) // 2, (N - tw) // 2)
    idx = fock.dets_to_fock_index(dets, L)
    assert abs(P).sum() == pytest.approx(abs(P[idx]).sum(), abs=1e-12)
    P = P[idx]
    return dict(cfg=cfg, h=h, V=V, tabs=tabs, ints=ints, Lb=Lb, Rb=Rb, ts=ts, P=P, H=H,
                vL=vL, vR=vR, isoL=isoL, isoR=isoR)


def _definition_ops(ints, first_site, m, L):
    """Every stored operator of a block of m sites from its Appendix-A2 definition, as
    dense matrices on the block's own Fock space (local Jordan-Wigner strings)."""
    c = fock.jw_creators(m)
    orbs = list(range(2 * first_site, 2 * (first_site + m)))
    cr = {i: c[i - 2 * first_site] for i in orbs}
    an = {i: cr[i].T for i in orbs}
    t, v = ints.t, ints.v
    dim = 4 ** m
    out = {}
    H = np.zeros((dim, dim))
    for i in orbs:
        for j in orbs:
            H += t[i, j] * cr[i] @ an[j]
            for k in orbs:
                for l in orbs:
                    if i != k and l != j and v[i, j, k, l] != 0:
                        H += 0.5 * v[i, j, k, l] * cr[i] @ cr[k] @ an[l] @ an[j]
    out[("H",)] = H
    for i in orbs:
        out[("C", i)] = cr[i]
        for k in orbs:
            if i < k:
                out[("A", i, k)] = cr[i] @ cr[k]
            out[("B", i, k)] = cr[i] @ an[k]
    for x in range(2 * L):
        if x in orbs:
            continue
        S = np.zeros((dim, dim))
        for j in orbs:
            S += 0.5 * t[x, j] * an[j]
            for k in orbs:
                for l in orbs:
                    if v[x, j, k, l] != 0:
                        S += v[x, j, k, l] * cr[k] @ an[l] @ an[j]
        out[("S", x)] = S
    return out


@pytest.mark.parametrize("L,N,tw,D,bond", [(4, 4, 0, 3, 1), (4, 4, 0, 16, 1), (4, 3, 1, 4, 1),
                                           (5, 4, 0, 5, 2), (5, 6, 2, 6, 1), (5, 5, -1, 7, 0)])
def test_heff_equals_projected_hamiltonian(L, N, tw, D, bond):
    s = _setup(L, N, tw, D, bond)
    ts, P, H = s["ts"], s["P"], s["H"]
    assert abs(P.T @ P - np.eye(P.shape[1])).max() < 1e-12
    Heff = P.T @ H @ P
    psi = fx.random_psi(ts.n, 2)
    y = ts.apply(psi)
    yb = Heff @ psi
    assert np.linalg.norm(y - yb) / np.linalg.norm(yb) < 1e-13
    assert abs(ts.diagonal() - np.diag(Heff)).max() < 1e-12
    # hermiticity through the operator path: <u|H v> = <v|H u>
    u, w = fx.random_vector(ts.n, 11), fx.random_vector(ts.n, 12)
    assert abs(u @ ts.apply(w) - w @ ts.apply(u)) < 1e-12


@pytest.mark.parametrize("side", ["L", "R"])
def test_renormalized_operators_equal_definition(side):
    # c5 pinned to <l'|O|l> with O from its definition in the block's Fock space
    L = 5
    s = _setup(L, 5, 1, 9, 2)
    if side == "L":
        blk, vec, first, m = s["Lb"], s["vL"], 0, 2
    else:
        blk, vec, first, m = s["Rb"], s["vR"], 4, 1
    Vb = np.concatenate([vec[i] for i in range(len(blk.basis))], axis=1)
    ref = _definition_ops(s["ints"], first, m, L)
    assert set(ref) == set(blk.store)
    for key, O in ref.items():
        got = blk.store[key].dense(blk.basis)
        assert abs(got - Vb.T @ O @ Vb).max() < 1e-12, key


def test_complements_and_composite_blocking_equal_definition():
    # P, Q of a block (weighted sums of stored A+, B) and every Composite.op (Appendix A3)
    # against Jordan-Wigner definitions, with a saturated (complete) left block.
    L = 4
    cfg = Config("t", L=L, N=4, twoS=0, sym=0, D=64, n_chol=6, bond=2)
    h, V, _ = fx.make_integrals(L, 6, 0)
    ints = ab.Integrals(h, V)
    # complete 2-site basis: tables without the complement cap (use N=4 on L=4: all sectors reachable)
    tabs = fx.block_tables(cfg)
    iso = fx.random_isometries(cfg, tabs, 2, 3)
    Xb = ab.build_block(ints, tabs, iso, [0, 1], True)
    assert sum(Xb.basis.dims) == 16
    comp = ab.Composite(Xb, ab.site_block(ints, 2))
    vec = brute.block_vectors(tabs, iso, 2, True)
    cols = []
    for (ix, iy) in comp.pairs:
        e = np.zeros((4, 1))
        e[ab.SITE_STATE_OF_SECTOR[iy], 0] = 1.0
        cols.append(np.kron(vec[ix], e))
    U = np.concatenate(cols, axis=1)                      # 64 x 64 orthogonal
    assert abs(U.T @ U - np.eye(64)).max() < 1e-12
    ref = _definition_ops(ints, 0, 3, L)
    c = fock.jw_creators(3)
    orbs = list(range(6))
    v = ints.v
    for key, O in ref.items():
        got = comp.op(*key).dense(comp.basis)
        assert abs(got - U.T @ O @ U).max() < 1e-12, key
    for i, k in [(6, 7), (7, 6), (6, 6)]:
        Pd = sum(v[i, j, k, l] * c[l].T @ c[j].T for j in orbs for l in orbs)
        Qd = sum((v[i, k, kk, j] - v[i, j, kk, k]) * c[kk] @ c[j].T for kk in orbs for j in orbs)
        assert abs(comp.op("P", i, k).dense(comp.basis) - U.T @ Pd @ U).max() < 1e-12
        assert abs(comp.op("Q", i, k).dense(comp.basis) - U.T @ Qd @ U).max() < 1e-12


def test_cut_identity_as_operator_identity():
    # Appendix A2: H = H^A + H^B + cross terms, all cuts of L = 4, with complete bases.
    L = 4
    h, V, _ = fx.make_integrals(L, 6, 0)
    ints = ab.Integrals(h, V)
    H = fock.hamiltonian_dense(h, V)
    # complete block bases: tables of an L=8, N=8 system are the full Fock sectors for m <= 3
    big = Config("t", L=8, N=8, twoS=0, sym=0, D=256, n_chol=6, bond=3)
    tabs = fx.block_tables(big)
    assert [int(t[:, 2].sum()) for t in tabs[:4]] == [1, 4, 16, 64]
    for cut in (1, 2, 3):
        isoL = fx.random_isometries(big, tabs, cut, 5)
        isoR = fx.random_isometries(big, tabs, L - cut, 6)
        A = ab.build_block(ints, tabs, isoL, list(range(cut)), True)
        B = ab.build_block(ints, tabs, isoR, list(range(L - 1, cut - 1, -1)), False)
        comp = ab.Composite(A, B)
        vA = brute.block_vectors(tabs, isoL, cut, True)
        vB = brute.block_vectors(tabs, isoR, L - cut, False)
        cols = [np.kron(vA[ix], vB[iy]) for (ix, iy) in comp.pairs]
        U = np.concatenate(cols, axis=1)
        assert U.shape == (256, 256) and abs(U.T @ U - np.eye(256)).max() < 1e-12
        got = comp.op("H").dense(comp.basis)
        assert abs(got - U.T @ H @ U).max() < 1e-12


def test_identity_and_number_operator_survive_renormalization():
    s = _setup(5, 4, 0, 5, 2)
    blk = s["Lb"]
    nop = ab.Op((0, 0))
    for i in blk.orbs:
        nop.add(1.0, blk.store[("B", i, i)])
    M = nop.dense(blk.basis)
    off = np.concatenate([[0], np.cumsum(blk.basis.dims)])
    for i, q in enumerate(blk.basis.labels):
        assert abs(M[off[i]:off[i + 1], off[i]:off[i + 1]] - q[0] * np.eye(blk.basis.dims[i])).max() < 1e-12
    assert abs(M - np.diag(np.diag(M))).max() < 1e-12


def test_saturated_heff_is_fci():
    # X = complete bases: H_eff has the FCI spectrum (exact at saturated D)
    s = _setup(4, 4, 0, 16, 1)
    Hfci, _ = fock.fci_matrix(s["h"], s["V"], 2, 2)
    ts = s["ts"]
    assert ts.n == 36
    Heff = np.stack([ts.apply(e) for e in np.eye(ts.n)], axis=1)
    assert abs(Heff - Heff.T).max() < 1e-12
    assert abs(np.linalg.eigvalsh(Heff) - np.linalg.eigvalsh(Hfci)).max() < 1e-11


def test_davidson_monotone_and_bounded():
    s = _setup(5, 4, 0, 5, 2)
    ts = s["ts"]
    Heff = s["P"].T @ s["H"] @ s["P"]
    e0 = np.linalg.eigvalsh(Heff)[0]
    x, th, rs = davidson(ts.apply, ts.diagonal(), fx.random_psi(ts.n, 2), 12)
    assert len(th) == 12
    assert np.all(np.diff(th) <= 1e-12)
    assert np.all(th >= e0 - 1e-12)
    x, th, rs = davidson(ts.apply, ts.diagonal(), fx.random_psi(ts.n, 2), ts.n, tol=1e-10)
    assert th[-1] == pytest.approx(e0, abs=1e-10)
    assert abs(np.linalg.norm(x) - 1) < 1e-12


def test_two_site_sweeps_reach_fci_at_saturated_D():
    L, N = 4, 4
    cfg = Config("t", L=L, N=N, twoS=0, sym=0, D=16, n_chol=6, bond=1)
    h, V, _ = fx.make_integrals(L, 6, 0)
    tabs = fx.block_tables(cfg)
    isoR = fx.random_isometries(cfg, tabs, L - 2, 1001)
    E = two_site_sweeps(ab.Integrals(h, V), cfg, tabs, isoR, n_sweeps=2)
    Hf, _ = fock.fci_matrix(h, V, 2, 2)
    assert E[-1] == pytest.approx(np.linalg.eigvalsh(Hf)[0], abs=1e-9)


def test_psi_block_list_cfg0_is_fci_dimension():
    cfg = fx.get_config("cfg0")
    tabs = fx.block_tables(cfg)
    blocks, n = ab.psi_block_list(tabs[cfg.bond], tabs[cfg.L - cfg.bond - 2], cfg.N, cfg.twoS)
    assert n == 4900            # BASELINE.json configs[0]
    assert int(tabs[cfg.bond][:, 2].sum()) == 64
