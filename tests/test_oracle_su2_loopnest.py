"""Pins for oracle/su2_loopnest.py (oracle part c4 in reduced form).

The loop-nest oracle works on reduced matrix elements with its own 6j/9j recoupling; it is pinned to the
expansion oracle (oracle/su2.py: Clebsch-Gordan expansion into the U(1)xU(1) oracle, itself pinned to the
brute-force projected Hamiltonian), which shares none of that recoupling."""
import numpy as np
import pytest

import fixtures as fx
from oracle import su2, su2_loopnest as ln
from tests.helpers import make_case, oracle_su2, rel_err, su2_block_components

# (L, N, 2S, D, bond): singlet, doublet, triplet, quartet, odd N, empty left block, larger D
CASES = [(4, 4, 0, 6, 1), (5, 5, 1, 8, 2), (5, 4, 2, 8, 1), (6, 6, 0, 10, 2), (5, 5, 3, 9, 0), (6, 7, 1, 12, 3),
         (6, 6, 2, 30, 2), (7, 6, 0, 24, 3)]


def _blocks(case):
    cfg, h, V, tabs = case["cfg"], case["h"], case["V"], case["tabs"]
    opsL = ln.build_block(h, V, tabs, case["isoL"], list(range(case["nl"])), True)
    opsR = ln.build_block(h, V, tabs, case["isoR"], list(range(cfg.L - 1, cfg.bond + 1, -1)), False)
    return opsL, opsR


@pytest.mark.parametrize("L,N,S2,D,bond", CASES)
def test_loopnest_heff_equals_the_expansion_oracle(L, N, S2, D, bond):
    case = make_case(L, N, S2, D, bond, sym=1)
    ex = oracle_su2(case)
    opsL, opsR = _blocks(case)
    ts = ln.TwoSite(case["h"], case["V"], opsL, bond, bond + 1, opsR, N, S2)
    assert ts.n == ex.n and np.array_equal(ts.blocks, ex.blocks)
    psi = fx.random_psi(ts.n, 2)
    ref = ex.apply(psi)
    assert rel_err(ts.apply(psi), ref) <= 1e-12
    # the same sum evaluated pair by pair on enlarged (un-rotated) blocks: the form the full-size checks use
    assert rel_err(ts.apply_enlarged(psi), ref) <= 1e-12
    # the cut identity holds with the normal pair operators on either side of the cut (Appendix A2)
    mirror = ln.TwoSite(case["h"], case["V"], opsL, bond, bond + 1, opsR, N, S2, normal_on="B")
    assert set(mirror.terms) != set(ts.terms)
    assert rel_err(mirror.apply(psi), ref) <= 1e-12
    # sampled outputs: only the requested blocks are filled, and they are the same numbers
    pick = sorted({0, len(ts.blocks) // 2, len(ts.blocks) - 1})
    part = ts.apply(psi, outputs=pick)
    for n, b in enumerate(ts.blocks):
        seg = slice(int(b[8]), int(b[8]) + int(b[6]) * int(b[7]))
        if n in pick:
            assert np.abs(part[seg] - ref[seg]).max() <= 1e-12 * max(1.0, np.abs(ref).max())
        else:
            assert not part[seg].any()


@pytest.mark.parametrize("L,N,S2,D,bond", [(5, 5, 1, 8, 2), (6, 6, 0, 10, 2), (6, 7, 1, 12, 3), (5, 4, 2, 8, 1)])
def test_loopnest_renormalized_operators_are_the_reduced_elements(L, N, S2, D, bond):
    """c5 in reduced form: every stored operator of both blocks (H, a+, S~, A^k, B^k) equals the Wigner-Eckart
    projection of the expanded U(1)xU(1) oracle operator."""
    case = make_case(L, N, S2, D, bond, sym=1)
    ex = oracle_su2(case)
    opsL, opsR = _blocks(case)
    tabs, nl, nr = case["tabs"], case["nl"], case["nr"]
    for ops, blk, tab in ((opsL, ex.Lb, tabs[nl]), (opsR, ex.Rb, tabs[nr])):
        if not ops.orbs:
            continue
        n_checked = 0
        for (kind, k2, p, r) in ln.normal_set(ops.orbs, L):
            comps, rank = su2_block_components(blk, kind, p, r, k2)
            red, worst = su2.reduced_blocks(comps, rank, tab)
            assert worst < 1e-11
            for ib in range(len(tab)):
                for ik in range(len(tab)):
                    got = ops.block((kind, 0, k2, p, r), ib, ik)
                    want = red.get((ib, ik))
                    if want is None or not ops.allowed((kind, 0, k2, p, r), ib, ik):
                        assert got is None or np.abs(got).max() < 1e-12
                        continue
                    got = np.zeros_like(want) if got is None else got
                    assert np.abs(got - want).max() < 1e-12, (kind, k2, p, r, ib, ik)
                    n_checked += 1
        assert n_checked > 10


def test_tilde_rules_against_explicit_components():
    """A4 "Adjoint rule" on the site: the reduced matrix of T~ built from explicit components equals the rule
    applied to the reduced matrix of T; T~~ = (-1)^{2k} T."""
    h, V, _ = fx.make_integrals(3, 4, 0)
    site = ln.SitePart(h, V, 1)
    for kind, k2, i, k in [("C", 1, 1, -1), ("S", 1, 0, -1), ("A", 0, 1, 1), ("B", 0, 1, 1), ("B", 2, 1, 1), ("Q", 2, 0, 2)]:
        f = site.op(kind, k2, i, k)
        if kind == "C":
            comps = site.cre
        elif kind == "B":
            comps = ln._couple_components(site.cre, 1, site.ann, 1, k2)
        else:
            comps = None
        if comps is not None:
            want = ln._reduce_site(ln._tilde_components(comps, k2), k2)
            assert np.abs(f.tilde().m - want).max() < 1e-14
        back = f.tilde().tilde().m
        assert np.abs(back - (-1.0 if k2 & 1 else 1.0) * f.m).max() < 1e-14
    # reduced site elements quoted in SURVEY.md Appendix A4
    c = site.op("C", 1, 1).m
    assert c[1, 0] == pytest.approx(1.0) and c[2, 1] == pytest.approx(-np.sqrt(2.0))
    a = site.op("C", 1, 1).tilde().m
    assert a[0, 1] == pytest.approx(-np.sqrt(2.0)) and a[1, 2] == pytest.approx(-1.0)
    b0 = site.op("B", 0, 1, 1).m               # E_pp = n = -sqrt2 B^0_pp
    assert np.allclose(-np.sqrt(2.0) * np.diag(b0), [0.0, 1.0, 2.0])


def test_term_list_is_hermitian_and_particle_conserving():
    """Every term conserves N, and the reduced H_eff built from the term list is symmetric."""
    case = make_case(6, 6, 0, 10, 2, sym=1)
    opsL, opsR = _blocks(case)
    ts = ln.TwoSite(case["h"], case["V"], opsL, 2, 3, opsR, 6, 0)
    for key in ts.terms:
        symL, symR, s1p, s1, s2p, s2 = key[:6]
        assert ln.sym_dN(symL) + ln.sym_dN(symR) + (s1p - s1) + (s2p - s2) == 0
    H = np.stack([ts.apply(e) for e in np.eye(ts.n)], axis=1)
    assert np.abs(H - H.T).max() < 1e-12
