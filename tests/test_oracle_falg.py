"""F_alg (SURVEY.md 8(d) "Algorithmic work"): the oracle's enumerator (oracle/falg.py) against brute-force
enumeration, and the library's integer (DMRG_TAB_FALG, DMRG_TAB_FALG_BLOCKS of a planning context, no GPU)
against the oracle's."""
import numpy as np
import pytest

import fixtures as fx
import paper_2603_28648_b200 as pkg
from oracle import abelian as ab, abelian_terms as at, falg, su2, su2_loopnest as ln
from oracle.fock import spin_orbital_integrals
from tests.helpers import make_case, library_context


def _oracle_falg(case):
    cfg, tabs, nl, nr = case["cfg"], case["tabs"], case["nl"], case["nr"]
    L, bond = cfg.L, cfg.bond
    if cfg.sym == 1:
        terms = ln.two_site_terms(case["h"], case["V"], list(range(bond)), bond, bond + 1, list(range(bond + 2, L)))
        blocks, _ = su2.psi_blocks(tabs[nl], tabs[nr], cfg.N, cfg.twoS)
        return terms, blocks, falg.falg(terms, tabs[nl], tabs[nr], blocks, True, cfg.twoS)
    t, v = spin_orbital_integrals(case["h"], case["V"])
    so = lambda ps: [i for p in ps for i in (2 * p, 2 * p + 1)]
    terms = at.two_site_terms(t, v, so(range(bond)), bond, bond + 1, so(range(bond + 2, L)))
    blocks, _ = ab.psi_block_list(tabs[nl], tabs[nr], cfg.N, cfg.twoS)
    return terms, blocks, falg.falg(terms, tabs[nl], tabs[nr], blocks, False)


def _library_falg(case):
    d = library_context(case, plan_only=True)
    out = int(d.table(pkg.TAB_FALG)[0]), d.table(pkg.TAB_FALG_BLOCKS), d.table(pkg.TAB_COUNTS)
    d.close()
    return out


@pytest.mark.parametrize("L,N,S2,D,bond", [(4, 4, 0, 6, 1), (4, 3, 1, 6, 1), (4, 4, 2, 6, 1), (5, 5, 1, 8, 2)])
def test_enumerator_equals_brute_force_enumeration(L, N, S2, D, bond):
    case = make_case(L, N, S2, D, bond, sym=1)
    terms, blocks, (tot, per, f1, f2) = _oracle_falg(case)
    tabs = case["tabs"]
    assert tot == falg.brute_force_su2(terms, tabs[case["nl"]], tabs[case["nr"]], blocks, S2)
    assert tot == f1 + f2 == int(per.sum()) and tot > 0


def test_falg_counts_the_multiply_adds_of_a_literal_two_stage_evaluation():
    """One group, by hand: n operator pairs between one input and one output block cost
    2 dL dR (n dR') + 2 dL' (n dL) dR' flops; checked on a synthetic one-block table."""
    tabL = np.array([[0, 0, 3, 0], [1, 1, 5, 3]])
    tabR = np.array([[1, 1, 4, 0], [2, 0, 2, 4]])
    # two pairs C_p (x) C~-like partners: left symbols a+_0, a+_1 (dN = +1), right symbols S~_0, S~_1 (dN = -1)
    terms = {(("C", 0, 1, p, -1), ("S", 0, 1, p, -1), 0, 0, 0, 0, 1, 0, 1, 0, 1): 1.0 for p in (0, 1)}
    blocks = np.array([[0, 0, 0, 0, 1, 0, 3, 2, 0], [1, 0, 1, 0, 0, 1, 5, 4, 6]])     # input (iL=0, iR=1), output (iL=1, iR=0)
    tot, per, f1, f2 = falg.falg(terms, tabL, tabR, blocks, True, 0)
    dL, dR, dLp, dRp, n = 3, 2, 5, 4, 2
    assert f1 == 2 * dL * dR * n * dRp and f2 == 2 * dLp * n * dL * dRp
    assert list(per) == [0, f1 + f2]


SMALL = [(4, 4, 0, 6, 1, 1), (5, 5, 1, 8, 2, 1), (5, 4, 2, 8, 1, 1), (6, 6, 0, 10, 2, 1), (5, 5, 3, 9, 0, 1), (6, 7, 1, 12, 3, 1),
         (7, 6, 0, 24, 3, 1), (12, 18, 0, 64, 5, 1), (4, 4, 0, 6, 1, 0), (5, 5, 1, 8, 2, 0), (6, 6, 0, 10, 2, 0), (5, 5, -1, 9, 0, 0),
         (6, 7, 1, 12, 3, 0)]


@pytest.mark.parametrize("L,N,tw,D,bond,sym", SMALL)
def test_library_falg_equals_the_oracle_small(L, N, tw, D, bond, sym):
    case = make_case(L, N, tw, D, bond, sym=sym)
    _, _, (tot, per, f1, f2) = _oracle_falg(case)
    F, Fb, counts = _library_falg(case)
    assert F == tot
    assert np.array_equal(Fb, per)
    assert (int(counts[11]), int(counts[12])) == (f1, f2)


@pytest.mark.parametrize("name", ["cfg0", "cfg1"])
def test_library_falg_equals_the_oracle_on_the_abelian_configs(name):
    case = make_case(0, 0, 0, 0, 0, cfg=fx.get_config(name))
    _, _, (tot, per, f1, f2) = _oracle_falg(case)
    F, Fb, counts = _library_falg(case)
    assert F == tot and np.array_equal(Fb, per)


def test_library_falg_equals_the_oracle_on_the_cas5436_shape_at_d256():
    """The CAS(54,36)-shaped system of configs[2] at D_SU(2) = 256 (same operator set and term list as D = 2048)."""
    case = make_case(0, 0, 0, 0, 0, cfg=fx.get_config("cfg2").with_(D=256))
    _, _, (tot, per, f1, f2) = _oracle_falg(case)
    F, Fb, counts = _library_falg(case)
    assert F == tot and np.array_equal(Fb, per)
    assert (int(counts[11]), int(counts[12])) == (f1, f2)
