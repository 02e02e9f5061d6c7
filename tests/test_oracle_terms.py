"""Pins for oracle/abelian_terms.py: the symbolic two-site term list of U(1)xU(1) (Appendix A2/A3/A5) against the
enlarged-block oracle (oracle/abelian.py), which is pinned to the brute-force projected Hamiltonian."""
import numpy as np
import pytest

import fixtures as fx
from oracle import abelian_terms as at
from tests.helpers import make_case, oracle_two_site, rel_err

CASES = [(4, 4, 0, 6, 1), (5, 5, 1, 8, 2), (5, 4, 2, 8, 1), (6, 6, 0, 10, 2), (5, 5, -1, 9, 0), (6, 7, 1, 12, 3)]


@pytest.mark.parametrize("L,N,tw,D,bond", CASES)
def test_term_list_heff_equals_the_enlarged_block_oracle(L, N, tw, D, bond):
    case = make_case(L, N, tw, D, bond)
    ints, Lb, Rb, ts = oracle_two_site(case)
    psi = fx.random_psi(ts.n, 2)
    ref = ts.apply(psi)
    terms = at.two_site_terms(ints.t, ints.v, Lb.orbs, bond, bond + 1, Rb.orbs)
    assert rel_err(at.apply_terms(terms, Lb, Rb, N, tw, psi), ref) <= 1e-12
    for key in terms:                                   # every term conserves (N, S_z)
        ql, qr = at.sym_dq(key[0]), at.sym_dq(key[1])
        lab = at.SITE_LABELS
        assert ql[0] + qr[0] + lab[key[2]][0] - lab[key[3]][0] + lab[key[4]][0] - lab[key[5]][0] == 0
        assert ql[1] + qr[1] + lab[key[2]][1] - lab[key[3]][1] + lab[key[4]][1] - lab[key[5]][1] == 0
    # the mirror identity (normal pair operators on the B side) gives the same vector from a different list
    mirror = at.two_site_terms(ints.t, ints.v, Lb.orbs, bond, bond + 1, Rb.orbs, normal_on="B")
    assert set(mirror) != set(terms)
    assert rel_err(at.apply_terms(mirror, Lb, Rb, N, tw, psi), ref) <= 1e-12
