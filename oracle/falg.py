"""Algorithmic flop count F_alg of one H_eff.psi (TEST INFRASTRUCTURE ONLY; SURVEY.md 8(d)
"Algorithmic work": "The oracle's enumerator computes F_alg as an integer; the library must report the
same integer").

Definition ("F_alg"), on the oracle's own term list of the two-site H_eff
(oracle/su2_loopnest.two_site_terms / oracle/abelian_terms.two_site_terms, normal pair operators on the
A = (L, s1) side, reading s5):

  1. Terms c * O_L (x) unit (x) O_R with equal (O_L, O_R, site unit, ranks) are one term; c = 0 drops it.
  2. Terms form a GROUP when they agree in the class of both block operators -- the stored class the operator
     is made of, (kind, dN, second label [d2Sz or rank]), complements counting as the pair class they are
     contracted from (P -> A+, Q -> B), plus the dagger/tilde flag -- in the site unit (s1', s1, s2', s2) and,
     for SU(2), in the ranks (k1, k, k2).
  3. Within a group the normal/complementary form needs n = min(#distinct O_L, #distinct O_R) operator pairs
     (the side with more distinct operators is contracted with the integrals onto the other, A3).
  4. For every group, input block b = (q_L, s1, s2, q_R) and reachable right sector q_R':
       stage 1   2 d_L d_R (n d_R')          once, if at least one output block uses it,
       stage 2   2 d_L' (n d_L) d_R'         for every output block b' = (q_L', s1', s2', q_R') that exists and
                                              (SU(2)) whose three 9j symbols satisfy their triangle conditions;
     a one-sided group (O_R = identity, or else O_L = identity) is ONE product per pair and output block:
     2 d_L' d_L d_R, resp. 2 d_L d_R d_R'.
True block dimensions; no tile padding, slice products, recombination or slicing.

Per-output-block figures attribute a stage-1 product to the first output block that uses it, in ascending
(q_L', 2S_A', 2S_B') order.

Pins (tests/test_oracle_falg.py): brute-force enumeration of every (term pair, input block, output block)
instance on L = 4 systems; F_alg/2 = the multiply-adds a literal two-stage evaluation performs.
"""
import numpy as np

from .wigner import triangle

_SITE_J2 = [0, 1, 0]
_SITE_N3 = [0, 1, 2]
_SITE_AB = [(0, 0), (1, 1), (1, -1), (2, 0)]


def _class_su2(sym):
    """(stored kind, stored dN, rank, tilde flag relative to the stored operator) of an SU(2) symbol."""
    kind, til, k2, i, k = sym
    if kind == "P":                     # P~ = sum w A~: the A class, tilde flag flipped
        return ("A", 2, k2, 1 - til)
    if kind == "Q":
        return ("B", 0, k2, 0)
    dn = {"I": 0, "H": 0, "C": 1, "S": -1, "A": 2, "B": 0}[kind]
    return (kind, dn, k2, til if kind not in ("I", "H", "B") else 0)


def _class_u1(sym):
    from .abelian_terms import sym_dq
    kind, dag, i, k = sym
    if kind == "P":                     # P_ik = sum w (A_jl)+: the class of A with the same spins, daggered
        q = sym_dq(("A", 0, i, k))
        return ("A", q[0], q[1], 1 - dag)
    if kind == "Q":                     # Q_il = sum w B_kj with the spin change of Q_il
        q = sym_dq(("Q", 0, i, k))
        return ("B", q[0], q[1], 0)
    q = sym_dq((kind, 0, i, k))
    return (kind, q[0], q[1], dag if kind not in ("I", "H", "B") else 0)


def groups_of(terms, su2):
    """{group key: (n pairs, effective dq of O_L, effective dq of O_R, kindL, kindR)}."""
    byL, byR = {}, {}
    info = {}
    for key in terms:
        symL, symR = key[0], key[1]
        cl, cr = (_class_su2(symL), _class_su2(symR)) if su2 else (_class_u1(symL), _class_u1(symR))
        g = (cl, cr) + tuple(key[2:6]) + ((key[7], key[8], key[9]) if su2 else ())
        byL.setdefault(g, set()).add(symL)
        byR.setdefault(g, set()).add(symR)
        info[g] = (cl, cr)
    out = {}
    for g, (cl, cr) in info.items():
        eff = lambda c: ((-c[1] if c[3] else c[1]), (c[2] if su2 else (-c[2] if c[3] else c[2])))
        out[g] = (min(len(byL[g]), len(byR[g])), eff(cl), eff(cr), cl[0], cr[0])
    return out


def _bras(tab, index, q, dq, su2):
    """Sectors reachable from ket sector q by an operator of class dq = (dN, second label)."""
    N, S = int(q[0]), int(q[1])
    if not su2:
        i = index.get((N + dq[0], S + dq[1]))
        return [] if i is None else [i]
    return [index[(N + dq[0], S2)] for S2 in range(abs(S - dq[1]), S + dq[1] + 1, 2) if (N + dq[0], S2) in index]


def falg(terms, tabL, tabR, psi_blocks, su2, S2tot=0):
    """(F_alg, per-output-block F_alg, stage-1 part, stage-2 part) from a term list and the block tables.
    psi_blocks: rows (iL, s1, 2S_A, s2, iR, 2S_B, dL, dR, off) for SU(2), (iL, s1, s2, iR, dL, dR, off) for U(1)xU(1)."""
    tabL, tabR = np.asarray(tabL), np.asarray(tabR)
    idxL = {(int(r[0]), int(r[1])): i for i, r in enumerate(tabL)}
    idxR = {(int(r[0]), int(r[1])): i for i, r in enumerate(tabR)}
    if su2:
        pos = {tuple(int(x) for x in b[:6]): n for n, b in enumerate(psi_blocks)}
        rows = [(int(b[0]), int(b[1]), int(b[2]), int(b[3]), int(b[4]), int(b[5])) for b in psi_blocks]
    else:
        pos = {(int(b[0]), int(b[1]), 0, int(b[2]), int(b[3]), 0): n for n, b in enumerate(psi_blocks)}
        rows = [(int(b[0]), int(b[1]), 0, int(b[2]), int(b[3]), 0) for b in psi_blocks]
    per_block = np.zeros(len(rows), dtype=np.int64)
    f1 = f2 = 0
    by_unit = {}
    for n, (iL, s1, SA, s2, iR, SB) in enumerate(rows):
        by_unit.setdefault((s1, s2), []).append(n)
    fuse = (lambda S, s: range(abs(S - _SITE_J2[s]), S + _SITE_J2[s] + 1, 2)) if su2 else (lambda S, s: [0])
    for g, (n_pairs, dqL, dqR, kindL, kindR) in groups_of(terms, su2).items():
        s1p, s1, s2p, s2 = g[2:6]
        k1, kk, k2 = g[6:9] if su2 else (0, 0, 0)
        kL, kR = (g[0][2], g[1][2]) if su2 else (0, 0)
        for n in by_unit.get((s1, s2), []):
            iL, _, SA, _, iR, SB = rows[n]
            dL, dR = int(tabL[iL][2]), int(tabR[iR][2])
            SL, SR = int(tabL[iL][1]), int(tabR[iR][1])
            for iRp in _bras(tabR, idxR, tabR[iR], dqR, su2):
                dRp, SRp = int(tabR[iRp][2]), int(tabR[iRp][1])
                stage1_done = False
                for iLp in _bras(tabL, idxL, tabL[iL], dqL, su2):
                    dLp, SLp = int(tabL[iLp][2]), int(tabL[iLp][1])
                    for SAp in fuse(SLp, s1p):
                        for SBp in fuse(SRp, s2p):
                            o = pos.get((iLp, s1p, SAp, s2p, iRp, SBp))
                            if o is None:
                                continue
                            if su2 and not (_nine_j_allowed(SL, _SITE_J2[s1], SA, kL, k1, kk, SLp, _SITE_J2[s1p], SAp)
                                            and _nine_j_allowed(_SITE_J2[s2], SR, SB, k2, kR, kk, _SITE_J2[s2p], SRp, SBp)
                                            and _nine_j_allowed(SA, SB, S2tot, kk, kk, 0, SAp, SBp, S2tot)):
                                continue
                            if kindR == "I":
                                w = 2 * dLp * dL * dR * n_pairs
                                f2 += w
                                per_block[o] += w
                                continue
                            if kindL == "I":
                                w = 2 * dL * dR * dRp * n_pairs
                                f2 += w
                                per_block[o] += w
                                continue
                            if not stage1_done:
                                stage1_done = True
                                w = 2 * dL * dR * n_pairs * dRp
                                f1 += w
                                per_block[o] += w
                            w = 2 * dLp * n_pairs * dL * dRp
                            f2 += w
                            per_block[o] += w
    return f1 + f2, per_block, f1, f2


def _nine_j_allowed(j1, j2, J, k1, k2, K, j1p, j2p, Jp):
    """The six triangle conditions of {j1 j2 J; k1 k2 K; j1' j2' J'} (rows and columns)."""
    return (triangle(j1, j2, J) and triangle(k1, k2, K) and triangle(j1p, j2p, Jp)
            and triangle(j1, k1, j1p) and triangle(j2, k2, j2p) and triangle(J, K, Jp))


def brute_force_su2(terms, tabL, tabR, psi_blocks, S2tot):
    """The same count by literal enumeration of every (elementary term, input block, output block) instance that
    the A5 element formula touches, then collapsing instances to operator pairs: a stage-1 product is identified by
    (group, pair slot, b, q_R'), a stage-2 product by (group, pair slot, b, b').  Pair slots: the distinct operators
    of the side with fewer of them.  Independent of `falg` in structure (sets of instances, no per-group arithmetic)."""
    tabL, tabR = np.asarray(tabL), np.asarray(tabR)
    idxL = {(int(r[0]), int(r[1])): i for i, r in enumerate(tabL)}
    idxR = {(int(r[0]), int(r[1])): i for i, r in enumerate(tabR)}
    pos = {tuple(int(x) for x in b[:6]): n for n, b in enumerate(psi_blocks)}
    from .su2_loopnest import sym_dN
    # operator-pair slots per group
    gl, gr, gkey = {}, {}, {}
    for key in terms:
        g = (_class_su2(key[0]), _class_su2(key[1])) + tuple(key[2:6]) + (key[7], key[8], key[9])
        gkey[key] = g
        gl.setdefault(g, set()).add(key[0])
        gr.setdefault(g, set()).add(key[1])
    stage1, stage2, one_sided = set(), set(), set()
    for key in terms:
        symL, symR, s1p, s1, s2p, s2, kL, k1, kk, k2, kR = key
        g = gkey[key]
        slot = key[0] if len(gl[g]) <= len(gr[g]) else key[1]        # which side names the pair
        for n, b in enumerate(psi_blocks):
            iL, bs1, SA, bs2, iR, SB = (int(x) for x in b[:6])
            if bs1 != s1 or bs2 != s2:
                continue
            NL, SL, NR, SR = int(tabL[iL][0]), int(tabL[iL][1]), int(tabR[iR][0]), int(tabR[iR][1])
            for o, bo in enumerate(psi_blocks):
                iLp, os1, SAp, os2, iRp, SBp = (int(x) for x in bo[:6])
                if os1 != s1p or os2 != s2p:
                    continue
                NLp, SLp, NRp, SRp = int(tabL[iLp][0]), int(tabL[iLp][1]), int(tabR[iRp][0]), int(tabR[iRp][1])
                if NLp - NL != sym_dN(symL) or NRp - NR != sym_dN(symR):
                    continue
                if not (_nine_j_allowed(SL, _SITE_J2[s1], SA, kL, k1, kk, SLp, _SITE_J2[s1p], SAp)
                        and _nine_j_allowed(_SITE_J2[s2], SR, SB, k2, kR, kk, _SITE_J2[s2p], SRp, SBp)
                        and _nine_j_allowed(SA, SB, S2tot, kk, kk, 0, SAp, SBp, S2tot)):
                    continue
                dL, dR, dLp, dRp = int(tabL[iL][2]), int(tabR[iR][2]), int(tabL[iLp][2]), int(tabR[iRp][2])
                if symR[0] == "I":
                    one_sided.add((g, slot, n, o, 2 * dLp * dL * dR))
                elif symL[0] == "I":
                    one_sided.add((g, slot, n, o, 2 * dL * dR * dRp))
                else:
                    stage1.add((g, slot, n, iRp, 2 * dL * dR * dRp))
                    stage2.add((g, slot, n, o, 2 * dLp * dL * dRp))
    return sum(x[-1] for x in stage1) + sum(x[-1] for x in stage2) + sum(x[-1] for x in one_sided)
