"""Oracle part c4 for SU(2): the plain definition by expansion (test infrastructure).

A spin-adapted (reduced) MPS / wave function / operator MEANS its Wigner-Eckart expansion into
the S_z-resolved U(1)xU(1) representation ("Wigner-Eckart convention", last
bullet; reading s20 of section 8(c)):

  X_full[(qL mL a), (s ms), (qA mA a')] = X_red[qL, s, qA][a, a'] <S_L mL; s ms | S_A mA>   (left block)
  X_full[(qR mR a), (s ms), (qB mB a')] = X_red[qR, s, qB][a, a'] <s ms; S_R mR | S_B mB>   (right block:
                                                                   the site is on the left)
  psi_full = sum psi_red[(qL s1 qA), (s2 qR qB)] <S_L mL; s1 m1|S_A mA> <s2 m2; S_R mR|S_B mB>
                                                 <S_A mA; S_B mB | S_tot M>
  <a' j' m'| T^k_q |a j m> = <j m; k q | j' m'> <a' j' || T^k || a j>       (bare Clebsch-Gordan)

so the SU(2) oracle is: expand with Condon-Shortley Clebsch-Gordan coefficients, run the pinned
U(1)xU(1) oracle (abelian.py, itself pinned to the brute-force projected Hamiltonian), and project
back.  Nothing of the library's 6j/9j recoupling is used here.  All spins are passed DOUBLED
(integers: 2j, 2m).

Pins (tests/test_oracle_su2.py): Clebsch-Gordan orthogonality, closed forms and exact values;
expanded isometries are isometries; expansion preserves the norm; the expanded Hamiltonian action
stays inside the S_tot multiplet (H is a scalar) and is independent of M.
"""
from math import factorial, sqrt

import numpy as np

SITE_J2 = [0, 1, 0]            # doubled spin of the site multiplets N = 0, 1, 2
SITE_N = [0, 1, 2]


def cg(j1, m1, j2, m2, J, M):
    """<j1 m1; j2 m2 | J M>, Condon-Shortley phases, Racah's formula; arguments doubled."""
    if m1 + m2 != M or J < abs(j1 - j2) or J > j1 + j2 or (j1 + j2 + J) % 2:
        return 0.0
    if abs(m1) > j1 or abs(m2) > j2 or abs(M) > J or (j1 + m1) % 2 or (j2 + m2) % 2 or (J + M) % 2:
        return 0.0
    f = lambda x: factorial(x // 2)          # x is an even doubled integer
    pre = (J + 1) * f(J + j1 - j2) * f(J - j1 + j2) * f(j1 + j2 - J) / f(j1 + j2 + J + 2)
    pre *= f(J + M) * f(J - M) * f(j1 - m1) * f(j1 + m1) * f(j2 - m2) * f(j2 + m2)
    s = 0.0
    k = 0
    while True:
        a = [j1 + j2 - J - 2 * k, j1 - m1 - 2 * k, j2 + m2 - 2 * k, J - j2 + m1 + 2 * k, J - j1 - m2 + 2 * k]
        if a[0] < 0 or a[1] < 0 or a[2] < 0:
            break
        if a[3] >= 0 and a[4] >= 0:
            s += (-1) ** k / (factorial(k) * f(a[0]) * f(a[1]) * f(a[2]) * f(a[3]) * f(a[4]))
        k += 1
    return sqrt(pre) * s


def site_state_of(s, m2):
    """U(1)xU(1) site state index (PAPER.md:41 order) of the component m of site multiplet s."""
    if s == 0:
        return 0
    if s == 2:
        return 3                       # |ud> = a+_u a+_d |0> is the N = 2 singlet
    return 1 if m2 == 1 else 2


def expand_table(tab):
    """SU(2) bond table -> U(1)xU(1) table plus the map (i_su2, 2m) -> (i_abelian, offset in sector).
    Inside an abelian sector the multiplets are ordered by S ascending."""
    dims, where = {}, {}
    for i, (N, S2, d, _) in enumerate(tab):
        for m2 in range(-S2, S2 + 1, 2):
            key = (int(N), m2)
            where[(i, m2)] = (key, dims.get(key, 0))
            dims[key] = dims.get(key, 0) + int(d)
    keys = sorted(dims)
    index = {k: n for n, k in enumerate(keys)}
    rows, off = [], 0
    for k in keys:
        rows.append((k[0], k[1], dims[k], off))
        off += dims[k]
    out = np.array(rows, dtype=np.int64).reshape(-1, 4)
    return out, {k: (index[v[0]], v[1]) for k, v in where.items()}


def expand_isometry(tab_prev, tab_next, blocks, data, site_is_right):
    """Packed reduced isometry -> packed U(1)xU(1) isometry (fixtures.mps layout)."""
    from fixtures.mps import isometry_blocks
    ta, wa = expand_table(tab_prev)
    tb, wb = expand_table(tab_next)
    ab_blocks, n = isometry_blocks(0, ta, tb)
    pos = {(int(b[0]), int(b[1]), int(b[2])): b for b in ab_blocks}
    out = np.zeros(n)
    for (ip, s, inext, rows, cols, off) in blocks:
        X = data[off:off + rows * cols].reshape(rows, cols)
        jp, jn, js = int(tab_prev[ip][1]), int(tab_next[inext][1]), SITE_J2[s]
        for mp in range(-jp, jp + 1, 2):
            for ms in range(-js, js + 1, 2):
                mn = mp + ms
                c = cg(jp, mp, js, ms, jn, mn) if site_is_right else cg(js, ms, jp, mp, jn, mn)
                if c == 0.0:
                    continue
                (ia, oa), (ib, ob) = wa[(ip, mp)], wb[(inext, mn)]
                b = pos[(ia, site_state_of(s, ms), ib)]
                view = out[b[5]:b[5] + b[3] * b[4]].reshape(b[3], b[4])
                view[oa:oa + rows, ob:ob + cols] += c * X
    return ta, tb, ab_blocks, out


def psi_blocks(tabL, tabR, N, S2tot):
    """Reduced psi layout: rows (iL, s1, 2S_A, s2, iR, 2S_B, dL, dR, offset), lexicographic."""
    rl = {(int(r[0]), int(r[1])): i for i, r in enumerate(tabR)}
    rows, off = [], 0
    for iL, (NL, SL, dL, _) in enumerate(tabL):
        for s1 in range(3):
            for SA in range(abs(SL - SITE_J2[s1]), SL + SITE_J2[s1] + 1, 2):
                NA = NL + SITE_N[s1]
                for s2 in range(3):
                    for iR, (NR, SR, dR, _) in enumerate(tabR):
                        if NA + SITE_N[s2] + NR != N:
                            continue
                        for SB in range(abs(SR - SITE_J2[s2]), SR + SITE_J2[s2] + 1, 2):
                            if abs(SA - SB) <= S2tot <= SA + SB and (SA + SB + S2tot) % 2 == 0:
                                rows.append((iL, s1, SA, s2, iR, SB, int(dL), int(dR), off))
                                off += int(dL) * int(dR)
    rows.sort(key=lambda r: r[:6])
    off = 0
    out = []
    for r in rows:
        out.append(r[:8] + (off,))
        off += r[6] * r[7]
    return np.array(out, dtype=np.int64).reshape(-1, 9), off


def _psi_map(tabL, tabR, N, S2tot, M2):
    """For every reduced block and spin component: (abelian block row, row/col offsets, coefficient)."""
    from .abelian import psi_block_list
    ta, wa = expand_table(tabL)
    tb, wb = expand_table(tabR)
    ab_blocks, n_ab = psi_block_list(ta, tb, N, M2)
    pos = {tuple(int(x) for x in b[:4]): b for b in ab_blocks}
    red, n_red = psi_blocks(tabL, tabR, N, S2tot)
    items = []
    for (iL, s1, SA, s2, iR, SB, dL, dR, off) in red:
        SL, SR = int(tabL[iL][1]), int(tabR[iR][1])
        j1, j2 = SITE_J2[s1], SITE_J2[s2]
        for mL in range(-SL, SL + 1, 2):
            for m1 in range(-j1, j1 + 1, 2):
                for m2 in range(-j2, j2 + 1, 2):
                    mR = M2 - mL - m1 - m2
                    if abs(mR) > SR:
                        continue
                    c = (cg(SL, mL, j1, m1, SA, mL + m1) * cg(j2, m2, SR, mR, SB, m2 + mR)
                         * cg(SA, mL + m1, SB, m2 + mR, S2tot, M2))
                    if c == 0.0:
                        continue
                    (ia, oa), (ib, ob) = wa[(iL, mL)], wb[(iR, mR)]
                    b = pos[(ia, site_state_of(s1, m1), site_state_of(s2, m2), ib)]
                    items.append((int(off), int(dL), int(dR), b, oa, ob, c))
    return items, n_red, n_ab


def expand_psi(psi_red, tabL, tabR, N, S2tot, M2):
    items, n_red, n_ab = _psi_map(tabL, tabR, N, S2tot, M2)
    assert len(psi_red) == n_red
    out = np.zeros(n_ab)
    for off, dL, dR, b, oa, ob, c in items:
        view = out[b[6]:b[6] + b[4] * b[5]].reshape(b[4], b[5])
        view[oa:oa + dL, ob:ob + dR] += c * psi_red[off:off + dL * dR].reshape(dL, dR)
    return out


def project_psi(psi_full, tabL, tabR, N, S2tot, M2):
    """Overlap with the coupled basis states |(L s1)A, (s2 R)B; S_tot M>: the reduced coefficients."""
    items, n_red, n_ab = _psi_map(tabL, tabR, N, S2tot, M2)
    assert len(psi_full) == n_ab
    out = np.zeros(n_red)
    for off, dL, dR, b, oa, ob, c in items:
        view = psi_full[b[6]:b[6] + b[4] * b[5]].reshape(b[4], b[5])
        out[off:off + dL * dR] += c * view[oa:oa + dL, ob:ob + dR].reshape(-1)
    return out


class ExpandedTwoSite:
    """H_eff of a spin-adapted two-site problem, defined by expansion into U(1)xU(1)."""

    def __init__(self, h, V, N, S2tot, bond, tabs_left, isos_left, tabs_right, isos_right, M2=None):
        from . import abelian as ab
        L = h.shape[0]
        self.N, self.S2, self.M2 = N, S2tot, (S2tot if M2 is None else M2)
        self.tabL, self.tabR = tabs_left[-1], tabs_right[-1]
        ints = ab.Integrals(h, V)
        self.ints = ints

        def grow(tabs, isos, sites, site_is_right):
            blk = ab.vacuum_block(ints)
            for m, p in enumerate(sites):
                ta, tb, bl, dat = expand_isometry(tabs[m], tabs[m + 1], isos[m][0], isos[m][1], site_is_right)
                blk = ab.renormalize(blk, ab.site_block(ints, p), bl, dat, tb, site_is_right)
            return blk
        self.Lb = grow(tabs_left, isos_left, list(range(bond)), True)
        self.Rb = grow(tabs_right, isos_right, list(range(L - 1, bond + 1, -1)), False)
        self.ts = ab.TwoSite(self.Lb, ab.site_block(ints, bond), ab.site_block(ints, bond + 1), self.Rb,
                             N, self.M2)
        self.blocks, self.n = psi_blocks(self.tabL, self.tabR, N, S2tot)

    def expand(self, psi_red):
        return expand_psi(psi_red, self.tabL, self.tabR, self.N, self.S2, self.M2)

    def project(self, psi_full):
        return project_psi(psi_full, self.tabL, self.tabR, self.N, self.S2, self.M2)

    def apply(self, psi_red):
        return self.project(self.ts.apply(self.expand(psi_red)))

    def leakage(self, psi_red):
        """|H psi - P H psi| in the expanded space: zero when H is a scalar and the basis is complete
        within the multiplet structure (a pin of the expansion itself)."""
        y = self.ts.apply(self.expand(psi_red))
        return float(np.linalg.norm(y - self.expand(self.project(y))))


def reduced_blocks(components, k2, tab):
    """Wigner-Eckart projection: components {2q: dense matrix in the expanded basis of `tab`} of a
    rank-k tensor operator -> ({(i_bra, i_ket): reduced matrix}, max inconsistency over m)."""
    ta, where = expand_table(tab)
    offs = ta[:, 3]
    out, worst = {}, 0.0
    for i, (N, S2, d, _) in enumerate(tab):
        for ip, (Np, Sp2, dp, _) in enumerate(tab):
            vals = []
            for q2, Mx in components.items():
                for m2 in range(-S2, S2 + 1, 2):
                    mp2 = m2 + q2
                    c = cg(int(S2), m2, k2, q2, int(Sp2), mp2)
                    if abs(c) < 1e-12 or abs(mp2) > Sp2:
                        continue
                    (ia, oa), (ib, ob) = where[(i, m2)], where[(ip, mp2)]
                    r0, c0 = offs[ib] + ob, offs[ia] + oa
                    vals.append(Mx[r0:r0 + dp, c0:c0 + d] / c)
            if not vals:
                continue
            ref = vals[0]
            worst = max([worst] + [float(np.abs(v - ref).max()) for v in vals[1:]])
            if np.abs(ref).max() > 0 or True:
                out[(ip, i)] = ref
    return out, worst
