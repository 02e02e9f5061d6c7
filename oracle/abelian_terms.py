"""Oracle part c3 in un-enlarged form: the two-site term list for U(1)xU(1) and its loop nest
(TEST INFRASTRUCTURE ONLY).

oracle/abelian.py evaluates H_eff.psi on ENLARGED blocks (numeric Kronecker products).  This module
expands the same identities symbolically -- block operators stay symbols, site operators are explicit
4x4 matrices -- into the term list of Appendix A3 "Two-site H_eff",

    H_eff = sum  c * O_L (x) E[s1',s1] (x) E[s2',s2] (x) O_R        (left-to-right order),

and applies it with the element formula of A5 (fermion sign from the block labels).  It exists for two
reasons: it is the loop nest of SURVEY.md 8(c) c3 in the form whose flops F_alg counts (oracle/falg.py),
and it is a second, structurally different evaluation that the enlarged-block oracle pins.

Symbols: (kind, dag, i, k) over spin-orbitals i = 2p + sigma; kinds I, H, C (a+_i), S, A (i < k), B stored,
P, Q complements (A2).  dag marks the Hermitian conjugate; B+_il = B_li and Q+_il = Q_li carry no flag.

Pins (tests/test_oracle_terms.py): H_eff.psi from the term list equals oracle/abelian.py (itself pinned to
the brute-force projected Hamiltonian) on six small systems to 1e-12.
"""
import numpy as np

from .abelian import SITE_LABELS, _spin, psi_block_list
from .fock import site_creators

def sym_dq(sym):
    """(dN, d2Sz) of a block symbol."""
    kind, dag, i, k = sym
    if kind in ("I", "H"):
        q = (0, 0)
    elif kind == "C":
        q = (1, _spin(i))
    elif kind == "S":
        q = (-1, -_spin(i))
    elif kind == "A":
        q = (2, _spin(i) + _spin(k))
    elif kind == "B":
        q = (0, _spin(i) - _spin(k))
    elif kind == "P":
        q = (-2, -_spin(i) - _spin(k))
    elif kind == "Q":
        q = (0, _spin(k) - _spin(i))
    else:
        raise KeyError(kind)
    return (-q[0], -q[1]) if dag else q


def sym_dagger(sym):
    kind, dag, i, k = sym
    if kind in ("I", "H"):
        return sym
    if kind in ("B", "Q"):                   # (a+_i a_l)+ = a+_l a_i;  (Q_il)+ = Q_li
        return (kind, 0, k, i)
    return (kind, 1 - dag, i, k)


class Fac:
    """A factor: linear combination of block symbols, or an explicit 4x4 site matrix."""

    def __init__(self, lc=None, m=None):
        self.lc, self.m = lc, m

    @property
    def is_site(self):
        return self.m is not None

    def dagger(self):
        if self.is_site:
            return Fac(m=self.m.T.copy())
        return Fac(lc=[(sym_dagger(s), c) for s, c in self.lc])


class SitePart:
    """One orbital p: every operator evaluated from its Appendix-A2 definition with 4x4 matrices."""
    is_site = True

    def __init__(self, t, v, p):
        self.t, self.v = t, v
        self.orbs = [2 * p, 2 * p + 1]
        cu, cd = site_creators()
        self.c = {self.orbs[0]: cu, self.orbs[1]: cd}
        self.a = {i: m.T for i, m in self.c.items()}

    def op(self, kind, i=-1, k=-1):
        t, v, c, a, orbs = self.t, self.v, self.c, self.a, self.orbs
        M = np.zeros((4, 4))
        if kind == "I":
            M = np.eye(4)
        elif kind == "C":
            M = c[i]
        elif kind == "A":
            M = c[i] @ c[k]
        elif kind == "B":
            M = c[i] @ a[k]
        elif kind == "H":
            for x in orbs:
                for y in orbs:
                    M = M + t[x, y] * c[x] @ a[y]
                    for z in orbs:
                        for w in orbs:
                            M = M + 0.5 * v[x, y, z, w] * c[x] @ c[z] @ a[w] @ a[y]
        elif kind == "S":                    # S_x = 1/2 sum_j t_xj a_j + sum_jkl v_xjkl a+_k a_l a_j
            for j in orbs:
                M = M + 0.5 * t[i, j] * a[j]
                for kk in orbs:
                    for l in orbs:
                        M = M + v[i, j, kk, l] * c[kk] @ a[l] @ a[j]
        elif kind == "P":                    # P_ik = sum_jl v_ijkl a_l a_j
            for j in orbs:
                for l in orbs:
                    M = M + v[i, j, k, l] * a[l] @ a[j]
        elif kind == "Q":                    # Q_il = sum_kj (v_ilkj - v_ijkl) a+_k a_j
            for kk in orbs:
                for j in orbs:
                    M = M + (v[i, k, kk, j] - v[i, j, kk, k]) * c[kk] @ a[j]
        else:
            raise KeyError(kind)
        return Fac(m=M) if np.any(M != 0.0) else None


class BlockPart:
    """A renormalized block: answers with symbols of its normal set and of the complements (A2)."""
    is_site = False

    def __init__(self, orbs):
        self.orbs = sorted(orbs)

    def op(self, kind, i=-1, k=-1):
        one = lambda sym, c=1.0: Fac(lc=[(sym, c)])
        if kind == "I":
            return one(("I", 0, -1, -1))
        if not self.orbs:
            return None
        if kind == "H":
            return one(("H", 0, -1, -1))
        if kind == "C":
            return one(("C", 0, i, -1))
        if kind == "S":
            return one(("S", 0, i, -1))
        if kind in ("A", "P"):               # A_ik = -A_ki, P_ik = -P_ki
            if i == k or (kind == "P" and len(self.orbs) < 2):
                return None
            return one((kind, 0, i, k)) if i < k else one((kind, 0, k, i), -1.0)
        if kind in ("B", "Q"):
            return one((kind, 0, i, k))
        raise KeyError(kind)


class Op2:
    """Operator on X u Y (one of them a site): {symbol: 4x4 matrix}, in left-to-right order."""

    def __init__(self):
        self.e = {}

    def add(self, sym, m, coef):
        if coef != 0.0:
            self.e[sym] = self.e.get(sym, 0.0) + coef * m

    def dagger(self):
        """(X Y)+ = Y+ X+ = (-1)^{pi_X pi_Y} X+ Y+, the parity of the site factor read per element."""
        out = Op2()
        n = [0, 1, 1, 2]
        for sym, m in self.e.items():
            pis = sym_dq(sym)[0] & 1
            t = np.zeros((4, 4))
            for a in range(4):
                for b in range(4):
                    if m[a, b] != 0.0:
                        t[b, a] = -m[a, b] if (pis and ((n[a] - n[b]) & 1)) else m[a, b]
            out.add(sym_dagger(sym), t, 1.0)
        return out


def cut_cross_terms(opX, opY, orbsX, orbsY, normal_on_x, emit):
    """Cross terms of the cut identity (A2) for X | Y, each in left-to-right order with its reorder sign;
    emit(coef, x, y, hc) adds coef x (x) y (and its Hermitian conjugate when hc)."""
    for i in orbsY:                          # a+_i S^X_i + h.c. = -S^X_i a+_i + h.c.
        s, c = opX("S", i), opY("C", i)
        if s is not None and c is not None:
            emit(-1.0, s, c, True)
    for i in orbsX:                          # a+_i S^Y_i + h.c.
        c, s = opX("C", i), opY("S", i)
        if s is not None and c is not None:
            emit(1.0, c, s, True)
    opN, opC, orbsN = (opX, opY, orbsX) if normal_on_x else (opY, opX, orbsY)
    put = (lambda w, n, c, hc: emit(w, n, c, hc)) if normal_on_x else (lambda w, n, c, hc: emit(w, c, n, hc))
    for a, i in enumerate(orbsN):
        for k in orbsN[a + 1:]:              # 1/2 sum_{ik} (A_ik P_ik + h.c.) = sum_{i<k}; even operators commute
            an, pc = opN("A", i, k), opC("P", i, k)
            if an is not None and pc is not None:
                put(1.0, an, pc, True)
    for i in orbsN:
        for l in orbsN:
            bn, qc = opN("B", i, l), opC("Q", i, l)
            if bn is not None and qc is not None:
                put(1.0, bn, qc, False)


class Composite:
    """R = X u Y, X left of Y, exactly one of them a site; blocking rules of Appendix A3."""

    def __init__(self, X, Y, v):
        self.X, self.Y, self.v = X, Y, v
        self.orbs = sorted(X.orbs + Y.orbs)

    def _tensor(self, out, x, y, coef):
        if x is None or y is None:
            return
        blk, site = (x, y) if y.is_site else (y, x)
        for sym, c in blk.lc:
            out.add(sym, site.m, coef * c)

    def op(self, kind, i=-1, k=-1):
        X, Y, v, T = self.X, self.Y, self.v, self._tensor
        IX, IY = X.op("I"), Y.op("I")
        inX = lambda p: p in X.orbs
        cre = lambda P, p: P.op("C", p)
        ann = lambda P, p: (lambda f: None if f is None else f.dagger())(P.op("C", p))
        out = Op2()
        if kind == "I":
            T(out, IX, IY, 1.0)
        elif kind == "C":
            T(out, cre(X, i), IY, 1.0) if inX(i) else T(out, IX, cre(Y, i), 1.0)
        elif kind == "A":
            if inX(i) and inX(k):
                T(out, X.op("A", i, k), IY, 1.0)
            elif not inX(i) and not inX(k):
                T(out, IX, Y.op("A", i, k), 1.0)
            elif inX(i):
                T(out, cre(X, i), cre(Y, k), 1.0)
            else:
                T(out, cre(X, k), cre(Y, i), -1.0)          # a+_i a+_k = -a+_k a+_i
        elif kind == "B":
            l = k
            if inX(i) and inX(l):
                T(out, X.op("B", i, l), IY, 1.0)
            elif not inX(i) and not inX(l):
                T(out, IX, Y.op("B", i, l), 1.0)
            elif inX(i):
                T(out, cre(X, i), ann(Y, l), 1.0)
            else:
                T(out, ann(X, l), cre(Y, i), -1.0)          # a+_i a_l = -a_l a+_i
        elif kind == "S":
            x = i
            T(out, X.op("S", x), IY, 1.0)
            T(out, IX, Y.op("S", x), 1.0)
            for j in Y.orbs:
                T(out, X.op("Q", x, j), ann(Y, j), 1.0)     # Q^X_xj a_j
                T(out, X.op("P", x, j), cre(Y, j), 1.0)     # a+_j P^X_xj
            for j in X.orbs:
                T(out, ann(X, j), Y.op("Q", x, j), 1.0)     # Q^Y_xj a_j
                T(out, cre(X, j), Y.op("P", x, j), 1.0)     # a+_j P^Y_xj
        elif kind == "P":
            T(out, X.op("P", i, k), IY, 1.0)
            T(out, IX, Y.op("P", i, k), 1.0)
            for j in X.orbs:
                for l in Y.orbs:
                    w = v[i, j, k, l] - v[i, l, k, j]
                    if w != 0.0:
                        T(out, ann(X, j), ann(Y, l), -w)    # a_l a_j = -a_j a_l
        elif kind == "Q":
            l = k
            T(out, X.op("Q", i, l), IY, 1.0)
            T(out, IX, Y.op("Q", i, l), 1.0)
            for kk in X.orbs:
                for j in Y.orbs:
                    w1 = v[i, l, kk, j] - v[i, j, kk, l]
                    w2 = v[i, l, j, kk] - v[i, kk, j, l]
                    if w1 != 0.0:
                        T(out, cre(X, kk), ann(Y, j), w1)   # a+_k a_j
                    if w2 != 0.0:
                        T(out, ann(X, kk), cre(Y, j), -w2)  # a+_j a_k = -a_k a+_j
        elif kind == "H":
            T(out, X.op("H"), IY, 1.0)
            T(out, IX, Y.op("H"), 1.0)

            def emit(coef, x, y, hc):
                T(out, x, y, coef)
                if hc:                                      # (x y)+ = (-1)^{pi_x pi_y} x+ y+, pi_x = pi_y here
                    blk = y if x.is_site else x
                    par = sym_dq(blk.lc[0][0])[0] & 1
                    T(out, x.dagger(), y.dagger(), -coef if par else coef)
            cut_cross_terms(X.op, Y.op, X.orbs, Y.orbs, X.is_site, emit)
        else:
            raise KeyError(kind)
        return out if out.e else None


def two_site_terms(t, v, orbsL, p1, p2, orbsR, normal_on="A"):
    """{(symL, symR, s1', s1, s2', s2): c} of the two-site H_eff: cut identity on A = (L, s1) | B = (s2, R),
    every A-side and B-side operator expanded by the blocking rules (A3 "Two-site H_eff")."""
    A = Composite(BlockPart(orbsL), SitePart(t, v, p1), v)
    B = Composite(SitePart(t, v, p2), BlockPart(orbsR), v)
    terms = {}

    def product(coef, a, b):
        for sa, ma in a.e.items():
            for sb, mb in b.e.items():
                for s1p, s1 in zip(*np.nonzero(ma)):
                    for s2p, s2 in zip(*np.nonzero(mb)):
                        key = (sa, sb, int(s1p), int(s1), int(s2p), int(s2))
                        terms[key] = terms.get(key, 0.0) + coef * ma[s1p, s1] * mb[s2p, s2]

    def emit(coef, a, b, hc):
        product(coef, a, b)
        if hc:                                              # (a b)+ = (-1)^{pi_a pi_b} a+ b+, pi_a = pi_b here
            sym, m = next(iter(a.e.items()))
            sp, s = (int(x[0]) for x in np.nonzero(m))
            par = (sym_dq(sym)[0] + SITE_LABELS[sp][0] - SITE_LABELS[s][0]) & 1
            product(-coef if par else coef, a.dagger(), b.dagger())

    product(1.0, A.op("H"), B.op("I"))
    product(1.0, A.op("I"), B.op("H"))
    cut_cross_terms(A.op, B.op, A.orbs, B.orbs, normal_on == "A", emit)
    return {k: c for k, c in terms.items() if c != 0.0}


def block_of(blk, sym, ibra, iket):
    """Numeric block <ibra|sym|iket> from a Block of oracle/abelian.py (stored normal set; P, Q from A2)."""
    kind, dag, i, k = sym
    if kind == "I":
        return np.eye(blk.basis.dims[ibra]) if ibra == iket else None
    key = {"H": ("H",), "C": ("C", i), "S": ("S", i), "A": ("A", i, k), "B": ("B", i, k), "P": ("P", i, k), "Q": ("Q", i, k)}[kind]
    op = blk.op(*key)
    if dag:
        op = op.dagger()
    return op.blocks.get((ibra, iket))


def apply_terms(terms, Lblk, Rblk, N, twoSz, psi, outputs=None):
    """psi' = H_eff psi by the element formula of A5, one (term, input block) at a time:
    psi'[l',s1',s2',r'] += c (-1)^{N_l(pi1+pi2+piR) + N_s1(pi2+piR) + N_s2 piR} O_L[l',l] psi[l,s1,s2,r] O_R[r',r]."""
    tabL = [(q[0], q[1], d, 0) for q, d in zip(Lblk.basis.labels, Lblk.basis.dims)]
    tabR = [(q[0], q[1], d, 0) for q, d in zip(Rblk.basis.labels, Rblk.basis.dims)]
    blocks, n = psi_block_list(tabL, tabR, N, twoSz)
    index = {tuple(int(x) for x in b[:4]): m for m, b in enumerate(blocks)}
    y = np.zeros(n)
    nsite = [q[0] for q in SITE_LABELS]
    for (symL, symR, s1p, s1, s2p, s2), c in terms.items():
        dqL, dqR = sym_dq(symL), sym_dq(symR)
        pi1, pi2, piR = (nsite[s1p] - nsite[s1]) & 1, (nsite[s2p] - nsite[s2]) & 1, dqR[0] & 1
        for (iL, a, b, iR, dL, dR, off) in blocks:
            if a != s1 or b != s2:
                continue
            qL, qR = Lblk.basis.labels[iL], Rblk.basis.labels[iR]
            iLp = Lblk.basis.index.get((qL[0] + dqL[0], qL[1] + dqL[1]))
            iRp = Rblk.basis.index.get((qR[0] + dqR[0], qR[1] + dqR[1]))
            if iLp is None or iRp is None:
                continue
            o = index.get((iLp, s1p, s2p, iRp))
            if o is None or (outputs is not None and o not in outputs):
                continue
            OL, OR = block_of(Lblk, symL, iLp, iL), block_of(Rblk, symR, iRp, iR)
            if OL is None or OR is None:
                continue
            e = qL[0] * (pi1 + pi2 + piR) + nsite[s1] * (pi2 + piR) + nsite[s2] * piR
            bo = blocks[o]
            x = psi[off: off + dL * dR].reshape(dL, dR)
            y[bo[6]: bo[6] + bo[4] * bo[5]] += ((-c if e & 1 else c) * (OL @ x @ OR.T)).reshape(-1)
    return y
