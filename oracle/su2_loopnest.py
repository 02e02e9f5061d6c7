"""Oracle part c4 (and c5 in reduced form): loop-nest H_eff.psi and renormalization for SU(2).
TEST INFRASTRUCTURE ONLY (Appendix A4, A5; reading s15).

Where oracle/su2.py DEFINES the spin-adapted result by Clebsch-Gordan expansion into the U(1)xU(1)
oracle (and therefore cannot reach D > ~300), this module computes the same result directly on reduced
matrix elements, in the paper's "fixed number of SU(2) multiplets" representation, so that
sampled output blocks of the full-size configurations can be checked.  It follows Appendix A4/A5 in
their order and notation:

  1. site tensors: explicit spherical components on the 4-dimensional site space, reduced by the
     Wigner-Eckart theorem with a bare Clebsch-Gordan factor (A4 "Wigner-Eckart convention");
  2. block operators are SYMBOLS (kind, tilde, rank, indices) of the stored normal set
     {H, a+_p, S~_x, A^k_pr, B^k_ps} and of the complements P~^k_pr, Q~^k_ps (A4 "Spin-adapted cut identity");
  3. blocking rules for R = X u Y (A4 "SU(2) blocking of the complements"), written as in the appendix;
     a product written Y-first is brought to X-first order by the swap rule;
  4. the two-site term list: the cut identity on A = (L, s1) | B = (s2, R), every A-side and B-side
     operator expanded by 3 (A3 "Two-site H_eff");
  5. the element formula of A5:  psi'[b'] += c F6 F9_A F9_B  O_L[qL',qL] psi[b] O_R[qR',qR]^T  with the
     9j product rule of A4 and the oracle's own Wigner symbols (oracle/wigner.py);
  6. renormalization (A5 last formula): O'[a',a] = sum f X[(qL',s')->a']^T O_L[qL',qL] X[(qL,s)->a].

Numeric operator blocks come from a callback `get_stored(kind, k2, i, k, ibra, iket)`: the oracle's own
renormalized blocks for small systems, or blocks downloaded from the device (`dmrg_op_export_block`) for
the sampled checks at full size, so that errors do not chain.  A matmul is the only
library primitive used; there is no blocking, stacking or two-stage reordering.

All spins are DOUBLED integers.  Site multiplet index s = 0, 1, 2 = particle number (spins 0, 1/2, 0).

Pins (tests/test_oracle_su2_loopnest.py, -m "not gpu"): every renormalized reduced operator equals the
Wigner-Eckart projection of the expanded U(1)xU(1) oracle operator, and H_eff.psi equals the expansion
oracle (oracle/su2.py, itself pinned to the brute-force projected Hamiltonian) on eight small systems
(singlet to quartet, odd N, empty block) to 1e-12; the result does not depend on which side of the cut
carries the normal pair operators; the tilde/adjoint rules against explicit components.
"""
from math import sqrt

import numpy as np

from .fock import site_creators
from .su2 import SITE_J2, SITE_N, cg, psi_blocks, site_state_of
from .wigner import triangle, wigner_9j

# ----------------------------------------------------------------------------- symbols
# A block-operator symbol is (kind, tilde, k2, i, k):
#   'I' identity, 'H' block Hamiltonian                           rank 0
#   'C' a+_p (p inside), 'S' the stored S~_x (x outside)          rank 1/2
#   'A' A^k_pr = [a+_p x a+_r]^k (p <= r), 'B' B^k_ps = [a+_p x a~_s]^k       rank k
#   'P' P~^k_pr, 'Q' Q~^k_ps  complements (lincombs of stored A~, B; A4)      rank k
# tilde = 1 marks T~ of the symbol, T~_m = (-1)^{k-m} (T_{-m})^+ (A4 "Adjoint rule").
_DN = {"I": 0, "H": 0, "C": 1, "S": -1, "A": 2, "B": 0, "P": -2, "Q": 0}


def sym_dN(sym):
    return -_DN[sym[0]] if sym[1] else _DN[sym[0]]


def sym_parity(sym):
    return _DN[sym[0]] & 1


def sym_tilde(sym):
    """(symbol, coefficient) of the tilde of a symbol.  T~~ = (-1)^{2k} T; B~^k_ps = (-1)^k B^k_sp and the
    same for Q~ (A4 identities); I and H are self-tilde (hermitian scalars)."""
    kind, til, k2, i, k = sym
    if kind in ("I", "H"):
        return sym, 1.0
    if kind in ("B", "Q"):
        return (kind, 0, k2, k, i), (-1.0 if k2 == 2 else 1.0)
    if til == 0:
        return (kind, 1, k2, i, k), 1.0
    return (kind, 0, k2, i, k), (-1.0 if k2 & 1 else 1.0)


def reduced_tilde(S_bra, S_ket, k2):
    """<j||T~||j'> = (-1)^{j'-j+k} sqrt((2j'+1)/(2j+1)) <j'||T||j>  (A4 "Adjoint rule"); j = S_bra, j' = S_ket."""
    e = (S_ket - S_bra + k2) // 2
    return (-1.0 if e & 1 else 1.0) * sqrt((S_ket + 1.0) / (S_bra + 1.0))


def f9(j1, j2, J, k1, k2, K, j1p, j2p, Jp):
    """sqrt((2K+1)(2J+1)(2j1'+1)(2j2'+1)) {j1 j2 J; k1 k2 K; j1' j2' J'}: the 9j factor of the product rule."""
    w = wigner_9j(j1, j2, J, k1, k2, K, j1p, j2p, Jp)
    return 0.0 if w == 0.0 else sqrt((K + 1.0) * (J + 1.0) * (j1p + 1.0) * (j2p + 1.0)) * w


# ----------------------------------------------------------------------------- factors
class Fac:
    """One factor of a product: a linear combination of block symbols (all of one rank and parity) or a
    site tensor given by its reduced 3x3 matrix m[s', s]."""
    __slots__ = ("is_site", "k2", "par", "lc", "m")

    def __init__(self, is_site, k2, par, lc=None, m=None):
        self.is_site, self.k2, self.par, self.lc, self.m = is_site, k2, par, lc, m

    def tilde(self):
        if self.is_site:
            m = np.zeros((3, 3))
            for a in range(3):
                for b in range(3):
                    if self.m[b, a] != 0.0:
                        m[a, b] = reduced_tilde(SITE_J2[a], SITE_J2[b], self.k2) * self.m[b, a]
            return Fac(True, self.k2, self.par, m=m)
        lc = []
        for sym, c in self.lc:
            t, ct = sym_tilde(sym)
            lc.append((t, c * ct))
        return Fac(False, self.k2, self.par, lc=lc)


# ----------------------------------------------------------------------------- site tensors
def _tilde_components(comps, k2):
    return {m: (-1.0) ** ((k2 - m) // 2) * comps[-m].T for m in comps}


def _couple_components(a, ka, b, kb, K):
    """[a x b]^K on the same site: sum_q <ka q1; kb q2|K Q> a_q1 b_q2."""
    out = {}
    for Q in range(-K, K + 1, 2):
        M = np.zeros((4, 4))
        for q1, A in a.items():
            q2 = Q - q1
            if q2 in b:
                M = M + cg(ka, q1, kb, q2, K, Q) * (A @ b[q2])
        out[Q] = M
    return out


def _reduce_site(comps, k2):
    """Reduced 3x3 matrix of a site tensor from its spherical components:
    <s' m'|T_q|s m> = <j m; k q|j' m'> <s'||T||s>."""
    red = np.zeros((3, 3))
    for sp in range(3):
        for s in range(3):
            vals = []
            for q, M in comps.items():
                for m in range(-SITE_J2[s], SITE_J2[s] + 1, 2):
                    mp = m + q
                    if abs(mp) > SITE_J2[sp] or (SITE_J2[sp] + mp) % 2:
                        continue
                    c = cg(SITE_J2[s], m, k2, q, SITE_J2[sp], mp)
                    x = M[site_state_of(sp, mp), site_state_of(s, m)]
                    if abs(c) < 1e-14:
                        assert abs(x) < 1e-12, "site operator is not a tensor operator"
                        continue
                    vals.append(x / c)
            if vals:
                assert max(vals) - min(vals) < 1e-12, "site operator violates the Wigner-Eckart theorem"
                red[sp, s] = vals[0]
    return red


class SitePart:
    """One orbital t: every operator from its definition (A4) with explicit 4x4 components."""
    is_site = True

    def __init__(self, h, V, t):
        self.h, self.V, self.t = h, V, t
        self.orbs = [t]
        cu, cd = site_creators()
        self.cre = {1: cu, -1: cd}                                   # a+_q, q = +-1/2
        self.ann = _tilde_components(self.cre, 1)                    # a~_{+1/2} = a_dn, a~_{-1/2} = -a_up
        self.n = cu @ cu.T + cd @ cd.T
        self._memo = {}

    def op(self, kind, k2=0, i=-1, k=-1):
        key = (kind, k2, i, k)
        if key not in self._memo:
            self._memo[key] = self._op(kind, k2, i, k)
        return self._memo[key]

    def _op(self, kind, k2, i, k):
        h, V, t = self.h, self.V, self.t
        au, ad = self.cre[1].T, self.cre[-1].T
        if kind == "I":
            comps, par = {0: np.eye(4)}, 0
        elif kind == "H":      # sum_s h_tt a+a + 1/2 (tt|tt) sum_{s,s'} a+_s a+_s' a_s' a_s = h_tt n + 1/2 (tt|tt) n (n - 1)
            comps, par = {0: h[t, t] * self.n + 0.5 * V[t, t, t, t] * (self.n @ self.n - self.n)}, 0
        elif kind == "C":
            comps, par = self.cre, 1
        elif kind == "S":      # S_{x s} = 1/2 h_xt a_ts + (xt|tt) n_t a_ts;  S~_m = (-1)^{1/2-m} S_{x,-m}
            x = i
            Su = 0.5 * h[x, t] * au + V[x, t, t, t] * (self.n @ au)
            Sd = 0.5 * h[x, t] * ad + V[x, t, t, t] * (self.n @ ad)
            comps, par = {1: Sd, -1: -Su}, 1
        elif kind == "A":
            comps, par = _couple_components(self.cre, 1, self.cre, 1, k2), 0
        elif kind == "B":
            comps, par = _couple_components(self.cre, 1, self.ann, 1, k2), 0
        elif kind == "P":      # P~^k_pr = (pt|rt) A~^k_tt
            a = _tilde_components(_couple_components(self.cre, 1, self.cre, 1, k2), k2)
            comps, par = {q: V[i, t, k, t] * M for q, M in a.items()}, 0
        elif kind == "Q":      # Q~^0_ps = [2(ps|tt) - (pt|ts)] B^0_tt,  Q~^1_ps = (pt|ts) B^1_tt
            b = _couple_components(self.cre, 1, self.ann, 1, k2)
            w = 2.0 * V[i, k, t, t] - V[i, t, t, k] if k2 == 0 else V[i, t, t, k]
            comps, par = {q: w * M for q, M in b.items()}, 0
        else:
            raise KeyError(kind)
        m = _reduce_site(comps, k2)
        return Fac(True, k2, par, m=m) if np.any(m != 0.0) else None


class BlockPart:
    """A renormalized block over the spatial orbitals `orbs`: answers with symbols (A4; the stored normal
    set and the complements).  An empty block (vacuum) has only the identity."""
    is_site = False

    def __init__(self, orbs):
        self.orbs = sorted(orbs)
        self.inside = set(self.orbs)

    def op(self, kind, k2=0, i=-1, k=-1):
        n = len(self.orbs)
        one = lambda sym, c=1.0: Fac(False, sym[2], sym_parity(sym), lc=[(sym, c)])
        sg = -1.0 if k2 == 2 else 1.0                                  # (-1)^k
        if kind == "I":
            return one(("I", 0, 0, -1, -1))
        if n == 0:
            return None
        if kind == "H":
            return one(("H", 0, 0, -1, -1))
        if kind == "C":
            return one(("C", 0, 1, i, -1)) if i in self.inside else None
        if kind == "S":
            return one(("S", 0, 1, i, -1))
        if kind in ("A", "P"):      # A^0_pr = A^0_rp, A^1_pr = -A^1_rp, A^1_pp = 0; the same for P~ (A4 identities)
            if i == k:
                return one((kind, 0, 0, i, k)) if k2 == 0 else None
            if n < 2 and kind == "P" and k2 == 2:
                return None                                            # no stored A^1 to build it from
            return one((kind, 0, k2, i, k)) if i < k else one((kind, 0, k2, k, i), sg)
        if kind in ("B", "Q"):
            return one((kind, 0, k2, i, k))
        raise KeyError(kind)


# ----------------------------------------------------------------------------- composites
class Entry:
    """coef-free piece [sym^kB x site^kS]^K (block-left) or [site^kS x sym^kB]^K (site-left); the reduced
    site matrix m carries the coefficient."""
    __slots__ = ("sym", "kB", "kS", "K", "parS", "m")

    def __init__(self, sym, kB, kS, K, parS, m):
        self.sym, self.kB, self.kS, self.K, self.parS, self.m = sym, kB, kS, K, parS, m


class Op2:
    """Operator on a composite X u Y: sum of entries, all of rank K."""

    def __init__(self, K=0):
        self.K = K
        self.e = {}

    def add(self, sym, kB, kS, K, parS, m, coef):
        if coef == 0.0:
            return
        self.K = K
        key = (sym, kS, K)
        if key in self.e:
            self.e[key].m = self.e[key].m + coef * m
        else:
            self.e[key] = Entry(sym, kB, kS, K, parS, coef * m)

    @property
    def par(self):
        for en in self.e.values():
            return (sym_parity(en.sym) + en.parS) & 1
        return 0

    def entries(self):
        return list(self.e.values())

    def tilde(self):
        """tilde([T x U]^K) = (-1)^{pi_T pi_U} [T~ x U~]^K for operators on different parts."""
        out = Op2(self.K)
        for en in self.e.values():
            t, ct = sym_tilde(en.sym)
            sgn = -1.0 if (sym_parity(en.sym) and en.parS) else 1.0
            mt = Fac(True, en.kS, en.parS, m=en.m).tilde().m
            out.add(t, en.kB, en.kS, en.K, en.parS, mt, ct * sgn)
        return out


def swap_factor(k1, k2, K, par1, par2):
    """[T^k1 x U^k2]^K = (-1)^{k1+k2-K} (-1)^{pi_T pi_U} [U^k2 x T^k1]^K (A4 "Swap rule")."""
    s = -1.0 if ((k1 + k2 - K) // 2) & 1 else 1.0
    return -s if (par1 and par2) else s


def cut_cross_terms(opX, opY, orbsX, orbsY, normal_on_x, pair):
    """Cross terms of the spin-adapted cut identity for X | Y (A4):
        - sqrt2 sum_{x in Y} ([a+_x x S~^X_x]^0 + h.c.) - sqrt2 sum_{y in X} ([a+_y x S~^Y_y]^0 + h.c.)
        + sum_{p<=r in N} sum_k w sqrt(2k+1) ([A^k_pr x P~^k_pr]^0 + h.c.),  w = 1 (p < r), 1/2 (p = r; k = 0 only)
        + sum_{p,s in N} ([B^0_ps x Q~^0_ps]^0 + sqrt3 [B^1_ps x Q~^1_ps]^0),
    N = the side carrying the normal pair operators, the complements summed over the other side.
    opX / opY(kind, k2, i, k) give the operators of the two sides (None = zero);
    pair(first, second, coef, first_on, hc) accumulates coef [first x second]^0 (+ its h.c. when hc)."""
    r2, r3 = sqrt(2.0), sqrt(3.0)
    for x in orbsY:
        c, s = opY("C", 1, x), opX("S", 1, x)
        if c is not None and s is not None:
            pair(c, s, -r2, "Y", True)                   # [a+_x x S~^X_x]^0: the first factor lives on Y
    for y in orbsX:
        c, s = opX("C", 1, y), opY("S", 1, y)
        if c is not None and s is not None:
            pair(c, s, -r2, "X", True)
    opN, opC, orbsN, side = (opX, opY, orbsX, "X") if normal_on_x else (opY, opX, orbsY, "Y")
    for a, p in enumerate(orbsN):
        for r in orbsN[a:]:
            for k2 in (0, 2):
                if p == r and k2 == 2:
                    continue
                an, pc = opN("A", k2, p, r), opC("P", k2, p, r)
                if an is not None and pc is not None:
                    pair(an, pc, (0.5 if p == r else 1.0) * sqrt(k2 + 1.0), side, True)
    for p in orbsN:
        for s in orbsN:
            for k2, w in ((0, 1.0), (2, r3)):
                bn, qc = opN("B", k2, p, s), opC("Q", k2, p, s)
                if bn is not None and qc is not None:
                    pair(bn, qc, w, side, False)


class Composite:
    """R = X u Y with X left of Y, exactly one of them a site; operators by the blocking rules of A4."""

    def __init__(self, X, Y, V):
        self.X, self.Y, self.V = X, Y, V
        self.orbs = sorted(X.orbs + Y.orbs)
        self.site_is_right = Y.is_site

    def _couple(self, out, first, second, K, coef, first_on="X"):
        """out += coef [first x second]^K; a product written Y-first is swapped to X-first order."""
        if first is None or second is None or not triangle(first.k2, second.k2, K):
            return
        if first_on == "Y":
            coef = coef * swap_factor(first.k2, second.k2, K, first.par, second.par)
            first, second = second, first
        blk, site = (first, second) if second.is_site else (second, first)
        assert site.is_site and not blk.is_site
        for sym, c in blk.lc:
            out.add(sym, blk.k2, site.k2, K, site.par, site.m, coef * c)

    def op(self, kind, k2=0, i=-1, k=-1):
        X, Y, V, cp = self.X, self.Y, self.V, self._couple
        IX, IY = X.op("I"), Y.op("I")
        inX = lambda p: p in X.orbs
        sg = -1.0 if k2 == 2 else 1.0
        cre = lambda P, p: P.op("C", 1, p)
        ann = lambda P, p: (lambda f: None if f is None else f.tilde())(P.op("C", 1, p))
        out = Op2(k2)
        if kind == "I":
            cp(out, IX, IY, 0, 1.0)
        elif kind == "C":
            if inX(i):
                cp(out, cre(X, i), IY, 1, 1.0)
            else:
                cp(out, IX, cre(Y, i), 1, 1.0)
        elif kind == "A":          # A^k_pr = [a+_p x a+_r]^k
            p, r = i, k
            if inX(p) and inX(r):
                cp(out, X.op("A", k2, p, r), IY, k2, 1.0)
            elif not inX(p) and not inX(r):
                cp(out, IX, Y.op("A", k2, p, r), k2, 1.0)
            else:
                cp(out, cre(X if inX(p) else Y, p), cre(X if inX(r) else Y, r), k2, 1.0, "X" if inX(p) else "Y")
        elif kind == "B":          # B^k_ps = [a+_p x a~_s]^k
            p, s = i, k
            if inX(p) and inX(s):
                cp(out, X.op("B", k2, p, s), IY, k2, 1.0)
            elif not inX(p) and not inX(s):
                cp(out, IX, Y.op("B", k2, p, s), k2, 1.0)
            else:
                cp(out, cre(X if inX(p) else Y, p), ann(X if inX(s) else Y, s), k2, 1.0, "X" if inX(p) else "Y")
        elif kind == "S":          # A4: S~^R_x
            x = i
            c0, c1 = 1.0 / sqrt(2.0), sqrt(1.5)
            cp(out, X.op("S", 1, x), IY, 1, 1.0)
            cp(out, IX, Y.op("S", 1, x), 1, 1.0)
            for y in Y.orbs:
                cp(out, X.op("Q", 0, x, y), ann(Y, y), 1, -c0)
                cp(out, cre(Y, y), X.op("P", 0, x, y), 1, -c0, "Y")
                cp(out, X.op("Q", 2, x, y), ann(Y, y), 1, +c1)
                cp(out, cre(Y, y), X.op("P", 2, x, y), 1, -c1, "Y")
            for q in X.orbs:
                cp(out, ann(X, q), Y.op("Q", 0, x, q), 1, -c0)
                cp(out, cre(X, q), Y.op("P", 0, x, q), 1, -c0)
                cp(out, ann(X, q), Y.op("Q", 2, x, q), 1, -c1)
                cp(out, cre(X, q), Y.op("P", 2, x, q), 1, -c1)
        elif kind == "P":          # P~^{R,k}_pr = P~^X + P~^Y + sum_{q in X, s in Y} [(pq|rs) + (-1)^k (ps|rq)] A~^k_qs
            p, r = i, k
            cp(out, X.op("P", k2, p, r), IY, k2, 1.0)
            cp(out, IX, Y.op("P", k2, p, r), k2, 1.0)
            for q in X.orbs:
                for s in Y.orbs:
                    w = V[p, q, r, s] + sg * V[p, s, r, q]
                    cp(out, ann(X, q), ann(Y, s), k2, -w)              # A~^k_qs = -[a~_q x a~_s]^k
        elif kind == "Q":
            p, s = i, k
            cp(out, X.op("Q", k2, p, s), IY, k2, 1.0)
            cp(out, IX, Y.op("Q", k2, p, s), k2, 1.0)
            for q in X.orbs:
                for r in Y.orbs:
                    if k2 == 0:    # [2(ps|qr) - (pr|qs)] B^0_qr + [2(ps|rq) - (pq|rs)] B^0_rq,  B^0_rq = +[a~_q x a+_r]^0
                        cp(out, cre(X, q), ann(Y, r), 0, 2.0 * V[p, s, q, r] - V[p, r, q, s])
                        cp(out, ann(X, q), cre(Y, r), 0, 2.0 * V[p, s, r, q] - V[p, q, r, s])
                    else:          # (pr|qs) B^1_qr + (pq|rs) B^1_rq,  B^1_rq = -[a~_q x a+_r]^1
                        cp(out, cre(X, q), ann(Y, r), 2, V[p, r, q, s])
                        cp(out, ann(X, q), cre(Y, r), 2, -V[p, q, r, s])
        elif kind == "H":          # H^R = H^X + H^Y + cut identity on X | Y; the site carries the normal pairs
            cp(out, X.op("H"), IY, 0, 1.0)
            cp(out, IX, Y.op("H"), 0, 1.0)

            def pair(first, second, coef, first_on, hc):
                cp(out, first, second, 0, coef, first_on)
                if hc:             # ([T x U]^0)^+ = (-1)^{pi_T pi_U} [T~ x U~]^0, T on the left part
                    if first_on == "Y":
                        coef = coef * swap_factor(first.k2, second.k2, 0, first.par, second.par)
                        first, second = second, first
                    cp(out, first.tilde(), second.tilde(), 0, -coef if (first.par and second.par) else coef)
            cut_cross_terms(X.op, Y.op, X.orbs, Y.orbs, X.is_site, pair)
        else:
            raise KeyError(kind)
        return out if out.e else None


# ----------------------------------------------------------------------------- two-site term list
def cut_pairs(h, V, orbsL, t1, t2, orbsR, normal_on="A"):
    """The two-site Hamiltonian as scalar-coupled operator pairs: (A, B, [(coef, T_A, U_B)]) with
    H = sum coef [T_A^k x U_B^k]^0 in A-first order (A3 "Two-site H_eff": the cut identity of A4 on
    A = (L, s1) | B = (s2, R)); T_A and U_B are operators (Op2) on the composites A and B.
    normal_on: which side of the cut carries A^k, B^k ("A": DESIGN.md reading s5; "B": the mirror
    identity, used as a pin)."""
    A = Composite(BlockPart(orbsL), SitePart(h, V, t1), V)
    B = Composite(SitePart(h, V, t2), BlockPart(orbsR), V)
    pairs = []

    def pair(first, second, coef, first_on, hc):
        if first_on == "Y":        # written B-first: swap to A-first order
            coef = coef * swap_factor(first.K, second.K, 0, first.par, second.par)
            first, second = second, first
        pairs.append((coef, first, second))
        if hc:                     # ([T x U]^0)^+ = (-1)^{pi_T pi_U} [T~ x U~]^0
            pairs.append((-coef if (first.par and second.par) else coef, first.tilde(), second.tilde()))

    pairs.append((1.0, A.op("H"), B.op("I")))
    pairs.append((1.0, A.op("I"), B.op("H")))
    cut_cross_terms(A.op, B.op, A.orbs, B.orbs, normal_on == "A", pair)
    return A, B, pairs


def two_site_terms(h, V, orbsL, t1, t2, orbsR, normal_on="A"):
    """Elementary terms c [[O_L^kL x o1^k1]^kk x [o2^k2 x O_R^kR]^kk]^0 of the two-site H_eff: every operator
    of `cut_pairs` expanded into (block operator) x (site operator) pieces.  dict key -> c with
    key = (symL, symR, s1', s1, s2', s2, kL, k1, kk, k2, kR); c includes <s1'||o1||s1> <s2'||o2||s2>."""
    terms = {}
    for coef, a, b in cut_pairs(h, V, orbsL, t1, t2, orbsR, normal_on)[2]:
        for ea in a.entries():
            for eb in b.entries():
                if ea.K != eb.K:
                    continue
                for s1p, s1 in zip(*np.nonzero(ea.m)):
                    for s2p, s2 in zip(*np.nonzero(eb.m)):
                        key = (ea.sym, eb.sym, int(s1p), int(s1), int(s2p), int(s2), ea.kB, ea.kS, ea.K, eb.kS, eb.kB)
                        terms[key] = terms.get(key, 0.0) + coef * ea.m[s1p, s1] * eb.m[s2p, s2]
    return {k: c for k, c in terms.items() if c != 0.0}


# ----------------------------------------------------------------------------- numeric block operators
class BlockOps:
    """Reduced operator blocks <i_bra|| sym ||i_ket> of one renormalized block.  Stored operators come
    from `get_stored(kind, k2, i, k, ibra, iket)` (None = no such block); tildes and complements are
    formed here from their A4 definitions."""

    def __init__(self, table, orbs, V, get_stored):
        self.table = np.asarray(table, dtype=np.int64).reshape(-1, 4)
        self.orbs = sorted(orbs)
        self.V = V
        self.get_stored = get_stored
        self._cache = {}

    def allowed(self, sym, ibra, iket):
        (Nb, Sb), (Nk, Sk) = self.table[ibra][:2], self.table[iket][:2]
        return Nb - Nk == sym_dN(sym) and triangle(int(Sk), sym[2], int(Sb))

    def kets(self, sym, ibra):
        return [ik for ik in range(len(self.table)) if self.allowed(sym, ibra, ik)]

    def block(self, sym, ibra, iket):
        key = (sym, ibra, iket)
        if key not in self._cache:
            self._cache[key] = self._block(sym, ibra, iket) if self.allowed(sym, ibra, iket) else None
        return self._cache[key]

    def _block(self, sym, ibra, iket):
        kind, til, k2, i, k = sym
        V, tab = self.V, self.table
        if kind == "I":
            return np.eye(int(tab[ibra][2])) if ibra == iket else None
        if kind in ("H", "C", "S", "A", "B"):
            if til == 0:
                return self.get_stored(kind, k2, i, k, ibra, iket)
            m = self.get_stored(kind, k2, i, k, iket, ibra)           # <bra||T~||ket> from <ket||T||bra>
            return None if m is None else reduced_tilde(int(tab[ibra][1]), int(tab[iket][1]), k2) * m.T
        # complements: integral-weighted sums over the stored pair operators of this block (A4).  All complements
        # of one class and sector pair are formed together, as the one matrix product W . stack
        index, data = self._complements(kind, til, k2, ibra, iket)
        if data is None:
            return None
        if (i, k) not in index:
            raise KeyError(sym)
        return data[index[(i, k)]]

    def _complements(self, kind, til, k2, ibra, iket):
        """P~^k_pr (p <= r) or Q~^k_ps for every pair of orbitals outside this block, for one sector pair."""
        key = ("complements", kind, til, k2, ibra, iket)
        if key in self._cache:
            return self._cache[key]
        V = self.V
        L = V.shape[0]
        out = [x for x in range(L) if x not in set(self.orbs)]
        sg = -1.0 if k2 == 2 else 1.0
        if kind == "P":            # P~^k_pr = sum_{q,s} (pq|rs) A~^k_qs, A~^k_sq = (-1)^k A~^k_qs;  tilde: A~ -> A
            members, stack = self._stack("A", 1 - til, k2, ibra, iket)
            pairs = [(p, r) for a, p in enumerate(out) for r in out[a:] if not (p == r and k2 == 2)]
        elif kind == "Q":          # Q~^0_ps = sum [2(ps|qr) - (pr|qs)] B^0_qr,  Q~^1_ps = sum (pr|qs) B^1_qr
            assert til == 0
            members, stack = self._stack("B", 0, k2, ibra, iket)
            pairs = [(p, s) for p in out for s in out]
        else:
            raise KeyError(kind)
        if not members or not pairs:
            res = ({}, None)
        else:
            # W[(p, r), (q, s)]: rows = complements, columns = stored members (index arrays broadcast over V)
            P = np.array([x[0] for x in pairs])[:, None]
            R = np.array([x[1] for x in pairs])[:, None]
            Q = np.array([x[0] for x in members])[None, :]
            S = np.array([x[1] for x in members])[None, :]
            if kind == "P":        # q < s: (pq|rs) + (-1)^k (ps|rq);  q = s: (pq|rq)
                W = np.where(Q == S, V[P, Q, R, Q], V[P, Q, R, S] + sg * V[P, S, R, Q])
            elif k2 == 0:          # rows (p, s), columns (q, r): 2 (ps|qr) - (pr|qs)
                W = 2.0 * V[P, R, Q, S] - V[P, S, Q, R]
            else:                  # (pr|qs)
                W = V[P, S, Q, R]
            res = ({pr: n for n, pr in enumerate(pairs)}, np.tensordot(W, stack, 1))
        self._cache[key] = res
        return res

    def _stack(self, kind, til, k2, ibra, iket):
        """All stored pair operators (A^k_qs with q <= s, or B^k_qr) of this block that have a block for the
        sector pair, stacked: (member labels, array [n, d_bra, d_ket])."""
        key = ("stack", kind, til, k2, ibra, iket)
        if key not in self._cache:
            members, mats = [], []
            for a, q in enumerate(self.orbs):
                for s in (self.orbs[a:] if kind == "A" else self.orbs):
                    if kind == "A" and q == s and k2 == 2:
                        continue
                    m = self.block((kind, til, k2, q, s), ibra, iket)
                    if m is not None:
                        members.append((q, s))
                        mats.append(m)
            self._cache[key] = (members, np.stack(mats) if mats else None)
        return self._cache[key]


def dict_store(store):
    """get_stored callback over {(kind, k2, i, k): {(ibra, iket): matrix}}."""
    def get(kind, k2, i, k, ibra, iket):
        return store.get((kind, k2, i, k), {}).get((ibra, iket))
    return get


def vacuum_ops(V):
    return BlockOps([(0, 0, 1, 0)], [], V, dict_store({}))


def normal_set(orbs, L):
    """Targets (kind, k2, i, k) of the stored normal operator set of a block over `orbs` (A2, A4)."""
    orbs = sorted(orbs)
    out = [("H", 0, -1, -1)] + [("C", 1, p, -1) for p in orbs] + [("S", 1, x, -1) for x in range(L) if x not in orbs]
    for a, p in enumerate(orbs):
        for r in orbs[a:]:
            out.append(("A", 0, p, r))
            if r != p:
                out.append(("A", 2, p, r))
    for p in orbs:
        for s in orbs:
            out += [("B", 0, p, s), ("B", 2, p, s)]
    return out


# ----------------------------------------------------------------------------- renormalization (c5, reduced)
def renormalize_blocks(h, V, ops, t, iso_blocks, iso_data, new_table, site_is_right, targets, only=None):
    """A5 "Renormalization": O'[a',a] = sum_pieces sum_{(q',s'),(q,s)} f X[(q',s')->a']^T O[q',q] X[(q,s)->a] with
    f = <s'||o||s> * 9j product-rule factor * (-1)^{N_1 pi_U}.  Returns {target: {(a', a): matrix}}.
    only: optional set of (target, a', a) to compute (the sampled check at full size)."""
    new_table = np.asarray(new_table, dtype=np.int64).reshape(-1, 4)
    tab = ops.table
    blk, site = BlockPart(ops.orbs), SitePart(h, V, t)
    comp = Composite(blk, site, V) if site_is_right else Composite(site, blk, V)
    into = {}                                              # new sector -> [(i_prev, s, X)]
    for b in iso_blocks:
        ip, s, inext, rows, cols, off = (int(v) for v in b)
        into.setdefault(inext, []).append((ip, s, iso_data[off:off + rows * cols].reshape(rows, cols)))
    out = {}
    for tg in targets:
        kind, k2, i, k = tg
        o2 = comp.op(kind, k2, i, k)
        res = {}
        if o2 is not None:
            dN = _DN[kind]
            for ap in range(len(new_table)):
                for a in range(len(new_table)):
                    if only is not None and (tg, ap, a) not in only:
                        continue
                    (Np, Sp), (Nk, Sk) = new_table[ap][:2], new_table[a][:2]
                    if Np - Nk != dN or not triangle(int(Sk), k2, int(Sp)):
                        continue
                    acc = None
                    for en in o2.entries():
                        parB = sym_parity(en.sym)
                        for (ipp, sp, Xp) in into.get(ap, []):
                            for (ip, s, X) in into.get(a, []):
                                ms = en.m[sp, s]
                                if ms == 0.0:
                                    continue
                                O = ops.block(en.sym, ipp, ip)
                                if O is None:
                                    continue
                                jb, jbp = int(tab[ip][1]), int(tab[ipp][1])
                                if site_is_right:          # subsystem 1 = block, 2 = site
                                    f = f9(jb, SITE_J2[s], int(Sk), en.kB, en.kS, en.K, jbp, SITE_J2[sp], int(Sp))
                                    odd = int(tab[ip][0]) & en.parS
                                else:                      # subsystem 1 = site, 2 = block
                                    f = f9(SITE_J2[s], jb, int(Sk), en.kS, en.kB, en.K, SITE_J2[sp], jbp, int(Sp))
                                    odd = SITE_N[s] & parB
                                if f == 0.0:
                                    continue
                                val = ((-f if odd & 1 else f) * ms) * (Xp.T @ O @ X)
                                acc = val if acc is None else acc + val
                    if acc is not None:
                        res[(ap, a)] = acc
        out[tg] = res
    return out


def renormalize(h, V, ops, t, iso_blocks, iso_data, new_table, site_is_right, L):
    """The next block's BlockOps (whole normal set), for the oracle's own environments on small systems."""
    orbs = sorted(ops.orbs + [t])
    store = renormalize_blocks(h, V, ops, t, iso_blocks, iso_data, new_table, site_is_right, normal_set(orbs, L))
    return BlockOps(new_table, orbs, V, dict_store(store))


def build_block(h, V, tables, isos, sites, site_is_right):
    ops = vacuum_ops(V)
    for m, p in enumerate(sites):
        ops = renormalize(h, V, ops, p, isos[m][0], isos[m][1], tables[m + 1], site_is_right, h.shape[0])
    return ops


# ----------------------------------------------------------------------------- H_eff.psi on output blocks
def op2_dN(o2):
    """Particle-number change of a composite operator (every entry has the same)."""
    for en in o2.entries():
        sp, s = (int(v[0]) for v in np.nonzero(en.m))
        return sym_dN(en.sym) + SITE_N[sp] - SITE_N[s]
    return 0


def enlarged_block(o2, ops, site_is_right, bra, ket):
    """Reduced block <(q', s') J'|| T ||(q, s) J> of a composite operator T = sum [sym x site]^K between
    the coupled sectors bra = (i_block', s', 2J') and ket = (i_block, s, 2J): the 9j product rule of A4
    with the sign (-1)^{N_1 pi_U} (site to the right of the block: subsystem 1 = block; else = site).
    The un-rotated (enlarged) form of the A5 renormalization formula.  None if it vanishes."""
    ipp, sp, Jp = bra
    ip, s, J = ket
    tab = ops.table
    jb, jbp = int(tab[ip][1]), int(tab[ipp][1])
    acc = None
    for en in o2.entries():
        ms = en.m[sp, s]
        if ms == 0.0:
            continue
        O = ops.block(en.sym, ipp, ip)
        if O is None:
            continue
        if site_is_right:
            f = f9(jb, SITE_J2[s], J, en.kB, en.kS, en.K, jbp, SITE_J2[sp], Jp)
            odd = int(tab[ip][0]) & en.parS
        else:
            f = f9(SITE_J2[s], jb, J, en.kS, en.kB, en.K, SITE_J2[sp], jbp, Jp)
            odd = SITE_N[s] & sym_parity(en.sym)
        if f == 0.0:
            continue
        val = ((-f if odd & 1 else f) * ms) * O
        acc = val if acc is None else acc + val
    return acc


class TwoSite:
    """Two-site H_eff in reduced form (A5).  psi blocks (iL, s1, 2S_A, s2, iR, 2S_B), packed as in the ABI.

    Two evaluations of the same sum, both plain loop nests over one output block at a time:
      apply            term by term, the element formula of A5 with the composed prefactor c F6 F9_A F9_B
                       (one pair of matmuls per elementary term and input block);
      apply_enlarged   pair by pair of the cut identity: the A-side and B-side operators of each scalar pair
                       [T_A x U_B]^0 are first assembled as numeric blocks on the coupled sectors of (L, s1) and
                       (s2, R) (`enlarged_block`), then  psi'[a',b'] += coef F6 T_A[a',a] psi[a,b] U_B[b',b]^T.
                       Same result with ~100x fewer matmuls at the full-size configurations (the elementary
                       terms of one pair share their psi block), which is what makes the sampled checks there
                       affordable."""

    def __init__(self, h, V, opsL, t1, t2, opsR, N, S2tot, normal_on="A"):
        self.opsL, self.opsR, self.N, self.S2 = opsL, opsR, N, S2tot
        self.blocks, self.n = psi_blocks(opsL.table, opsR.table, N, S2tot)
        self._args = (h, V, opsL.orbs, t1, t2, opsR.orbs, normal_on)
        self.A, self.B, self.pairs = cut_pairs(*self._args)
        self._terms = None
        tL, tR = opsL.table, opsR.table
        # input blocks indexed by (s1, N_L, s2, N_R): the spins are the only freedom left
        self._by = {}
        for n, b in enumerate(self.blocks):
            self._by.setdefault((int(b[1]), int(tL[b[0]][0]), int(b[3]), int(tR[b[4]][0])), []).append(n)

    @property
    def terms(self):
        if self._terms is None:
            self._terms = two_site_terms(*self._args)
            self._terms_by = {}
            for key, c in self._terms.items():
                self._terms_by.setdefault((key[2], key[4]), []).append((key, c))
        return self._terms

    def factor(self, key, bo, bi):
        """F6 F9_A F9_B with the signs (-1)^{N_1 pi_U} of the three product rules (A5); 0 if forbidden."""
        symL, symR, s1p, s1, s2p, s2, kL, k1, kk, k2, kR = key
        tL, tR = self.opsL.table, self.opsR.table
        iLp, _, SAp, _, iRp, SBp = (int(v) for v in bo[:6])
        iL, _, SA, _, iR, SB = (int(v) for v in bi[:6])
        NL, SL, SLp = int(tL[iL][0]), int(tL[iL][1]), int(tL[iLp][1])
        SR, SRp = int(tR[iR][1]), int(tR[iRp][1])
        par1, par2, parR = (SITE_N[s1p] - SITE_N[s1]) & 1, (SITE_N[s2p] - SITE_N[s2]) & 1, sym_parity(symR)
        fa = f9(SL, SITE_J2[s1], SA, kL, k1, kk, SLp, SITE_J2[s1p], SAp)
        if fa == 0.0:
            return 0.0
        fb = f9(SITE_J2[s2], SR, SB, k2, kR, kk, SITE_J2[s2p], SRp, SBp)
        if fb == 0.0:
            return 0.0
        f6 = f9(SA, SB, self.S2, kk, kk, 0, SAp, SBp, self.S2)
        e = NL * par1 + SITE_N[s2] * parR + (NL + SITE_N[s1]) * ((par2 + parR) & 1)
        f = fa * fb * f6
        return -f if e & 1 else f

    def _view(self, psi, n):
        b = self.blocks[n]
        return psi[int(b[8]): int(b[8]) + int(b[6]) * int(b[7])].reshape(int(b[6]), int(b[7]))

    def apply(self, psi, outputs=None):
        """psi' on the output blocks `outputs` (indices into self.blocks; default all); zero elsewhere."""
        tL, tR = self.opsL.table, self.opsR.table
        self.terms
        y = np.zeros(self.n)
        for o in (range(len(self.blocks)) if outputs is None else outputs):
            bo = self.blocks[o]
            iLp, s1p, SAp, s2p, iRp, SBp, dLp, dRp, offo = (int(v) for v in bo)
            acc = np.zeros((dLp, dRp))
            for key, c in self._terms_by.get((s1p, s2p), []):
                symL, symR = key[0], key[1]
                NL, NR = int(tL[iLp][0]) - sym_dN(symL), int(tR[iRp][0]) - sym_dN(symR)
                for n in self._by.get((key[3], NL, key[5], NR), []):
                    bi = self.blocks[n]
                    f = self.factor(key, bo, bi)
                    if f == 0.0:
                        continue
                    OL = self.opsL.block(symL, iLp, int(bi[0]))
                    if OL is None:
                        continue
                    OR = self.opsR.block(symR, iRp, int(bi[4]))
                    if OR is None:
                        continue
                    acc += (c * f) * (OL @ self._view(psi, n) @ OR.T)
            y[offo: offo + dLp * dRp] = acc.reshape(-1)
        return y

    def apply_enlarged(self, psi, outputs=None):
        """Same result, pair by pair of the cut identity on enlarged (un-rotated) blocks."""
        tL, tR = self.opsL.table, self.opsR.table
        y = np.zeros(self.n)
        info = []                         # per pair: rank, dN and reachable (s, dN_sym) of both operators
        for coef, a, b in self.pairs:
            reach = lambda o2: sorted({(int(sp), int(s), sym_dN(en.sym)) for en in o2.entries() for sp, s in zip(*np.nonzero(en.m))})
            info.append((a.K, reach(a), reach(b), b.par))
        for o in (range(len(self.blocks)) if outputs is None else outputs):
            bo = self.blocks[o]
            iLp, s1p, SAp, s2p, iRp, SBp, dLp, dRp, offo = (int(v) for v in bo)
            NLp, NRp = int(tL[iLp][0]), int(tR[iRp][0])
            acc = np.zeros((dLp, dRp))
            for (coef, a, b), (K, ra, rb, parB) in zip(self.pairs, info):
                cand = set()
                for (sp1, s1, dnl) in ra:
                    if sp1 != s1p:
                        continue
                    for (sp2, s2, dnr) in rb:
                        if sp2 == s2p:
                            cand.update(self._by.get((s1, NLp - dnl, s2, NRp - dnr), []))
                memoA, memoB = {}, {}
                for n in sorted(cand):
                    bi = self.blocks[n]
                    iL, s1, SA, s2, iR, SB = (int(v) for v in bi[:6])
                    f6 = f9(SA, SB, self.S2, K, K, 0, SAp, SBp, self.S2)
                    if f6 == 0.0:
                        continue
                    if (iL, s1, SA) not in memoA:
                        memoA[(iL, s1, SA)] = enlarged_block(a, self.opsL, True, (iLp, s1p, SAp), (iL, s1, SA))
                    TA = memoA[(iL, s1, SA)]
                    if TA is None:
                        continue
                    if (s2, iR, SB) not in memoB:
                        memoB[(s2, iR, SB)] = enlarged_block(b, self.opsR, False, (iRp, s2p, SBp), (iR, s2, SB))
                    UB = memoB[(s2, iR, SB)]
                    if UB is None:
                        continue
                    if ((int(tL[iL][0]) + SITE_N[s1]) & parB) & 1:       # (-1)^{N_A pi_{U_B}}
                        f6 = -f6
                    acc += (coef * f6) * (TA @ self._view(psi, n) @ UB.T)
            y[offo: offo + dLp * dRp] = acc.reshape(-1)
        return y
