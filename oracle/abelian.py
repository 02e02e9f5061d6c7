"""Oracle parts c3/c5 for U(1)xU(1): block operators, blocking, renormalization,
H_eff.psi (test infrastructure).

Everything is written as (operator on X) (x) (operator on Y) with X left of Y and
the sign rule of Appendix A1:  (X-op)(Y-op) -> X_loc (x) Y_loc * (-1)^{N_x pi_Y},
N_x the particle number of the KET state of X, pi_Y the parity of the Y operator.

Operator definitions for a region R and outside spin-orbitals i,k,l (Appendix A2):
  H^R    all indices in R
  C_i    = a+_i                        (i in R)
  A_ik   = a+_i a+_k,  B_il = a+_i a_l (i,k,l in R)
  S^R_i  = 1/2 sum_j t_ij a_j + sum_jkl v_ijkl a+_k a_l a_j
  P^R_ik = sum_jl v_ijkl a_l a_j
  Q^R_il = sum_kj (v_ilkj - v_ijkl) a+_k a_j
Cut identity (Appendix A2) and blocking rules (Appendix A3) are implemented in
`Composite.op`; they are pinned against Jordan-Wigner matrices in the tests.

A block stores the NORMAL set {H, C_i, S_x, A_ik (i<k), B_il}; P and Q are formed
from their definitions as integral-weighted sums of the stored A+ and B.
"""
import numpy as np

from .fock import site_creators, spin_orbital_integrals

SITE_LABELS = [(0, 0), (1, 1), (1, -1), (2, 0)]          # site state s -> (N, 2Sz)
SITE_TABLE = [(0, 0), (1, -1), (1, 1), (2, 0)]           # sorted sector order of one site
SITE_SECTOR_OF_STATE = [0, 2, 1, 3]                      # site state s -> index in SITE_TABLE
SITE_STATE_OF_SECTOR = [0, 2, 1, 3]


class Op:
    """Block-sparse operator: blocks[(i_bra, i_ket)] = dense matrix; dq = (dN, d2Sz)."""
    __slots__ = ("blocks", "dq")

    def __init__(self, dq, blocks=None):
        self.dq = dq
        self.blocks = blocks if blocks is not None else {}

    @property
    def parity(self):
        return self.dq[0] & 1

    def dagger(self):
        return Op((-self.dq[0], -self.dq[1]), {(j, i): m.T for (i, j), m in self.blocks.items()})

    def add(self, c, other):
        assert other.dq == self.dq
        for key, m in other.blocks.items():
            if key in self.blocks:
                self.blocks[key] = self.blocks[key] + c * m
            else:
                self.blocks[key] = c * m
        return self

    def scaled(self, c):
        return Op(self.dq, {k: c * m for k, m in self.blocks.items()})

    def dense(self, basis):
        off = np.concatenate([[0], np.cumsum(basis.dims)])
        M = np.zeros((off[-1], off[-1]))
        for (i, j), m in self.blocks.items():
            M[off[i]:off[i + 1], off[j]:off[j + 1]] = m
        return M


class Basis:
    """Ordered list of sectors with labels (N, 2Sz) and dimensions."""

    def __init__(self, labels, dims):
        self.labels = [tuple(int(x) for x in q) for q in labels]
        self.dims = [int(d) for d in dims]
        self.index = {q: i for i, q in enumerate(self.labels)}

    @staticmethod
    def from_table(tab):
        return Basis([(r[0], r[1]) for r in tab], [r[2] for r in tab])

    def __len__(self):
        return len(self.labels)


def identity_op(basis):
    return Op((0, 0), {(i, i): np.eye(d) for i, d in enumerate(basis.dims)})


class Integrals:
    def __init__(self, h, V):
        self.L = h.shape[0]
        self.t, self.v = spin_orbital_integrals(h, V)
        self.n = 2 * self.L


class Block:
    """A region with stored normal operators in a given basis."""

    def __init__(self, ints, orbs, basis):
        self.ints = ints
        self.orbs = list(orbs)                       # spin-orbital indices in the region
        self.outside = [i for i in range(ints.n) if i not in set(self.orbs)]
        self.basis = basis
        self.store = {}                              # key -> Op

    # -- access -------------------------------------------------------------
    def op(self, *key):
        kind = key[0]
        if kind == "I":
            return identity_op(self.basis)
        if kind == "A":
            _, i, k = key
            if i == k:
                return Op((2, _spin(i) + _spin(k)))
            if i > k:
                return self.store[("A", k, i)].scaled(-1.0)
        if kind == "P":
            return self._P(key[1], key[2])
        if kind == "Q":
            return self._Q(key[1], key[2])
        return self.store[key]

    def _P(self, i, k):
        """P_ik = sum_{j,l in R} v_ijkl a_l a_j = sum_{j<l} (v_ijkl - v_ilkj) (A_jl)+."""
        v = self.ints.v
        out = Op((-2, -_spin(i) - _spin(k)))
        for a, j in enumerate(self.orbs):
            for l in self.orbs[a + 1:]:
                w = v[i, j, k, l] - v[i, l, k, j]
                if w != 0.0:
                    out.add(w, self.store[("A", j, l)].dagger())
        return out

    def _Q(self, i, l):
        """Q_il = sum_{k,j in R} (v_ilkj - v_ijkl) a+_k a_j."""
        v = self.ints.v
        out = Op((0, _spin(l) - _spin(i)))
        for k in self.orbs:
            for j in self.orbs:
                w = v[i, l, k, j] - v[i, j, k, l]
                if w != 0.0:
                    out.add(w, self.store[("B", k, j)])
        return out


def _spin(i):
    return 1 if (i & 1) == 0 else -1


def site_block(ints, p):
    """One-site block: every operator evaluated from its definition with 4x4 matrices."""
    cu, cd = site_creators()
    orbs = [2 * p, 2 * p + 1]
    c = {orbs[0]: cu, orbs[1]: cd}
    a = {i: m.T for i, m in c.items()}
    t, v = ints.t, ints.v
    basis = Basis(SITE_TABLE, [1, 1, 1, 1])
    blk = Block(ints, orbs, basis)

    def to_op(M, dq):
        o = Op(dq)
        for sp in range(4):
            for s in range(4):
                if M[sp, s] != 0.0:
                    o.blocks[(SITE_SECTOR_OF_STATE[sp], SITE_SECTOR_OF_STATE[s])] = np.array([[M[sp, s]]])
        return o

    H = np.zeros((4, 4))
    for i in orbs:
        for j in orbs:
            H += t[i, j] * c[i] @ a[j]
            for k in orbs:
                for l in orbs:
                    H += 0.5 * v[i, j, k, l] * c[i] @ c[k] @ a[l] @ a[j]
    blk.store[("H",)] = to_op(H, (0, 0))
    for i in orbs:
        blk.store[("C", i)] = to_op(c[i], (1, _spin(i)))
    blk.store[("A", orbs[0], orbs[1])] = to_op(c[orbs[0]] @ c[orbs[1]], (2, 0))
    for i in orbs:
        for l in orbs:
            blk.store[("B", i, l)] = to_op(c[i] @ a[l], (0, _spin(i) - _spin(l)))
    for x in blk.outside:
        S = np.zeros((4, 4))
        for j in orbs:
            S += 0.5 * t[x, j] * a[j]
            for k in orbs:
                for l in orbs:
                    S += v[x, j, k, l] * c[k] @ a[l] @ a[j]
        blk.store[("S", x)] = to_op(S, (-1, -_spin(x)))
    return blk


def vacuum_block(ints):
    """Block with no orbitals: one state, all operators zero."""
    blk = Block(ints, [], Basis([(0, 0)], [1]))
    blk.store[("H",)] = Op((0, 0))
    for x in blk.outside:
        blk.store[("S", x)] = Op((-1, -_spin(x)))
    return blk


class Composite:
    """R = X u Y (X left of Y), un-rotated product basis; operators by Appendix A3."""

    def __init__(self, X, Y, keep=None):
        self.X, self.Y = X, Y
        self.ints = X.ints
        self.orbs = X.orbs + Y.orbs
        inside = set(self.orbs)
        self.outside = [i for i in range(self.ints.n) if i not in inside]
        labels, dims, self.pairs = [], [], []
        for ix, (qx, dx) in enumerate(zip(X.basis.labels, X.basis.dims)):
            for iy, (qy, dy) in enumerate(zip(Y.basis.labels, Y.basis.dims)):
                q = (qx[0] + qy[0], qx[1] + qy[1])
                if keep is not None and not keep(q):
                    continue
                labels.append(q)
                dims.append(dx * dy)
                self.pairs.append((ix, iy))
        # NB: several composite sectors may share a label; Basis.index is not used here.
        self.basis = Basis(labels, dims)
        self.pair_index = {p: i for i, p in enumerate(self.pairs)}
        self._inX = set(X.orbs)

    # -- tensor product with the A1 sign rule ---------------------------------
    def tensor(self, ox, oy, coef=1.0, out=None):
        dq = (ox.dq[0] + oy.dq[0], ox.dq[1] + oy.dq[1])
        out = out if out is not None else Op(dq)
        assert out.dq == dq
        piy = oy.parity
        for (ixp, ix), mx in ox.blocks.items():
            sgn = -1.0 if (piy and (self.X.basis.labels[ix][0] & 1)) else 1.0
            for (iyp, iy), my in oy.blocks.items():
                kb = self.pair_index.get((ixp, iyp))
                kk = self.pair_index.get((ix, iy))
                if kb is None or kk is None:
                    continue
                m = (coef * sgn) * np.kron(mx, my)
                if (kb, kk) in out.blocks:
                    out.blocks[(kb, kk)] = out.blocks[(kb, kk)] + m
                else:
                    out.blocks[(kb, kk)] = m
        return out

    def op(self, *key):
        X, Y, T = self.X, self.Y, self.tensor
        IX, IY = X.op("I"), Y.op("I")
        v, inX = self.ints.v, self._inX
        kind = key[0]
        if kind == "I":
            return identity_op(self.basis)
        if kind == "C":
            i = key[1]
            return T(X.op("C", i), IY) if i in inX else T(IX, Y.op("C", i))
        if kind == "A":
            _, i, k = key
            if i in inX and k in inX:
                return T(X.op("A", i, k), IY)
            if i not in inX and k not in inX:
                return T(IX, Y.op("A", i, k))
            if i in inX:
                return T(X.op("C", i), Y.op("C", k))
            return T(X.op("C", k), Y.op("C", i), -1.0)             # a+_i a+_k = -a+_k a+_i
        if kind == "B":
            _, i, l = key
            if i in inX and l in inX:
                return T(X.op("B", i, l), IY)
            if i not in inX and l not in inX:
                return T(IX, Y.op("B", i, l))
            if i in inX:
                return T(X.op("C", i), Y.op("C", l).dagger())
            return T(X.op("C", l).dagger(), Y.op("C", i), -1.0)    # a+_i a_l = -a_l a+_i
        if kind == "S":
            x = key[1]
            out = T(X.op("S", x), IY)
            T(IX, Y.op("S", x), 1.0, out)
            for j in Y.orbs:
                T(X.op("Q", x, j), Y.op("C", j).dagger(), 1.0, out)   # Q^X_xj a_j
                T(X.op("P", x, j), Y.op("C", j), 1.0, out)            # a+_j P^X_xj
            for j in X.orbs:
                T(X.op("C", j).dagger(), Y.op("Q", x, j), 1.0, out)   # Q^Y_xj a_j
                T(X.op("C", j), Y.op("P", x, j), 1.0, out)            # a+_j P^Y_xj
            return out
        if kind == "P":
            _, i, k = key
            out = T(X.op("P", i, k), IY)
            T(IX, Y.op("P", i, k), 1.0, out)
            for j in X.orbs:
                for l in Y.orbs:
                    w = v[i, j, k, l] - v[i, l, k, j]
                    if w != 0.0:                                       # a_l a_j = -a_j a_l
                        T(X.op("C", j).dagger(), Y.op("C", l).dagger(), -w, out)
            return out
        if kind == "Q":
            _, i, l = key
            out = T(X.op("Q", i, l), IY)
            T(IX, Y.op("Q", i, l), 1.0, out)
            for k in X.orbs:
                for j in Y.orbs:
                    w1 = v[i, l, k, j] - v[i, j, k, l]
                    w2 = v[i, l, j, k] - v[i, k, j, l]
                    if w1 != 0.0:
                        T(X.op("C", k), Y.op("C", j).dagger(), w1, out)      # a+_k a_j
                    if w2 != 0.0:
                        T(X.op("C", k).dagger(), Y.op("C", j), -w2, out)     # a+_j a_k
            return out
        if kind == "H":
            out = T(X.op("H"), IY)
            T(IX, Y.op("H"), 1.0, out)
            for coef, ox, oy in cut_terms(X, Y):
                T(ox, oy, coef, out)
            return out
        raise KeyError(key)


def cut_terms(X, Y):
    """Cross terms of the cut identity (Appendix A2) as (coef, op on X, op on Y),
    already in left-to-right order.  The side with fewer orbitals (tie: X) carries the
    normal pair operators A, B; the other side carries P, Q."""
    terms = []
    for i in Y.orbs:                                   # a+_i S^X_i + h.c.,  i in Y
        sx, cy = X.op("S", i), Y.op("C", i)
        terms.append((-1.0, sx, cy))                   # a+_i S^X_i = -S^X_i a+_i
        terms.append((1.0, sx.dagger(), cy.dagger()))  # (S^X_i)+ a_i
    for i in X.orbs:                                   # a+_i S^Y_i + h.c.,  i in X
        cx, sy = X.op("C", i), Y.op("S", i)
        terms.append((1.0, cx, sy))
        terms.append((-1.0, cx.dagger(), sy.dagger())) # (S^Y_i)+ a_i = -a_i (S^Y_i)+
    if len(X.orbs) <= len(Y.orbs):
        for a, i in enumerate(X.orbs):
            for k in X.orbs[a + 1:]:                   # 1/2 sum_{ik} = sum_{i<k}
                ax, py = X.op("A", i, k), Y.op("P", i, k)
                terms.append((1.0, ax, py))
                terms.append((1.0, ax.dagger(), py.dagger()))
        for i in X.orbs:
            for l in X.orbs:
                terms.append((1.0, X.op("B", i, l), Y.op("Q", i, l)))
    else:
        for a, i in enumerate(Y.orbs):
            for k in Y.orbs[a + 1:]:
                px, ay = X.op("P", i, k), Y.op("A", i, k)
                terms.append((1.0, px, ay))
                terms.append((1.0, px.dagger(), ay.dagger()))
        for i in Y.orbs:
            for l in Y.orbs:
                terms.append((1.0, X.op("Q", i, l), Y.op("B", i, l)))
    return terms


# ------------------------------------------------------------------ renormalization


def isometry_dict(blocks, data):
    """Packed isometry (fixtures.mps layout) -> {(i_prev, s, i_next): matrix}."""
    return {(int(b[0]), int(b[1]), int(b[2])):
            data[int(b[5]): int(b[5]) + int(b[3]) * int(b[4])].reshape(int(b[3]), int(b[4]))
            for b in blocks}


def rotate(op, comp, iso, new_basis, site_is_right):
    """O' = X^T O X (Appendix A5): X maps composite sectors (block sector, site state)
    to the new sectors."""
    out = Op(op.dq)
    maps = {}                                # composite index -> list of (i_next, matrix)
    for (ip, s, inext), m in iso.items():
        sec = SITE_SECTOR_OF_STATE[s]
        pair = (ip, sec) if site_is_right else (sec, ip)
        ci = comp.pair_index.get(pair)
        if ci is not None:
            maps.setdefault(ci, []).append((inext, m))
    for (cb, ck), m in op.blocks.items():
        for (nb, xb) in maps.get(cb, []):
            for (nk, xk) in maps.get(ck, []):
                val = xb.T @ m @ xk
                if (nb, nk) in out.blocks:
                    out.blocks[(nb, nk)] += val
                else:
                    out.blocks[(nb, nk)] = val
    return out


def renormalize(block, site, iso_blocks, iso_data, new_table, site_is_right, pair_orbs=None):
    """Oracle c5: the next block's normal operator set from (block, site) and an isometry.
    pair_orbs limits the spin-orbitals for which A, B are kept (default: all inside)."""
    comp = Composite(block, site) if site_is_right else Composite(site, block)
    iso = isometry_dict(iso_blocks, iso_data)
    nb = Basis.from_table(new_table)
    new = Block(block.ints, comp.orbs, nb)
    new.orbs = sorted(comp.orbs)
    rot = lambda o: rotate(o, comp, iso, nb, site_is_right)
    new.store[("H",)] = rot(comp.op("H"))
    for i in new.orbs:
        new.store[("C", i)] = rot(comp.op("C", i))
    for x in new.outside:
        new.store[("S", x)] = rot(comp.op("S", x))
    po = new.orbs if pair_orbs is None else [i for i in new.orbs if i in pair_orbs]
    for a, i in enumerate(po):
        for k in po[a + 1:]:
            new.store[("A", i, k)] = rot(comp.op("A", i, k))
    for i in po:
        for l in po:
            new.store[("B", i, l)] = rot(comp.op("B", i, l))
    return new


def build_block(ints, tables, isos, sites, site_is_right):
    """Grow a block over `sites` (in absorption order) from the vacuum."""
    blk = vacuum_block(ints)
    for m, p in enumerate(sites):
        blocks, data = isos[m]
        blk = renormalize(blk, site_block(ints, p), blocks, data, tables[m + 1], site_is_right)
    return blk


# ------------------------------------------------------------------ two-site H_eff


def psi_block_list(tabL, tabR, N, twoSz):
    """Packed psi layout: rows (iL, s1, s2, iR, dL, dR, offset), lexicographic."""
    rl = {(int(r[0]), int(r[1])): i for i, r in enumerate(tabR)}
    rows, off = [], 0
    for iL, r in enumerate(tabL):
        for s1 in range(4):
            for s2 in range(4):
                NR = N - int(r[0]) - SITE_LABELS[s1][0] - SITE_LABELS[s2][0]
                tR = twoSz - int(r[1]) - SITE_LABELS[s1][1] - SITE_LABELS[s2][1]
                iR = rl.get((NR, tR))
                if iR is None:
                    continue
                dL, dR = int(r[2]), int(tabR[iR][2])
                rows.append((iL, s1, s2, iR, dL, dR, off))
                off += dL * dR
    return np.array(rows, dtype=np.int64).reshape(-1, 7), off


class TwoSite:
    """H_eff of the window (L, s1 | s2, R) by the cut identity on A=(L,s1) | B=(s2,R)."""

    def __init__(self, Lblk, s1blk, s2blk, Rblk, N, twoSz):
        self.A = Composite(Lblk, s1blk)
        self.B = Composite(s2blk, Rblk)
        self.N, self.twoSz = N, twoSz
        tabL = [(q[0], q[1], d, 0) for q, d in zip(Lblk.basis.labels, Lblk.basis.dims)]
        tabR = [(q[0], q[1], d, 0) for q, d in zip(Rblk.basis.labels, Rblk.basis.dims)]
        self.blocks, self.n = psi_block_list(tabL, tabR, N, twoSz)
        self._terms = None

    def terms(self):
        if self._terms is None:
            A, B = self.A, self.B
            t = [(1.0, A.op("H"), B.op("I")), (1.0, A.op("I"), B.op("H"))]
            t += cut_terms(A, B)
            self._terms = t
        return self._terms

    def unpack(self, psi):
        out = {}
        for (iL, s1, s2, iR, dL, dR, off) in self.blocks:
            a = self.A.pair_index[(iL, SITE_SECTOR_OF_STATE[s1])]
            b = self.B.pair_index[(SITE_SECTOR_OF_STATE[s2], iR)]
            out[(a, b)] = psi[off: off + dL * dR].reshape(dL, dR)
        return out

    def pack(self, d):
        psi = np.zeros(self.n)
        for (iL, s1, s2, iR, dL, dR, off) in self.blocks:
            a = self.A.pair_index[(iL, SITE_SECTOR_OF_STATE[s1])]
            b = self.B.pair_index[(SITE_SECTOR_OF_STATE[s2], iR)]
            if (a, b) in d:
                psi[off: off + dL * dR] = d[(a, b)].reshape(-1)
        return psi

    def apply(self, psi, only_outputs=None):
        """psi' = H_eff psi (packed in, packed out).  only_outputs: set of output
        (a, b) keys to compute (the 5 % sample); others are left zero."""
        x = self.unpack(psi)
        y = {k: np.zeros_like(m) for k, m in x.items()}
        by_a = {}
        for (a, b) in x:
            by_a.setdefault(a, []).append(b)
        NA = [q[0] for q in self.A.basis.labels]
        for coef, oa, ob in self.terms():
            pib = ob.parity
            bmap = {}
            for (bp, b), m in ob.blocks.items():
                bmap.setdefault(b, []).append((bp, m))
            for (ap, a), ma in oa.blocks.items():
                sgn = -coef if (pib and (NA[a] & 1)) else coef
                for b in by_a.get(a, []):
                    for (bp, mb) in bmap.get(b, []):
                        if (ap, bp) not in y:
                            continue
                        if only_outputs is not None and (ap, bp) not in only_outputs:
                            continue
                        y[(ap, bp)] += sgn * (ma @ x[(a, b)] @ mb.T)
        return self.pack(y)

    def diagonal(self):
        """diag(H_eff), packed (Davidson preconditioner)."""
        y = {k: np.zeros_like(m) for k, m in self.unpack(np.zeros(self.n)).items()}
        NA = [q[0] for q in self.A.basis.labels]
        for coef, oa, ob in self.terms():
            if oa.dq != (0, 0) or ob.dq != (0, 0):
                continue
            for (a, b) in y:
                ma, mb = oa.blocks.get((a, a)), ob.blocks.get((b, b))
                if ma is None or mb is None:
                    continue
                sgn = -coef if (ob.parity and (NA[a] & 1)) else coef
                y[(a, b)] += sgn * np.outer(np.diag(ma), np.diag(mb))
        return self.pack(y)
