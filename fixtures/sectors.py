"""Synthetic bond sector tables ("Bond sector dimensions").

A table describes the basis of a block holding m orbitals: int64 rows
(N, twoS, dim, offset) sorted by (N, twoS); twoS is 2*Sz for U(1)xU(1) and 2*S
for SU(2).  The recipe is the same from either edge, so `block_tables(cfg)[m]`
serves the left block with m orbitals (bond p = m) and the right block with m
orbitals (bond p = L - m, the block's OWN labels).

Only sector bookkeeping and a Gaussian weight recipe live here: no operators,
no Hamiltonian.
"""
from math import comb, exp

import numpy as np

from .configs import SYM_SU2, SYM_U1U1


def site_states(sym):
    """Site basis labels (N, twoS) in index order (PAPER.md:41 order for U1U1)."""
    if sym == SYM_U1U1:
        return [(0, 0), (1, 1), (1, -1), (2, 0)]
    return [(0, 0), (1, 1), (2, 0)]


def fuse(sym, q, s):
    """Labels reachable by fusing block label q with site state index s."""
    Ns, ts = site_states(sym)[s]
    N, t = q
    if sym == SYM_U1U1:
        return [(N + Ns, t + ts)]
    if ts == 0:
        return [(N + Ns, t)]
    out = []
    if t >= 1:
        out.append((N + Ns, t - 1))
    out.append((N + Ns, t + 1))
    return out


def fock_count(sym, m, q):
    """Number of states (U1U1) or multiplets (SU2, Weyl-Paldus) of label q on m orbitals."""
    N, t = q
    if sym == SYM_U1U1:
        if (N + t) % 2:
            return 0
        nu, nd = (N + t) // 2, (N - t) // 2
        if nu < 0 or nd < 0 or nu > m or nd > m:
            return 0
        return comb(m, nu) * comb(m, nd)
    if t < 0 or (N - t) % 2 or N < 0:
        return 0
    a = (N - t) // 2          # N/2 - S
    b = (N + t) // 2 + 1      # N/2 + S + 1
    if a < 0 or b > m + 1:
        return 0
    return (t + 1) * comb(m + 1, a) * comb(m + 1, b) // (m + 1)


def _complement_count(cfg, m, q):
    """States/multiplets on the other L-m orbitals that can pair q to the target."""
    mc = cfg.L - m
    N, t = q
    if cfg.sym == SYM_U1U1:
        return fock_count(cfg.sym, mc, (cfg.N - N, cfg.twoS - t))
    tot = 0
    for tr in range(abs(t - cfg.twoS), t + cfg.twoS + 1, 2):
        tot += fock_count(cfg.sym, mc, (cfg.N - N, tr))
    return tot


def _distribute(keys, w, caps, D):
    """Distribute D over keys proportionally to w under caps (Appendix C)."""
    n = len(keys)
    if sum(caps) <= D:
        return list(caps)
    fixed = [None] * n
    rem = D
    free = [i for i in range(n) if w[i] > 0 and caps[i] > 0]
    for i in range(n):
        if i not in free:
            fixed[i] = 0
    while True:
        sw = sum(w[i] for i in free)
        over = [i for i in free if rem * w[i] / sw >= caps[i]]
        if not over:
            break
        for i in over:
            fixed[i] = caps[i]
            rem -= caps[i]
            free.remove(i)
        if not free:
            break
    if free:
        sw = sum(w[i] for i in free)
        alloc = {i: rem * w[i] / sw for i in free}
        for i in free:
            fixed[i] = int(alloc[i])
        left = D - sum(fixed)
        order = sorted(free, key=lambda i: (-(alloc[i] - int(alloc[i])), keys[i]))
        k = 0
        while left > 0 and order:
            i = order[k % len(order)]
            if fixed[i] < caps[i]:
                fixed[i] += 1
                left -= 1
            k += 1
            if k > 4 * len(order) + 4 * D:
                break
    return fixed


def block_tables(cfg):
    """Tables for blocks of m = 0..L orbitals grown from an edge (vacuum at m=0)."""
    sym = cfg.sym
    ns = len(site_states(sym))
    tables = []
    prev = {(0, 0): 1}
    tables.append(_to_table(prev))
    for m in range(1, cfg.L + 1):
        reach = {}
        for q, d in prev.items():
            for s in range(ns):
                for q2 in fuse(sym, q, s):
                    reach[q2] = reach.get(q2, 0) + d
        keys, w, caps = [], [], []
        for q in sorted(reach):
            cc = _complement_count(cfg, m, q)
            fc = fock_count(sym, m, q)
            if cc <= 0 or fc <= 0:
                continue
            N, t = q
            cN = cfg.N * m / cfg.L
            ct = cfg.twoS * m / cfg.L
            if sym == SYM_U1U1:
                wt = exp(-(N - cN) ** 2 / (2 * cfg.sigma_N ** 2)) \
                    * exp(-(t - ct) ** 2 / (2 * cfg.sigma_Z ** 2))
            else:
                wt = exp(-(N - cN) ** 2 / (2 * cfg.sigma_N ** 2)) * (t + 1) \
                    * exp(-((t - ct) / 2.0) ** 2 / (2 * cfg.sigma_S ** 2))
            keys.append(q)
            w.append(wt)
            caps.append(min(fc, cc, reach[q]))
        dims = _distribute(keys, w, caps, cfg.D)
        prev = {q: d for q, d in zip(keys, dims) if d > 0}
        tables.append(_to_table(prev))
    return tables


def _to_table(dims):
    rows, off = [], 0
    for q in sorted(dims):
        rows.append((q[0], q[1], dims[q], off))
        off += dims[q]
    return np.array(rows, dtype=np.int64).reshape(-1, 4)


def left_bond_tables(cfg):
    """tables[p] for p = 0..bond+1: left block with p orbitals."""
    return block_tables(cfg)[: cfg.bond + 2]


def right_bond_tables(cfg):
    """tables[m] for m = 0..L-bond-1: right block with m orbitals (own labels)."""
    return block_tables(cfg)[: cfg.L - cfg.bond]


def bond_tables_for(cfg):
    t = block_tables(cfg)
    return t[: cfg.bond + 2], t[: cfg.L - cfg.bond]
