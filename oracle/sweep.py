"""Oracle support a10 + sweep driver for tiny systems (test infrastructure).

Split and truncate (SURVEY.md Appendix A5 "Truncation", reading s9): per composite
sector q_A, rho = sum over B-side blocks psi psi^T; eigen-decompose; keep the D
largest eigenvalues over all sectors (ties: sector label ascending, then eigen-index);
the isometry is made of the kept eigenvectors.  Discarded weight = truncation error
(PAPER.md:49).  Two-site sweeps at saturated D reproduce E_FCI.
"""
import numpy as np

from . import abelian as ab
from .davidson import davidson


def split(ts, psi, D, absorb_left):
    """Returns (new_table, iso_blocks, iso_data, discarded_weight) for the grown block."""
    x = ts.unpack(psi)
    comp = ts.A if absorb_left else ts.B
    groups = {}                                           # label -> list of composite idx
    for (a, b) in x:
        c = a if absorb_left else b
        groups.setdefault(comp.basis.labels[c], set()).add(c)
    cand = []                                             # (weight, label, eig index)
    eig = {}
    for q, cs in groups.items():
        # rows ordered by (i_prev, s) as in the packed isometry layout
        def key(c):
            ix, iy = comp.pairs[c]
            return (ix, ab.SITE_STATE_OF_SECTOR[iy]) if absorb_left else (iy, ab.SITE_STATE_OF_SECTOR[ix])
        cs = sorted(cs, key=key)
        rows = []
        for c in cs:
            mats = []
            for (a, b), m in sorted(x.items()):
                if (a if absorb_left else b) == c:
                    mats.append(m if absorb_left else m.T)
            rows.append(np.concatenate(mats, axis=1))
        # different rows may see different column sets: assemble rho block-wise
        dims = [r.shape[0] for r in rows]
        off = np.concatenate([[0], np.cumsum(dims)])
        rho = np.zeros((off[-1], off[-1]))
        for i, ci in enumerate(cs):
            for j, cj in enumerate(cs):
                acc = np.zeros((dims[i], dims[j]))
                for (a, b), m in x.items():
                    ka, kb = (a, b) if absorb_left else (b, a)
                    if ka != ci:
                        continue
                    other = (cj, kb) if absorb_left else (kb, cj)
                    if other in x:
                        m2 = x[other]
                        acc += (m @ m2.T) if absorb_left else (m.T @ m2)
                rho[off[i]:off[i + 1], off[j]:off[j + 1]] = acc
        w, U = np.linalg.eigh(rho)
        w, U = w[::-1], U[:, ::-1]
        eig[q] = (cs, off, U, key)
        for e in range(len(w)):
            cand.append((-w[e], q, e))
    cand.sort()
    keep = cand[:D]
    disc = -sum(c[0] for c in cand[D:])
    kept = {}
    for _, q, e in keep:
        kept.setdefault(q, []).append(e)
    labels = sorted(kept)
    table, o = [], 0
    for q in labels:
        table.append((q[0], q[1], len(kept[q]), o))
        o += len(kept[q])
    table = np.array(table, dtype=np.int64).reshape(-1, 4)
    blocks, chunks = [], []
    for inext, q in enumerate(labels):
        cs, off, U, key = eig[q]
        Uk = U[:, sorted(kept[q])]
        for i, c in enumerate(cs):
            ip, s = key(c)
            blocks.append([ip, s, inext, off[i + 1] - off[i], Uk.shape[1], Uk[off[i]:off[i + 1]]])
    blocks.sort(key=lambda b: (b[0], b[1], b[2]))
    rows, o = [], 0
    for b in blocks:
        rows.append((b[0], b[1], b[2], b[3], b[4], o))
        chunks.append(b[5].reshape(-1))
        o += b[3] * b[4]
    data = np.concatenate(chunks) if chunks else np.zeros(0)
    return table, np.array(rows, dtype=np.int64).reshape(-1, 6), data, disc


def two_site_sweeps(ints, cfg, tables, isosR, n_sweeps=4, n_dav=40, tol=1e-10, seed=5):
    """Plain two-site DMRG from a random right-canonical start; returns energies per step."""
    L, D = cfg.L, cfg.D
    rng = np.random.default_rng(seed)
    right = [ab.vacuum_block(ints)]
    for m in range(L - 2):
        right.append(ab.renormalize(right[-1], ab.site_block(ints, L - 1 - m), *isosR[m],
                                    tables[m + 1], False))
    left = [ab.vacuum_block(ints)]
    energies = []
    for sw in range(n_sweeps):
        for p in range(0, L - 1):                            # rightward
            ts = ab.TwoSite(left[p], ab.site_block(ints, p), ab.site_block(ints, p + 1),
                            right[L - 2 - p], cfg.N, cfg.twoS)
            x, th, rs = davidson(ts.apply, ts.diagonal(), rng.standard_normal(ts.n), n_dav, tol)
            energies.append(th[-1])
            if p < L - 2:
                tab, ib, idt, _ = split(ts, x, D, True)
                blk = ab.renormalize(left[p], ab.site_block(ints, p), ib, idt, tab, True)
                left[p + 1:] = [blk]
        for p in range(L - 2, -1, -1):                       # leftward
            ts = ab.TwoSite(left[p], ab.site_block(ints, p), ab.site_block(ints, p + 1),
                            right[L - 2 - p], cfg.N, cfg.twoS)
            x, th, rs = davidson(ts.apply, ts.diagonal(), rng.standard_normal(ts.n), n_dav, tol)
            energies.append(th[-1])
            if p > 0:
                tab, ib, idt, _ = split(ts, x, D, False)
                blk = ab.renormalize(right[L - 2 - p], ab.site_block(ints, p + 1), ib, idt, tab, False)
                right[L - 1 - p:] = [blk]
    return energies
