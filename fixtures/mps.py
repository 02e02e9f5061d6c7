"""Random mixed-canonical MPS tensors, psi and random operator data
(SURVEY.md Appendix C).  Pure input generation: Gaussian fills and a QR
orthonormalisation; nothing of the method's arithmetic.

Packed isometry layout (part of the ABI): blocks
(i_prev, s, i_next) -- indices into the smaller block's table, site state,
index into the grown block's table -- sorted lexicographically, each block
row-major [a_prev][a_next], blocks contiguous.
"""
import numpy as np

from .sectors import fuse, site_states


def isometry_blocks(sym, tab_prev, tab_next):
    """int64 rows (i_prev, s, i_next, rows, cols, offset) in packed order."""
    nxt = {(int(r[0]), int(r[1])): i for i, r in enumerate(tab_next)}
    rows = []
    for ip, r in enumerate(tab_prev):
        q = (int(r[0]), int(r[1]))
        for s in range(len(site_states(sym))):
            for q2 in fuse(sym, q, s):
                if q2 in nxt:
                    rows.append([ip, s, nxt[q2], int(r[2]), int(tab_next[nxt[q2]][2]), 0])
    rows.sort(key=lambda x: (x[0], x[1], x[2]))
    off = 0
    for r in rows:
        r[5] = off
        off += r[3] * r[4]
    return np.array(rows, dtype=np.int64).reshape(-1, 6), off


def random_isometry(sym, tab_prev, tab_next, rng):
    """Packed random isometry: for each grown sector, Q of a Gaussian matrix."""
    blocks, n = isometry_blocks(sym, tab_prev, tab_next)
    data = np.zeros(n, dtype=np.float64)
    for inext in range(len(tab_next)):
        sel = [b for b in blocks if b[2] == inext]          # already (i_prev, s) sorted
        nrow = sum(int(b[3]) for b in sel)
        ncol = int(tab_next[inext][2])
        if nrow < ncol:
            raise ValueError("sector table violates the isometry cap")
        G = rng.standard_normal((nrow, ncol))
        Q, R = np.linalg.qr(G)
        Q = Q * np.sign(np.diag(R))[None, :]
        r0 = 0
        for b in sel:
            nr = int(b[3])
            data[int(b[5]): int(b[5]) + nr * ncol] = Q[r0:r0 + nr].reshape(-1)
            r0 += nr
    return blocks, data


def random_isometries(cfg, tables, n_sites, seed):
    """Isometries growing a block from 0 to n_sites orbitals: list of (blocks, data)."""
    rng = np.random.Generator(np.random.Philox(seed))
    out = []
    for m in range(n_sites):
        out.append(random_isometry(cfg.sym, tables[m], tables[m + 1], rng))
    return out


def random_vector(n, seed, normalise=True):
    rng = np.random.Generator(np.random.Philox(seed))
    v = rng.standard_normal(n)
    if normalise:
        v /= np.linalg.norm(v)
    return v


def random_psi(n, seed=2):
    """psi: N(0,1) in every allowed block (flat, layout-agnostic), normalised."""
    return random_vector(n, seed, True)
