"""Oracle part c1: determinant-space Hamiltonian, Lanczos, Jacobi (test infrastructure).

Conventions (PAPER.md:41 for the site basis):
  spin-orbital i = 2p + sigma (sigma 0 = up, 1 = down), ordered (0u,0d,1u,1d,..);
  |n> = prod_i (a+_i)^{n_i} |0> in ascending i, so a_i carries (-1)^{sum_{j<i} n_j};
  site states 0=|0>, 1=|u>, 2=|d>, 3=|ud> = a+_u a+_d |0>;
  H = sum_ij t_ij a+_i a_j + 1/2 sum_ijkl v_ijkl a+_i a+_k a_l a_j  (+ e_core),
  t_ij = h_pq d(si,sj), v_ijkl = (pq|rs) d(si,sj) d(sk,sl), V[p,q,r,s] = (pq|rs).
"""
import numpy as np

# ---------------------------------------------------------------- site / JW matrices


def site_creators():
    """4x4 matrices of a+_up, a+_dn in the site basis (intra-site sign included)."""
    cu = np.zeros((4, 4))
    cd = np.zeros((4, 4))
    cu[1, 0] = 1.0      # |0> -> |u>
    cu[3, 2] = 1.0      # |d> -> a+u a+d|0> = |ud>
    cd[2, 0] = 1.0      # |0> -> |d>
    cd[3, 1] = -1.0     # a+d a+u|0> = -|ud>
    return cu, cd


SITE_PARITY = np.diag([1.0, -1.0, -1.0, 1.0])
SITE_N = np.array([0, 1, 1, 2])
SITE_2SZ = np.array([0, 1, -1, 0])


def jw_creators(L):
    """Dense a+_i (i = 0..2L-1) on the 4^L Fock space; site 0 is the most significant digit."""
    cu, cd = site_creators()
    out = []
    for p in range(L):
        for c in (cu, cd):
            m = np.ones((1, 1))
            for s in range(L):
                m = np.kron(m, SITE_PARITY if s < p else (c if s == p else np.eye(4)))
            out.append(m)
    return out


def spin_orbital_integrals(h, V):
    """t_ij and v_ijkl of Appendix A2 as dense arrays over spin-orbitals."""
    L = h.shape[0]
    n = 2 * L
    t = np.zeros((n, n))
    v = np.zeros((n, n, n, n))
    for s in range(2):
        t[s::2, s::2] = h
        for s2 in range(2):
            v[s::2, s::2, s2::2, s2::2] = V
    return t, v


def hamiltonian_dense(h, V, creators=None):
    """H on the full 4^L Fock space straight from the definition (small L only)."""
    L = h.shape[0]
    c = creators if creators is not None else jw_creators(L)
    a = [m.T for m in c]
    t, v = spin_orbital_integrals(h, V)
    n = 2 * L
    dim = c[0].shape[0]
    H = np.zeros((dim, dim))
    for i in range(n):
        for j in range(n):
            if t[i, j] != 0.0:
                H += t[i, j] * (c[i] @ a[j])
    for i in range(n):
        for k in range(n):
            if i == k:
                continue
            cik = c[i] @ c[k]
            for l in range(n):
                for j in range(n):
                    if l == j or v[i, j, k, l] == 0.0:
                        continue
                    H += 0.5 * v[i, j, k, l] * (cik @ (a[l] @ a[j]))
    return H


# ---------------------------------------------------------------- determinant FCI


def sector_dets(L, nup, ndn):
    """All occupation bit-strings with nup up and ndn down electrons, ascending."""
    n = 2 * L
    allb = np.arange(1 << n, dtype=np.int64)
    upmask = sum(1 << (2 * p) for p in range(L))
    dnmask = upmask << 1
    ok = (np.bitwise_count(allb & upmask) == nup) & (np.bitwise_count(allb & dnmask) == ndn)
    return allb[ok]


def dets_to_fock_index(dets, L):
    """Index of each determinant in the 4^L site-product basis (site 0 most significant)."""
    idx = np.zeros_like(dets)
    for p in range(L):
        s = ((dets >> (2 * p)) & 1) + 2 * ((dets >> (2 * p + 1)) & 1)
        idx = idx * 4 + s
    return idx


def _apply(op_is_create, i, dets, sign, alive):
    bit = np.int64(1) << i
    has = (dets & bit) != 0
    ok = alive & (~has if op_is_create else has)
    below = np.bitwise_count(dets & (bit - 1))
    sign = np.where(below & 1, -sign, sign)
    dets = dets ^ bit
    return dets, sign, ok


def fci_matrix(h, V, nup, ndn):
    """Dense H in the (nup, ndn) determinant sector, applied string by string."""
    L = h.shape[0]
    dets = sector_dets(L, nup, ndn)
    nd = len(dets)
    lookup = -np.ones(1 << (2 * L), dtype=np.int64)
    lookup[dets] = np.arange(nd)
    t, v = spin_orbital_integrals(h, V)
    n = 2 * L
    H = np.zeros((nd, nd))
    cols = np.arange(nd)
    one = np.ones(nd)
    alive0 = np.ones(nd, dtype=bool)
    for i in range(n):
        for j in range(n):
            if t[i, j] == 0.0:
                continue
            d, s, ok = _apply(False, j, dets, one, alive0)
            d, s, ok = _apply(True, i, d, s, ok)
            r = lookup[d[ok]]
            np.add.at(H, (r, cols[ok]), t[i, j] * s[ok])
    for j in range(n):
        d1, s1, ok1 = _apply(False, j, dets, one, alive0)
        for l in range(n):
            if l == j:
                continue
            d2, s2, ok2 = _apply(False, l, d1, s1, ok1)
            if not ok2.any():
                continue
            for k in range(n):
                if (k & 1) != (l & 1):
                    continue
                d3, s3, ok3 = _apply(True, k, d2, s2, ok2)
                for i in range(n):
                    if (i & 1) != (j & 1) or i == k or v[i, j, k, l] == 0.0:
                        continue
                    d4, s4, ok4 = _apply(True, i, d3, s3, ok3)
                    r = lookup[d4[ok4]]
                    np.add.at(H, (r, cols[ok4]), 0.5 * v[i, j, k, l] * s4[ok4])
    return H, dets


# ---------------------------------------------------------------- eigen-solvers


def jacobi_eigh(A, tol=1e-15, max_sweeps=30):
    """Cyclic Jacobi for a small symmetric matrix; eigenvalues ascending, vectors in columns."""
    A = np.array(A, dtype=np.float64)
    n = A.shape[0]
    Vv = np.eye(n)
    for _ in range(max_sweeps):
        off = np.linalg.norm(A - np.diag(np.diag(A)))
        nrm = max(np.linalg.norm(A), 1e-300)
        if off <= tol * nrm:
            break
        for p in range(n - 1):
            for q in range(p + 1, n):
                if abs(A[p, q]) <= 1e-18 * nrm:
                    continue
                theta = (A[q, q] - A[p, p]) / (2.0 * A[p, q])
                if abs(theta) > 1e100:
                    tt = 0.5 / theta
                elif theta != 0:
                    tt = np.sign(theta) / (abs(theta) + np.sqrt(theta * theta + 1.0))
                else:
                    tt = 1.0
                c = 1.0 / np.sqrt(tt * tt + 1.0)
                s = tt * c
                # A <- J^T A J, V <- V J with J the rotation in the (p, q) plane
                colp, colq = A[:, p].copy(), A[:, q].copy()
                A[:, p], A[:, q] = c * colp - s * colq, s * colp + c * colq
                rowp, rowq = A[p, :].copy(), A[q, :].copy()
                A[p, :], A[q, :] = c * rowp - s * rowq, s * rowp + c * rowq
                vp, vq = Vv[:, p].copy(), Vv[:, q].copy()
                Vv[:, p], Vv[:, q] = c * vp - s * vq, s * vp + c * vq
    w = np.diag(A).copy()
    order = np.argsort(w)
    return w[order], Vv[:, order]


def lanczos_lowest(matvec, n, v0=None, tol=1e-10, max_iter=500, seed=7):
    """Lowest eigenpair by Lanczos with full re-orthogonalisation; stops at residual tol."""
    rng = np.random.default_rng(seed)
    v = rng.standard_normal(n) if v0 is None else np.array(v0, dtype=np.float64)
    v /= np.linalg.norm(v)
    Q = [v]
    alphas, betas = [], []
    theta, x = 0.0, v
    for it in range(min(max_iter, n)):
        w = matvec(Q[-1])
        a = float(Q[-1] @ w)
        alphas.append(a)
        for _ in range(2):
            for q in Q:
                w = w - (q @ w) * q
        T = np.diag(alphas) + np.diag(betas, 1) + np.diag(betas, -1)
        ev, evec = np.linalg.eigh(T)
        theta = ev[0]
        y = evec[:, 0]
        b = float(np.linalg.norm(w))
        resid = abs(b * y[-1])
        if resid < tol or b < 1e-14:
            break
        betas.append(b)
        Q.append(w / b)
    x = np.stack(Q[: len(y)], axis=1) @ y
    x /= np.linalg.norm(x)
    return theta, x, it + 1
