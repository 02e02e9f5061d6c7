"""Oracle part c2: the plain definition of the result for tiny L (test infrastructure).

From the MPS tensors build the block basis vectors explicitly in Fock space
(|l_new> = sum X[l,s,l_new] |l>|s>; for the right block the site is on the left,
|r_new> = sum Y[r,s,r_new] |s>|r>), then H_eff = P^T H P with H the dense
Jordan-Wigner Hamiltonian of fock.py.
The site-product basis is the occupation basis of Appendix A1, so plain Kronecker
products carry no extra sign.
"""
import numpy as np

from .abelian import isometry_dict, psi_block_list


def block_vectors(tables, isos, n_sites, site_is_right):
    """Columns = block basis vectors in the 4^n_sites Fock space, ordered by the table."""
    vec = {0: np.ones((1, 1))}                       # sector index -> (dimFock, d)
    for m in range(n_sites):
        iso = isometry_dict(*isos[m])
        tab = tables[m + 1]
        dimF = 4 ** (m + 1)
        new = {i: np.zeros((dimF, int(r[2]))) for i, r in enumerate(tab)}
        for (ip, s, inext), X in iso.items():
            e = np.zeros((4, 1))
            e[s, 0] = 1.0
            for a in range(X.shape[0]):
                v = vec[ip][:, a:a + 1]
                ket = np.kron(v, e) if site_is_right else np.kron(e, v)
                new[inext] += ket @ X[a:a + 1, :]
        vec = new
    return vec


def projector(cfg_N, cfg_twoSz, tabL, vecL, tabR, vecR):
    """P: columns |l s1 s2 r> in packed psi order (abelian layout)."""
    blocks, n = psi_block_list(tabL, tabR, cfg_N, cfg_twoSz)
    dimL = next(iter(vecL.values())).shape[0]
    dimR = next(iter(vecR.values())).shape[0]
    P = np.zeros((dimL * 16 * dimR, n))
    for (iL, s1, s2, iR, dL, dR, off) in blocks:
        e = np.zeros((16, 1))
        e[s1 * 4 + s2, 0] = 1.0
        for a in range(dL):
            left = np.kron(vecL[iL][:, a:a + 1], e)
            P[:, off + a * dR: off + (a + 1) * dR] = np.kron(left, vecR[iR])
    return P, blocks
