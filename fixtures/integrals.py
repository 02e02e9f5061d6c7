"""Integral recipe R (BASELINE.json:configs[0]).

h_ii = -2 + N(0,0.5); h_ij = N(0,0.3) exp(-|i-j|/3) (i<j, symmetric);
B^c_ij = N(0,0.2) exp(-|i-j|/4) (i<=j, symmetric), V_ijkl = sum_c B^c_ij B^c_kl.
Variants: "spread" h_ii ~ U(-4,0) (configs[2,3]); "bands" for configs[4].
Returns plain numpy arrays; no Hamiltonian arithmetic happens here.
"""
import numpy as np


def make_integrals(L, n_chol, seed=0, hdiag="default", want_V=True):
    rng = np.random.Generator(np.random.Philox(seed))
    idx = np.arange(L)
    dist = np.abs(idx[:, None] - idx[None, :]).astype(np.float64)
    if hdiag == "default":
        d = -2.0 + 0.5 * rng.standard_normal(L)
    elif hdiag == "spread":
        d = rng.uniform(-4.0, 0.0, L)
    elif hdiag == "bands":
        n1 = (32 * L) // 102
        n2 = (25 * L) // 102
        d = np.empty(L)
        d[:n1] = -3.0 + 0.5 * rng.standard_normal(n1)
        d[n1:n1 + n2] = -1.0 + 0.05 * rng.standard_normal(n2)
        d[n1 + n2:] = 1.0 + 0.5 * rng.standard_normal(L - n1 - n2)
    else:
        raise ValueError(hdiag)
    off = 0.3 * rng.standard_normal((L, L)) * np.exp(-dist / 3.0)
    h = np.triu(off, 1)
    h = h + h.T + np.diag(d)
    chol = 0.2 * rng.standard_normal((n_chol, L, L)) * np.exp(-dist / 4.0)[None]
    chol = np.triu(chol)
    chol = chol + np.transpose(np.triu(chol, 1), (0, 2, 1))
    V = None
    if want_V:
        B = chol.reshape(n_chol, L * L)
        V = (B.T @ B).reshape(L, L, L, L)
    return np.ascontiguousarray(h), V, np.ascontiguousarray(chol)
