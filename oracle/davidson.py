"""Oracle part c6: Davidson reference (test infrastructure).

Start v0 = psi/|psi|.  Each iteration: w = H v_new; G = V^T W; lowest eigenpair
(theta, y) of G (symmetrised) by LAPACK eigh; x = V y; r = W y - theta x; t_i = r_i / (theta - diag_i)
with |theta - diag_i| < 1e-12 replaced by +-1e-12; orthogonalise t against V twice
(classical Gram-Schmidt); normalise; append.  No restart.  "n iterations" means
exactly n applications of H (tol <= 0 disables the early exit).
The paper's own solver is "Lanczos" with residual 1e-6; BASELINE.json
north_star asks for Davidson (reading s6).
"""
import numpy as np



def davidson(matvec, diag, psi0, n_iter, tol=0.0):
    v = np.array(psi0, dtype=np.float64)
    v /= np.linalg.norm(v)
    V, W = [v], []
    thetas, resids = [], []
    x = v
    for it in range(n_iter):
        W.append(matvec(V[-1]))
        Vm, Wm = np.stack(V, 1), np.stack(W, 1)
        G = Vm.T @ Wm
        G = 0.5 * (G + G.T)
        ev, evec = np.linalg.eigh(G)
        theta, y = ev[0], evec[:, 0]
        x = Vm @ y
        r = Wm @ y - theta * x
        rn = float(np.linalg.norm(r))
        thetas.append(float(theta))
        resids.append(rn)
        if (tol > 0 and rn < tol) or it == n_iter - 1:
            break
        den = theta - diag
        small = np.abs(den) < 1e-12
        den = np.where(small, np.where(den < 0, -1e-12, 1e-12), den)
        t = r / den
        for _ in range(2):
            t = t - Vm @ (Vm.T @ t)
        nt = np.linalg.norm(t)
        if nt < 1e-14:
            break
        V.append(t / nt)
    x = x / np.linalg.norm(x)
    return x, np.array(thetas), np.array(resids)
