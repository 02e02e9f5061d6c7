"""Shared test helpers: build seeded inputs, the oracle objects and a library context."""
import numpy as np

import fixtures as fx
from fixtures.configs import Config
from oracle import abelian as ab


def make_case(L, N, tw, D, bond, nchol=6, seed=1, cfg=None, hdiag="default", sym=0):
    cfg = cfg or Config("t", L=L, N=N, twoS=tw, sym=sym, D=D, n_chol=nchol, bond=bond, hdiag=hdiag)
    h, V, chol = fx.make_integrals(cfg.L, cfg.n_chol, 0, cfg.hdiag)
    tabs = fx.block_tables(cfg)
    nl, nr = cfg.bond, cfg.L - cfg.bond - 2
    isoL = fx.random_isometries(cfg, tabs, nl, seed)
    isoR = fx.random_isometries(cfg, tabs, nr, seed + 1000)
    return dict(cfg=cfg, h=h, V=V, chol=chol, tabs=tabs, nl=nl, nr=nr, isoL=isoL, isoR=isoR)


def oracle_two_site(case):
    cfg = case["cfg"]
    ints = ab.Integrals(case["h"], case["V"])
    Lb = ab.build_block(ints, case["tabs"], case["isoL"], list(range(case["nl"])), True)
    Rb = ab.build_block(ints, case["tabs"], case["isoR"], list(range(cfg.L - 1, cfg.bond + 1, -1)), False)
    ts = ab.TwoSite(Lb, ab.site_block(ints, cfg.bond), ab.site_block(ints, cfg.bond + 1), Rb, cfg.N, cfg.twoS)
    return ints, Lb, Rb, ts


EMU_EVERYTHING = {k: 1 for k in ("emu_mink", "emu_minm", "emu_minn", "emu_mink1", "emu_minm1", "emu_minn1")}


def library_context(case, device=0, stream=None, plan_only=False, options=None, use_chol=False, precision=0, slices=0):
    """options: {key: value} for dmrg_set_option (e.g. EMU_EVERYTHING: every stage-1 job and two-sided stage-2
    segment runs on the tensor-core path whatever its size); use_chol: ingest the Cholesky vectors with V = NULL."""
    import paper_2603_28648_b200 as pkg
    cfg = case["cfg"]
    d = pkg.Dmrg(-1 if plan_only else device, stream)
    for k, v in (options or {}).items():
        d.set_option(k, v)
    if use_chol:
        d.init_integrals(case["h"], None, case["chol"], 0.0, cfg.N, cfg.twoS, cfg.sym, cfg.D)
    else:
        d.init_integrals(case["h"], case["V"], None, 0.0, cfg.N, cfg.twoS, cfg.sym, cfg.D)
    d.set_mps(cfg.bond, case["tabs"][:case["nl"] + 1], [x[1] for x in case["isoL"]],
              case["tabs"][:case["nr"] + 1], [x[1] for x in case["isoR"]])
    if plan_only:
        d.plan_bond()
    else:
        d.build_env(precision, slices)
    return d


def rel_err(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def oracle_su2(case, M2=None):
    """SU(2) oracle: Wigner-Eckart expansion into the pinned U(1)xU(1) oracle (oracle/su2.py)."""
    from oracle import su2
    cfg = case["cfg"]
    return su2.ExpandedTwoSite(case["h"], case["V"], cfg.N, cfg.twoS, cfg.bond, case["tabs"][:case["nl"] + 1],
                               case["isoL"], case["tabs"][:case["nr"] + 1], case["isoR"], M2)


def su2_block_components(blk, kind, p, r, rank):
    """Spherical components {2q: dense matrix} of a stored SU(2) operator, built from the U(1)xU(1)
    oracle block `blk` (spin-orbital operators) by the definitions of SURVEY.md Appendix A4:
    a+_q = a+_{p,sigma}; a~_{+1/2} = a_dn, a~_{-1/2} = -a_up; [T x U]^K_Q = sum CG T_q1 U_q2."""
    from oracle import su2
    dense = lambda *key: blk.op(*key).dense(blk.basis)
    so = lambda orb, q2: 2 * orb + (0 if q2 == 1 else 1)
    if kind == "H":
        return {0: dense("H")}, 0
    if kind == "C":
        return {1: dense("C", so(p, 1)), -1: dense("C", so(p, -1))}, 1
    if kind == "S":      # S~_m = (-1)^{1/2-m} S_{x,-m}
        return {1: dense("S", so(p, -1)), -1: -dense("S", so(p, 1))}, 1
    out = {}
    for Q in range(-rank, rank + 1, 2):
        M = 0.0
        for q1 in (1, -1):
            q2 = Q - q1
            if abs(q2) != 1:
                continue
            c = su2.cg(1, q1, 1, q2, rank, Q)
            if c == 0.0:
                continue
            if kind == "A":
                M = M + c * dense("A", so(p, q1), so(r, q2))
            else:        # B^k_ps = [a+_p x a~_s]^k with a~_{q2} = (-1)^{1/2 - q2} a_{s,-q2}
                sgn = 1.0 if q2 == 1 else -1.0
                M = M + c * sgn * dense("B", so(p, q1), so(r, -q2))
        out[Q] = M if not np.isscalar(M) else np.zeros((sum(blk.basis.dims),) * 2)
    return out, rank


# ------------------------------------------------------------------ sampled checks at full size (oracle c4)
class DeviceStore:
    """`get_stored` callback of oracle/su2_loopnest.BlockOps over operator blocks downloaded from the device
    ("taking the environment operator blocks ... as input data downloaded from the device").
    One download per (operator class, sector pair): dmrg_op_export_class."""

    def __init__(self, d, side):
        import paper_2603_28648_b200 as pkg
        self.d, self.side = d, side
        self.code = {"H": pkg.OP_H, "C": pkg.OP_C, "S": pkg.OP_S, "A": pkg.OP_A, "B": pkg.OP_B}
        self.cache = {}

    def __call__(self, kind, k2, i, k, ibra, iket):
        key = (kind, k2, ibra, iket)
        if key not in self.cache:
            code = self.code[kind] | ((k2 << 8) if kind in ("A", "B") else 0)
            mem, data = self.d.op_export_class(self.side, code, 0, 0, ibra, iket)
            self.cache[key] = None if mem is None else ({(int(a), int(b)): n for n, (a, b) in enumerate(mem)}, data)
        hit = self.cache[key]
        if hit is None:
            return None
        n = hit[0].get((i, k))
        return None if n is None else hit[1][n]


def sample_blocks(blocks, frac, at_least, seed=3, dims=(6, 7)):
    """Seeded sample of psi blocks (reading s15): `frac` of the blocks, at least `at_least`, always including
    the largest."""
    nb = len(blocks)
    want = min(nb, max(at_least, int(round(frac * nb))))
    sizes = blocks[:, dims[0]] * blocks[:, dims[1]]
    pick = [int(np.argmax(sizes))]
    rng = np.random.Generator(np.random.Philox(seed))
    for i in rng.permutation(nb):
        if len(pick) >= want:
            break
        if int(i) not in pick:
            pick.append(int(i))
    return sorted(pick)


def gather_blocks(vec, blocks, pick, dims=(6, 7), off=8):
    return np.concatenate([vec[int(blocks[n][off]): int(blocks[n][off]) + int(blocks[n][dims[0]]) * int(blocks[n][dims[1]])]
                           for n in pick])


# ------------------------------------------------------------------ Davidson: tolerance derived from the arithmetic
def davidson_envelope(matvec, diag, psi0, n_iter, eps=2.0 ** -50, trials=6, safety=8.0, seed=9):
    """Per-iteration bound on |theta_it - theta_it(reference)| and on the residual norm for two CORRECT FP64
    implementations of SURVEY.md 8(c) c6 on this input.  Two implementations differ by rounding in the matvec and in
    the vector work; that is modelled by running the oracle's Davidson with the matvec perturbed by componentwise
    relative noise of size eps ~ 4 ulp (seeded), several times, and taking the largest deviation from the unperturbed
    run, times a safety factor, plus a floor of 1e-12 |theta|.  The preconditioner r_i / (theta - diag_i) has
    near-singular denominators on random environments, so the envelope grows by orders of magnitude per iteration
    (tests/test_oracle_davidson.py shows it): the envelope is what a test may ask of iteration it, not more.
    Returns (theta_ref, resid_ref, env_theta, env_resid)."""
    from oracle.davidson import davidson
    _, th0, rs0 = davidson(matvec, diag, psi0, n_iter)
    rng = np.random.Generator(np.random.Philox(seed))
    dev_t, dev_r = np.zeros(len(th0)), np.zeros(len(rs0))
    for _ in range(trials):
        noisy = lambda v: (lambda y: y * (1.0 + eps * rng.standard_normal(len(y))))(matvec(v))
        _, th, rs = davidson(noisy, diag, psi0, n_iter)
        m = min(len(th), len(th0))
        dev_t[:m] = np.maximum(dev_t[:m], np.abs(th[:m] - th0[:m]))
        dev_r[:m] = np.maximum(dev_r[:m], np.abs(rs[:m] - rs0[:m]))
    env_t = safety * np.maximum.accumulate(dev_t) + 1e-12 * np.abs(th0)
    env_r = safety * np.maximum.accumulate(dev_r) + 1e-12 * np.maximum(1.0, rs0)
    return th0, rs0, env_t, env_r
