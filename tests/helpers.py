"""Shared test helpers: build seeded inputs, the oracle objects and a library context."""
import numpy as np

import fixtures as fx
from fixtures.configs import Config
from oracle import abelian as ab


def make_case(L, N, tw, D, bond, nchol=6, seed=1, cfg=None, hdiag="default"):
    cfg = cfg or Config("t", L=L, N=N, twoS=tw, sym=0, D=D, n_chol=nchol, bond=bond, hdiag=hdiag)
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


def library_context(case, device=0, stream=None, plan_only=False):
    import paper_2603_28648_b200 as pkg
    cfg = case["cfg"]
    d = pkg.Dmrg(-1 if plan_only else device, stream)
    d.init_integrals(case["h"], case["V"], None, 0.0, cfg.N, cfg.twoS, pkg.SYM_U1U1, cfg.D)
    d.set_mps(cfg.bond, case["tabs"][:case["nl"] + 1], [x[1] for x in case["isoL"]],
              case["tabs"][:case["nr"] + 1], [x[1] for x in case["isoR"]])
    if plan_only:
        d.plan_bond()
    else:
        d.build_env()
    return d


def rel_err(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))
