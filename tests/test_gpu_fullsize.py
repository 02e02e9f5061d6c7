"""-m gpu: parity of the CUDA path with the loop-nest oracle (oracle/su2_loopnest.py, part c4) at the FULL size of
BASELINE.json configs[2], [3] and [4], on a seeded sample of output psi blocks (reading s15,
8(d) table "Checked"), in the launch configuration bench.py times (default plans, no forced code paths).

The oracle takes the environment operator blocks and psi as data downloaded from the device, so that errors do not
chain; each sampled output block is computed in full (every term) with the oracle's own 6j/9j recoupling.  The same
is done for sampled blocks of one renormalization of the enlarged block (row a9).  Error measure (reading s16):
relative Frobenius norm over the compared blocks.  Tolerances: BASELINE.json north_star (1e-11 native FP64,
1e-10 emulated FP64 at the default kappa = 6, 1e-5 for the 3xTF32 mode).

Sample sizes: configs[2] and configs[3] 5 % of the output blocks (BASELINE.json configs[2]); configs[4] 10 blocks at the centre and 16 at site 10, the largest always included: its ~5500 blocks are tiny and the plain numpy oracle spends ~10 s of Python on each,
so 5 % (275 blocks) would not fit the driver's time limit for the GPU suite."""
import time

import numpy as np
import pytest

import fixtures as fx
from oracle import su2_loopnest as ln
from tests.helpers import DeviceStore, gather_blocks, make_case, rel_err, sample_blocks

pytestmark = pytest.mark.gpu
TOL = {"fp64": 1e-11, "emu": 1e-10, "perf": 1e-10, "tf32": 1e-5}


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    assert torch.cuda.is_available()
    return torch


def _context(torch, case):
    import paper_2603_28648_b200 as pkg
    cfg = case["cfg"]
    d = pkg.Dmrg(0, torch.cuda.current_stream().cuda_stream)
    d.init_integrals(case["h"], None, case["chol"], 0.0, cfg.N, cfg.twoS, cfg.sym, cfg.D)   # Cholesky ingest (a1)
    d.set_mps(cfg.bond, case["tabs"][:case["nl"] + 1], [x[1] for x in case["isoL"]],
              case["tabs"][:case["nr"] + 1], [x[1] for x in case["isoR"]])
    d.build_env()
    return d


def _oracle(case, d):
    cfg = case["cfg"]
    sL, sR = DeviceStore(d, 0), DeviceStore(d, 1)
    opsL = ln.BlockOps(case["tabs"][case["nl"]], list(range(cfg.bond)), case["V"], sL)
    opsR = ln.BlockOps(case["tabs"][case["nr"]], list(range(cfg.bond + 2, cfg.L)), case["V"], sR)
    ts = ln.TwoSite(case["h"], case["V"], opsL, cfg.bond, cfg.bond + 1, opsR, cfg.N, cfg.twoS)
    return ts, (sL, sR, opsL, opsR)


def _oracle_blocks(ts, stores, psi, pick):
    """Oracle psi' on the sampled blocks, one block at a time (the downloaded operator blocks are dropped in between)."""
    ref = np.zeros(ts.n)
    for o in pick:
        ref += ts.apply_enlarged(psi, outputs=[o])
        for s in stores:
            (s.cache if hasattr(s, "cache") else s._cache).clear()
    return ref


def _apply(torch, d, psi, prec, kappa=0):
    x = torch.from_numpy(psi).cuda()
    y = torch.empty_like(x)
    d.heff_apply(x, y, prec, kappa)
    torch.cuda.synchronize()
    return y.cpu().numpy()


def _renorm_sample(torch, case, d, stores, modes):
    """Row a9 at full size: sampled blocks of the grown left block's operators against oracle c5 (reduced form), in
    every precision mode of `modes` (a fresh environment per mode: dmrg_renormalize replaces the block).  The error
    is relative to the largest element of the sampled reference blocks of the operator."""
    import paper_2603_28648_b200 as pkg
    cfg, tabs, nl = case["cfg"], case["tabs"], case["nl"]
    sL, opsL = stores[0], stores[2]
    rng = np.random.Generator(np.random.Philox(77))
    iso_blocks, iso_data = fx.random_isometry(cfg.sym, tabs[nl], tabs[nl + 1], rng)
    new_tab = tabs[nl + 1]
    orbs = list(range(cfg.bond + 1))
    outside = [x for x in range(cfg.L) if x not in orbs]
    p, r = orbs[0], orbs[-1]                      # r = the absorbed site: mixed block x site pieces
    targets = [("H", 0, -1, -1), ("C", 1, p, -1), ("C", 1, r, -1), ("S", 1, outside[0], -1), ("S", 1, outside[-1], -1),
               ("A", 0, p, r), ("A", 2, p, r), ("A", 0, r, r), ("B", 0, p, r), ("B", 2, r, p), ("B", 2, r, r), ("B", 0, p, orbs[1])]
    big = int(np.argmax(new_tab[:, 2]))
    only = set()
    for tg in targets:                            # the block with the largest ket sector, and a random one
        dN = ln._DN[tg[0]]
        for a in (big, int(rng.integers(len(new_tab)))):
            for ap in range(len(new_tab)):
                if new_tab[ap][0] - new_tab[a][0] == dN and ln.triangle(int(new_tab[a][1]), tg[1], int(new_tab[ap][1])):
                    only.add((tg, ap, a))
                    break
    want = ln.renormalize_blocks(case["h"], case["V"], opsL, cfg.bond, iso_blocks, iso_data, new_tab, True, targets, only)
    out = {}
    for mi, mode in enumerate(modes):
        if mi > 0:
            d.close()
            d = _context(torch, case)
        prec, kappa = MODES(pkg)[mode]
        d.renormalize(pkg.LEFT_TO_RIGHT, new_tab, iso_data, precision=prec, slices=kappa)
        new_store = DeviceStore(d, 0)
        n, worst = 0, 0.0
        for (tg, ap, a) in sorted(only):
            ref = want[tg].get((ap, a))
            got = new_store(tg[0], tg[1], tg[2], tg[3], ap, a)
            if ref is None:
                assert got is None or np.abs(got).max() < 1e-9, (tg, ap, a)
                continue
            assert got is not None, (tg, ap, a)
            scale = max(1.0, float(np.abs(ref).max()))
            worst = max(worst, float(np.abs(got - ref).max()) / scale)
            n += 1
        assert n >= 8
        out[mode] = (n, worst)
        assert worst <= TOL[mode], (mode, worst)
    return out, d


def MODES(pkg):
    return {"fp64": (pkg.PREC_FP64, 0), "emu": (pkg.PREC_FP64_EMU, 6), "tf32": (pkg.PREC_TF32X3, 0),
            "perf": (pkg.PREC_FP64_EMU_PERF, 6)}        # the paper's performant mode (reading s21)


def _run(torch, name, frac, at_least, modes, bond=None, renorm_modes=None):
    import paper_2603_28648_b200 as pkg
    cfg = fx.get_config(name)
    if bond is not None:
        cfg = cfg.with_(bond=bond)
    t0 = time.time()
    case = make_case(0, 0, 0, 0, 0, cfg=cfg)
    d = _context(torch, case)
    t1 = time.time()
    ts, stores = _oracle(case, d)
    n = d.psi_length()
    assert n == ts.n
    assert np.array_equal(d.table(pkg.TAB_PSI_BLOCKS, 9), ts.blocks)
    pick = sample_blocks(ts.blocks, frac, at_least)
    psi = fx.random_psi(n, 2)
    ref = gather_blocks(_oracle_blocks(ts, stores, psi, pick), ts.blocks, pick)
    t2 = time.time()
    assert np.linalg.norm(ref) > 0
    errs = {}
    for mode in modes:
        prec, kappa = MODES(pkg)[mode]
        got = gather_blocks(_apply(torch, d, psi, prec, kappa), ts.blocks, pick)
        errs[mode] = rel_err(got, ref)
        if mode == "emu":      # the emulated lists really ran (default thresholds, as in bench.py)
            counts = d.table(pkg.TAB_COUNTS)
            assert counts[15] > 0 and counts[18] > 0
        if mode == "perf":     # slice products were really let go, and the eager count is the plan's
            kept, eager = d.last_emu_products()
            assert 0 < kept < eager
            print(f"performant mode kept {kept / eager:.3f} of the stage-2 slice products")
    rn, d = _renorm_sample(torch, case, d, stores, renorm_modes or [m for m in modes if m != "perf"])
    d.close()
    print(f"\n{cfg.name} bond {cfg.bond}: {len(pick)} of {len(ts.blocks)} output blocks, rel. errors {errs}, renormalized "
          f"blocks (n, worst) {rn}; setup {t1 - t0:.0f} s, oracle {t2 - t1:.0f} s, total {time.time() - t0:.0f} s")
    for mode in modes:
        assert errs[mode] <= TOL[mode], (mode, errs)
    if "tf32" in errs:
        assert errs["tf32"] > 1e-10          # it is not the FP64 path


def test_cfg2_sampled_blocks_all_modes(torch_mod):
    """BASELINE.json configs[2]: CAS(54,36)-shaped, SU(2), D = 2048; "the oracle is checked on a seeded 5 % sample"."""
    _run(torch_mod, "cfg2", 0.05, 8, ["fp64", "emu", "perf", "tf32"])


def test_cfg3_sampled_blocks_all_modes(torch_mod):
    """configs[3]: D = 4096; the three precision modes on identical inputs, and one renormalization."""
    _run(torch_mod, "cfg3", 0.05, 8, ["fp64", "emu", "tf32"])


def test_cfg4_centre_sampled_blocks(torch_mod):
    """configs[4]: CAS(89,102)-shaped sextet, D = 1024, emulated FP64 (and native), centre site."""
    _run(torch_mod, "cfg4", 0.0, 10, ["fp64", "emu"], renorm_modes=["emu"])


def test_cfg4_site_10_from_the_edge(torch_mod):
    """configs[4] "plus at a site 10 from the edge" (left block of 10 orbitals)."""
    _run(torch_mod, "cfg4", 0.0, 16, ["fp64", "emu"], bond=10, renorm_modes=["emu"])
