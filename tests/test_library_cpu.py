"""-m "not gpu": the C-ABI library loads, exports every symbol include/dmrg.h declares, its
integer tables are bit-exact against the oracle / fixtures enumerators, and compute calls fail
loudly without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

import fixtures as fx
from fixtures.configs import Config
from fixtures.mps import isometry_blocks
from oracle import abelian as ab
from tests.helpers import make_case, library_context

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    import paper_2603_28648_b200 as p
    p.build_library()
    return p


def test_library_exports_every_declared_symbol(pkg):
    hdr = open(os.path.join(ROOT, "include", "dmrg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)           # prototypes only, not comment text
    declared = set(re.findall(r"\b(dmrg_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(pkg.EXPORTS)
    lib = ctypes.CDLL(pkg.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name


def test_compute_calls_fail_loudly_without_gpu(pkg):
    case = make_case(5, 4, 0, 5, 2)
    d = library_context(case, plan_only=True)
    n = d.psi_length()
    x = np.zeros(n)
    y = np.zeros(n)
    for call in (lambda: d.heff_apply(x, y), lambda: d.heff_apply_host(x, y), lambda: d.heff_diag(y),
                 lambda: d.davidson_step(x, 2), lambda: d.build_env(), lambda: d.measure_peak()):
        with pytest.raises(pkg.DmrgError) as e:
            call()
        assert e.value.code == pkg.EUNSUPPORTED
    d.close()


def test_call_order_and_argument_errors(pkg):
    d = pkg.Dmrg(-1)
    with pytest.raises(pkg.DmrgError) as e:
        d.psi_length()
    assert e.value.code == pkg.ESTATE
    h, V, _ = fx.make_integrals(4, 4, 0)
    with pytest.raises(pkg.DmrgError) as e:
        d.init_integrals(h, V, None, 0.0, 3, 0, pkg.SYM_U1U1, 8)      # N + 2Sz odd
    assert e.value.code == pkg.EINVAL
    with pytest.raises(pkg.DmrgError) as e:
        d.init_integrals(h, V, None, 0.0, 4, -2, pkg.SYM_SU2, 8)      # 2S must be non-negative
    assert e.value.code == pkg.EINVAL
    with pytest.raises(pkg.DmrgError) as e:
        d.init_integrals(h, V, None, 0.0, 4, 0, 7, 8)                  # unknown symmetry
    assert e.value.code == pkg.EINVAL
    d.init_integrals(h, V, None, 0.0, 4, 0, pkg.SYM_U1U1, 8)
    bad = np.array([[0, 0, 1, 0], [0, 0, 1, 1]], dtype=np.int64)       # duplicate sector
    with pytest.raises(pkg.DmrgError) as e:
        d.set_mps(1, [bad, bad], [np.zeros(1)], [bad, bad], [np.zeros(1)])
    assert e.value.code == pkg.EINVAL
    d.close()


@pytest.mark.parametrize("name,L,N,tw,D,bond", [("s", 6, 6, 0, 12, 2), ("odd", 5, 5, 1, 9, 2),
                                                 ("cfg0", 0, 0, 0, 0, 0), ("cfg1", 0, 0, 0, 0, 0)])
def test_tables_bit_exact(pkg, name, L, N, tw, D, bond):
    """psi block table vs the oracle's enumerator; bond and isometry tables vs fixtures."""
    cfg = fx.get_config(name) if name.startswith("cfg") else None
    if cfg is None:
        case = make_case(L, N, tw, D, bond)
    else:   # tables only: no isometry data needed for a planning context
        tabs = fx.block_tables(cfg)
        nl, nr = cfg.bond, cfg.L - cfg.bond - 2
        h, _, chol = fx.make_integrals(cfg.L, cfg.n_chol, 0, cfg.hdiag, want_V=False)
        case = dict(cfg=cfg, tabs=tabs, nl=nl, nr=nr)
    cfg = case["cfg"]
    tabs, nl, nr = case["tabs"], case["nl"], case["nr"]
    d = pkg.Dmrg(-1)
    if "h" in case:
        d.init_integrals(case["h"], case["V"], None, 0.0, cfg.N, cfg.twoS, pkg.SYM_U1U1, cfg.D)
    else:
        d.init_integrals(h, None, chol, 0.0, cfg.N, cfg.twoS, pkg.SYM_U1U1, cfg.D)
    d.set_mps(cfg.bond, tabs[:nl + 1], [], tabs[:nr + 1], [])
    d.plan_bond()
    blocks, n = ab.psi_block_list(tabs[nl], tabs[nr], cfg.N, cfg.twoS)
    assert d.psi_length() == n
    assert np.array_equal(d.table(pkg.TAB_PSI_BLOCKS, 7), blocks)
    assert np.array_equal(d.table(pkg.TAB_BOND_L, 4), tabs[nl])
    assert np.array_equal(d.table(pkg.TAB_BOND_R, 4), tabs[nr])
    if nl >= 1:
        ib, _ = isometry_blocks(cfg.sym, tabs[nl - 1], tabs[nl])
        assert np.array_equal(d.table(pkg.TAB_ISO_BLOCKS_L, 6), ib)
    if nr >= 1:
        ib, _ = isometry_blocks(cfg.sym, tabs[nr - 1], tabs[nr])
        assert np.array_equal(d.table(pkg.TAB_ISO_BLOCKS_R, 6), ib)
    # operator block table: every (kind, dq) class lists exactly the sector pairs q' = q + dq
    for tab_id, tab in ((pkg.TAB_OP_BLOCKS_L, tabs[nl]), (pkg.TAB_OP_BLOCKS_R, tabs[nr])):
        ob = d.table(tab_id, 7)
        labels = {(int(r[0]), int(r[1])): i for i, r in enumerate(tab)}
        seen = {}
        off = 0
        for kind, dN, dS, nmem, ibra, iket, o in ob:
            assert o == off
            off += nmem * tab[ibra][2] * tab[iket][2]
            assert (tab[iket][0] + dN, tab[iket][1] + dS) == (tab[ibra][0], tab[ibra][1])
            seen.setdefault((kind, dN, dS), set()).add((ibra, iket))
        for (kind, dN, dS), pairs in seen.items():
            want = {(labels[(q[0] + dN, q[1] + dS)], i) for q, i in labels.items()
                    if (q[0] + dN, q[1] + dS) in labels}
            assert pairs == want
    falg = int(d.table(pkg.TAB_FALG)[0])
    assert falg > 0
    d.close()


def test_cfg0_psi_length_is_fci_dimension(pkg):
    cfg = fx.get_config("cfg0")
    tabs = fx.block_tables(cfg)
    nl, nr = cfg.bond, cfg.L - cfg.bond - 2
    h, V, _ = fx.make_integrals(cfg.L, cfg.n_chol, 0)
    d = pkg.Dmrg(-1)
    d.init_integrals(h, V, None, 0.0, cfg.N, cfg.twoS, pkg.SYM_U1U1, cfg.D)
    d.set_mps(cfg.bond, tabs[:nl + 1], [], tabs[:nr + 1], [])
    d.plan_bond()
    assert d.psi_length() == 4900      # BASELINE.json configs[0]
    d.close()


@pytest.mark.parametrize("name,L,N,S2,D,bond", [("s", 6, 6, 0, 10, 2), ("q", 5, 5, 3, 9, 1), ("cfg2", 0, 0, 0, 0, 0)])
def test_su2_tables_bit_exact(pkg, name, L, N, S2, D, bond):
    """SU(2): psi block table (iL, s1, 2S_A, s2, iR, 2S_B, dL, dR, offset) against the oracle's own
    enumerator (oracle/su2.py psi_blocks), isometry block tables against fixtures, and the triangle
    rule of every reduced-operator class."""
    from oracle import su2
    if name == "cfg2":
        cfg = fx.get_config("cfg2")
    else:
        cfg = Config("t", L=L, N=N, twoS=S2, sym=1, D=D, n_chol=6, bond=bond)
    tabs = fx.block_tables(cfg)
    nl, nr = cfg.bond, cfg.L - cfg.bond - 2
    h, _, chol = fx.make_integrals(cfg.L, cfg.n_chol, 0, cfg.hdiag, want_V=False)
    d = pkg.Dmrg(-1)
    d.init_integrals(h, None, chol, 0.0, cfg.N, cfg.twoS, pkg.SYM_SU2, cfg.D)
    d.set_mps(cfg.bond, tabs[:nl + 1], [], tabs[:nr + 1], [])
    d.plan_bond()
    blocks, n = su2.psi_blocks(tabs[nl], tabs[nr], cfg.N, cfg.twoS)
    assert d.psi_length() == n
    assert np.array_equal(d.table(pkg.TAB_PSI_BLOCKS, 9), blocks)
    if nl >= 1:
        ib, _ = isometry_blocks(1, tabs[nl - 1], tabs[nl])
        assert np.array_equal(d.table(pkg.TAB_ISO_BLOCKS_L, 6), ib)
    if nr >= 1:
        ib, _ = isometry_blocks(1, tabs[nr - 1], tabs[nr])
        assert np.array_equal(d.table(pkg.TAB_ISO_BLOCKS_R, 6), ib)
    for tab_id, tab in ((pkg.TAB_OP_BLOCKS_L, tabs[nl]), (pkg.TAB_OP_BLOCKS_R, tabs[nr])):
        labels = {(int(r[0]), int(r[1])): i for i, r in enumerate(tab)}
        seen = {}
        for kind, dN, k2, nmem, ibra, iket, o in d.table(tab_id, 7):
            seen.setdefault((kind, dN, k2), set()).add((ibra, iket))
        for (kind, dN, k2), pairs in seen.items():
            want = set()
            for (Nq, Sq), i in labels.items():
                for Sp in range(abs(Sq - k2), Sq + k2 + 1, 2):
                    if (Nq + dN, Sp) in labels:
                        want.add((labels[(Nq + dN, Sp)], i))
            assert pairs == want
    counts = d.table(pkg.TAB_COUNTS)
    assert int(d.table(pkg.TAB_FALG)[0]) == int(counts[11] + counts[12]) > 0
    assert int(d.table(pkg.TAB_FALG_BLOCKS).sum()) == int(d.table(pkg.TAB_FALG)[0])
    d.close()


@pytest.mark.parametrize("name", ["cfg1", "cfg2"])
def test_emulated_plan_tables_without_a_gpu(name):
    """dmrg_replan on a planning context: the emulated plan moves stage-1 jobs and stage-2 segments to the INT8
    lists without changing what is computed (same psi blocks, same F_alg and per-stage flops); every emulated
    descriptor lies inside its slice buffer (checked by the planner, which throws otherwise)."""
    import paper_2603_28648_b200 as pkg
    case = make_case(0, 0, 0, 0, 0, cfg=fx.get_config(name))
    d = library_context(case, plan_only=True)
    c0, falg, blocks = d.table(pkg.TAB_COUNTS).copy(), int(d.table(pkg.TAB_FALG)[0]), d.table(pkg.TAB_PSI_BLOCKS).copy()
    assert c0[15] == 0 and c0[16] == 0 and c0[17] == 0 and c0[18] == 0
    d.replan(pkg.PREC_FP64_EMU, 6)
    c1 = d.table(pkg.TAB_COUNTS).copy()
    assert int(d.table(pkg.TAB_FALG)[0]) == falg and c1[11] == c0[11] and c1[12] == c0[12]
    assert np.array_equal(d.table(pkg.TAB_PSI_BLOCKS), blocks)
    assert 0 < c1[15] <= c1[12] and 0 < c1[18] <= c1[11]          # emulated part of stage 2 / stage 1
    assert c1[16] > 0 and c1[17] > 0 and c1[3] < c0[3]             # segments left the FP64 stage-2 list
    d.replan(pkg.PREC_FP64)
    assert np.array_equal(d.table(pkg.TAB_COUNTS), c0)
    with pytest.raises(pkg.DmrgError):
        d.replan(pkg.PREC_FP64_EMU, 8)
    d.replan(pkg.PREC_TF32X3)                                      # the 3xTF32 lists: same split, no fused emission
    c2 = d.table(pkg.TAB_COUNTS)
    assert c2[15] == c1[15] and c2[18] == c1[18] and c2[11] == c0[11] and c2[12] == c0[12]
    d.close()


def test_row_threshold_of_stage2_follows_the_sector_sizes():
    """Option emu_minm = 0 (default): output blocks of 8..31 rows join the tensor path only when the largest sector of
    the two blocks reaches 96 (plan_heff_jobs.cpp).  cfg1 (sectors <= 56) plans as with emu_minm = 32;
    configs[2] (sectors up to 125) as with emu_minm = 8."""
    import paper_2603_28648_b200 as pkg

    def emulated_stage2_flops(case, minm):
        d = library_context(case, plan_only=True, options={"emu_minm": minm})
        d.replan(pkg.PREC_FP64_EMU, 6)
        out = int(d.table(pkg.TAB_COUNTS)[15]), int(max(d.table(pkg.TAB_BOND_L, 4)[:, 2].max(), d.table(pkg.TAB_BOND_R, 4)[:, 2].max()))
        d.close()
        return out

    small = make_case(0, 0, 0, 0, 0, cfg=fx.get_config("cfg1"))
    a, maxdim = emulated_stage2_flops(small, 0)
    assert maxdim < 96
    assert a == emulated_stage2_flops(small, 32)[0] and a < emulated_stage2_flops(small, 8)[0]
    large = make_case(0, 0, 0, 0, 0, cfg=fx.get_config("cfg2"))
    b, maxdim = emulated_stage2_flops(large, 0)
    assert maxdim >= 96
    assert b == emulated_stage2_flops(large, 8)[0] and b > emulated_stage2_flops(large, 32)[0]


def _projectors(rows, data):
    """Per new sector: projector U U^T of the stacked isometry blocks (gauge free)."""
    out = {}
    for inext in sorted(set(int(r[2]) for r in rows)):
        blk = [data[int(r[5]):int(r[5]) + int(r[3]) * int(r[4])].reshape(int(r[3]), int(r[4])) for r in rows if int(r[2]) == inext]
        U = np.concatenate(blk, axis=0)
        out[inext] = U @ U.T
    return out


@pytest.mark.parametrize("args,D", [((5, 4, 0, 5, 2), 6), ((6, 6, 0, 12, 2), 9), ((5, 5, 1, 9, 2), 30), ((6, 6, 0, 12, 1), 4)])
@pytest.mark.parametrize("grow_left", [True, False])
def test_split_truncate_matches_the_oracle(args, D, grow_left):
    """Row a10 (host Jacobi in the library) against oracle/sweep.py: same kept sectors and counts (bit-exact
    table), same discarded weight, and the same kept subspaces (projectors; eigenvector signs are a gauge)."""
    import paper_2603_28648_b200 as pkg
    from oracle.sweep import split
    from tests.helpers import oracle_two_site
    case = make_case(*args)
    _, _, _, ts = oracle_two_site(case)
    d = library_context(case, plan_only=True)
    psi = fx.random_psi(ts.n, 9)
    tab_o, rows_o, data_o, disc_o = split(ts, psi, D, grow_left)
    tab_l, data_l, disc_l = d.split_truncate(psi, pkg.LEFT_TO_RIGHT if grow_left else pkg.RIGHT_TO_LEFT, D, on_device=False)
    assert np.array_equal(tab_l, tab_o)
    assert abs(disc_l - disc_o) < 1e-13
    assert len(data_l) == len(data_o)
    po, pl = _projectors(rows_o, data_o), _projectors(rows_o, data_l)
    for k in po:
        assert np.abs(po[k] - pl[k]).max() < 1e-9
    assert int(tab_l[:, 2].sum()) <= D and 0.0 <= disc_l < 1.0
    d.close()
