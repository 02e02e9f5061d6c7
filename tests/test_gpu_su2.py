"""-m gpu: SU(2) spin-adapted path through the C ABI against the expansion oracle (oracle/su2.py):
SURVEY.md 8(c) c4 / reading s20 -- expand(H_eff psi) = H_eff^{U(1)} expand(psi)."""
import numpy as np
import pytest

import fixtures as fx
from oracle import su2
from oracle.davidson import davidson
from tests.helpers import EMU_EVERYTHING, davidson_envelope, make_case, oracle_su2, library_context, rel_err, su2_block_components

pytestmark = pytest.mark.gpu
TOL_FP64 = 1e-11
# (L, N, 2S, D, bond): singlet, doublet, triplet, quartet, odd N, empty left block, larger D
CASES = [(4, 4, 0, 6, 1), (5, 5, 1, 8, 2), (5, 4, 2, 8, 1), (6, 6, 0, 10, 2), (5, 5, 3, 9, 0), (6, 7, 1, 12, 3),
         (6, 6, 2, 30, 2), (7, 6, 0, 24, 3)]


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    assert torch.cuda.is_available()
    return torch


def _apply(torch, d, psi):
    x = torch.from_numpy(psi).cuda()
    y = torch.empty_like(x)
    d.heff_apply(x, y)
    torch.cuda.synchronize()
    return y.cpu().numpy()


@pytest.mark.parametrize("L,N,S2,D,bond", CASES)
def test_su2_heff_diag_davidson(torch_mod, L, N, S2, D, bond):
    import paper_2603_28648_b200 as pkg
    torch = torch_mod
    case = make_case(L, N, S2, D, bond, sym=1)
    ex = oracle_su2(case)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream)
    n = d.psi_length()
    assert n == ex.n
    assert np.array_equal(d.table(pkg.TAB_PSI_BLOCKS, 9), ex.blocks)
    psi = fx.random_psi(n, 2)
    ref = ex.apply(psi)
    got = _apply(torch, d, psi)
    assert rel_err(got, ref) <= TOL_FP64
    u, w = fx.random_vector(n, 11), fx.random_vector(n, 12)
    assert abs(u @ _apply(torch, d, w) - w @ _apply(torch, d, u)) < 1e-12
    # a7 and a8 against the full reduced H_eff matrix of the oracle
    if n <= 250:
        H = np.stack([ex.apply(e) for e in np.eye(n)], axis=1)
        assert np.abs(H - H.T).max() < 1e-11
        dg = torch.empty(n, dtype=torch.float64, device="cuda")
        d.heff_diag(dg)
        assert np.abs(dg.cpu().numpy() - np.diag(H)).max() < 1e-11
        e0 = np.linalg.eigvalsh(0.5 * (H + H.T))[0]
        x = torch.from_numpy(psi).cuda()
        nit = min(8, n)
        theta, resid = d.davidson_step(x, nit)
        th0, rs0, env_t, env_r = davidson_envelope(lambda v: H @ v, np.diag(H).copy(), psi, nit)
        assert np.all(np.abs(theta - th0) <= env_t), (np.abs(theta - th0), env_t)     # every iteration (derived tolerance)
        assert np.abs(theta[:2] - th0[:2]).max() < 1e-9
        assert np.all(np.diff(theta) <= 1e-10) and np.all(theta >= e0 - 1e-10)
        xv = x.cpu().numpy()
        assert abs(xv @ H @ xv - theta[-1]) < 1e-9
        x2 = torch.from_numpy(psi).cuda()
        th2, rs2 = d.davidson_step(x2, min(32, n), tol=1e-9)
        if rs2[-1] < 1e-9:
            assert abs(th2[-1] - e0) < 1e-8
    d.close()


@pytest.mark.parametrize("mode,tol", [(0, 1e-11), (1, 1e-10), (2, 1e-5)])
@pytest.mark.parametrize("L,N,S2,D,bond", [(5, 5, 1, 8, 2), (6, 6, 0, 10, 2), (6, 7, 1, 12, 3)])
def test_su2_renormalized_operators_are_the_reduced_elements(torch_mod, L, N, S2, D, bond, mode, tol):
    """a9 in SU(2): every stored reduced operator equals the Wigner-Eckart projection of the expanded
    U(1)xU(1) oracle operator (and that projection is m-independent, i.e. the operators are tensors)."""
    import paper_2603_28648_b200 as pkg
    torch = torch_mod
    case = make_case(L, N, S2, D, bond, sym=1)
    ex = oracle_su2(case)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream, precision=mode, slices=6)   # a9 in every mode
    tabs, nl, nr = case["tabs"], case["nl"], case["nr"]
    for side, blk, tab, orbs in ((0, ex.Lb, tabs[nl], list(range(nl))), (1, ex.Rb, tabs[nr], list(range(bond + 2, L)))):
        if not orbs:
            continue
        outside = [x for x in range(L) if x not in orbs]
        todo = [("H", -1, -1, 0)] + [("C", p, -1, 0) for p in orbs] + [("S", x, -1, 0) for x in outside]
        for p in orbs:
            for r in orbs:
                todo += [("B", p, r, 0), ("B", p, r, 2)]
                if p <= r:
                    todo.append(("A", p, r, 0))
                if p < r:
                    todo.append(("A", p, r, 2))
        offs = np.concatenate([[0], np.cumsum(tab[:, 2])])
        kind_id = {"H": pkg.OP_H, "C": pkg.OP_C, "S": pkg.OP_S, "A": pkg.OP_A, "B": pkg.OP_B}
        for kind, p, r, rank in todo:
            comps, k2 = su2_block_components(blk, kind, p, r, rank)
            red, worst = su2.reduced_blocks(comps, k2, tab)
            assert worst < 1e-11, (kind, p, r, rank)
            got = d.op_export(side, kind_id[kind] | (rank << 8), p, r)
            ref = np.zeros_like(got)
            for (ib, ik), m in red.items():
                ref[offs[ib]:offs[ib + 1], offs[ik]:offs[ik + 1]] = m
            assert np.abs(got - ref).max() <= tol * max(1.0, np.abs(ref).max()), (side, kind, p, r, rank)
    d.close()


def _abelian_library_on_expansion(torch, case, M2):
    """The library's own U(1)xU(1) path fed with the Wigner-Eckart expansion of an SU(2) state."""
    import paper_2603_28648_b200 as pkg
    cfg, tabs, nl, nr = case["cfg"], case["tabs"], case["nl"], case["nr"]
    lt, li, rt, ri = [su2.expand_table(tabs[0])[0]], [], [su2.expand_table(tabs[0])[0]], []
    for m in range(nl):
        ta, tb, _, dat = su2.expand_isometry(tabs[m], tabs[m + 1], case["isoL"][m][0], case["isoL"][m][1], True)
        lt.append(tb); li.append(dat)
    for m in range(nr):
        ta, tb, _, dat = su2.expand_isometry(tabs[m], tabs[m + 1], case["isoR"][m][0], case["isoR"][m][1], False)
        rt.append(tb); ri.append(dat)
    d = pkg.Dmrg(0, torch.cuda.current_stream().cuda_stream)
    d.init_integrals(case["h"], case["V"], None, 0.0, cfg.N, M2, pkg.SYM_U1U1, cfg.D)
    d.set_mps(cfg.bond, lt, li, rt, ri)
    d.build_env()
    return d


@pytest.mark.parametrize("L,N,S2,D,bond", [(12, 18, 0, 64, 5), (12, 15, 3, 48, 5), (36, 54, 0, 256, 17)])
def test_su2_equals_abelian_on_the_expanded_state(torch_mod, L, N, S2, D, bond):
    """Reading s20 (BASELINE.json configs[2]: "abelian-vs-SU(2) singlet equivalence at D=256"):
    expand(H_eff psi) = H_eff^{U(1)} expand(psi) and equal <psi|H_eff|psi>, with the two symmetry
    paths of the library on the GPU and the oracle's Clebsch-Gordan expansion in between.  The last
    case is the CAS(54,36)-shaped system itself (L=36, N=54, singlet) at D_SU(2) = 256."""
    torch = torch_mod
    hdiag = "spread" if L == 36 else "default"
    case = make_case(L, N, S2, D, bond, nchol=48 if L == 36 else 8, sym=1, hdiag=hdiag)
    cfg, tabs, nl, nr = case["cfg"], case["tabs"], case["nl"], case["nr"]
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream)
    n = d.psi_length()
    psi = fx.random_psi(n, 2)
    y = _apply(torch, d, psi)
    d.close()
    M2 = S2
    da = _abelian_library_on_expansion(torch, case, M2)
    full = su2.expand_psi(psi, tabs[nl], tabs[nr], cfg.N, S2, M2)
    assert len(full) == da.psi_length()
    yf = _apply(torch, da, full)
    da.close()
    ref = su2.expand_psi(y, tabs[nl], tabs[nr], cfg.N, S2, M2)
    assert rel_err(ref, yf) <= TOL_FP64
    assert abs(psi @ y - full @ yf) < 1e-10 * max(1.0, abs(psi @ y))


def test_cfg2_full_size_invariants(torch_mod):
    """configs[2] at full size (D_SU(2) = 2048, len psi ~ 2e6): no oracle reaches this size, so parity
    is pinned at D = 256 above and here only the invariants are checked: H_eff symmetric through the
    CUDA path and Davidson Ritz values monotone and consistent with H_eff."""
    torch = torch_mod
    cfg = fx.get_config("cfg2")
    case = make_case(0, 0, 0, 0, 0, cfg=cfg)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream)
    n = d.psi_length()
    u, w = fx.random_vector(n, 11), fx.random_vector(n, 12)
    Hu, Hw = _apply(torch, d, u), _apply(torch, d, w)
    assert abs(w @ Hu - u @ Hw) < 1e-10 * np.linalg.norm(Hu)
    x = torch.from_numpy(u).cuda()
    theta, resid = d.davidson_step(x, 6)
    assert abs(theta[0] - u @ Hu) < 1e-9 * abs(theta[0])
    assert np.all(np.diff(theta) <= 1e-9)
    xv = x.cpu().numpy()
    Hx = _apply(torch, d, xv)
    assert abs(xv @ Hx - theta[-1]) < 1e-8 * abs(theta[-1])
    assert abs(np.linalg.norm(Hx - theta[-1] * xv) - resid[-1]) < 1e-7 * max(1.0, resid[-1])
    d.close()


def _fci_lowest_with_spin(h, V, N, S2):
    """Lowest FCI eigenvalue of total spin exactly S = S2 / 2: the S_z = S sector holds every multiplet
    with S' >= S, the S_z = S + 1 sector those with S' >= S + 1; the difference of the two spectra (as
    multisets) is the spin-S spectrum."""
    from oracle import fock
    nup, ndn = (N + S2) // 2, (N - S2) // 2
    lo = np.linalg.eigvalsh(fock.fci_matrix(h, V, nup, ndn)[0])
    hi = np.linalg.eigvalsh(fock.fci_matrix(h, V, nup + 1, ndn - 1)[0]) if ndn >= 1 and nup + 1 <= h.shape[0] else np.array([])
    hi = list(hi)
    for e in lo:
        j = next((i for i, x in enumerate(hi) if abs(x - e) < 1e-9), None)
        if j is None:
            return float(e)
        hi.pop(j)
    raise AssertionError("no state of the requested spin")


@pytest.mark.parametrize("L,N,S2,bond,emulated", [(6, 6, 0, 2, False), (6, 6, 2, 2, False), (6, 5, 1, 2, False),
                                                 (6, 7, 1, 2, False), (6, 6, 0, 2, True)])
def test_su2_saturated_bond_has_the_fci_energy_of_its_spin(torch_mod, L, N, S2, bond, emulated):
    """At saturated bond dimension the reduced two-site space is the whole (N, S) sector in a rotated basis
    (the isometries are square), so the lowest eigenvalue of the spin-adapted H_eff is the FCI energy of the
    lowest state with that total spin, whatever the random isometries are."""
    import paper_2603_28648_b200 as pkg
    case = make_case(L, N, S2, 4096, bond, sym=1)
    d = library_context(case, stream=torch_mod.cuda.current_stream().cuda_stream,
                        options=EMU_EVERYTHING if emulated else None)
    n = d.psi_length()
    from math import comb                              # Weyl's dimension of the (N, S) sector: the bond is saturated
    assert n == (S2 + 1) * comb(L + 1, (N - S2) // 2) * comb(L + 1, (N + S2) // 2 + 1) // (L + 1)
    x = torch_mod.from_numpy(fx.random_psi(n, 11)).cuda()
    prec, kap = (pkg.PREC_FP64_EMU, 7) if emulated else (pkg.PREC_FP64, 0)
    theta = resid = None
    for _ in range(20):                              # restarted Davidson
        theta, resid = d.davidson_step(x, min(24, n), 1e-10, prec, kap)
        if resid[-1] < 1e-9:
            break
    assert resid[-1] < 1e-8
    e_fci = _fci_lowest_with_spin(case["h"], case["V"], N, S2)
    assert abs(theta[-1] - e_fci) < 1e-8
    d.close()


@pytest.mark.parametrize("L,N,S2", [(6, 6, 0), (6, 5, 1)])
def test_su2_sweeps_with_the_library_split_reach_fci(torch_mod, L, N, S2):
    """Full spin-adapted two-site sweeps through the C ABI alone (dmrg_set_mps / dmrg_build_env /
    dmrg_davidson_step / dmrg_split_truncate, rows a2-a10) at saturated bond dimension end at the FCI energy
    of the target spin."""
    import paper_2603_28648_b200 as pkg
    from fixtures.configs import Config
    torch = torch_mod
    cfg = Config("t", L=L, N=N, twoS=S2, sym=1, D=4096, n_chol=6, bond=2)
    h, V, _ = fx.make_integrals(L, cfg.n_chol, 0)
    tabs = fx.block_tables(cfg)
    e_fci = _fci_lowest_with_spin(h, V, N, S2)
    lt, li = [tabs[0]], []
    rt = [tabs[m] for m in range(L - 1)]
    ri = [x[1] for x in fx.random_isometries(cfg, tabs, L - 2, 1001)]
    d = pkg.Dmrg(0, torch.cuda.current_stream().cuda_stream)
    d.init_integrals(h, V, None, 0.0, N, S2, pkg.SYM_SU2, cfg.D)

    def solve(p):
        nl, nr = p, L - p - 2
        d.set_mps(p, lt[:nl + 1], li[:nl], rt[:nr + 1], ri[:nr])
        d.build_env()
        n = d.psi_length()
        x = torch.from_numpy(fx.random_psi(n, 100 + p)).cuda()
        theta = resid = None
        for _ in range(20):
            theta, resid = d.davidson_step(x, min(24, n), tol=1e-10)
            if resid[-1] < 1e-9:
                break
        return theta[-1], x

    energies = []
    for sweep in range(2):
        for p in range(0, L - 1):
            e, psi = solve(p)
            energies.append(e)
            if p < L - 2:
                tab, data, _ = d.split_truncate(psi, pkg.LEFT_TO_RIGHT, cfg.D)
                lt[p + 1:] = [tab]
                li[p:] = [data]
        for p in range(L - 2, -1, -1):
            e, psi = solve(p)
            energies.append(e)
            if p > 0:
                tab, data, _ = d.split_truncate(psi, pkg.RIGHT_TO_LEFT, cfg.D)
                m = L - p - 2
                rt[m + 1:] = [tab]
                ri[m:] = [data]
    d.close()
    assert abs(energies[-1] - e_fci) < 1e-8, (energies[-4:], e_fci)
    assert min(energies) > e_fci - 1e-8


@pytest.mark.parametrize("L,N,S2,D,bond", [(5, 5, 1, 8, 2), (6, 6, 0, 10, 2), (6, 7, 1, 12, 3), (6, 6, 2, 30, 2), (7, 6, 0, 24, 3)])
def test_su2_reduced_precision_modes_against_the_oracle(torch_mod, L, N, S2, D, bond):
    """Emulated FP64 at kappa = 6 (<= 1e-10) and 3xTF32 (<= 1e-5) on SU(2) systems against oracle/su2.py, every stage-1
    job and two-sided stage-2 segment forced onto the tensor cores (round 1 compared these modes with the native
    path only)."""
    import paper_2603_28648_b200 as pkg
    torch = torch_mod
    case = make_case(L, N, S2, D, bond, sym=1)
    ex = oracle_su2(case)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream, options=EMU_EVERYTHING)
    psi = fx.random_psi(ex.n, 2)
    ref = ex.apply(psi)
    x = torch.from_numpy(psi).cuda()
    y = torch.empty_like(x)
    d.heff_apply(x, y, pkg.PREC_FP64_EMU, 6)
    torch.cuda.synchronize()
    c = d.table(pkg.TAB_COUNTS)
    assert c[15] > 0 and c[18] > 0
    assert rel_err(y.cpu().numpy(), ref) <= 1e-10
    d.heff_apply(x, y, pkg.PREC_TF32X3, 0)
    torch.cuda.synchronize()
    e = rel_err(y.cpu().numpy(), ref)
    assert 1e-10 < e <= 1e-5
    d.close()
