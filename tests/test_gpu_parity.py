"""-m gpu: the CUDA path through the C ABI against the CPU oracle, element by element
(tolerances of BASELINE.json north_star: H_eff.psi relative Frobenius error
<= 1e-11 in native FP64; tables bit-exact)."""
import numpy as np
import pytest

import fixtures as fx
from oracle.davidson import davidson
from tests.helpers import davidson_envelope, make_case, oracle_two_site, library_context, rel_err

pytestmark = pytest.mark.gpu

TOL_FP64 = 1e-11
KIND = {"H": 1, "C": 2, "S": 3, "A": 4, "B": 5}


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


def _check_davidson(torch, d, ts, psi, nit, Heff):
    """Davidson (oracle c6), EVERY iteration against the oracle's sequence within a tolerance derived from the
    arithmetic (tests/helpers.py davidson_envelope; pinned in tests/test_oracle_davidson.py): the preconditioner
    r_i / (theta - diag_i) has near-singular denominators on random environments, so rounding-level differences
    between two correct implementations grow by orders of magnitude per iteration; the envelope is that growth,
    measured on the oracle with rounding-level noise.  Then what is unique whatever the rounding: monotone Ritz
    values, the variational bound, and that the returned vector, Ritz value and residual norm are consistent
    with the oracle's H_eff."""
    x = torch.from_numpy(psi).cuda()
    theta, resid = d.davidson_step(x, nit)
    big = len(psi) > 5000                      # cfg1: one oracle matvec takes seconds
    th0, rs0, env_t, env_r = davidson_envelope(ts.apply, ts.diagonal(), psi, nit, trials=1 if big else 6,
                                               safety=30.0 if big else 8.0)
    assert len(theta) == nit
    assert np.all(np.abs(theta - th0) <= env_t), (np.abs(theta - th0), env_t)
    assert np.all(np.abs(resid - rs0) <= env_r + 1e-9 * np.maximum(1.0, rs0)), (np.abs(resid - rs0), env_r)
    assert np.abs(theta[:2] - th0[:2]).max() < 1e-9          # and the first two tightly, as before
    assert np.all(np.diff(theta) <= 1e-10)
    xv = x.cpu().numpy()
    assert abs(np.linalg.norm(xv) - 1) < 1e-12
    Hx = ts.apply(xv)
    assert abs(xv @ Hx - theta[-1]) < 1e-9
    assert abs(np.linalg.norm(Hx - theta[-1] * xv) - resid[-1]) < 1e-8
    if Heff is not None:
        e0 = np.linalg.eigvalsh(0.5 * (Heff + Heff.T))[0]
        assert np.all(theta >= e0 - 1e-10)
        # run to convergence: the eigenvalue is unique
        x2 = torch.from_numpy(psi).cuda()
        th2, rs2 = d.davidson_step(x2, min(32, len(psi)), tol=1e-9)
        if rs2[-1] < 1e-9:
            assert abs(th2[-1] - e0) < 1e-8


# small cases: several sectors, ragged block sizes (1..7), odd N, Sz != 0, edge bond (empty left block)
SMALL = [(4, 4, 0, 16, 1), (5, 4, 0, 5, 2), (5, 5, 1, 9, 2), (6, 6, 0, 12, 2), (5, 6, 2, 6, 1),
         (5, 5, -1, 7, 0), (6, 5, 1, 40, 3), (7, 7, 1, 30, 3)]


@pytest.mark.parametrize("L,N,tw,D,bond", SMALL)
def test_small_cases_full_parity(torch_mod, L, N, tw, D, bond):
    import paper_2603_28648_b200 as pkg
    torch = torch_mod
    case = make_case(L, N, tw, D, bond)
    ints, Lb, Rb, ts = oracle_two_site(case)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream)
    n = d.psi_length()
    assert n == ts.n
    assert np.array_equal(d.table(pkg.TAB_PSI_BLOCKS, 7), ts.blocks)
    # a9: every renormalized operator of both blocks
    for side, blk in ((0, Lb), (1, Rb)):
        if not blk.orbs:
            continue
        for key, op in blk.store.items():
            i = key[1] if len(key) > 1 else -1
            k = key[2] if len(key) > 2 else -1
            got = d.op_export(side, KIND[key[0]], i, k)
            assert np.abs(got - op.dense(blk.basis)).max() < 1e-12, (side, key)
    # a5 + a6
    psi = fx.random_psi(n, 2)
    ref = ts.apply(psi)
    got = _apply(torch, d, psi)
    assert rel_err(got, ref) <= TOL_FP64
    # host-buffer entry point gives the same bits
    out = np.zeros(n)
    d.heff_apply_host(psi, out)
    assert np.array_equal(out, got)
    # a7
    dg = torch.empty(n, dtype=torch.float64, device="cuda")
    d.heff_diag(dg)
    assert np.abs(dg.cpu().numpy() - ts.diagonal()).max() < 1e-12
    # hermiticity through the CUDA path
    u, w = fx.random_vector(n, 11), fx.random_vector(n, 12)
    assert abs(u @ _apply(torch, d, w) - w @ _apply(torch, d, u)) < 1e-12
    # a8
    Heff = np.stack([ts.apply(e) for e in np.eye(n)], axis=1) if n <= 400 else None
    _check_davidson(torch, d, ts, psi, min(8, n), Heff)
    d.close()


def test_renormalize_call_matches_oracle(torch_mod):
    """dmrg_renormalize absorbs one more site with a caller-given isometry (oracle c5)."""
    import paper_2603_28648_b200 as pkg
    from fixtures.configs import Config
    from oracle import abelian as ab
    torch = torch_mod
    case = make_case(6, 6, 0, 14, 2)
    cfg, tabs = case["cfg"], case["tabs"]
    ints, Lb, Rb, ts = oracle_two_site(case)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream)
    rng = np.random.Generator(np.random.Philox(77))
    # left block absorbs site `bond`; right block absorbs site bond+1
    blocksL, dataL = fx.random_isometry(cfg.sym, tabs[2], tabs[3], rng)
    blocksR, dataR = fx.random_isometry(cfg.sym, tabs[2], tabs[3], rng)
    newL = ab.renormalize(Lb, ab.site_block(ints, cfg.bond), blocksL, dataL, tabs[3], True)
    newR = ab.renormalize(Rb, ab.site_block(ints, cfg.bond + 1), blocksR, dataR, tabs[3], False)
    d.renormalize(pkg.LEFT_TO_RIGHT, tabs[3], dataL)
    d.renormalize(pkg.RIGHT_TO_LEFT, tabs[3], torch.from_numpy(dataR).cuda(), on_device=True)
    for side, blk in ((0, newL), (1, newR)):
        for key, op in blk.store.items():
            i = key[1] if len(key) > 1 else -1
            k = key[2] if len(key) > 2 else -1
            got = d.op_export(side, KIND[key[0]], i, k)
            assert np.abs(got - op.dense(blk.basis)).max() < 1e-12, (side, key)
    with pytest.raises(pkg.DmrgError):          # the old bond's plan is gone
        d.psi_length()
    d.close()


def test_cfg0_centre_bond(torch_mod):
    """BASELINE.json configs[0]: L=8, N=8, D=256 (saturated), centre bond; len(psi) = 4900."""
    torch = torch_mod
    cfg = fx.get_config("cfg0")
    case = make_case(0, 0, 0, 0, 0, cfg=cfg)
    ints, Lb, Rb, ts = oracle_two_site(case)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream)
    assert d.psi_length() == 4900
    psi = fx.random_psi(4900, 2)
    ref = ts.apply(psi)
    got = _apply(torch, d, psi)
    assert rel_err(got, ref) <= TOL_FP64
    dg = torch.empty(4900, dtype=torch.float64, device="cuda")
    d.heff_diag(dg)
    assert np.abs(dg.cpu().numpy() - ts.diagonal()).max() < 1e-11
    _check_davidson(torch, d, ts, psi, 8, None)
    d.close()


def test_cfg1_centre_bond_all_sector_pairs(torch_mod):
    """BASELINE.json configs[1]: L=24, N=24, D=512; the oracle (c3) is checked on the full set of
    sector pairs: every psi block, the diagonal, hermiticity, and the Davidson step (8 iterations).
    The oracle needs about 3-4 minutes of CPU time for its environment and term list."""
    import paper_2603_28648_b200 as pkg
    torch = torch_mod
    cfg = fx.get_config("cfg1")
    case = make_case(0, 0, 0, 0, 0, cfg=cfg)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream)
    n = d.psi_length()
    psi = fx.random_psi(n, 2)
    got = _apply(torch, d, psi)
    ints, Lb, Rb, ts = oracle_two_site(case)
    assert n == ts.n and np.array_equal(d.table(pkg.TAB_PSI_BLOCKS, 7), ts.blocks)
    ref = ts.apply(psi)
    assert rel_err(got, ref) <= TOL_FP64
    for (iL, s1, s2, iR, dL, dR, off) in ts.blocks:          # block by block, not only in the norm
        a, b = got[off:off + dL * dR], ref[off:off + dL * dR]
        assert np.linalg.norm(a - b) <= 1e-11 * max(np.linalg.norm(ref), 1.0)
    dg = torch.empty(n, dtype=torch.float64, device="cuda")
    d.heff_diag(dg)
    assert np.abs(dg.cpu().numpy() - ts.diagonal()).max() < 1e-10
    u, w = fx.random_vector(n, 11), fx.random_vector(n, 12)
    assert abs(u @ _apply(torch, d, w) - w @ _apply(torch, d, u)) < 1e-11
    _check_davidson(torch, d, ts, psi, 8, None)
    # a sample of renormalized operators of both blocks (a9 chained over 11 sites each)
    for side, blk in ((0, Lb), (1, Rb)):
        keys = sorted(blk.store.keys(), key=str)
        for key in keys[:: max(1, len(keys) // 12)]:
            i = key[1] if len(key) > 1 else -1
            k = key[2] if len(key) > 2 else -1
            got_op = d.op_export(side, KIND[key[0]], i, k)
            ref_op = blk.store[key].dense(blk.basis)
            assert np.abs(got_op - ref_op).max() < 1e-11 * max(1.0, np.abs(ref_op).max()), (side, key)
    d.close()


@pytest.mark.parametrize("tile", [32, 48, 64])
def test_every_tile_size_matches_oracle(torch_mod, tile):
    """The three instantiations of k_gemm_f64 (CTA tile 32/48/64) on a case with ragged sectors
    (dimensions 1..40, so tiles have partial rows, columns and K blocks, and strips/split-K kick in)."""
    torch = torch_mod
    case = make_case(7, 7, 1, 120, 3)
    ints, Lb, Rb, ts = oracle_two_site(case)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream, options={"tile": tile})
    n = d.psi_length()
    psi = fx.random_psi(n, 2)
    assert rel_err(_apply(torch, d, psi), ts.apply(psi)) <= TOL_FP64
    for side, blk in ((0, Lb), (1, Rb)):
        for key in list(blk.store.keys())[::7]:
            i = key[1] if len(key) > 1 else -1
            k = key[2] if len(key) > 2 else -1
            assert np.abs(d.op_export(side, KIND[key[0]], i, k) - blk.store[key].dense(blk.basis)).max() < 1e-12
    d.close()


@pytest.mark.parametrize("library_split", [False, True])
def test_cfg0_sweeps_reach_fci_energy(torch_mod, library_split):
    """BASELINE.json configs[0]: full two-site sweeps at D=256 (saturated) through the C ABI
    (dmrg_set_mps / dmrg_build_env / dmrg_davidson_step per bond; the split-and-truncate support
    step a10 is the library's dmrg_split_truncate or, as a cross-check, the oracle's) reach the
    determinant-FCI energy within 1e-8 Eh (exact at saturated bond dimension;
    BASELINE.json north_star)."""
    import paper_2603_28648_b200 as pkg
    from oracle import abelian as ab
    from oracle import fock
    from oracle.sweep import split
    torch = torch_mod
    cfg = fx.get_config("cfg0")
    L, D = cfg.L, cfg.D
    h, V, _ = fx.make_integrals(L, cfg.n_chol, 0)
    tabs = fx.block_tables(cfg)
    ints = ab.Integrals(h, V)
    Hf, _ = fock.fci_matrix(h, V, cfg.N // 2, cfg.N // 2)
    e_fci = np.linalg.eigvalsh(Hf)[0]
    lt, li = [tabs[0]], []                              # left block grows from the vacuum
    rt = [tabs[m] for m in range(L - 1)]                # random right-canonical start
    ri = [x[1] for x in fx.random_isometries(cfg, tabs, L - 2, 1001)]
    d = pkg.Dmrg(0, torch.cuda.current_stream().cuda_stream)
    d.init_integrals(h, V, None, 0.0, cfg.N, cfg.twoS, pkg.SYM_U1U1, D)

    def shell(tab, first, n):                           # oracle block with a basis and no operators
        orbs = [i for p in range(first, first + n) for i in (2 * p, 2 * p + 1)]
        return ab.Block(ints, orbs, ab.Basis.from_table(tab))

    def solve(p):
        nl, nr = p, L - p - 2
        d.set_mps(p, lt[:nl + 1], li[:nl], rt[:nr + 1], ri[:nr])
        d.build_env()
        n = d.psi_length()
        x = torch.from_numpy(fx.random_psi(n, 100 + p)).cuda()
        for _ in range(12):
            theta, resid = d.davidson_step(x, min(24, n), tol=1e-10)
            if resid[-1] < 1e-9:
                break
        ts = ab.TwoSite(shell(lt[nl], 0, nl), ab.site_block(ints, p), ab.site_block(ints, p + 1),
                        shell(rt[nr], p + 2, nr), cfg.N, cfg.twoS)
        assert ts.n == n
        return theta[-1], resid[-1], ts, x

    energies = []
    for sweep in range(2):
        for p in range(0, L - 1):                       # rightward
            e, r, ts, psi = solve(p)
            energies.append(e)
            if p < L - 2:
                if library_split:
                    tab, data, _ = d.split_truncate(psi, pkg.LEFT_TO_RIGHT, D)
                else:
                    tab, _, data, _ = split(ts, psi.cpu().numpy(), D, True)
                lt[p + 1:] = [tab]
                li[p:] = [data]
        for p in range(L - 2, -1, -1):                  # leftward
            e, r, ts, psi = solve(p)
            energies.append(e)
            if p > 0:
                if library_split:
                    tab, data, _ = d.split_truncate(psi, pkg.RIGHT_TO_LEFT, D)
                else:
                    tab, _, data, _ = split(ts, psi.cpu().numpy(), D, False)
                m = L - p - 2
                rt[m + 1:] = [tab]
                ri[m:] = [data]
    d.close()
    assert abs(energies[-1] - e_fci) < 1e-8, (energies[-6:], e_fci)
    assert min(energies) > e_fci - 1e-8                 # variational


@pytest.mark.parametrize("name,L,N,S2,sym", [("cfg0", 8, 8, 0, 0), ("su2", 6, 6, 0, 1), ("su2", 6, 5, 1, 1)])
def test_device_sweep_driver_reaches_fci(torch_mod, name, L, N, S2, sym):
    """dmrg_sweep: two-site sweeps entirely inside the library (H_eff plan, Davidson, split
    and truncate, renormalization; blocks of both sides resident on the device) at saturated bond dimension end at
    the FCI energy of the target sector; every bond energy obeys the variational bound."""
    import paper_2603_28648_b200 as pkg
    from fixtures.configs import Config
    from oracle import fock
    torch = torch_mod
    cfg = fx.get_config("cfg0") if name == "cfg0" else Config("t", L=L, N=N, twoS=S2, sym=1, D=4096, n_chol=6, bond=0)
    h, V, _ = fx.make_integrals(cfg.L, cfg.n_chol, 0)
    tabs = fx.block_tables(cfg)
    if sym == 0:
        e_fci = np.linalg.eigvalsh(fock.fci_matrix(h, V, cfg.N // 2, cfg.N // 2)[0])[0]
    else:
        from tests.test_gpu_su2 import _fci_lowest_with_spin
        e_fci = _fci_lowest_with_spin(h, V, N, S2)
    rt = [tabs[m] for m in range(cfg.L - 1)]
    ri = [x[1] for x in fx.random_isometries(cfg, tabs, cfg.L - 2, 1001)]
    d = pkg.Dmrg(0, torch.cuda.current_stream().cuda_stream)
    d.init_integrals(h, V, None, 0.0, cfg.N, cfg.twoS, sym, cfg.D)
    d.set_mps(0, [tabs[0]], [], rt, ri)
    energies, disc = d.sweep(2, cfg.D, davidson_iters=24, max_restarts=20, tol=1e-9, seed=3)
    assert len(energies) == 2 * 2 * (cfg.L - 1)
    assert abs(energies[-1] - e_fci) < 1e-8, (energies[-4:], e_fci)
    assert energies.min() > e_fci - 1e-8 and disc < 1e-12
    d.close()


def test_cholesky_ingest_equals_the_four_index_ingest(torch_mod):
    """a1: dmrg_init_integrals with chol != NULL and V = NULL (V_ijkl = sum_c B^c_ij B^c_kl) against the oracle, which
    takes the four-index V of the fixture; and the Davidson driver is safe when asked for more iterations than the
    space has dimensions or started from an exact eigenvector."""
    torch = torch_mod
    case = make_case(6, 6, 0, 12, 2)
    ints, Lb, Rb, ts = oracle_two_site(case)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream, use_chol=True)
    psi = fx.random_psi(ts.n, 2)
    assert rel_err(_apply(torch, d, psi), ts.apply(psi)) <= TOL_FP64
    d.close()
    # n_iter > dim: the basis is clamped to the dimension and n_done says so
    small = make_case(4, 3, 1, 16, 1)
    _, _, _, ts2 = oracle_two_site(small)
    d = library_context(small, stream=torch.cuda.current_stream().cuda_stream)
    n = d.psi_length()
    assert n < 32
    H = np.stack([ts2.apply(e) for e in np.eye(n)], axis=1)
    x = torch.from_numpy(fx.random_psi(n, 3)).cuda()
    theta, resid = d.davidson_step(x, 32)
    assert len(theta) <= n and np.all(np.isfinite(theta)) and np.all(np.isfinite(x.cpu().numpy()))
    e0 = np.linalg.eigvalsh(0.5 * (H + H.T))[0]
    assert theta[-1] >= e0 - 1e-10 and abs(theta[-1] - e0) < 1e-8       # the full space was spanned
    # exact eigenvector start with tol <= 0: no NaN, the Ritz value stays, the expansion stops
    w, U = np.linalg.eigh(0.5 * (H + H.T))
    x = torch.from_numpy(U[:, 0].copy()).cuda()
    theta, resid = d.davidson_step(x, 6)
    assert np.all(np.isfinite(theta)) and abs(theta[-1] - w[0]) < 1e-10 and np.all(theta >= w[0] - 1e-10)
    assert np.all(np.isfinite(x.cpu().numpy()))
    d.close()


RENORM_TOL = {1: 1e-10, 2: 1e-5}       # emulated FP64 (kappa = 6), 3xTF32: BASELINE.json north_star tolerances


@pytest.mark.parametrize("mode", [1, 2])
@pytest.mark.parametrize("L,N,tw,D,bond", [(6, 6, 0, 12, 2), (7, 7, 1, 30, 3), (8, 8, 0, 40, 3)])
def test_renormalization_in_reduced_precision_modes(torch_mod, L, N, tw, D, bond, mode):
    """a9 in the emulated and 3xTF32 modes (SURVEY.md 8(a) a9 "FP64 / emulated / 3xTF32"; PAPER.md:53-59 runs all GEMMs
    emulated): dmrg_build_env with the mode renormalizes every site through the tensor-core rotation; every stored
    operator of both blocks against oracle c5, relative to the operator's largest element (errors of the earlier
    sites ride along, as in a sweep)."""
    import paper_2603_28648_b200 as pkg
    torch = torch_mod
    case = make_case(L, N, tw, D, bond)
    ints, Lb, Rb, ts = oracle_two_site(case)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream, precision=mode, slices=6)
    KIND = {"H": pkg.OP_H, "C": pkg.OP_C, "S": pkg.OP_S, "A": pkg.OP_A, "B": pkg.OP_B}
    worst, n_ops = 0.0, 0
    for side, blk in ((0, Lb), (1, Rb)):
        for key, op in blk.store.items():
            i, k = (list(key[1:]) + [-1, -1])[:2]
            got = d.op_export(side, KIND[key[0]], i, k)
            ref = op.dense(blk.basis)
            scale = max(1.0, np.abs(ref).max())
            worst = max(worst, np.abs(got - ref).max() / scale)
            n_ops += 1
    assert n_ops > 50
    assert worst <= RENORM_TOL[mode], worst
    if mode == 2:
        assert worst > 1e-10                               # it really is the TF32 path
    # and the H_eff built on those operators, in the same mode, stays within the mode's tolerance of the oracle
    psi = fx.random_psi(ts.n, 2)
    x = torch.from_numpy(psi).cuda()
    y = torch.empty_like(x)
    d.heff_apply(x, y, mode, 6)
    torch.cuda.synchronize()
    assert rel_err(y.cpu().numpy(), ts.apply(psi)) <= 10 * RENORM_TOL[mode]
    d.close()


def test_sweeps_stop_at_eps_sweep(torch_mod):
    """the sweeps end "once the energy difference between three subsequent sweeps dropped below
    eps_sweep" (option sweep_eps).  A truncated run (D = 12 on L = 6) asked for 10 sweeps stops early, after at least
    three; its sweep energies stay above E_FCI, and the last three differ by less than eps."""
    import paper_2603_28648_b200 as pkg
    from fixtures.configs import Config
    from oracle import fock
    torch = torch_mod
    cfg = Config("t", L=6, N=6, twoS=0, sym=0, D=12, n_chol=6, bond=0)
    h, V, _ = fx.make_integrals(cfg.L, cfg.n_chol, 0)
    tabs = fx.block_tables(cfg)
    e_fci = np.linalg.eigvalsh(fock.fci_matrix(h, V, 3, 3)[0])[0]
    rt = [tabs[m] for m in range(cfg.L - 1)]
    ri = [x[1] for x in fx.random_isometries(cfg, tabs, cfg.L - 2, 1001)]
    eps = 1e-6
    d = pkg.Dmrg(0, torch.cuda.current_stream().cuda_stream)
    d.set_option("sweep_eps", eps)
    d.init_integrals(h, V, None, 0.0, cfg.N, cfg.twoS, 0, cfg.D)
    d.set_mps(0, [tabs[0]], [], rt, ri)
    energies, disc = d.sweep(10, cfg.D, davidson_iters=24, max_restarts=20, tol=1e-10, seed=3)
    per = 2 * (cfg.L - 1)
    assert len(energies) % per == 0
    n_run = len(energies) // per
    assert 3 <= n_run < 10, n_run
    e_sw = energies.reshape(n_run, per).min(axis=1)
    assert e_sw.min() > e_fci - 1e-9              # variational (a truncated two-site sweep need not be monotone)
    assert abs(e_sw[-1] - e_sw[-2]) < eps and abs(e_sw[-2] - e_sw[-3]) < eps
    if n_run > 3:                                   # it did not stop a sweep too late
        assert not (abs(e_sw[-2] - e_sw[-3]) < eps and abs(e_sw[-3] - e_sw[-4]) < eps)
    with pytest.raises(pkg.DmrgError):
        d.set_option("sweep_eps", -1.0)
    d.close()
