"""Performant mode (DMRG_PREC_FP64_EMU_PERF; reading s21) against
oracle/ozaki.py: the kept-product arithmetic and the device's slice-count decisions bit for bit, the host rule entry
(no GPU), and H_eff.psi in performant mode against the FP64 oracle at the eager mode's tolerance."""
import numpy as np
import pytest

import fixtures as fx
from oracle import ozaki
from tests.helpers import EMU_EVERYTHING, make_case, oracle_two_site, oracle_su2, library_context, rel_err

TOL_EMU = 1e-10


def test_keep_rule_entry_matches_the_oracle_rule():
    """dmrg_emu_keep_rule needs no device: the library's rule (the function its kernel calls) against performant_keep."""
    import paper_2603_28648_b200 as pkg
    d = pkg.Dmrg(-1, None)
    rng = np.random.default_rng(5)
    for trial in range(200):
        n = int(rng.integers(1, 20))
        E_all = rng.integers(-200, 200, size=n).tolist()
        E_nz = [None if rng.random() < 0.2 else int(e - rng.integers(0, 12)) for e in E_all]
        for kappa, kmin in ((6, 3), (7, 2), (4, 4), (5, 1)):
            assert d.emu_keep_rule(E_all, E_nz, kappa, kmin) == ozaki.performant_keep(E_all, E_nz, kappa, kmin)
    assert d.emu_keep_rule([], [], 6, 3) == []
    with pytest.raises(pkg.DmrgError):
        d.emu_keep_rule([1], [1], 9, 3)
    d.close()


@pytest.fixture(scope="module")
def env():
    import torch
    import paper_2603_28648_b200 as pkg
    assert torch.cuda.is_available()
    d = pkg.Dmrg(0, torch.cuda.current_stream().cuda_stream)
    yield torch, d
    d.close()


def _wide(shape, seed):
    rng = np.random.Generator(np.random.Philox(seed))
    return rng.standard_normal(shape) * 10.0 ** rng.uniform(-6, 0, shape)


@pytest.mark.gpu
@pytest.mark.parametrize("M,N,K", [(150, 70, 200), (128, 64, 32), (37, 130, 4100)])
@pytest.mark.parametrize("kappa,keeps", [(6, (1, 3, 5, 6)), (7, (2, 6)), (4, (2,))])
def test_kept_products_bit_exact(env, M, N, K, kappa, keeps):
    torch, d = env
    A, B = _wide((M, K), 4), _wide((K, N), 5)
    Ad, Bd = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    for keep in keeps:
        Cd = torch.zeros((M, N), dtype=torch.float64, device="cuda")
        d.emu_gemm_kept(M, N, K, Ad, Bd, Cd, kappa, keep)
        assert np.array_equal(Cd.cpu().numpy(), ozaki.emulated_gemm(A, B, kappa, kc=16384, keep=keep)), (keep,)


@pytest.mark.gpu
def test_kept_products_argument_checks(env):
    import paper_2603_28648_b200 as pkg
    torch, d = env
    x = torch.zeros((32, 32), dtype=torch.float64, device="cuda")
    for keep in (0, 7):
        with pytest.raises(pkg.DmrgError):
            d.emu_gemm_kept(32, 32, 32, x, x, x.clone(), 6, keep)


@pytest.mark.gpu
@pytest.mark.parametrize("M,N,K", [(150, 70, 200), (60, 200, 96)])
@pytest.mark.parametrize("kappa,kmin", [(6, 3), (7, 2), (5, 5)])
def test_device_decisions_and_sum_bit_exact(env, M, N, K, kappa, kmin):
    """Classes spread over 40 bits, one with an all-zero B column and one with an all-zero A (exponent 0 everywhere):
    the device's slice counts equal the oracle's, and the sum equals emulated_sum bit for bit (alpha = +-2^j, so the
    kernel's fused multiply-add and the model's multiply-then-add round alike)."""
    torch, d = env
    rng = np.random.Generator(np.random.Philox(11))
    shifts = [3, -6, -7, -14, -23, -40, 2, -1]
    alpha = [1.0, -2.0, 0.5, 1.0, -4.0, 1.0, 0.25, 1.0]
    A = np.stack([rng.standard_normal((M, K)) * 2.0 ** 2 for _ in shifts])
    B = np.stack([rng.standard_normal((K, N)) * 2.0 ** s for s in shifts])
    B[2][:, 3] = 0.0
    A[6][:] = 0.0
    Ad, Bd = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    Cd = torch.zeros((M, N), dtype=torch.float64, device="cuda")
    keep = d.emu_sum_perf(M, N, K, Ad, Bd, alpha, Cd, kappa, kmin)
    want, keep_oracle = ozaki.emulated_sum([(al, a, b) for al, a, b in zip(alpha, A, B)], kappa, kmin)
    assert keep == keep_oracle
    assert len(set(keep)) > 1 or kappa == kmin              # the spread really lowers some classes
    assert np.array_equal(Cd.cpu().numpy(), want)
    exact = sum(al * (a @ b) for al, a, b in zip(alpha, A, B))
    ref_bound = max(ozaki.truncation_bound(ozaki.exponents(a, 1), ozaki.exponents(b, 0), K, kappa, kappa).max() * abs(al)
                    for al, a, b in zip(alpha, A, B))
    assert np.abs(Cd.cpu().numpy() - exact).max() <= len(shifts) * ref_bound * 1.01 or kappa == kmin


def _apply(torch, d, psi, precision, slices=0):
    x = torch.from_numpy(psi).cuda()
    y = torch.empty_like(x)
    d.heff_apply(x, y, precision, slices)
    return y.cpu().numpy()


@pytest.mark.gpu
@pytest.mark.parametrize("args,sym", [((6, 6, 0, 12, 2), 0), ((8, 8, 0, 40, 3), 0), ((6, 6, 2, 30, 2), 1), ((7, 6, 0, 24, 3), 1)])
def test_performant_apply_matches_oracle(args, sym):
    import torch
    import paper_2603_28648_b200 as pkg
    case = make_case(*args, sym=sym)
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream, options=EMU_EVERYTHING)
    if sym == 0:
        _, _, _, ts = oracle_two_site(case)
        psi = fx.random_psi(ts.n, 2)
        want = ts.apply(psi)
    else:
        o = oracle_su2(case)
        psi = fx.random_psi(d.psi_length(), 2)
        want = o.apply(psi)
    eager = _apply(torch, d, psi, pkg.PREC_FP64_EMU, 6)
    got = _apply(torch, d, psi, pkg.PREC_FP64_EMU_PERF, 6)
    kept, all_ = d.last_emu_products()
    assert 0 < kept <= all_
    assert rel_err(got, want) < TOL_EMU
    assert rel_err(eager, want) < TOL_EMU
    # the eager mode on the same plan afterwards: no decision of the performant call lingers
    again = _apply(torch, d, psi, pkg.PREC_FP64_EMU, 6)
    assert np.array_equal(again, eager)
    # kmin = kappa switches the truncation off: bit-identical to the eager mode
    d.set_option("emu_kmin", 6)
    same = _apply(torch, d, psi, pkg.PREC_FP64_EMU_PERF, 6)
    assert np.array_equal(same, eager)
    k2, a2 = d.last_emu_products()
    assert k2 == a2 == all_
    d.close()


@pytest.mark.gpu
def test_performant_apply_drops_products_when_the_classes_spread():
    """Two-electron integrals scaled by 2^-22: the classes that carry only V (A.P, B.Q, the V part of C.S) fall
    more than 16 bits below the one-electron classes, so the rule lets slices go; the result stays at the eager
    tolerance against the FP64 oracle of the same (scaled) Hamiltonian."""
    import torch
    import paper_2603_28648_b200 as pkg
    case = make_case(8, 8, 0, 40, 3)
    case["V"] = case["V"] * 2.0 ** -22
    d = library_context(case, stream=torch.cuda.current_stream().cuda_stream, options=EMU_EVERYTHING)
    _, _, _, ts = oracle_two_site(case)
    psi = fx.random_psi(ts.n, 2)
    want = ts.apply(psi)
    got = _apply(torch, d, psi, pkg.PREC_FP64_EMU_PERF, 6)
    kept, all_ = d.last_emu_products()
    assert kept < 0.9 * all_
    assert rel_err(got, want) < TOL_EMU
    d.close()


@pytest.mark.gpu
def test_sweep_in_performant_mode_reaches_fci():
    """dmrg_sweep with DMRG_PREC_FP64_EMU_PERF (every emulated job forced onto the tensor path; renormalization in the
    eager emulated mode, as the header says): an SU(2) singlet at saturated bond dimension ends at the FCI energy of its
    spin sector, to the accuracy of the 47-bit arithmetic."""
    import torch
    import paper_2603_28648_b200 as pkg
    from fixtures.configs import Config
    from tests.test_gpu_su2 import _fci_lowest_with_spin
    cfg = Config("t", L=6, N=6, twoS=0, sym=1, D=4096, n_chol=6, bond=0)
    h, V, _ = fx.make_integrals(cfg.L, cfg.n_chol, 0)
    tabs = fx.block_tables(cfg)
    e_fci = _fci_lowest_with_spin(h, V, cfg.N, cfg.twoS)
    rt = [tabs[m] for m in range(cfg.L - 1)]
    ri = [x[1] for x in fx.random_isometries(cfg, tabs, cfg.L - 2, 1001)]
    d = pkg.Dmrg(0, torch.cuda.current_stream().cuda_stream)
    for k, v in EMU_EVERYTHING.items():
        d.set_option(k, v)
    d.init_integrals(h, V, None, 0.0, cfg.N, cfg.twoS, 1, cfg.D)
    d.set_mps(0, [tabs[0]], [], rt, ri)
    energies, disc = d.sweep(2, cfg.D, davidson_iters=24, max_restarts=20, tol=1e-8, precision=pkg.PREC_FP64_EMU_PERF, slices=6, seed=3)
    assert len(energies) == 2 * 2 * (cfg.L - 1)
    assert abs(energies[-1] - e_fci) < 1e-7, (energies[-4:], e_fci)
    assert energies.min() > e_fci - 1e-7 and disc < 1e-10
    d.close()
