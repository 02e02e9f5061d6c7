"""-m gpu: H_eff.psi in the emulated-FP64 mode (DMRG_PREC_FP64_EMU: stage 2 on the INT8 tensor cores,
rows a4/a6 of SURVEY.md section 8) against the CPU oracle and against the native FP64 path of the library
(north_star tolerance: relative Frobenius error <= 1e-10 in emulated mode)."""
import numpy as np
import pytest

import fixtures as fx
from tests.helpers import EMU_EVERYTHING, make_case, oracle_two_site, library_context, rel_err

pytestmark = pytest.mark.gpu

TOL_EMU = 1e-10


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture
def emu_everything():
    """Options (dmrg_set_option) that lower the size thresholds so that every stage-1 job and every two-sided
    stage-2 segment runs emulated."""
    return dict(EMU_EVERYTHING)


def _apply(torch, d, psi, precision=0, slices=0):
    x = torch.from_numpy(psi).cuda()
    y = torch.empty_like(x)
    d.heff_apply(x, y, precision, slices)
    torch.cuda.synchronize()
    return y.cpu().numpy()


def _counts(d):
    import paper_2603_28648_b200 as pkg
    return d.table(pkg.TAB_COUNTS)


@pytest.mark.parametrize("args", [(4, 4, 0, 16, 1), (6, 6, 0, 12, 2), (5, 5, 1, 9, 2), (8, 8, 0, 40, 3)])
@pytest.mark.parametrize("kappa", [6, 7])
def test_emulated_apply_matches_oracle(torch_mod, emu_everything, args, kappa):
    OPTS = emu_everything
    import paper_2603_28648_b200 as pkg
    case = make_case(*args)
    _, _, _, ts = oracle_two_site(case)
    d = library_context(case, stream=torch_mod.cuda.current_stream().cuda_stream, options=OPTS)
    psi = fx.random_psi(ts.n, 2)
    want = ts.apply(psi)
    n_fp64_segs = _counts(d)[3]
    got = _apply(torch_mod, d, psi, pkg.PREC_FP64_EMU, kappa)   # 6: the paper's 47-bit mode, what bench.py times
    c = _counts(d)
    assert c[3] < n_fp64_segs                   # segments really moved to the emulated lists
    assert c[15] > 0 and c[18] == c[11]         # stage 2 partly, stage 1 entirely on the INT8 tensor cores
    assert rel_err(got, want) < TOL_EMU
    back = _apply(torch_mod, d, psi)             # switching back re-plans for native FP64
    assert _counts(d)[3] == n_fp64_segs
    assert rel_err(back, want) < 1e-11
    d.close()


@pytest.mark.parametrize("sym", [0, 1])
def test_emulated_error_falls_with_slices(torch_mod, emu_everything, sym):
    OPTS = emu_everything
    import paper_2603_28648_b200 as pkg
    case = make_case(8, 8, 0, 48, 3, sym=sym)
    d = library_context(case, stream=torch_mod.cuda.current_stream().cuda_stream, options=OPTS)
    psi = fx.random_psi(d.psi_length(), 3)
    ref = _apply(torch_mod, d, psi)
    errs = [rel_err(_apply(torch_mod, d, psi, pkg.PREC_FP64_EMU, k), ref) for k in (3, 4, 5, 6, 7)]
    assert errs[-1] < 1e-13 and errs[-2] < 1e-11
    for a, b in zip(errs[:-2], errs[1:-1]):       # ~2^-8 per added slice until the FP64 floor
        assert b < a / 32
    assert 1e-9 < errs[0] < 1e-4
    d.close()


def test_emulated_multi_pass_and_mixed_lists(torch_mod):
    """Thresholds that leave part of the two-sided segments in FP64 (both kinds meet in the split-K partial
    slots); a small T budget then forces several passes."""
    OPTS = {}
    import paper_2603_28648_b200 as pkg
    opts = {"emu_mink": 64, "emu_minm": 16, "emu_minn": 16, "emu_minm1": 24}
    case = make_case(10, 10, 0, 300, 4)
    stream = torch_mod.cuda.current_stream().cuda_stream
    d = library_context(case, stream=stream, options=opts)
    psi = fx.random_psi(d.psi_length(), 4)
    ref = _apply(torch_mod, d, psi)
    segs_fp64 = _counts(d)[3]
    one = _apply(torch_mod, d, psi, pkg.PREC_FP64_EMU)
    c = _counts(d)
    assert c[3] < segs_fp64 and c[14] == 1 and 0 < c[18] < c[11]
    assert rel_err(one, ref) < 1e-12
    d.close()
    d2 = library_context(case, stream=stream, options=dict(opts, scratch_gb=0.002))
    many = _apply(torch_mod, d2, psi, pkg.PREC_FP64_EMU)
    assert _counts(d2)[14] > 1
    assert rel_err(many, ref) < 1e-12
    d2.close()


def test_emulated_davidson(torch_mod, emu_everything):
    OPTS = emu_everything
    import paper_2603_28648_b200 as pkg
    case = make_case(8, 8, 0, 40, 3)
    d = library_context(case, stream=torch_mod.cuda.current_stream().cuda_stream, options=OPTS)
    psi = fx.random_psi(d.psi_length(), 5)
    x0 = torch_mod.from_numpy(psi).cuda()
    th0, rs0 = d.davidson_step(x0, 4)
    x1 = torch_mod.from_numpy(psi).cuda()
    th1, rs1 = d.davidson_step(x1, 4, 0.0, pkg.PREC_FP64_EMU, 7)
    assert np.abs(th1[:2] - th0[:2]).max() < 1e-9
    assert np.all(np.diff(th1) <= 1e-10)
    assert abs(th1[-1] - th0[-1]) < 1e-6
    d.close()


def test_emulated_rejects_bad_slices(torch_mod):
    OPTS = {}
    import paper_2603_28648_b200 as pkg
    case = make_case(4, 4, 0, 16, 1)
    d = library_context(case, stream=torch_mod.cuda.current_stream().cuda_stream, options=OPTS)
    x = torch_mod.zeros(d.psi_length(), dtype=torch_mod.float64, device="cuda")
    y = torch_mod.zeros_like(x)
    with pytest.raises(Exception):
        d.heff_apply(x, y, pkg.PREC_FP64_EMU, 9)
    with pytest.raises(Exception):
        d.heff_apply(x, y, 7, 0)                  # unknown precision mode
    d.close()


TOL_TF32 = 1e-5


@pytest.mark.parametrize("args,sym", [((6, 6, 0, 12, 2), 0), ((5, 5, 1, 9, 2), 0), ((8, 8, 0, 40, 3), 0), ((8, 8, 0, 48, 3), 1)])
def test_tf32x3_apply_within_its_tolerance(torch_mod, emu_everything, args, sym):
    """3xTF32 mode (hi/lo TF32 split, three products, FP32 accumulation in TMEM): <= 1e-5 relative Frobenius
    error (BASELINE.json north_star), and visibly not the FP64 path."""
    OPTS = emu_everything
    import paper_2603_28648_b200 as pkg
    case = make_case(*args, sym=sym)
    d = library_context(case, stream=torch_mod.cuda.current_stream().cuda_stream, options=OPTS)
    psi = fx.random_psi(d.psi_length(), 6)
    ref = _apply(torch_mod, d, psi)
    if sym == 0:
        _, _, _, ts = oracle_two_site(case)
        assert rel_err(ref, ts.apply(psi)) < 1e-11
    got = _apply(torch_mod, d, psi, pkg.PREC_TF32X3)
    c = _counts(d)
    assert c[15] > 0 and c[18] == c[11]
    err = rel_err(got, ref)
    assert 1e-10 < err < TOL_TF32
    x = torch_mod.from_numpy(psi).cuda()
    th, rs = d.davidson_step(x, 3, 0.0, pkg.PREC_TF32X3)
    x0 = torch_mod.from_numpy(psi).cuda()
    th0, rs0 = d.davidson_step(x0, 3)
    assert abs(th[0] - th0[0]) < 1e-4 * max(1.0, abs(th0[0]))
    d.close()


def test_emulated_stage2_gangs_multi_tile_blocks(torch_mod):
    """psi' blocks wider than one 128 x 64 tile (d_R' = 94): their stage-2 tiles run as gangs (kernels.cu up_tiles,
    GangSync).  Sampled output blocks against the oracle (seeded sample, largest included), and
    the schedule must not change a bit of the result."""
    OPTS = {}
    import paper_2603_28648_b200 as pkg
    case = make_case(12, 12, 0, 900, 5)
    _, _, _, ts = oracle_two_site(case)
    stream = torch_mod.cuda.current_stream().cuda_stream
    d = library_context(case, stream=stream)
    blocks = np.asarray(d.table(pkg.TAB_PSI_BLOCKS)).reshape(-1, 7)
    assert (blocks[:, 5] > 64).sum() > 0                      # jobs with more than one n-tile exist
    psi = fx.random_psi(ts.n, 2)
    shapes = {k: m.shape for k, m in ts.unpack(psi).items()}
    keys = sorted(shapes, key=lambda k: (-shapes[k][0] * shapes[k][1], k))
    rng = np.random.Generator(np.random.Philox(5))
    sample = set(keys[:3]) | {keys[i] for i in rng.choice(len(keys), 5, replace=False)}
    want = ts.unpack(ts.apply(psi, only_outputs=sample))
    got_flat = _apply(torch_mod, d, psi, pkg.PREC_FP64_EMU, 6)
    c = _counts(d)
    assert c[15] > 0 and c[18] > 0                            # both stages have emulated lists
    got = ts.unpack(got_flat)
    num = sum(np.linalg.norm(got[k] - want[k]) ** 2 for k in sample)
    den = sum(np.linalg.norm(want[k]) ** 2 for k in sample)
    assert den > 0 and (num / den) ** 0.5 < TOL_EMU
    d.close()
    d2 = library_context(case, stream=stream, options={"emu_gang": 0})
    plain = _apply(torch_mod, d2, psi, pkg.PREC_FP64_EMU, 6)
    d2.close()
    assert np.array_equal(got_flat, plain)


def test_emulated_stage2_piece_cutting_against_the_oracle(torch_mod, emu_everything):
    """Stage-2 contractions longer than one piece are cut at operator-member boundaries into pieces with their own
    exponent sets.  With the default piece length (K <= 16384) that happens at configs[2..4] (K up to 1e5), which
    tests/test_gpu_fullsize.py compares with the oracle; here the option emu_kpiece shortens the pieces so that
    the same cutting runs on a system the oracle covers completely."""
    import paper_2603_28648_b200 as pkg
    case = make_case(8, 8, 0, 60, 3)
    _, _, _, ts = oracle_two_site(case)
    psi = fx.random_psi(ts.n, 2)
    want = ts.apply(psi)
    stream = torch_mod.cuda.current_stream().cuda_stream
    d = library_context(case, stream=stream, options=emu_everything)
    whole = _apply(torch_mod, d, psi, pkg.PREC_FP64_EMU, 6)
    n_whole = _counts(d)[16]
    d.close()
    d = library_context(case, stream=stream, options=dict(emu_everything, emu_kpiece=64))
    cut = _apply(torch_mod, d, psi, pkg.PREC_FP64_EMU, 6)
    assert _counts(d)[16] > n_whole                       # more emulated segments: the pieces
    d.close()
    assert rel_err(whole, want) < TOL_EMU and rel_err(cut, want) < TOL_EMU


def test_options_are_validated(torch_mod):
    import paper_2603_28648_b200 as pkg
    d = pkg.Dmrg(0, torch_mod.cuda.current_stream().cuda_stream)
    for key, val in (("no_such_option", 1), ("tile", 40), ("emu_gang", 2), ("emu_kpiece", 8), ("scratch_gb", -1.0), ("emu_mink", 1.5)):
        with pytest.raises(pkg.DmrgError) as ei:
            d.set_option(key, val)
        assert ei.value.code == pkg.EINVAL
    d.set_option("tile", 48)
    d.close()
