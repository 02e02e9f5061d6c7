"""-m gpu: the Ozaki-emulated FP64 engine (INT8 tcgen05) against oracle/ozaki.py (SURVEY.md 8(c)
"Emulated mode": digits bit-exact, INT32 partial sums through a bit-exact final result, <= 1e-10 against
the FP64 product, error falling ~2^-8 per added slice)."""
import numpy as np
import pytest

from oracle import ozaki

pytestmark = pytest.mark.gpu


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


@pytest.mark.parametrize("kappa", [3, 6, 7])
def test_slices_and_exponents_bit_exact(env, kappa):
    torch, d = env
    a = _wide((45, 333), 1)
    a[3] = 0.0
    A = torch.from_numpy(a).cuda()
    for by_rows in (True, False):          # rows of A, and columns of A (the B-operand orientation)
        lines, K = (45, 333) if by_rows else (333, 45)
        ls, ks = (333, 1) if by_rows else (1, 333)
        out = torch.zeros((kappa, lines, K), dtype=torch.int8, device="cuda")
        ex = torch.zeros(lines, dtype=torch.int32, device="cuda")
        d.emu_slice(A, lines, K, ls, ks, kappa, out, ex)
        src = a if by_rows else a.T
        e = ozaki.exponents(src, 1)
        dig, _ = ozaki.slice_lines(src, e, kappa, 1)
        assert np.array_equal(ex.cpu().numpy().astype(np.int64), e)
        assert np.array_equal(out.cpu().numpy().astype(np.int64), dig)


@pytest.mark.parametrize("M,N,K", [(128, 64, 32), (200, 100, 1000), (37, 130, 77), (300, 64, 4096), (64, 64, 40000)])
def test_emulated_gemm_matches_the_integer_model(env, M, N, K):
    torch, d = env
    A, B = _wide((M, K), 2), _wide((K, N), 3)
    Ad, Bd = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    Cd = torch.zeros((M, N), dtype=torch.float64, device="cuda")
    d.emu_gemm(M, N, K, Ad, Bd, Cd, 6)
    got = Cd.cpu().numpy()
    model = ozaki.emulated_gemm(A, B, 6, kc=16384)         # same K chunking as the kernel
    assert np.array_equal(got, model)                      # digits, INT32 sums and recombination order agree bit for bit
    ref = A @ B
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 1e-10


def test_error_falls_with_the_slice_count(env):
    torch, d = env
    rng = np.random.Generator(np.random.Philox(9))
    A, B = rng.standard_normal((256, 2048)), rng.standard_normal((2048, 128))
    ref = A @ B
    Ad, Bd = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    errs = []
    for kappa in (3, 4, 5, 6, 7):
        Cd = torch.zeros((256, 128), dtype=torch.float64, device="cuda")
        d.emu_gemm(256, 128, 2048, Ad, Bd, Cd, kappa)
        errs.append(np.linalg.norm(Cd.cpu().numpy() - ref) / np.linalg.norm(ref))
    for a, b in zip(errs[:3], errs[1:4]):
        assert b < a / 50
    assert errs[3] < 1e-11 and errs[4] < 1e-13


def test_int8_tensor_pipe_self_check_and_peak(env):
    """dmrg_measure_peak(EMU) first checks one tcgen05 kind::i8 MMA (and an accumulating sequence)
    element by element against the integer definition, then times full-tile MMAs on every SM."""
    import paper_2603_28648_b200 as pkg
    torch, d = env
    p = d.measure_peak(pkg.PREC_FP64_EMU)
    assert 2.0e15 < p < 5.0e15          # nominal 4.5 Pop/s dense INT8 on B200


def test_tf32_self_check_and_peak(env):
    """dmrg_measure_peak(TF32X3) first checks accumulating tcgen05 kind::tf32 MMAs against their exact value."""
    import paper_2603_28648_b200 as pkg
    torch, d = env
    p = d.measure_peak(pkg.PREC_TF32X3)
    assert 2e14 < p < 3e15


def test_tf32_split_bit_exact(env):
    """Row a4 of the 3xTF32 mode: the device split against oracle/ozaki.py tf32_split, bit for bit, on wide-range data,
    ties, zeros and values near the FP32 rounding boundary."""
    torch, d = env
    rng = np.random.Generator(np.random.Philox(21))
    x = np.concatenate([rng.standard_normal(100003) * 10.0 ** rng.uniform(-12, 12, 100003),
                        [0.0, -0.0, 1.0 + 2.0 ** -11, -(1.0 + 2.0 ** -11), 1.0 + 2.0 ** -24, 1.0 + 2.0 ** -12 + 2.0 ** -40, 3.0e38, 1e-30]])
    xd = torch.from_numpy(x).cuda()
    hi = torch.zeros(len(x), dtype=torch.int32, device="cuda")
    lo = torch.zeros(len(x), dtype=torch.int32, device="cuda")
    d.tf32_split(xd, len(x), hi, lo)
    h0, l0 = ozaki.tf32_split(x)
    assert np.array_equal(hi.cpu().numpy().view(np.uint32), h0.view(np.uint32))
    assert np.array_equal(lo.cpu().numpy().view(np.uint32), l0.view(np.uint32))
