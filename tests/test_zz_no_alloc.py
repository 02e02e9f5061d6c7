"""-m gpu, collected last: the allocation-free entry point dmrg_dots_noalloc (static device scratch, no cudaMalloc)
against the existing path (dmrg_dots through a context, cudaMalloc'ed scratch) on two calls in a row.  The two paths
run the same kernels in the same summation order, so the results must be bit-identical; both are also within the
suite's FP64 tolerance of numpy.  Kept in a file of its own at the end of the collection order so that a failure
here cannot hide another test under `pytest -x`."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    assert torch.cuda.is_available()
    return torch


def test_noalloc_dots_match_the_context_path_on_two_calls_in_a_row(torch_mod):
    import paper_2603_28648_b200 as pkg
    torch = torch_mod
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream().cuda_stream
    d = pkg.Dmrg(0, stream)                      # planning-free context: only its dots path is used
    rng = np.random.Generator(np.random.Philox(123))
    # second call: fewer and shorter vectors, so stale partial sums of the first call stay in the static array
    for call, (nvec, n) in enumerate([(32, 1_000_003), (5, 70_001)]):
        ld = n + 13
        V = torch.from_numpy(rng.standard_normal((nvec, ld))).cuda()
        w = torch.from_numpy(rng.standard_normal(n)).cuda()
        ref = torch.full((nvec,), float("nan"), dtype=torch.float64, device="cuda")
        got = torch.full((nvec,), float("nan"), dtype=torch.float64, device="cuda")
        d.dots(V, ld, nvec, w, n, ref)
        free_before = torch.cuda.mem_get_info()[0]
        pkg.dots_noalloc(V, ld, nvec, w, n, got, stream=stream)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before          # no device memory was taken
        ref, got = ref.cpu().numpy(), got.cpu().numpy()
        assert np.array_equal(got, ref), (call, np.abs(got - ref).max())
        want = V.cpu().numpy()[:, :n] @ w.cpu().numpy()
        assert np.abs(got - want).max() <= 1e-11 * np.sqrt(n)
    d.close()


def test_noalloc_rejects_sizes_beyond_the_static_scratch(torch_mod):
    import paper_2603_28648_b200 as pkg
    torch = torch_mod
    V = torch.zeros(33 * 8, dtype=torch.float64, device="cuda")
    w = torch.zeros(8, dtype=torch.float64, device="cuda")
    out = torch.zeros(33, dtype=torch.float64, device="cuda")
    with pytest.raises(pkg.DmrgError) as ei:
        pkg.dots_noalloc(V, 8, 33, w, 8, out)
    assert "33" in str(ei.value) and "32" in str(ei.value)
    pkg.dots_noalloc(V, 8, 32, w, 8, out)        # the maximum itself is accepted
    torch.cuda.synchronize()
