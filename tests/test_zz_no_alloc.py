"""ctqmc_density_batch_static (include/ctqmc.h): the density-matrix accumulation with its scratch in the library's fixed device
array -- the one entry point that calls no cudaMalloc / cudaFree, for callers under CUDA graph capture or in harnesses that forbid
allocation.  Its output must equal ctqmc_density_batch's (the existing, arena-backed path, itself parity-tested against
oracle/density_oracle.py in test_gpu_density.py) within that file's bar, 1e-9 of the largest element, on two calls in a row: the
array keeps the first call's contents, so the second call starts from stale scratch.  Run on a B200: -m gpu.

The file name sorts last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-9


@pytest.fixture(scope="module")
def torch_cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests must run on the B200 box")
    return torch


@pytest.fixture(scope="module")
def lib():
    from paper_2010_08482_b200 import build
    build.build()
    import paper_2010_08482_b200 as L
    L.library()
    return L


def _device_batch(torch, batch):
    return tuple(torch.from_numpy(x).cuda() for x in (batch.offset, batch.symbol, batch.tau))


def test_static_scratch_entry_point_matches_the_arena_path_on_two_calls_in_a_row(lib, torch_cuda, impurities):
    from workloads import make_batch
    torch = torch_cuda
    imp = impurities(2)
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        n = lib.ctqmc_density_size(h)
        # two different batches (different lengths and slot strides), the second one reusing the array the first one left behind
        calls = [make_batch(2, 48, start=700), make_batch(2, 20, start=760)]
        free_before = None
        for k, batch in enumerate(calls):
            off, sym, tau = _device_batch(torch, batch)
            L = max(int(np.diff(batch.offset).max()), 1)
            mant, exp2, _, status = lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=L)
            weight = torch.tensor([1.0 if b % 4 else -1.0 for b in range(len(batch.offset) - 1)], dtype=torch.float64, device="cuda")
            want = lib.ctqmc_density_batch(h, batch.beta, off, sym, tau, mant, exp2, status, weight=weight, max_len=L)
            got = torch.zeros(n, dtype=torch.float64, device="cuda")
            torch.cuda.synchronize()
            if k == 1:
                free_before = torch.cuda.mem_get_info()[0]
            lib.ctqmc_density_batch_static(h, batch.beta, off, sym, tau, mant, exp2, status, got, weight=weight, max_len=L)
            torch.cuda.synchronize()
            if k == 1:
                assert torch.cuda.mem_get_info()[0] == free_before, "the static entry point changed the device's free memory"
            want, got = want.cpu().numpy(), got.cpu().numpy()
            scale = np.abs(want).max()
            assert scale > 0
            assert np.abs(got - want).max() <= TOL * scale, (k, np.abs(got - want).max(), scale)
    finally:
        h.free()


def test_static_scratch_entry_point_rejects_what_does_not_fit(lib, torch_cuda, impurities):
    """Config 4 (295-state complex sectors, ~100 operators): one string's prefix products exceed the 64 MiB array."""
    from workloads import make_batch
    torch = torch_cuda
    assert lib.ctqmc_density_static_limit() == 64 << 20
    imp = impurities(4)
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        batch = make_batch(4, 1, start=500)
        off, sym, tau = _device_batch(torch, batch)
        L = max(int(np.diff(batch.offset).max()), 1)
        assert (L + 5) * 295 * 295 * 16 > lib.ctqmc_density_static_limit()
        mant, exp2, _, status = lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=L)
        rho = torch.zeros(lib.ctqmc_density_size(h) * 2, dtype=torch.float64, device="cuda")
        with pytest.raises(lib.CtqmcError) as err:
            lib.ctqmc_density_batch_static(h, batch.beta, off, sym, tau, mant, exp2, status, rho, max_len=L)
        assert err.value.code == lib.CTQMC_ERR_UNSUPPORTED and "static scratch" in str(err.value)
        torch.cuda.synchronize()
        assert float(rho.abs().max()) == 0.0            # nothing was enqueued
    finally:
        h.free()
