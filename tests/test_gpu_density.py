"""Parity of ctqmc_density_batch (reduced density matrix estimator, Eq. 27) with
oracle/density_oracle.py on the same seeded batches.  Run on a B200: -m gpu.

Bar: every element of the accumulated rho within 1e-9 of the batch's largest element (the elements are sums of terms of both
signs whose natural scale is the weight of the configuration, i.e. O(1) per configuration), and trace(rho) = sum of the weights
of the contributing configurations to 1e-10 (pin D1 on the CUDA side)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


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


def _run(lib, torch, imp, batch, weight=None):
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        off, sym, tau = (torch.from_numpy(x).cuda() for x in (batch.offset, batch.symbol, batch.tau))
        L = max(int(np.diff(batch.offset).max()), 1)
        mant, exp2, _, status = lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=L)
        w = None if weight is None else torch.from_numpy(np.asarray(weight, dtype=np.float64)).cuda()
        rho = lib.ctqmc_density_batch(h, batch.beta, off, sym, tau, mant, exp2, status, weight=w, max_len=L)
        torch.cuda.synchronize()
        rho = rho.cpu().numpy()
        if imp.is_complex:
            rho = rho[0::2] + 1j * rho[1::2]
        return rho, status.cpu().numpy(), mant.cpu().numpy()
    finally:
        h.free()


def _trace_of(imp, rho):
    off2 = np.concatenate([[0], np.cumsum(np.asarray(imp.dims, dtype=np.int64) ** 2)])
    return sum(np.trace(rho[off2[q]:off2[q + 1]].reshape((int(imp.dims[q]),) * 2, order="F")) for q in range(len(imp.dims)))


@pytest.mark.parametrize("cfg,n", [(1, 24), (2, 12), (3, 2), (4, 1)])
def test_density_parity(lib, torch_cuda, impurities, cfg, n):
    from oracle import density_oracle as D
    from test_lazy_oracle import _imp_for
    from workloads import make_batch
    imp = _imp_for(impurities, cfg) if cfg == 3 else impurities(cfg)     # config 3 with all its quantum numbers (reading A8 (ii))
    batch = make_batch(cfg, n, start=500)
    weight = [1.0 if b % 3 else -1.0 for b in range(n)]
    rho, status, mant = _run(lib, torch_cuda, imp, batch, weight)
    want = D.density_batch(imp, batch.beta, batch.offset, batch.symbol, batch.tau, weight)
    scale = np.abs(want).max()
    assert scale > 0
    assert np.abs(rho - want).max() <= 1e-9 * scale, (cfg, np.abs(rho - want).max(), scale)
    wsum = sum(w for b, w in enumerate(weight) if status[b] == 0 and (mant[b] != 0).any())
    assert abs(_trace_of(imp, rho) - wsum) <= 1e-10 * n


def test_density_edge_cases(lib, torch_cuda, impurities):
    """Empty configuration (thermal state), an invalid and a structurally vanishing configuration (both contribute nothing),
    accumulation over two calls."""
    from oracle import density_oracle as D
    from workloads import Batch, make_batch
    imp = impurities(2)
    good = make_batch(2, 2, start=510)
    cfgs = [good.config(0), ([], []), ([1, 1, 1, 1], [1.0, 2.0, 3.0, 4.0]), ([1, 0], [3.0, 2.0]), good.config(1)]
    batch = Batch.from_lists(imp.beta, cfgs)
    rho, status, mant = _run(lib, torch_cuda, imp, batch)
    assert status.tolist() == [0, 0, 1, 2, 0]
    want = D.density_batch(imp, batch.beta, batch.offset, batch.symbol, batch.tau)
    assert np.abs(rho - want).max() <= 1e-9 * np.abs(want).max()
    assert abs(_trace_of(imp, rho) - 3.0) <= 1e-10
    # the empty configuration alone: diag(exp(-beta E)) / Z
    only = Batch.from_lists(imp.beta, [([], [])])
    rho1, _, _ = _run(lib, torch_cuda, imp, only)
    en = np.asarray(imp.energy)
    p = np.exp(-imp.beta * (en - en.min()))
    off = np.concatenate([[0], np.cumsum(imp.dims)])
    off2 = np.concatenate([[0], np.cumsum(np.asarray(imp.dims, dtype=np.int64) ** 2)])
    for q in range(imp.n_sectors):
        blk = rho1[off2[q]:off2[q + 1]].reshape((int(imp.dims[q]),) * 2, order="F")
        assert np.abs(blk - np.diag(p[off[q]:off[q + 1]] / p.sum())).max() <= 1e-14


def test_density_at_bench_size_has_the_weight_sum_as_its_trace(lib, torch_cuda, impurities):
    """BASELINE's batch of config 2 (4096 configurations, the launch bench.py times): pin D1 -- every contributing configuration
    adds a matrix of unit trace -- holds at any size, so trace(rho) must equal the sum of the weights of the configurations with
    status 0 and a non-zero weight; the first 16 configurations are also compared with the oracle element by element."""
    from oracle import density_oracle as D
    from workloads import Batch, make_batch
    imp = impurities(2)
    n = 4096
    batch = make_batch(2, n)
    weight = [1.0 if b % 5 else -1.0 for b in range(n)]
    rho, status, mant = _run(lib, torch_cuda, imp, batch, weight)
    wsum = sum(w for b, w in enumerate(weight) if status[b] == 0 and (mant[b] != 0).any())
    assert abs(_trace_of(imp, rho) - wsum) <= 1e-10 * n
    head = Batch.from_lists(imp.beta, [batch.config(b) for b in range(16)])
    rho16, _, _ = _run(lib, torch_cuda, imp, head, weight[:16])
    want = D.density_batch(imp, head.beta, head.offset, head.symbol, head.tau, weight[:16])
    assert np.abs(rho16 - want).max() <= 1e-9 * np.abs(want).max()
