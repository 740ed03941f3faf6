"""Pins for oracle/density_oracle.py (Eq. 27): the analytically integrated estimator of the
reduced density matrix must (D1) have unit trace for every configuration, because sum_u P_uu = 1 turns the integrand into
w_loc(C) / w_loc(C); (D2) reduce to diag(exp(-beta E)) / Z on the empty configuration; (D3) equal the Gauss-Legendre quadrature
over tau of oracle.trace_oracle.trace_config -- itself pinned by brute force -- with the projector |v><u| inserted as one more
operator symbol, element by element including off-diagonal ones."""
import math
import types

import numpy as np
import pytest

from oracle import density_oracle as D
from oracle import trace_oracle as O
from workloads import make_batch


def _with_projector(base, q, u, v):
    """`base` plus one symbol (index n_symbols) whose only block is |v><u| inside sector q (element (m, n) = <m|O|n>)."""
    d = int(base.dims[q])
    blk = np.zeros((d, d), dtype=np.complex128 if base.is_complex else np.float64)
    blk[v, u] = 1.0
    data = np.asarray(base.blk_data)
    return types.SimpleNamespace(dims=base.dims, energy=base.energy, n_symbols=base.n_symbols + 1, is_complex=base.is_complex,
                                 blk_symbol=np.append(base.blk_symbol, base.n_symbols).astype(np.int32),
                                 blk_src=np.append(base.blk_src, q).astype(np.int32), blk_dst=np.append(base.blk_dst, q).astype(np.int32),
                                 blk_offset=np.append(base.blk_offset, len(data)).astype(np.int64),
                                 blk_data=np.concatenate([data, blk.ravel(order="F")]))


def _value(r):
    return complex(r["mant"]) * 2.0 ** r["exp2"] if r["mant"] != 0 else 0j


@pytest.mark.parametrize("cfg,n", [(1, 6), (2, 4), (4, 1)])
def test_D1_unit_trace_for_every_configuration(impurities, cfg, n):
    imp = impurities(cfg)
    batch = make_batch(cfg, n, start=60)
    for b in range(n):
        s, t = batch.config(b)
        r = D.density_config(imp, batch.beta, s, t)
        assert r["status"] == 0
        tr = sum(np.trace(m) for m in r["rho"])
        assert abs(tr - 1.0) < 1e-10, (cfg, b, tr)


def test_D2_empty_configuration_is_the_thermal_state(impurities):
    imp = impurities(2)
    r = D.density_config(imp, imp.beta, np.zeros(0, np.int32), np.zeros(0))
    en = np.asarray(imp.energy)
    Z = math.fsum(np.exp(-imp.beta * (en - en.min())))
    off = np.concatenate([[0], np.cumsum(imp.dims)])
    for q in range(imp.n_sectors):
        want = np.diag(np.exp(-imp.beta * (en[off[q]:off[q + 1]] - en.min()))) / Z
        assert np.max(np.abs(r["rho"][q] - want)) < 1e-14


@pytest.mark.parametrize("cfg,b", [(1, 3), (2, 1)])
def test_D3_equals_the_quadrature_of_the_trace_with_an_inserted_projector(impurities, cfg, b):
    imp = impurities(cfg)
    batch = make_batch(cfg, b + 1, start=70)
    s, t = batch.config(b)
    beta = batch.beta
    r = D.density_config(imp, beta, s, t)
    w = _value(O.trace_config(imp, beta, s, t))
    # the sector with the largest weight, its two largest diagonal entries and the largest off-diagonal entries
    q = int(np.argmax([abs(np.trace(m)) for m in r["rho"]]))
    rho = r["rho"][q]
    d = rho.shape[0]
    pairs = [(u, u) for u in np.argsort(-np.abs(np.diag(rho)))[:2]]
    offd = np.abs(rho - np.diag(np.diag(rho)))
    if d > 1 and offd.max() > 0:
        u, v = np.unravel_index(int(np.argmax(offd)), offd.shape)
        pairs += [(int(u), int(v)), (int(v), int(u))]
    x, wt = np.polynomial.legendre.leggauss(8)
    edges = [0.0] + [float(z) for z in t] + [float(beta)]
    scale = max(np.abs(rho).max(), 1e-300)
    for u, v in pairs:
        ext = _with_projector(imp, q, u, v)
        total = 0j
        for a, c in zip(edges[:-1], edges[1:]):
            if c <= a:
                continue
            for xi, wi in zip(x, wt):
                tau = 0.5 * (a + c) + 0.5 * (c - a) * xi
                k = int(np.searchsorted(t, tau))
                s2 = np.insert(s, k, imp.n_symbols).astype(np.int32)
                t2 = np.insert(t, k, tau)
                total += 0.5 * (c - a) * wi * _value(O.trace_config(ext, beta, s2, t2))
        want = total / (beta * w)
        got = rho[u, v]
        assert abs(got - want) <= 1e-9 * scale, (cfg, q, u, v, got, want)
