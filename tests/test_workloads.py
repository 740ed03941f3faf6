"""Pins for the input builder: things the paper and textbook atomic physics fix."""
import os

import numpy as np
import pytest

from workloads import impurity as wi
from workloads import make_batch, BASELINE_CONFIGS


def _golden():
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_pins.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                out[k.strip()] = float(v)
    return out


def test_paper_block_ranks():
    g = _golden()
    _, _, twomj = wi.f_shell_coupled([4.5, 6.1, 4.1, 3.0], 0.3)
    qn_f = [(1, m) for m in twomj]
    d = wi.sector_dimensions(14, qn_f)
    assert sum(d.values()) == g["fock_dim_f_shell"]
    assert max(d.values()) == g["max_block_f_high_symmetry"]
    assert max(wi.sector_dimensions(14, qn_f, modulo=(0, 8)).values()) == g["max_block_f_low_symmetry"]
    qn_d = [(1, -1, m) for m in range(-2, 3)] + [(1, 1, m) for m in range(-2, 3)]
    dd = wi.sector_dimensions(10, qn_d, modulo=(0, 0, 4))
    assert sum(dd.values()) == g["fock_dim_d_shell"]
    assert max(dd.values()) == g["max_block_d_fig1"]


def test_delta_pu_parameters():
    g = _golden()
    F2, F4, F6 = 6.1, 4.1, 3.0
    assert abs((286 * F2 + 195 * F4 + 250 * F6) / 6435 - g["delta_pu_J"]) < 5e-4
    assert g["delta_pu_U"] == 4.5


def test_kanamori_spectra():
    U, J = 4.0, 0.8
    h1, u, qn = wi._kanamori(2, U, J, 0.0)
    imp = wi.build_impurity("k2", h1, u, qn, 1.0)
    e = np.sort(np.concatenate([imp.energy_of(q) for q, l in enumerate(imp.labels) if l[0] == 2]))
    np.testing.assert_allclose(e, sorted([U - 3 * J] * 3 + [U - J] * 2 + [U + J]), atol=1e-12)
    U, J = 3.0, 0.5
    h1, u, qn = wi._kanamori(3, U, J, 0.0)
    imp = wi.build_impurity("k3", h1, u, qn, 1.0)
    e = np.sort(np.concatenate([imp.energy_of(q) for q, l in enumerate(imp.labels) if l[0] == 2]))
    np.testing.assert_allclose(e, sorted([U - 3 * J] * 9 + [U - J] * 5 + [U + 2 * J]), atol=1e-12)


def test_slater_d2_terms():
    F0, F2, F4 = 6.0, 8.4, 5.3
    u = wi.spin_orbital_tensor(wi.slater_orbital_tensor(2, [F0, F2, F4]))
    imp = wi.build_impurity("d", np.zeros((10, 10)), u, [(1,)] * 10, 1.0)
    f2, f4 = F2 / 49, F4 / 441
    expect = sorted([F0 - 8 * f2 - 9 * f4] * 21 + [F0 + 7 * f2 - 84 * f4] * 9 + [F0 + 4 * f2 + f4] * 9
                    + [F0 - 3 * f2 + 36 * f4] * 5 + [F0 + 14 * f2 + 126 * f4])
    np.testing.assert_allclose(np.sort(imp.energy_of(2)), expect, atol=1e-10)


def test_slater_f2_degeneracies_and_basis_invariance():
    F = [4.5, 6.1, 4.1, 3.0]
    u = wi.spin_orbital_tensor(wi.slater_orbital_tensor(3, F))
    u[np.abs(u) < 1e-14] = 0
    imp = wi.build_impurity("f", np.zeros((14, 14)), u, [(1,)] * 14, 1.0, n_window=(2, 2))
    e = np.sort(imp.energy_of(0))
    _, counts = np.unique(np.round(e, 8), return_counts=True)
    assert sorted(counts.tolist()) == sorted([33, 21, 9, 13, 9, 5, 1])      # 3H 3F 3P 1I 1G 1D 1S
    uc, _, twomj = wi.f_shell_coupled(F, 0.0)
    impc = wi.build_impurity("fc", np.zeros((14, 14)), uc, [(1,)] * 14, 1.0, n_window=(2, 2))
    np.testing.assert_allclose(np.sort(impc.energy_of(0)), e, atol=1e-10)     # CG rotation leaves the spectrum alone
    # with SOC, J_z labelling must still block-diagonalise H (assert inside build_impurity) and keep the N=1 levels
    uc, soc, twomj = wi.f_shell_coupled(F, 0.3)
    imp1 = wi.build_impurity("f1", np.diag(soc), uc, [(1, m) for m in twomj], 1.0, n_window=(1, 1))
    np.testing.assert_allclose(np.sort(imp1.energy), sorted([-0.6] * 6 + [0.45] * 8), atol=1e-12)


def test_cfg3_particle_hole_symmetric_spectrum(impurities):
    imp = impurities(3)
    for n in range(11):
        np.testing.assert_allclose(np.sort(imp.energy_of(n)), np.sort(imp.energy_of(10 - n)), atol=1e-9)


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_operator_block_invariants(impurities, cfg):
    """P10: F^H F is the projector n_f (or 1-n_f) in the sector, so sigma in {0,1}, ||F||_F^2 integer; c = (c^dag)^H;
    sum_f F_{c^dag f}(q')^H... N_q identity."""
    imp = impurities(cfg)
    where = {(int(a), int(s)): b for b, (a, s) in enumerate(zip(imp.blk_symbol, imp.blk_src))}
    for b in range(imp.n_blocks):
        F = imp.block(b)
        sv = np.linalg.svd(F, compute_uv=False)
        assert np.all((np.abs(sv) < 1e-9) | (np.abs(sv - 1) < 1e-9))
        a, s, d = int(imp.blk_symbol[b]), int(imp.blk_src[b]), int(imp.blk_dst[b])
        fro2 = float(np.sum(np.abs(F) ** 2))
        st = imp.sector_states[s]
        f = a // 2
        occ = int(np.sum((st >> f) & 1))
        assert abs(fro2 - (len(st) - occ if a & 1 else occ)) < 1e-9
        partner = where[(a ^ 1, d)]
        assert int(imp.blk_dst[partner]) == s
        np.testing.assert_allclose(imp.block(partner), F.conj().T, atol=1e-13)
    for q, lab in enumerate(imp.labels):
        acc = np.zeros((imp.dims[q], imp.dims[q]), dtype=imp.blk_data.dtype)
        for f in range(imp.n_flavours):
            b = where.get((2 * f, q))
            if b is not None:
                F = imp.block(b)
                acc += F.conj().T @ F
        np.testing.assert_allclose(acc, lab[0] * np.eye(imp.dims[q]), atol=1e-9)


def test_config_tables(impurities):
    """Sector tables of SURVEY.md §8 for configs 1-4 (config 5: dimensions only, without diagonalising)."""
    assert sorted(impurities(1).dims.tolist()) == sorted([1, 2, 2, 1, 4, 1, 2, 2, 1])
    assert sorted(impurities(2).dims.tolist()) == sorted([1, 3, 3, 3, 9, 3, 1, 9, 9, 1, 3, 9, 3, 3, 3, 1])
    assert impurities(3).dims.tolist() == [1, 10, 45, 120, 210, 252, 210, 120, 45, 10, 1]
    i4 = impurities(4)
    assert i4.n_sectors == 70 and int(i4.dims.max()) == 295 and int(i4.dims.sum()) == 6006 and i4.is_complex
    assert np.abs(i4.blk_data.imag).max() > 0.1
    d5 = wi.sector_dimensions(14, [(1,)] * 14, n_window=(4, 6))
    assert sorted(d5.values()) == [1001, 2002, 3003]
    # ground state of the delta-Pu-like model sits at N = 5 (reading A16)
    q = int(np.argmin([i4.energy_of(q).min() for q in range(i4.n_sectors)]))
    assert i4.labels[q][0] == 5


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_batches_are_valid_and_reproducible(cfg):
    p = BASELINE_CONFIGS[cfg]
    n = 64 if cfg < 4 else 6
    b = make_batch(cfg, n)
    b2 = make_batch(cfg, n // 2, start=n // 2)
    assert b.n_configs == n
    for i in range(n):
        s, t = b.config(i)
        assert len(s) % 2 == 0 and np.all(np.diff(t) >= 0) and (len(t) == 0 or (t[0] >= 0 and t[-1] < p["beta"]))
        for f in range(p["n_flavours"]):                    # per flavour c^dag and c alternate
            ty = (s[(s // 2) == f] & 1)
            assert np.all(ty[1:] != ty[:-1]) and len(ty) % 2 == 0
        if i >= n // 2:                                      # prefix property of the seeding
            s2, t2 = b2.config(i - n // 2)
            assert np.array_equal(s, s2) and np.array_equal(t, t2)
    L = np.diff(b.offset)
    if cfg == 1:
        assert np.all(L == 40)
    else:
        assert abs(L.mean() / (2 * p["mean_pairs"]) - 1) < 0.2
