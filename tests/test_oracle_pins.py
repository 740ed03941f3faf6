"""Pins for the oracle: closed forms, invariants and brute force, chosen so that a
dropped term, wrong sign or index, or transposed operand in oracle/trace_oracle.py fails at least one of them."""
import copy
import math

import numpy as np
import pytest

from oracle import brute_force as BF
from oracle import trace_oracle as O
from workloads import impurity as wi
from workloads import make_batch
from workloads.configs import Batch
from util import rel_diff, scaled_ge


def _shifted(imp, c):
    j = copy.copy(imp)
    j.energy = imp.energy + c
    if hasattr(j, "_oracle_view"):
        del j._oracle_view
    return j


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_P1_empty_configuration_is_Z(impurities, cfg):
    imp = impurities(cfg)
    r = O.trace_config(imp, imp.beta, [], [])
    e0 = imp.energy.min()
    z = math.fsum(np.exp(-imp.beta * (imp.energy - e0)))
    assert r["status"] == 0 and r["survive"].all()
    lnw = O.to_log(r["mant"], r["exp2"])
    assert abs(lnw - (math.log(z) - imp.beta * e0)) < 1e-9 * max(1.0, abs(lnw))
    assert r["mant"].imag == 0 and r["mant"].real > 0


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_P2_cyclicity(impurities, cfg):
    imp = impurities(cfg)
    b = make_batch(cfg, 3)
    for i in range(3):
        s, t = b.config(i)
        r = O.trace_config(imp, imp.beta, s, t)
        for delta in (0.37 * imp.beta, 0.81 * imp.beta):
            t2 = (t + delta) % imp.beta
            o = np.argsort(t2, kind="stable")
            r2 = O.trace_config(imp, imp.beta, s[o], t2[o])
            assert rel_diff(r2["mant"], r2["exp2"], r["mant"], r["exp2"]) < 1e-10


@pytest.mark.parametrize("cfg", [1, 2])
def test_P3_brute_force_kanamori(impurities, cfg):
    imp = impurities(cfg)
    b = make_batch(cfg, 4)
    for i in range(4):
        s, t = b.config(i)
        r = O.trace_config(imp, imp.beta, s, t)
        m, e = BF.trace(imp.h1, imp.u, imp.beta, s, t)
        assert rel_diff(r["mant"], r["exp2"], m, e) < 1e-10


def _p_shell_toy(seed=11):
    """3-orbital l=1 Slater + SOC + random Hermitian crystal field: complex, only N conserved, Fock dim 64."""
    from workloads.rng import Stream
    l = 1
    u = wi.spin_orbital_tensor(wi.slater_orbital_tensor(l, [2.0, 1.2]))
    T = wi.clebsch_gordan_l_half(l)
    uc = wi.rotate_tensor(u, T)
    uc[np.abs(uc) < 1e-14] = 0
    soc = np.array([-0.3 * (l + 1) / 2.0] * (2 * l) + [0.3 * l / 2.0] * (2 * l + 2))
    rng = Stream(seed)
    cf = np.zeros((6, 6), dtype=np.complex128)
    for i in range(6):
        for j in range(i, 6):
            if i == j:
                cf[i, i] = 0.2 * rng.normal()
            else:
                cf[i, j] = 0.2 * (rng.normal() + 1j * rng.normal())
                cf[j, i] = np.conj(cf[i, j])
    h1 = np.diag(soc - 1.5) + cf
    return wi.build_impurity("ptoy", h1, uc, [(1,)] * 6, beta=6.0)


def _toy_batch(n_flavours, beta, n, seed=77, pairs=3):
    from workloads.configs import _uniform_alternating
    return _uniform_alternating(seed, 0, n, n_flavours, beta, pairs, None)


def test_P3_brute_force_complex_toy():
    imp = _p_shell_toy()
    assert imp.is_complex
    b = _toy_batch(6, imp.beta, 4)
    nontrivial = 0
    for i in range(4):
        s, t = b.config(i)
        r = O.trace_config(imp, imp.beta, s, t)
        m, e = BF.trace(imp.h1, imp.u, imp.beta, s, t)
        assert rel_diff(r["mant"], r["exp2"], m, e) < 1e-10
        nontrivial += abs(r["mant"].imag) > 1e-3
    assert nontrivial >= 2          # the complex path is really exercised


def test_P4_gauge_shift_and_time_reversal(impurities):
    imp = _p_shell_toy()
    b = _toy_batch(6, imp.beta, 3)
    # (i) random eigenvector phases do not change any trace
    imp_ph = wi.build_impurity("ptoy-ph", imp.h1, imp.u, [(1,)] * 6, beta=imp.beta, phase_seed=3)
    # (ii) H -> H + c multiplies w by exp(-beta c)
    c = 0.73
    imp_sh = _shifted(imp, c)
    for i in range(3):
        s, t = b.config(i)
        r = O.trace_config(imp, imp.beta, s, t)
        r1 = O.trace_config(imp_ph, imp.beta, s, t)
        assert rel_diff(r1["mant"], r1["exp2"], r["mant"], r["exp2"]) < 1e-10
        r2 = O.trace_config(imp_sh, imp.beta, s, t)
        lg = -imp.beta * c * O.LOG2E
        k = math.floor(lg)
        assert rel_diff(r2["mant"], r2["exp2"], r["mant"] * 2.0 ** (lg - k), r["exp2"] + k) < 1e-10
        # (iv) time reversal: tau -> beta - tau, c <-> c^dag, order reversed gives conj(w)   [Tr X^H = conj Tr X]
        keep = t > 0
        s3, t3 = (s[keep] ^ 1)[::-1], (imp.beta - t[keep])[::-1]
        if keep.all():
            r3 = O.trace_config(imp, imp.beta, s3, t3)
            assert rel_diff(r3["mant"], r3["exp2"], np.conj(r["mant"]), r["exp2"]) < 1e-10


def test_P4_sector_coarsening_d_shell():
    """(iii) the same d-shell model with sectors (N, 2Sz, Lz), (N, 2Sz) and N only gives the same traces; pins routing
    tables and block assembly at d = 252 where brute force is impossible."""
    u = wi.spin_orbital_tensor(wi.slater_orbital_tensor(2, [6.0, 8.4, 5.3]))
    u[np.abs(u) < 1e-14] = 0
    h1 = -wi.symmetric_mu(u) * np.eye(10)
    fine = [(1, -1, m) for m in range(-2, 3)] + [(1, 1, m) for m in range(-2, 3)]
    imps = [wi.build_impurity("d-fine", h1, u, fine, beta=4.0),
            wi.build_impurity("d-mid", h1, u, [q[:2] for q in fine], beta=4.0),
            wi.build_impurity("d-N", h1, u, [(1,)] * 10, beta=4.0)]
    assert [int(i.dims.max()) for i in imps] == [16, 100, 252]
    b = _toy_batch(10, 4.0, 2, pairs=2)
    for i in range(2):
        s, t = b.config(i)
        rs = [O.trace_config(im, 4.0, s, t) for im in imps]
        assert rs[0]["mant"] != 0
        for r in rs[1:]:
            assert rel_diff(r["mant"], r["exp2"], rs[0]["mant"], rs[0]["exp2"]) < 1e-9


def test_P5_ising_limit_closed_form():
    """Density-density interaction, diagonal t: every sector has d = 1 and
    w = sign * exp(-int_0^beta E[n(tau)] dtau) with the Jordan-Wigner sign of the operator sequence."""
    n, beta = 4, 7.0
    Umat = np.array([[0, 2.0, 1.1, 0.7], [2.0, 0, 0.9, 1.3], [1.1, 0.9, 0, 2.2], [0.7, 1.3, 2.2, 0]])
    eps = np.array([-1.0, -0.4, -1.7, -0.2])
    u = np.zeros((n,) * 4)
    for a in range(n):
        for b_ in range(n):
            if a != b_:
                u[a, b_, b_, a] = Umat[a, b_]
    qn = [(1,) + tuple(int(i == f) for i in range(n)) for f in range(n)]
    imp = wi.build_impurity("ising", np.diag(eps), u, qn, beta=beta)
    assert int(imp.dims.max()) == 1 and imp.n_sectors == 16
    b = _toy_batch(n, beta, 5, seed=5, pairs=4)

    def energy(occ):
        return float(eps @ occ + 0.5 * occ @ Umat @ occ)

    for i in range(5):
        s, t = b.config(i)
        # initial occupation: flavour f is occupied at tau=0 iff its first operator is an annihilator
        occ = np.zeros(n)
        for f in range(n):
            sf = s[(s // 2) == f]
            occ[f] = 1.0 if (len(sf) and sf[0] % 2 == 0) else 0.0
        state = sum(1 << f for f in range(n) if occ[f])
        sign, integral, t_prev = 1.0, 0.0, 0.0
        for a, tt in zip(s, t):
            integral += (tt - t_prev) * energy(occ)
            f = int(a) // 2
            sign *= (-1) ** bin(state & ((1 << f) - 1)).count("1")
            occ[f] = a % 2
            state ^= (1 << f)
            t_prev = tt
        integral += (beta - t_prev) * energy(occ)
        r = O.trace_config(imp, beta, s, t)
        assert r["survive"].sum() == 1
        assert math.copysign(1.0, r["mant"].real) == sign
        assert abs(O.to_log(r["mant"], r["exp2"]) + integral) < 1e-9 * max(1.0, abs(integral))


def test_P5_coarse_sectors_do_not_underflow():
    """Ising limit again, but with sectors labelled by N only (so d > 1 and E_n - Emin is large inside a sector) and
    level splittings times time differences far beyond 745: exp(-Delta (E_n - Emin)) underflows a double, the value of
    Eq. 65 does not.  Closed form per start sector: each Fock state is its own invariant subspace, so
    t(q0) = sum over Fock states s in q0 that survive the operator sequence of sign(s) exp(-int E[n(tau)] dtau)."""
    n, beta = 3, 60.0
    eps = np.array([-2.0, 31.0, 75.0])
    Umat = np.array([[0, 3.0, 1.0], [3.0, 0, 2.0], [1.0, 2.0, 0]])
    u = np.zeros((n,) * 4)
    for a in range(n):
        for b_ in range(n):
            if a != b_:
                u[a, b_, b_, a] = Umat[a, b_]
    imp = wi.build_impurity("ising-coarse", np.diag(eps), u, [(1,)] * n, beta=beta)
    assert list(imp.dims) == [1, 3, 3, 1]

    def energy(state):
        occ = np.array([(state >> f) & 1 for f in range(n)], dtype=float)
        return float(eps @ occ + 0.5 * occ @ Umat @ occ)

    # flavour 2 (the expensive one) is created and kept for 40 time units; flavour 1 flips in between
    configs = [([5, 3, 2, 4], [1.0, 7.0, 19.5, 41.0]),
               ([5, 4], [3.0, 58.0]),
               ([3, 5, 4, 2, 1, 0], [2.0, 2.5, 30.0, 44.0, 50.0, 59.0])]
    import mpmath
    mpmath.mp.dps = 60
    beyond = 0
    for s, t in configs:
        r = O.trace_config(imp, beta, s, t)
        assert r["status"] == 0
        for q0 in range(imp.n_sectors):
            terms = []
            for st0 in imp.sector_states[q0]:
                state, sign, integral, t_prev, ok = int(st0), 1.0, 0.0, 0.0, True
                for a, tt in zip(s, t):
                    integral += (tt - t_prev) * energy(state)
                    f, create = int(a) // 2, int(a) % 2
                    if ((state >> f) & 1) == create:
                        ok = False
                        break
                    sign *= (-1) ** bin(state & ((1 << f) - 1)).count("1")
                    state ^= (1 << f)
                    t_prev = tt
                if ok and state == int(st0):
                    terms.append((sign, integral + (beta - t_prev) * energy(state)))
            if r["sector"][q0] is None:
                assert not terms
                continue
            zs, es = r["sector"][q0]
            if not terms:
                assert zs == 0
                continue
            top = min(i for _, i in terms)
            # the closed form evaluated in 60-digit arithmetic and compared as a VALUE at the oracle's own exponent: a relative
            # error of 1e-10 in the mantissa / row-exponent split of oracle._propagate fails here (a comparison of logarithms
            # at |log| ~ 4000 would let 4e-6 through)
            exact = sum(mpmath.mpf(sg) * mpmath.exp(-mpmath.mpf(i)) for sg, i in terms)
            got = mpmath.mpf(zs.real) * mpmath.mpf(2) ** es
            assert zs.imag == 0.0
            assert abs(got - exact) <= mpmath.mpf(1e-10) * abs(exact), (q0, float(abs(got - exact) / abs(exact)))
            assert (es * math.log(2.0) < -745.0) or top < 745.0   # at least some sectors are beyond exp()'s range
            beyond += es * math.log(2.0) < -745.0
            bd = O.bound_config(imp, beta, s, t, 0, 1)
            assert scaled_ge(bd["sector"][q0][0], bd["sector"][q0][1], abs(zs), es)
    # the middle configuration keeps flavour 2 for 55 time units: within the N=1 sector that is 77*55 = 4235 >> 745
    r = O.trace_config(imp, beta, *configs[1])
    assert r["sector"][0] is not None and r["sector"][0][0] != 0
    assert beyond >= 2


def test_P6_atomic_green_function():
    """One orbital: c^dag_up at 0+, c_up at tau:  w = e^{mu tau} + e^{-tau (U - 2 mu) + mu (beta - tau)}  (textbook)."""
    U, mu, beta, tau = 2.5, 0.9, 3.0, 1.234
    h1, u, qn = wi._kanamori(1, U, 0.0, mu)
    imp = wi.build_impurity("atom", h1, u, qn, beta=beta)
    up = 1   # flavour order Eq. A.4: down = 0, up = 1
    r = O.trace_config(imp, beta, [2 * up + 1, 2 * up], [0.0, tau])
    # states during (0, tau): up added.  start |0>: weight e^{-tau(-mu)};  start |dn>: e^{-tau(U-2mu)} e^{-(beta-tau)(-mu)}
    expect = math.exp(mu * tau) + math.exp(-tau * (U - 2 * mu) + mu * (beta - tau))
    val = r["mant"].real * 2.0 ** r["exp2"]
    assert abs(val - expect) < 1e-12 * expect
    assert r["survive"].sum() == 2


def test_zero_sector_and_status(impurities):
    imp = impurities(1)
    # three creators of spin-down flavours leave the (N, S_z) label set from every start sector (only 2 such flavours)
    r = O.trace_config(imp, imp.beta, [1, 3, 1, 0, 2, 0], [0.1, 0.2, 0.3, 0.4, 0.5, 0.6])
    assert r["status"] == 1 and r["mant"] == 0 and r["exp2"] == 0 and not r["survive"].any()
    for bad in ([[1, 0], [0.5, 0.4]], [[1, 0], [0.5, imp.beta]], [[1, 99], [0.1, 0.2]], [[1, 0], [-0.1, 0.2]]):
        r = O.trace_config(imp, imp.beta, *bad)
        assert r["status"] == 2 and math.isnan(r["mant"].real)
    # tau = 0 and equal times are legal (reading A7)
    r = O.trace_config(imp, imp.beta, [1, 0], [0.0, 0.0])
    assert r["status"] == 0


# ----------------------------------------------------------------------------------------------- bounds
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_PB1_bound_dominates_trace_and_PB2_monotone(impurities, cfg):
    imp = impurities(cfg)
    b = make_batch(cfg, 3)
    for i in range(3):
        s, t = b.config(i)
        r = O.trace_config(imp, imp.beta, s, t)
        prev = None
        for S in (1, 2, 4, 8, 0):
            for kind in (0, 1):
                if kind == 1 and cfg == 3 and S not in (1, 0):
                    continue
                bd = O.bound_config(imp, imp.beta, s, t, kind, S)
                assert scaled_ge(bd["mant"], bd["exp2"], abs(r["mant"]), r["exp2"])
                for q0 in range(imp.n_sectors):
                    if r["sector"][q0] is not None:
                        zs, es = r["sector"][q0]
                        assert scaled_ge(bd["sector"][q0][0], bd["sector"][q0][1], abs(zs), es)
                    else:
                        assert bd["sector"][q0] is None
            bd = O.bound_config(imp, imp.beta, s, t, 0, S)
            if prev is not None:      # S' multiple of S  =>  bound(S') <= bound(S) (1 + eps)
                assert scaled_ge(prev[0] * (1 + 1e-9), prev[1], bd["mant"], bd["exp2"])
            prev = (bd["mant"], bd["exp2"])


def test_PB3_S1_closed_forms(impurities):
    imp = impurities(2)
    view = O._imp(imp)
    b = make_batch(2, 2)
    for i in range(2):
        s, t = b.config(i)
        deltas = O._factor_deltas(imp.beta, t)
        fro = O.bound_config(imp, imp.beta, s, t, 0, 1)
        spec = O.bound_config(imp, imp.beta, s, t, 1, 1)
        for q0 in range(imp.n_sectors):
            vis = O.route(imp, s, q0)
            if vis is None:
                continue
            dmin = min(int(imp.dims[q]) for q in vis)
            # Frobenius: ||diag(p) F||_F^2 = sum_n p_n^2 r_n, r_n = squared row norms of F
            ln_f = 0.5 * math.log(dmin)
            ln_s = math.log(dmin)
            for k, a in enumerate(s):
                F = view.F[(int(a), vis[k])]
                rn = np.sum(np.abs(F) ** 2, axis=1)
                p = np.exp(-deltas[k] * view.E[vis[k + 1]])
                ln_f += 0.5 * math.log(float(np.sum(p * p * rn)))
                ln_s += -deltas[k] * view.Emin[vis[k + 1]]          # sigma_max(c or c^dag block) = 1 (P10)
            assert abs(O.to_log(*fro["sector"][q0]) - ln_f) < 1e-9 * max(1, abs(ln_f))
            assert abs(O.to_log(*spec["sector"][q0]) - ln_s) < 1e-9 * max(1, abs(ln_s))


def test_PB4_equality_in_one_dimensional_sectors():
    """Strings living entirely in d = 1 sectors: bound = |t| (before the outward rounding)."""
    h1, u, qn = wi._kanamori(1, 2.0, 0.0, 0.7)
    imp = wi.build_impurity("atom", h1, u, qn, beta=2.0)
    s, t = [3, 2, 1, 0], [0.2, 0.5, 0.9, 1.4]
    r = O.trace_config(imp, 2.0, s, t)
    for kind in (0, 1):
        for S in (1, 2, 0):
            bd = O.bound_config(imp, 2.0, s, t, kind, S)
            for q0 in range(imp.n_sectors):
                if r["sector"][q0] is not None:
                    zs, es = r["sector"][q0]
                    assert rel_diff(bd["sector"][q0][0], bd["sector"][q0][1], abs(zs), es) < 1e-11
                    assert scaled_ge(bd["sector"][q0][0], bd["sector"][q0][1], abs(zs), es)


def test_PB2_whole_chain_frobenius_matches_trace_matrix(impurities):
    """S = 0, Frobenius: sqrt(d_min) * ||A_L ... A_1||_F, recomputed here from explicit numpy products."""
    imp = impurities(1)
    view = O._imp(imp)
    b = make_batch(1, 2)
    for i in range(2):
        s, t = b.config(i)
        deltas = O._factor_deltas(imp.beta, t)
        bd = O.bound_config(imp, imp.beta, s, t, 0, 0)
        for q0 in range(imp.n_sectors):
            vis = O.route(imp, s, q0)
            if vis is None:
                continue
            e0 = view.Emin.min()
            M = np.eye(int(imp.dims[q0]))
            for k, a in enumerate(s):
                M = np.diag(np.exp(-deltas[k] * (view.E[vis[k + 1]] - e0))) @ view.F[(int(a), vis[k])] @ M
            ln = 0.5 * math.log(min(int(imp.dims[q]) for q in vis)) + math.log(np.linalg.norm(M)) - imp.beta * e0
            assert abs(O.to_log(*bd["sector"][q0]) - ln) < 1e-9 * max(1, abs(ln))


def test_A8_config3_coarse_sectors_are_ill_conditioned_in_fp64(impurities):
    """DESIGN.md reading A8 (ii), established with the oracle alone: configuration 45 of BASELINE config 3 is not determined by
    fp64 in the N-only sector basis (its value moves by orders of magnitude under the exact cyclic shifts of pin P2), while
    the same Hamiltonian in (N, 2S_z, L_z) sectors gives a value stable to 1e-10 -- the trace itself is basis independent
    (pin P4 (iii)).  A well-conditioned neighbour (configuration 1) agrees between the two bases to 1e-10."""
    coarse = impurities(3)
    u = wi.spin_orbital_tensor(wi.slater_orbital_tensor(2, [6.0, 8.4, 5.3]))
    u[np.abs(u) < 1e-14] = 0
    h1 = -wi.symmetric_mu(u) * np.eye(10)
    fineqn = [(1, -1, m) for m in range(-2, 3)] + [(1, 1, m) for m in range(-2, 3)]
    fine = wi.build_impurity("d-fine", h1, u, fineqn, beta=coarse.beta, keep_eigvecs=False)
    b = make_batch(3, 46)

    def spread(imp, s, t, r):
        out = 0.0
        for frac in (0.23, 0.52, 0.77):
            t2 = (t + frac * imp.beta) % imp.beta
            o = np.argsort(t2, kind="stable")
            r2 = O.trace_config(imp, imp.beta, s[o], t2[o])
            out = max(out, rel_diff(r2["mant"], r2["exp2"], r["mant"], r["exp2"]))
        return out

    s, t = b.config(45)
    rc, rf = O.trace_config(coarse, coarse.beta, s, t), O.trace_config(fine, fine.beta, s, t)
    assert spread(fine, s, t, rf) < 1e-10
    assert spread(coarse, s, t, rc) > 1e-3
    s, t = b.config(1)
    rc, rf = O.trace_config(coarse, coarse.beta, s, t), O.trace_config(fine, fine.beta, s, t)
    assert rel_diff(rc["mant"], rc["exp2"], rf["mant"], rf["exp2"]) < 1e-10


@pytest.mark.parametrize("cfg,S", [(1, 2), (2, 3), (2, 0)])
def test_PB5_certified_spectral_estimate_lies_between_the_exact_spectral_and_the_frobenius_bound(impurities, cfg, S):
    """norm_kind 2 (reading A1: min(||G_j||_F, prod sigma_max(F_i)) per segment) is pinned by the two inequalities that make it
    a bound -- it dominates the exact spectral-norm product (SVD) and, the prefactor aside, never exceeds the Frobenius
    product -- by bound >= |trace| per sector, and by the case where it must coincide with the exact value: c / c^dag blocks have
    sigma_max = 1 (pin P10), so with segment length 1 it equals the factorised closed form P-B3."""
    imp = impurities(cfg)
    batch = make_batch(cfg, 6, start=900)
    for b in range(batch.n_configs):
        s, t = batch.config(b)
        est = O.bound_config(imp, batch.beta, s, t, 2, S)
        exact = O.bound_config(imp, batch.beta, s, t, 1, S)
        fro = O.bound_config(imp, batch.beta, s, t, 0, S)
        tr = O.trace_config(imp, batch.beta, s, t)
        dmin_max = math.sqrt(max(int(d) for d in imp.dims))
        for q0, se in enumerate(est["sector"]):
            if se is None:
                assert exact["sector"][q0] is None
                continue
            ex, fr = exact["sector"][q0], fro["sector"][q0]
            assert scaled_ge(se[0] * (1 + 1e-12), se[1], ex[0], ex[1])
            assert scaled_ge(fr[0] * dmin_max * (1 + 1e-12), fr[1], se[0], se[1])
            z, e = tr["sector"][q0]
            assert scaled_ge(se[0], se[1], abs(z), e)
        one = O.bound_config(imp, batch.beta, s, t, 2, 1)
        closed = O.bound_config(imp, batch.beta, s, t, 1, 1)
        assert rel_diff(one["mant"], one["exp2"], closed["mant"], closed["exp2"]) < 1e-14
