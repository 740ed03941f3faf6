"""Pins for oracle/lazy_oracle.py: the incremental tree of stored sub-products must
give exactly Eq. 65 of the edited configuration (against oracle.trace_oracle, itself pinned by brute force), with O(log k)
products per edit; its bounds must dominate; its lazy decision must equal the decision taken with the exact trace for every
threshold."""
import math

import numpy as np
import pytest

from oracle import lazy_oracle as LZ
from oracle import trace_oracle as O
from util import rel_diff, scaled_ge
from workloads import make_batch
from workloads.rng import Stream


def _ops_of(batch, b):
    s, t = batch.config(b)
    return [(float(tt), int(a)) for a, tt in zip(s, t)]


def _exact(imp, beta, ops):
    ops = sorted(ops, key=lambda o: o[0])
    return O.trace_config(imp, beta, np.array([a for _, a in ops], np.int32), np.array([t for t, _ in ops], np.float64))


def _determined(imp, beta, ops, r) -> bool:
    """False for configurations whose trace vanishes by a symmetry the sector labels do not resolve (e.g. the orbital parities
    of the Kanamori pair hopping): every fp64 evaluation of them is rounding noise, 40+ binary orders below the bound, and no
    two evaluation orders agree.  Detected with the exact oracle alone: its value must survive an exact cyclic shift."""
    if r["mant"] == 0:
        return False
    ops = sorted(ops, key=lambda o: o[0])
    t = (np.array([x for x, _ in ops]) + 0.41 * beta) % beta
    o = np.argsort(t, kind="stable")
    r2 = O.trace_config(imp, beta, np.array([a for _, a in ops], np.int32)[o], t[o])
    return rel_diff(r2["mant"], r2["exp2"], r["mant"], r["exp2"]) < 1e-8


def _random_pair(rng, imp, beta, ops):
    """A pair (c^dag_f, c_f) at two random times, or the removal of two existing operators of one flavour (adjacent in that
    flavour's own sequence, so that alternation is kept).  Input generation only."""
    nf = imp.n_symbols // 2
    f = rng.integer(nf)
    mine = [o for o in ops if o[1] // 2 == f]
    if mine and rng.uniform() < 0.4 and len(mine) >= 2:
        i = rng.integer(len(mine))
        return [], [mine[i], mine[(i + 1) % len(mine)]]
    t1, t2 = sorted((beta * rng.uniform(), beta * rng.uniform()))
    # type of the earlier operator: opposite of the flavour's operator just before t1 (cyclically), else a coin
    before = [o for o in mine if o[0] < t1] or mine
    first = (1 - (before[-1][1] & 1)) if before else rng.integer(2)
    return [(t1, 2 * f + first), (t2, 2 * f + 1 - first)], []


def _imp_for(impurities, cfg):
    """Config 3 enters with all its Abelian quantum numbers (N, 2S_z, L_z): in the N-only basis fp64 does not determine a few
    per cent of its configurations at all (reading A8 (ii)), which would test conditioning, not the tree."""
    if cfg != 3:
        return impurities(cfg)
    from golden.make_golden import _fine_cfg3
    return _fine_cfg3()


@pytest.mark.parametrize("cfg,depth,n_edits", [(1, 3, 24), (2, 5, 24), (3, 5, 5)])
def test_F1_root_equals_full_recomputation_on_edit_sequences(impurities, cfg, depth, n_edits):
    imp = _imp_for(impurities, cfg)
    beta = imp.beta
    rng = Stream(400 + cfg)
    chain = LZ.LazyChain(imp, beta, depth)
    # the empty configuration: Z (pin P1 through the tree)
    w, e, _ = chain.trace()
    r = _exact(imp, beta, [])
    assert rel_diff(w, e, r["mant"], r["exp2"]) < 1e-12
    # load a BASELINE configuration as one big insertion, then edit it pair by pair
    start = _ops_of(make_batch(cfg, 1, start=31), 0)
    res = chain.propose(insert=start)
    assert res["accept"] and res["decided_by"] in ("partial", "full")
    chain.commit(res)
    accepted = 0
    for _ in range(n_edits):
        ins, rem = _random_pair(rng, imp, beta, chain.ops)
        res = chain.propose(insert=ins, remove=rem)          # threshold -inf: accepted unless the trace vanishes
        r = _exact(imp, beta, res["ops"])
        if r["mant"] == 0:
            assert not res["accept"]
            continue
        if not _determined(imp, beta, res["ops"], r):
            continue
        assert res["accept"]
        assert rel_diff(res["trace"][0], res["trace"][1], r["mant"], r["exp2"]) < 1e-9 * max(1.0, r["kappa"] * 1e-5)
        chain.commit(res)
        accepted += 1
        w, e, terms = chain.trace()                           # the stored root after the commit
        assert rel_diff(w, e, r["mant"], r["exp2"]) < 1e-9 * max(1.0, r["kappa"] * 1e-5)
        for q0, se in enumerate(r["sector"]):
            assert (se is not None) == (q0 in terms)
    assert accepted >= n_edits // 3


def test_F2_products_per_edit_are_logarithmic(impurities):
    """A pair insertion multiplies at most 2 (depth + 1) nodes per start sector plus the operators of two leaves -- not the
    k operators of the configuration."""
    imp = impurities(2)
    beta = imp.beta
    depth = 6
    chain = LZ.LazyChain(imp, beta, depth)
    start = _ops_of(make_batch(2, 1, start=77), 0)
    res = chain.propose(insert=start)
    chain.commit(res)
    k = len(chain.ops)
    assert k >= 80
    rng = Stream(9)
    for _ in range(6):
        ins, rem = _random_pair(rng, imp, beta, chain.ops)
        before = chain.n_products
        res = chain.propose(insert=ins, remove=rem)
        if res["accept"]:
            chain.commit(res)
        used = chain.n_products - before
        leaf_ops = 2 * (3 + 2 * k // (1 << depth))            # the two dirty leaves hold O(k / 2^depth) operators each
        assert used <= imp.n_sectors * (2 * (depth + 1) + 2 * leaf_ops), (used, k)
        assert used < imp.n_sectors * k / 2                   # well below one product per operator and sector


@pytest.mark.parametrize("cfg,depth", [(1, 3), (2, 5), (3, 4)])
def test_F3_bounds_dominate_and_F4_decision_equals_exact_decision(impurities, cfg, depth):
    imp = _imp_for(impurities, cfg)
    beta = imp.beta
    rng = Stream(800 + cfg)
    chain = LZ.LazyChain(imp, beta, depth)
    chain.commit(chain.propose(insert=_ops_of(make_batch(cfg, 1, start=5), 0)))
    early = 0
    for _ in range(6 if cfg < 3 else 2):
        ins, rem = _random_pair(rng, imp, beta, chain.ops)
        free = chain.propose(insert=ins, remove=rem)
        r = _exact(imp, beta, free["ops"])
        # F3: per-sector and total bounds dominate the exact values
        for q0, se in enumerate(r["sector"]):
            if se is not None:
                assert q0 in free["sector_bound"]
                assert scaled_ge(free["sector_bound"][q0][0], free["sector_bound"][q0][1], abs(se[0]), se[1])
        assert scaled_ge(free["bound"][0], free["bound"][1], abs(r["mant"]), r["exp2"])
        if not _determined(imp, beta, free["ops"], r):
            continue
        lw = math.log2(abs(r["mant"])) + r["exp2"]
        lb = math.log2(free["bound"][0]) + free["bound"][1]
        # F4: thresholds from far below |w| to above the bound, and a hair on either side of |w|
        for thr in [lw - 60, lw - 3, lw - 1e-6, lw + 1e-6, lw + 0.5 * (lb - lw), lb + 1e-9, lb + 5]:
            res = chain.propose(insert=ins, remove=rem, log2_threshold=thr)
            assert res["accept"] == (lw > thr), (thr, lw, lb, res["decided_by"])
            if thr > lb:
                assert res["decided_by"] == "bound" and res["n_sectors_evaluated"] == 0
            early += res["decided_by"] != "full"
            if res["accept"]:
                assert rel_diff(res["trace"][0], res["trace"][1], r["mant"], r["exp2"]) < 1e-9 * max(1.0, r["kappa"] * 1e-5)
        if free["accept"]:
            chain.commit(free)
    assert early > 0       # the lazy path really decides without the full trace
