"""Parity of the chain-set calls (ctqmc_chains_*: incremental lazy trace) with
oracle/lazy_oracle.py on the same seeded edit sequences.  Run on a B200: -m gpu.

Bars: accept / decided_by / n_sectors_evaluated / status identical (integers; the thresholds are placed away from the exact
values, so no decision hangs on a rounding); bounds and traces within 1e-9 (x max(1, kappa 1e-5), reading A8 (i)); after a
commit the stored root equals Eq. 65 of the edited configuration computed from scratch by oracle.trace_oracle."""
import math

import numpy as np
import pytest

from test_lazy_oracle import _determined, _exact, _imp_for, _ops_of, _random_pair
from util import rel_diff, scaled_ge

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


def _edits(torch, per_chain):
    """per_chain: list (one per chain) of (insert list, remove list) of (tau, symbol) -> CSR device tensors."""
    off, tau, sym, kind = [0], [], [], []
    for ins, rem in per_chain:
        for t, a in rem:
            tau.append(t); sym.append(a); kind.append(-1)
        for t, a in ins:
            tau.append(t); sym.append(a); kind.append(1)
        off.append(len(tau))
    return (torch.tensor(off, dtype=torch.int64, device="cuda"), torch.tensor(tau, dtype=torch.float64, device="cuda"),
            torch.tensor(sym, dtype=torch.int32, device="cuda"), torch.tensor(kind, dtype=torch.int32, device="cuda"))


def _log2(m, e):
    return -math.inf if m == 0 else math.log2(abs(m)) + e


def _check_traces(lib, torch, ch, oracles, imp, beta, label):
    mant, exp2 = lib.ctqmc_chains_trace(ch)
    torch.cuda.synchronize()
    mant, exp2 = mant.cpu().numpy(), exp2.cpu().numpy()
    for c, oc in enumerate(oracles):
        r = _exact(imp, beta, oc.ops)
        g = complex(mant[c, 0], mant[c, 1])
        if r["mant"] == 0 or not _determined(imp, beta, oc.ops, r):
            # structurally zero (or zero by an unresolved symmetry): rounding noise at most, far below the bound
            b = oc.propose()
            assert g == 0 or _log2(abs(g), int(exp2[c])) < _log2(*b["bound"]) - 30, f"{label} chain {c}"
            continue
        d = rel_diff(g, int(exp2[c]), r["mant"], r["exp2"])
        assert d <= TOL * max(1.0, r["kappa"] * 1e-5), f"{label} chain {c}: stored root vs Eq. 65 from scratch {d:.3e}"


def _gauge_twisted(base):
    """The same impurity in a basis rotated by a diagonal unitary, |n> -> exp(i theta_n) |n>: every trace is unchanged, every
    operator block becomes complex.  Gives the small-impurity kernels (sector dimensions <= 16) a complex case."""
    import types
    from workloads.rng import Stream
    rng = Stream(515)
    dims = np.asarray(base.dims, dtype=np.int64)
    soff = np.concatenate([[0], np.cumsum(dims)])
    phase = np.exp(2j * np.pi * np.array([rng.uniform() for _ in range(int(soff[-1]))]))
    data = np.asarray(base.blk_data, dtype=np.complex128).copy()
    for b in range(len(base.blk_symbol)):
        qs, qd = int(base.blk_src[b]), int(base.blk_dst[b])
        m, n = int(dims[qd]), int(dims[qs])
        o = int(base.blk_offset[b])
        blk = data[o:o + m * n].reshape((m, n), order="F")
        blk *= phase[soff[qd]:soff[qd + 1], None] * np.conj(phase[soff[qs]:soff[qs + 1]])[None, :]
        data[o:o + m * n] = blk.ravel(order="F")
    return types.SimpleNamespace(dims=base.dims, energy=base.energy, n_symbols=base.n_symbols, is_complex=True, n_sectors=base.n_sectors,
                                 beta=base.beta, blk_symbol=base.blk_symbol, blk_src=base.blk_src, blk_dst=base.blk_dst,
                                 blk_offset=base.blk_offset, blk_data=data)


def _real_part(base):
    """Config 4's sectors and routing with the real parts of its operator blocks: not a physical impurity, but a real-valued
    block-sparse operator set with sectors of up to 295 states -- the tiled chain-set kernels in real arithmetic.  (Config 3 in its
    N-only basis would be the natural case, but fp64 does not determine its node norms to better than 1e-3: reading A8 (ii).)"""
    import types
    return types.SimpleNamespace(dims=base.dims, energy=base.energy, n_symbols=base.n_symbols, is_complex=False, n_sectors=base.n_sectors,
                                 beta=base.beta, blk_symbol=base.blk_symbol, blk_src=base.blk_src, blk_dst=base.blk_dst,
                                 blk_offset=base.blk_offset, blk_data=np.ascontiguousarray(np.asarray(base.blk_data).real, dtype=np.float64))


# kernel families behind the cases: configs 1, 2 and 3 (fine sectors, 16 states at most) take the warp-per-task kernels, real;
# "2twist" the same kernels, complex; config 4 the tiled kernels, complex; "4real" the tiled kernels, real
@pytest.mark.parametrize("cfg,depth,n_chains,n_steps,lazy_rounds", [(1, 3, 6, 10, 1), (2, 5, 5, 8, 2), (2, 4, 3, 5, 0), (3, 4, 2, 4, 1),
                                                                      (4, 3, 2, 7, 2), ("2twist", 4, 3, 6, 1), ("4real", 3, 2, 5, 1)])
def test_chains_follow_the_lazy_oracle(lib, torch_cuda, impurities, cfg, depth, n_chains, n_steps, lazy_rounds):
    from oracle import lazy_oracle as LZ
    from workloads import make_batch
    from workloads.rng import Stream
    torch = torch_cuda
    if cfg == "2twist":
        cfg, imp = 2, _gauge_twisted(impurities(2))
    elif cfg == "4real":
        cfg, imp = 4, _real_part(impurities(4))
    else:
        imp = _imp_for(impurities, cfg)
    beta = imp.beta
    h = lib.ctqmc_load_impurity(imp, 0)
    ch = None
    try:
        ch = lib.ctqmc_chains_create(h, beta, n_chains, depth, leaf_capacity=64 if cfg == 4 else 24, max_edits=8, lazy_rounds=lazy_rounds)
        oracles = [LZ.LazyChain(imp, beta, depth) for _ in range(n_chains)]
        _check_traces(lib, torch, ch, oracles, imp, beta, f"cfg{cfg} empty")          # Z through the tree
        # ---- load a BASELINE configuration per chain in chunks of 8 operators, commits forced by the mask (the intermediate
        #      configurations are arbitrary, most of them vanish)
        starts = [_ops_of(make_batch(cfg, 1, start=40 + c), 0) for c in range(n_chains)]
        if cfg == 4:
            starts = [[] for _ in starts]          # grown from the empty configuration by the pair moves below (keeps the oracle's share short)
        nchunk = max((len(s) + 7) // 8 for s in starts)
        ones = torch.ones(n_chains, dtype=torch.int32, device="cuda")
        for k in range(nchunk):
            per = [(s[8 * k:8 * k + 8], []) for s in starts]
            out = lib.ctqmc_chains_propose(ch, *_edits(torch, per))
            lib.ctqmc_chains_commit(ch, ones)
            torch.cuda.synchronize()
            assert (out["status"] == 0).all().item()
            for oc, (ins, _) in zip(oracles, per):
                res = oc.propose(insert=ins)
                res["accept"] = True
                oc.commit(res)
        _check_traces(lib, torch, ch, oracles, imp, beta, f"cfg{cfg} loaded")
        # ---- pair moves with thresholds placed by the oracle
        rngs = [Stream(9000 + 10 * cfg + c) for c in range(n_chains)]
        n_checked = n_early = 0
        for step in range(n_steps):
            per, free, thr, exact = [], [], [], []
            for c, oc in enumerate(oracles):
                ins, rem = _random_pair(rngs[c], imp, beta, oc.ops)
                fr = oc.propose(insert=ins, remove=rem)
                r = _exact(imp, beta, fr["ops"])
                lb = _log2(*fr["bound"])
                ok = r["mant"] != 0 and _determined(imp, beta, fr["ops"], r)
                lw = _log2(abs(r["mant"]), r["exp2"]) if ok else None
                choice = (step + c) % 4
                if not ok or choice == 0:
                    t = -math.inf if ok else lb + 3.0          # undetermined values: decide by the bound alone
                elif choice == 1:
                    t = lw - 2.0
                elif choice == 2:
                    t = lw + 0.5 * (lb - lw) if lb - lw > 1e-3 else lw + 2.0
                else:
                    t = lb + 5.0
                per.append((ins, rem)); free.append(fr); thr.append(t); exact.append((r, ok))
            out = lib.ctqmc_chains_propose(ch, *_edits(torch, per), torch.tensor(thr, dtype=torch.float64, device="cuda"))
            lib.ctqmc_chains_commit(ch)
            torch.cuda.synchronize()
            out = {k: v.cpu().numpy() for k, v in out.items()}
            for c, oc in enumerate(oracles):
                ins, rem = per[c]
                res = oc.propose(insert=ins, remove=rem, log2_threshold=thr[c])
                r, ok = exact[c]
                label = f"cfg{cfg} step {step} chain {c} thr {thr[c]:.3f}"
                assert out["status"][c] == 0, label
                d = rel_diff(out["bound_mant"][c], int(out["bound_exp2"][c]), res["bound"][0], res["bound"][1])
                assert d <= TOL, f"{label}: bound {d:.3e}"
                assert bool(out["accept"][c]) == res["accept"], f"{label}: accept {out['accept'][c]} vs {res['accept']} ({res['decided_by']})"
                assert out["decided_by"][c] == {"bound": 0, "partial": 1, "full": 2}[res["decided_by"]], label
                assert out["n_sectors_evaluated"][c] == res["n_sectors_evaluated"], label
                if ok:
                    assert res["accept"] == (_log2(abs(r["mant"]), r["exp2"]) > thr[c]), label      # the oracle's own pin, restated
                if res["accept"]:
                    g = complex(out["trace_mant"][c, 0], out["trace_mant"][c, 1])
                    d = rel_diff(g, int(out["trace_exp2"][c]), res["trace"][0], res["trace"][1])
                    assert d <= TOL * max(1.0, r["kappa"] * 1e-5), f"{label}: trace {d:.3e}"
                    assert scaled_ge(out["bound_mant"][c], int(out["bound_exp2"][c]), abs(g), int(out["trace_exp2"][c])), label
                    oc.commit(res)
                    n_checked += 1
                n_early += res["decided_by"] != "full"
        assert n_checked >= 1 and n_early >= 1
        _check_traces(lib, torch, ch, oracles, imp, beta, f"cfg{cfg} after moves")
        st = lib.ctqmc_chains_stats(ch)
        assert st["products"] > 0 and st["bytes"] > 0
    finally:
        if ch is not None:
            ch.destroy()
        h.free()


def test_chain_edit_errors_leave_the_chain_untouched(lib, torch_cuda, impurities):
    """Invalid proposals get a per-chain status, are never accepted, and a commit skips them."""
    from oracle import lazy_oracle as LZ
    torch = torch_cuda
    imp = impurities(1)
    beta = imp.beta
    h = lib.ctqmc_load_impurity(imp, 0)
    ch = lib.ctqmc_chains_create(h, beta, 6, 2, leaf_capacity=2, max_edits=4, lazy_rounds=1)
    try:
        pair = [(1.0, 1), (1.5, 0)]
        out = lib.ctqmc_chains_propose(ch, *_edits(torch, [(pair, [])] * 6))
        lib.ctqmc_chains_commit(ch)
        torch.cuda.synchronize()
        assert (out["status"] == 0).all().item() and (out["accept"] == 1).all().item()
        oc = LZ.LazyChain(imp, beta, 2)
        oc.commit(oc.propose(insert=pair))
        per = [([(3.0, 3), (3.2, 2)], []),                       # fine
               ([(beta, 1), (0.5, 0)], []),                      # tau = beta: bad edit
               ([], [(1.0, 1), (1.25, 0)]),                      # second operator is not in the chain
               ([(1.1, 3), (1.2, 2)], []),                       # leaf [0, beta/4) would hold 4 > 2 operators
               ([(0.1, 40), (0.2, 0)], []),                      # symbol out of range
               ([(6.0 + 0.1 * i, 2 + (i & 1)) for i in range(6)], [])]     # 6 edits > max_edits
        out = lib.ctqmc_chains_propose(ch, *_edits(torch, per))
        lib.ctqmc_chains_commit(ch, torch.ones(6, dtype=torch.int32, device="cuda"))
        torch.cuda.synchronize()
        assert out["status"].cpu().tolist() == [0, 2, 3, 4, 2, 2]
        assert out["accept"].cpu().tolist()[1:] == [0] * 5
        assert torch.isnan(out["bound_mant"][1:]).all().item()
        mant, exp2 = lib.ctqmc_chains_trace(ch)
        torch.cuda.synchronize()
        w, e, _ = oc.trace()
        for c in range(1, 6):
            assert rel_diff(complex(mant[c, 0].item(), mant[c, 1].item()), int(exp2[c].item()), w, e) <= 1e-12
        oc.commit(oc.propose(insert=per[0][0]))
        w, e, _ = oc.trace()
        assert rel_diff(complex(mant[0, 0].item(), mant[0, 1].item()), int(exp2[0].item()), w, e) <= 1e-12
    finally:
        ch.destroy()
        h.free()


def test_chain_set_products_are_logarithmic_and_create_reports_oom(lib, torch_cuda, impurities):
    """A pair move multiplies O(depth) nodes per sector, not the k operators of the configuration; a chain set
    that cannot be allocated is refused with the size it would need."""
    from workloads import make_batch
    torch = torch_cuda
    imp = impurities(2)
    beta = imp.beta
    h = lib.ctqmc_load_impurity(imp, 0)
    depth = 6
    ch = lib.ctqmc_chains_create(h, beta, 1, depth, leaf_capacity=16, max_edits=8, lazy_rounds=1)
    try:
        ops = _ops_of(make_batch(2, 1, start=77), 0)
        one = torch.ones(1, dtype=torch.int32, device="cuda")
        for k in range(0, len(ops), 8):
            lib.ctqmc_chains_propose(ch, *_edits(torch, [(ops[k:k + 8], [])]))
            lib.ctqmc_chains_commit(ch, one)
        before = lib.ctqmc_chains_stats(ch)["products"]
        lib.ctqmc_chains_propose(ch, *_edits(torch, [([(3.3, 1), (17.9, 0)], [])]))
        lib.ctqmc_chains_commit(ch, one)
        used = lib.ctqmc_chains_stats(ch)["products"] - before
        k = len(ops)
        assert k >= 80
        assert 0 < used <= imp.n_sectors * (2 * (depth + 1) + 2 * (3 + 2 * k // (1 << depth)) + 4), used
        assert used < imp.n_sectors * k / 2
        with pytest.raises(lib.CtqmcError) as ei:
            lib.ctqmc_chains_create(h, beta, 1 << 20, 12, leaf_capacity=16, max_edits=8)
        assert ei.value.code == lib.CTQMC_ERR_OOM
    finally:
        ch.destroy()
        h.free()


def test_chain_sets_at_bench_size_agree_with_the_stateless_trace(lib, torch_cuda, impurities):
    """The launch configuration bench.py times (config 2, 1024 chains, depth 6, leaf capacity 32, two lazy rounds): after loading a
    BASELINE configuration per chain and three Metropolis rounds of pair moves, the stored root of EVERY chain must equal
    ctqmc_trace_batch of the host's mirror of its configuration (a path that is itself held to the oracle on every output of config
    2), and a sample of chains is compared with oracle.trace_oracle directly.  A property that holds at any size."""
    from oracle import trace_oracle as O
    from workloads import Batch, apply_move, make_batch, random_pair_move
    from workloads.rng import Stream
    torch = torch_cuda
    imp = impurities(2)
    beta, nC, nf = imp.beta, 1024, imp.n_symbols // 2
    h = lib.ctqmc_load_impurity(imp, 0)
    ch = lib.ctqmc_chains_create(h, beta, nC, 6, leaf_capacity=32, max_edits=8, lazy_rounds=2)
    try:
        ops = [_ops_of(make_batch(2, 1, start=c % 64), 0) for c in range(nC)]
        ones = torch.ones(nC, dtype=torch.int32, device="cuda")
        for k in range(max((len(s) + 7) // 8 for s in ops)):
            out = lib.ctqmc_chains_propose(ch, *_edits(torch, [(s[8 * k:8 * k + 8], []) for s in ops]))
            lib.ctqmc_chains_commit(ch, ones)
        assert (out["status"] == 0).all().item()
        rngs = [Stream(880000 + c) for c in range(nC)]
        n_acc = 0
        for _ in range(3):
            moves = [random_pair_move(rngs[c], nf, beta, ops[c]) for c in range(nC)]
            u = torch.tensor([max(rngs[c].uniform(), 1e-300) for c in range(nC)], dtype=torch.float64, device="cuda")
            mant, exp2 = lib.ctqmc_chains_trace(ch)
            thr = torch.log2(torch.hypot(mant[:, 0], mant[:, 1])) + exp2.to(torch.float64) + torch.log2(u)
            out = lib.ctqmc_chains_propose(ch, *_edits(torch, moves), thr)
            lib.ctqmc_chains_commit(ch)
            torch.cuda.synchronize()
            acc, st = out["accept"].cpu().numpy(), out["status"].cpu().numpy()
            assert (st == 0).all()
            for c in range(nC):
                if acc[c]:
                    ops[c] = apply_move(ops[c], *moves[c])
            n_acc += int(acc.sum())
        assert 0 < n_acc < 3 * nC
        mant, exp2 = lib.ctqmc_chains_trace(ch)
        batch = Batch.from_lists(beta, [([a for _, a in s], [t for t, _ in s]) for s in ops])
        off, sym, tau = (torch.from_numpy(x).cuda() for x in (batch.offset, batch.symbol, batch.tau))
        m2, e2, _, status = lib.ctqmc_trace_batch(h, beta, off, sym, tau, max_len=int(np.diff(batch.offset).max()))
        torch.cuda.synchronize()
        mant, exp2, m2, e2 = mant.cpu().numpy(), exp2.cpu().numpy(), m2.cpu().numpy(), e2.cpu().numpy()
        assert (status.cpu().numpy() == 0).all()
        worst = 0.0
        for c in range(nC):
            assert m2[c, 0] != 0.0, c                      # an accepted configuration has a non-zero weight
            worst = max(worst, rel_diff(complex(*mant[c]), int(exp2[c]), complex(*m2[c]), int(e2[c])))
        assert worst <= TOL, worst
        for c in range(0, nC, 128):
            r = _exact(imp, beta, ops[c])
            assert rel_diff(complex(*mant[c]), int(exp2[c]), r["mant"], r["exp2"]) <= TOL * max(1.0, r["kappa"] * 1e-5), c
    finally:
        ch.destroy()
        h.free()
