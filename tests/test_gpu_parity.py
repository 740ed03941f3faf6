"""Parity of the CUDA path (through the C ABI) with the CPU oracle on the same seeded inputs.  Run on a B200: -m gpu.

Bars (BASELINE.json north_star):
  * routing (`survive`) and the vanishing pattern (`status`): bit-exact;
  * trace: |w_gpu - w_cpu| <= 1e-9 |w_cpu| at a common exponent (checks sign / phase too; reading A5), loosened only
    by the conditioning rule A8: (i) final cancellation, tolerance 1e-9 * max(1, kappa * 1e-5), at most 1 % of a batch;
    (ii) BASELINE config 3 only: its N-only sectors hide the S_z / L_z symmetries and fp64 does not determine a few per cent
    of its configurations in that basis -- on EITHER side.  There a true value exists: the same oracle on the same Hamiltonian
    labelled by (N, 2S_z, L_z) (equal by pin P4 (iii), stable to 1e-10 under the cyclic shifts of pin P2).  A configuration
    that misses 1e-9 against the coarse oracle is judged against that truth: |gpu - truth| <= max(1e-9, 10 |coarse - truth|),
    |coarse - truth| being the largest of four samples of the coarse oracle's own noise (the configuration as given and after
    three exact cyclic shifts), i.e. the GPU must be no worse than the fp64 oracle fed the same blocks.  Nothing is exempt;
  * bound: relative 1e-9 against the oracle's bound (plus, for segment products, the rounding floor 2^-40 x the product of
    the factor norms), bound >= |trace| per configuration AND per start sector.
"""
import math

import numpy as np
import pytest

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
    build.build()   # no-op when the in-tree library is newer than its sources (nvcc is in the image)
    import paper_2010_08482_b200 as L
    L.library()   # raises loudly if the extension is missing
    return L


@pytest.fixture(scope="module")
def handles(lib, impurities, torch_cuda):
    cache = {}

    def get(cfg):
        if cfg not in cache:
            cache[cfg] = lib.ctqmc_load_impurity(impurities(cfg), 0)
        return cache[cfg]
    yield get
    for h in cache.values():
        h.free()


def _dev(torch, batch):
    return (torch.from_numpy(batch.offset).cuda(), torch.from_numpy(batch.symbol).cuda(), torch.from_numpy(batch.tau).cuda())


_TRUTH = {}


def _truth_for(imp):
    """Config 3's Hamiltonian labelled by all its Abelian quantum numbers (N, 2S_z, L_z) (rule A8 (ii) above); None for
    every other impurity (they use all their quantum numbers already, or have none left to hide)."""
    if getattr(imp, "name", "") != "cfg3-dshell-N":
        return None
    if "cfg3" not in _TRUTH:
        from golden.make_golden import _fine_cfg3
        _TRUTH["cfg3"] = _fine_cfg3()
    return _TRUTH["cfg3"]


def _check_trace(lib, torch, imp, handle, batch, label, sample=None):
    """GPU against the oracle on every (sampled) configuration."""
    from oracle import trace_oracle as O
    truth_imp = _truth_for(imp)
    off, sym, tau = _dev(torch, batch)
    mant, exp2, surv, status = lib.ctqmc_trace_batch(handle, batch.beta, off, sym, tau)
    torch.cuda.synchronize()
    mant, exp2, surv, status = mant.cpu().numpy(), exp2.cpu().numpy(), surv.cpu().numpy(), status.cpu().numpy()
    worst = 0.0
    loosened = explained = 0
    checked = range(batch.n_configs) if sample is None else sample   # the GPU ran the whole batch; the oracle checks these
    for b in checked:
        s, t = batch.config(b)
        r = O.trace_config(imp, batch.beta, s, t)
        assert status[b] == r["status"], f"{label} config {b}: status {status[b]} != oracle {r['status']}"
        if r["status"] == 2:
            assert math.isnan(mant[b, 0]) and math.isnan(mant[b, 1])
            continue
        assert np.array_equal(surv[b], r["survive"]), f"{label} config {b}: survive mask differs"
        w = complex(mant[b, 0], mant[b, 1])
        if r["mant"] == 0:
            assert w == 0, f"{label} config {b}: oracle is exactly zero, gpu is {w}"
            continue
        mx = max(abs(w.real), abs(w.imag))
        assert 1.0 <= mx < 2.0, f"{label} config {b}: mantissa {w} not normalised"
        d = rel_diff(w, int(exp2[b]), r["mant"], r["exp2"])
        # kappa (final cancellation) loosens the bar only where no truth is available; with one, a miss is judged against it
        tol = TOL * max(1.0, r["kappa"] * 1e-5) if truth_imp is None else TOL
        if tol > TOL:
            loosened += 1
        if d > tol and truth_imp is not None and len(s) > 0:
            rt = O.trace_config(truth_imp, batch.beta, s, t)
            d_gpu = rel_diff(w, int(exp2[b]), rt["mant"], rt["exp2"])
            # the coarse oracle's own noise: its distance from the truth as computed, and after three exact cyclic shifts
            noise = [rel_diff(r["mant"], r["exp2"], rt["mant"], rt["exp2"])]
            for frac in (0.23, 0.52, 0.77):
                t2 = (t + frac * batch.beta) % batch.beta
                o = np.argsort(t2, kind="stable")
                r2 = O.trace_config(imp, batch.beta, s[o], t2[o])
                noise.append(rel_diff(r2["mant"], r2["exp2"], rt["mant"], rt["exp2"]))
            d_coarse = max(noise)
            print(f"{label} config {b}: coarse oracle is up to {d_coarse:.2e} from the (N,Sz,Lz) truth, gpu {d_gpu:.2e}, gpu-coarse {d:.2e}")
            assert d_gpu <= max(TOL, 10.0 * d_coarse), f"{label} config {b}: gpu {d_gpu:.3e} from the truth, coarse oracle {d_coarse:.3e}"
            explained += 1
            continue
        assert d <= tol, f"{label} config {b}: rel diff {d:.3e} > {tol:.1e} (kappa {r['kappa']:.2e})"
        if tol == TOL:
            worst = max(worst, d)          # worst difference among the configurations held to 1e-9
    n_checked = len(checked)
    assert loosened <= max(1, n_checked // 100), f"{label}: {loosened} configurations needed the kappa loosening"
    if explained:
        print(f"{label}: {explained} of {n_checked} configurations judged against the (N,Sz,Lz) truth")
    return worst


def _load_golden(cfg):
    import json
    import os
    from workloads import BASELINE_CONFIGS
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"cfg{cfg}_batch{BASELINE_CONFIGS[cfg]['batch']}.json")
    with open(path) as fh:
        return json.load(fh)


def _check_trace_golden(lib, torch, handle, batch, doc, label, records=None):
    """GPU against the stored oracle values (tests/golden/make_golden.py wrote them from oracle/ alone): EVERY record."""
    off, sym, tau = _dev(torch, batch)
    mant, exp2, surv, status = lib.ctqmc_trace_batch(handle, batch.beta, off, sym, tau)
    torch.cuda.synchronize()
    mant, exp2, surv, status = mant.cpu().numpy(), exp2.cpu().numpy(), surv.cpu().numpy(), status.cpu().numpy()
    recs = doc["records"] if records is None else records
    worst, judged_by_truth, loosened = 0.0, 0, 0
    for rec in recs:
        b = rec["b"]
        assert b < batch.n_configs and rec["n_ops"] == len(batch.config(b)[0]), f"{label}: golden record {b} is not this batch's configuration"
        assert status[b] == rec["status"], f"{label} config {b}: status"
        assert "".join(str(int(x)) for x in surv[b]) == rec["survive"], f"{label} config {b}: survive mask differs"
        w = complex(mant[b, 0], mant[b, 1])
        om, oe = complex(*rec["mant"]), rec["exp2"]
        assert om != 0 and 1.0 <= max(abs(w.real), abs(w.imag)) < 2.0
        d = rel_diff(w, int(exp2[b]), om, oe)
        tol = TOL * max(1.0, rec["kappa"] * 1e-5)
        loosened += tol > TOL and "coarse_shifts" not in rec     # kappa of a configuration fp64 does not determine means nothing
        if "fine" in rec and d > tol:
            tm, te = complex(*rec["fine"]["mant"]), rec["fine"]["exp2"]
            d_gpu = rel_diff(w, int(exp2[b]), tm, te)
            d_coarse = max([rel_diff(om, oe, tm, te)] + [rel_diff(complex(*x["mant"]), x["exp2"], tm, te) for x in rec.get("coarse_shifts", [])])
            assert d_gpu <= max(TOL, 10.0 * d_coarse), f"{label} config {b}: gpu {d_gpu:.3e} from the truth, coarse oracle {d_coarse:.3e}"
            judged_by_truth += 1
            continue
        assert d <= tol, f"{label} config {b}: rel diff {d:.3e} > {tol:.1e} (kappa {rec['kappa']:.2e})"
        worst = max(worst, d)
    assert loosened <= max(1, len(recs) // 100), f"{label}: {loosened} configurations needed the kappa loosening"
    print(f"{label}: {len(recs)} outputs against the golden file, worst relative difference {worst:.3e}, "
          f"{judged_by_truth} judged against the (N,Sz,Lz) truth")
    return worst


# --------------------------------------------------------------------------- trace parity on the BASELINE configs
@pytest.mark.parametrize("cfg,n", [(1, 1024), (2, 512), (3, 24), (4, 4)])
def test_trace_parity_baseline_configs(cfg, n, lib, torch_cuda, impurities, handles):
    from workloads import make_batch
    batch = make_batch(cfg, n)
    worst = _check_trace(lib, torch_cuda, impurities(cfg), handles(cfg), batch, f"cfg{cfg}")
    print(f"cfg{cfg}: worst relative difference {worst:.3e}")


@pytest.mark.parametrize("cfg", [1, 2])
def test_trace_parity_full_baseline_batch(cfg, lib, torch_cuda, impurities, handles):
    """BASELINE.json's full batch in the launch configuration bench.py times, EVERY output against the oracle run here
    (configs 1-2); configs 3-5: test_trace_parity_full_baseline_batch_golden."""
    from workloads import BASELINE_CONFIGS, make_batch
    B = BASELINE_CONFIGS[cfg]["batch"]
    worst = _check_trace(lib, torch_cuda, impurities(cfg), handles(cfg), make_batch(cfg, B), f"cfg{cfg}-full")
    print(f"cfg{cfg} full batch {B}, every output checked: worst relative difference {worst:.3e}")


@pytest.mark.parametrize("cfg", [3, 4])
def test_trace_parity_full_baseline_batch_golden(cfg, lib, torch_cuda, impurities, handles):
    """BASELINE.json's full batches of configs 3 (1024) and 4 (256) in the launch configuration bench.py times: EVERY output
    against the oracle values stored by tests/golden/make_golden.py; config 5: test_trace_parity_cfg5_*."""
    from workloads import BASELINE_CONFIGS, make_batch
    doc = _load_golden(cfg)
    B = BASELINE_CONFIGS[cfg]["batch"]
    assert doc["batch"] == B and len(doc["records"]) == B
    _check_trace_golden(lib, torch_cuda, handles(cfg), make_batch(cfg, B), doc, f"cfg{cfg}-full")


@pytest.mark.parametrize("cfg,n", [(1, 64), (2, 64), (3, 6), (4, 2)])
def test_trace_parity_literal_schedule(cfg, n, lib, torch_cuda, impurities, handles):
    """The literal order of Eq. 65 (start at q0, carry dim(q0) columns) must agree with the thin start."""
    from workloads import make_batch
    h = handles(cfg)
    lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_LITERAL)
    try:
        _check_trace(lib, torch_cuda, impurities(cfg), h, make_batch(cfg, n, start=5000), f"cfg{cfg}-literal")
    finally:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_THIN)


@pytest.mark.parametrize("cfg,width", [(2, 8), (2, 16), (3, 8), (3, 16), (3, 32)])
def test_trace_parity_panel_widths(cfg, width, lib, torch_cuda, impurities, handles):
    from workloads import make_batch
    h = handles(cfg)
    lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_PANEL)
    try:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PANEL_WIDTH, width)
    except lib.CtqmcError as e:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)
        if e.code == -4:
            pytest.skip(str(e))
        raise
    try:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_LITERAL)
        _check_trace(lib, torch_cuda, impurities(cfg), h, make_batch(cfg, 6, start=7000), f"cfg{cfg}-W{width}")
    finally:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_THIN)
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PANEL_WIDTH, 0)
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)


# --------------------------------------------------------------------------- kernel families
def test_small_path_is_the_default_for_small_sectors(lib, torch_cuda, impurities, handles):
    from workloads import make_batch
    for cfg in (1, 2):
        batch = make_batch(cfg, 8)
        off, sym, tau = _dev(torch_cuda, batch)
        lib.ctqmc_trace_batch(handles(cfg), batch.beta, off, sym, tau)
        st = lib.ctqmc_last_stats(handles(cfg))
        assert st["path"] == lib.CTQMC_PATH_SMALL and st["launches"] == 1, st
    with pytest.raises(lib.CtqmcError) as ei:
        lib.ctqmc_set_option(handles(3), lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_SMALL)
    assert ei.value.code == -4


@pytest.mark.parametrize("cfg,n", [(1, 256), (2, 128)])
@pytest.mark.parametrize("schedule", ["thin", "literal"])
def test_trace_parity_panel_path_forced(cfg, n, schedule, lib, torch_cuda, impurities, handles):
    """The shared-memory panel kernel (one-warp teams) on the small impurities, which default to the small path."""
    from workloads import make_batch
    h = handles(cfg)
    lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_PANEL)
    try:
        if schedule == "literal":
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_LITERAL)
        _check_trace(lib, torch_cuda, impurities(cfg), h, make_batch(cfg, n, start=11000), f"cfg{cfg}-panel-{schedule}")
        assert lib.ctqmc_last_stats(h)["path"] == lib.CTQMC_PATH_PANEL
    finally:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_THIN)
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)


@pytest.mark.parametrize("cfg,n", [(1, 300), (2, 200)])
def test_small_path_first_variant_on_real_impurities(cfg, n, lib, torch_cuda, impurities, monkeypatch):
    """Real small impurities default to the uniform (padded, DP lanes per configuration) variant; CTQMC_SMALL_V1=1 selects
    the element-per-lane variant that complex impurities use.  Both against the oracle, both schedules."""
    from workloads import make_batch
    imp = impurities(cfg)
    monkeypatch.setenv("CTQMC_SMALL_V1", "1")
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        for sched in (lib.CTQMC_SCHEDULE_THIN, lib.CTQMC_SCHEDULE_LITERAL):
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, sched)
            _check_trace(lib, torch_cuda, imp, h, make_batch(cfg, n, start=16000), f"cfg{cfg}-small-v1")
            st = lib.ctqmc_last_stats(h)
            assert st["path"] == lib.CTQMC_PATH_SMALL and st["panel_width"] in (8, 16, 32)   # lanes per configuration, not DP
    finally:
        h.free()


@pytest.mark.parametrize("dims", [(2, 1), (6, 5), (12, 7), (16, 12)])
def test_small_path_every_padded_size(dims, lib, torch_cuda):
    """The uniform small-sector kernels are instantiated for DP = 2, 4, 6, 9, 12, 16 lanes per configuration; BASELINE's
    impurities only reach 4 and 9.  Hand-built two-sector impurities with seeded random blocks (0 -> 1, 1 -> 0, 0 -> 0) and
    random closed walks cover the rest, traces and S = 1 bounds against the oracle."""
    import types
    from workloads import Batch
    from workloads.rng import Stream
    rng = Stream(100 * dims[0] + dims[1])
    d0, d1 = dims
    blocks = [(0, 0, 1), (1, 1, 0), (2, 0, 0)]          # (symbol, src, dst)
    data, off, pos = [], [], 0
    for _, s_, d_ in blocks:
        m, n = (d0, d1)[d_], (d0, d1)[s_]
        data.append(np.array([rng.normal() for _ in range(m * n)]) * (0.9 / np.sqrt(max(m, n))))
        off.append(pos); pos += m * n
    energy = np.array([0.3 * rng.normal() for _ in range(d0 + d1)])
    beta = 3.0
    imp = types.SimpleNamespace(dims=np.array([d0, d1], np.int32), energy=energy, n_symbols=3, is_complex=False, n_sectors=2,
                                beta=beta, blk_symbol=np.array([b[0] for b in blocks], np.int32),
                                blk_src=np.array([b[1] for b in blocks], np.int32), blk_dst=np.array([b[2] for b in blocks], np.int32),
                                blk_offset=np.array(off, np.int64), blk_data=np.concatenate(data))
    cfgs = []
    for _ in range(40):
        q, syms = 0, []
        for _ in range(2 + rng.integer(30)):             # random walk on the two sectors, closed at the end
            a = (rng.integer(2) * 2) if q == 0 else 1     # from 0: symbol 0 (to 1) or 2 (stay); from 1: symbol 1 (back)
            syms.append(a)
            q = 1 if a == 0 else 0
        if q == 1:
            syms.append(1)
        taus = np.sort(beta * rng.uniforms(len(syms)))
        cfgs.append((syms, taus))
    cfgs += [([], []), ([1, 0], [0.5, 1.0]), ([0, 0], [0.5, 1.0])]   # empty; closes from sector 1 only; hits the zero sector
    batch = Batch.from_lists(beta, cfgs)
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        for sched in (lib.CTQMC_SCHEDULE_THIN, lib.CTQMC_SCHEDULE_LITERAL):
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, sched)
            _check_trace(lib, torch_cuda, imp, h, batch, f"pad{dims}")
            st = lib.ctqmc_last_stats(h)
            assert st["path"] == lib.CTQMC_PATH_SMALL and st["panel_width"] >= max(dims)
        _check_bound(lib, torch_cuda, imp, h, batch, 0, 1, f"pad{dims}-frobenius")
    finally:
        h.free()


@pytest.mark.parametrize("lanes", [8, 16, 32])
def test_small_path_complex_and_group_sizes(lanes, lib, torch_cuda, monkeypatch):
    """Small path with complex blocks (config 1 with seeded eigenvector phases, reading A17) and every lanes-per-
    configuration variant, both schedules."""
    from workloads import impurity as wi
    from workloads import make_batch
    h1, u, qn = wi._kanamori(2, 4.0, 0.8, 2.0)
    imp = wi.build_impurity("cfg1-phases", h1, u, qn, beta=10.0, phase_seed=3)
    assert imp.is_complex
    monkeypatch.setenv("CTQMC_SMALL_G", str(lanes))
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        for sched in (lib.CTQMC_SCHEDULE_THIN, lib.CTQMC_SCHEDULE_LITERAL):
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, sched)
            _check_trace(lib, torch_cuda, imp, h, make_batch(1, 300, start=12000), f"small-complex-G{lanes}")
            st = lib.ctqmc_last_stats(h)
            assert st["path"] == lib.CTQMC_PATH_SMALL and st["panel_width"] == lanes
    finally:
        h.free()


def test_complex_toy_panel_and_large(lib, torch_cuda):
    """The complex p-shell toy of oracle pin P3 (only N conserved, d_max = 20) through the panel and the large path."""
    from test_oracle_pins import _p_shell_toy, _toy_batch
    imp = _p_shell_toy()
    batch = _toy_batch(6, imp.beta, 40, seed=78, pairs=4)
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        for path in (lib.CTQMC_PATH_PANEL, lib.CTQMC_PATH_LARGE):
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, path)
            _check_trace(lib, torch_cuda, imp, h, batch, f"ptoy-path{path}")
    finally:
        h.free()


# --------------------------------------------------------------------------- large-sector path (tiled GEMM, one launch per step)
@pytest.mark.parametrize("cfg,n", [(1, 64), (2, 64), (3, 12), (4, 3)])
@pytest.mark.parametrize("schedule", ["thin", "literal"])
def test_trace_parity_large_path_forced(cfg, n, schedule, lib, torch_cuda, impurities, handles):
    """The large-sector kernel family forced onto the small impurities: ragged tiles (dims 1..295 against 128 x 64
    tiles), real and complex, both schedules, element-wise against the oracle."""
    from workloads import make_batch
    h = handles(cfg)
    lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_LARGE)
    try:
        if schedule == "literal":
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_LITERAL)
        worst = _check_trace(lib, torch_cuda, impurities(cfg), h, make_batch(cfg, n, start=9000), f"cfg{cfg}-large-{schedule}")
        assert lib.ctqmc_last_stats(h)["path"] == lib.CTQMC_PATH_LARGE
        print(f"cfg{cfg} large path {schedule}: worst relative difference {worst:.3e}")
    finally:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_THIN)
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)


@pytest.mark.parametrize("cfg,n", [(1, 64), (2, 64), (3, 24), (4, 4)])
@pytest.mark.parametrize("schedule", ["thin", "literal"])
def test_trace_parity_grouped_path(cfg, n, schedule, lib, torch_cuda, impurities, handles):
    """Step-synchronous grouped GEMM path: strings sharing a block share a GEMM; columns gathered from / scattered to the
    strings' own matrices.  Ragged tiles, real and complex, both schedules, element-wise against the oracle."""
    from workloads import make_batch
    h = handles(cfg)
    lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_GROUPED)
    try:
        if schedule == "literal":
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_LITERAL)
        worst = _check_trace(lib, torch_cuda, impurities(cfg), h, make_batch(cfg, n, start=13000), f"cfg{cfg}-grouped-{schedule}")
        assert lib.ctqmc_last_stats(h)["path"] == lib.CTQMC_PATH_GROUPED
        print(f"cfg{cfg} grouped path {schedule}: worst relative difference {worst:.3e}")
    finally:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_THIN)
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)


def test_auto_path_by_batch_size(lib, torch_cuda, impurities, handles):
    """AUTO: batches of >= 64 configurations of a mid-size impurity take the grouped path, smaller ones the panel kernel;
    both agree with the oracle (checked on the larger batch here, on the smaller ones by the baseline-config tests)."""
    from workloads import make_batch
    h = handles(3)
    batch = make_batch(3, 72, start=15000)
    _check_trace(lib, torch_cuda, impurities(3), h, batch, "cfg3-auto-72")
    assert lib.ctqmc_last_stats(h)["path"] == lib.CTQMC_PATH_GROUPED
    off, sym, tau = _dev(torch_cuda, make_batch(3, 8, start=15000))
    lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau)
    assert lib.ctqmc_last_stats(h)["path"] == lib.CTQMC_PATH_PANEL


def test_grouped_scratch_limit_falls_back_to_panel(lib, torch_cuda, impurities, handles):
    """With a scratch limit too small for the grouped schedule AUTO runs the panel kernel (same results); an explicit
    request for the grouped path reports CTQMC_ERR_OOM."""
    from workloads import make_batch
    h = handles(3)
    batch = make_batch(3, 72, start=17000)
    lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCRATCH_LIMIT, 1 << 20)
    try:
        _check_trace(lib, torch_cuda, impurities(3), h, batch, "cfg3-auto-limited")
        assert lib.ctqmc_last_stats(h)["path"] == lib.CTQMC_PATH_PANEL
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_GROUPED)
        off, sym, tau = _dev(torch_cuda, batch)
        with pytest.raises(lib.CtqmcError) as ei:
            lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau)
        assert ei.value.code == -2
    finally:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCRATCH_LIMIT, 0)
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)
    _check_trace(lib, torch_cuda, impurities(3), h, batch, "cfg3-auto-unlimited")
    assert lib.ctqmc_last_stats(h)["path"] == lib.CTQMC_PATH_GROUPED


def test_grouped_path_edge_cases_and_repeatability(lib, torch_cuda, impurities, handles):
    from workloads import Batch, make_batch
    imp = impurities(2)
    h = handles(2)
    good = make_batch(2, 3, start=960)
    cfgs = [good.config(0), ([], []), ([1, 1, 1, 1], [1.0, 2.0, 3.0, 4.0]), ([1, 1], [1.0, 2.0]), ([1, 0], [3.0, 2.0]),
            good.config(1), ([1, 0], [0.0, 0.0]), good.config(2)]
    batch = Batch.from_lists(imp.beta, cfgs)
    lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_GROUPED)
    try:
        _check_trace(lib, torch_cuda, imp, h, batch, "grouped-edge")
    finally:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)
    # column order inside a group comes from atomics, the values must not depend on it
    h3 = handles(3)
    b3 = make_batch(3, 16, start=14000)
    off, sym, tau = _dev(torch_cuda, b3)
    lib.ctqmc_set_option(h3, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_GROUPED)
    try:
        a = lib.ctqmc_trace_batch(h3, b3.beta, off, sym, tau)
        torch_cuda.cuda.synchronize()
        b = lib.ctqmc_trace_batch(h3, b3.beta, off, sym, tau)
        torch_cuda.cuda.synchronize()
        for x, y in zip(a, b):
            assert torch_cuda.equal(x, y)
    finally:
        lib.ctqmc_set_option(h3, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)


def test_large_path_edge_cases(lib, torch_cuda, impurities, handles):
    """Empty, vanishing, invalid and off-diagonal configurations through the large-sector path."""
    from workloads import Batch, make_batch
    imp = impurities(2)
    h = handles(2)
    good = make_batch(2, 3, start=950)
    cfgs = [good.config(0), ([], []), ([1, 1, 1, 1], [1.0, 2.0, 3.0, 4.0]), ([1, 1], [1.0, 2.0]), ([1, 0], [3.0, 2.0]),
            good.config(1), ([1, 0], [0.0, 0.0]), good.config(2)]
    batch = Batch.from_lists(imp.beta, cfgs)
    lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_LARGE)
    try:
        _check_trace(lib, torch_cuda, imp, h, batch, "large-edge")
    finally:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)


def test_trace_parity_cfg5_crystal_field(lib, torch_cuda, impurities):
    """BASELINE config 5 (sectors 1001 / 2002 / 3003, complex), the config north_star's tensor-pipe target is stated on: the
    full batch of 64 at the launch configuration bench.py times (thin schedule), EVERY output against the stored oracle
    values (tests/golden/cfg5_batch64.json: 1.1e13 flop of numpy each, computed once by tests/golden/make_golden.py); then
    the literal schedule of Eq. 65 on the first 6, which must agree with the same file; then the S = 1 Frobenius bound."""
    from workloads import make_batch
    doc = _load_golden(5)
    assert doc["batch"] == 64 and len(doc["records"]) == 64
    imp = impurities(5)
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        assert lib.ctqmc_last_stats(h)["path"] == lib.CTQMC_PATH_LARGE
        _check_trace_golden(lib, torch_cuda, h, make_batch(5, 64), doc, "cfg5-thin")
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_LITERAL)
        _check_trace_golden(lib, torch_cuda, h, make_batch(5, 6), doc, "cfg5-literal", records=doc["records"][:6])
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, lib.CTQMC_SCHEDULE_THIN)
        _check_bound(lib, torch_cuda, imp, h, make_batch(5, 1), 0, 1, "cfg5-frobenius-S1", golden=doc)
    finally:
        h.free()


def test_split_precision_path_meets_the_same_bar(lib, torch_cuda, impurities):
    """CTQMC_PATH_SPLIT: every chain step as int8 slice products on the tcgen05 tensor pipe, exact
    int32 accumulation, FP64 recombination.  Kept only because it meets the bar of the FP64 path: ALL 64 golden outputs of config 5
    within 1e-9 (7 slices, the default), config 4 against the oracle element by element (thin and literal schedule, long and
    empty configurations, 8 slices too); survive / status bit-exact.  Real impurities are refused."""
    from workloads import Batch, make_batch
    doc = _load_golden(5)
    imp = impurities(5)
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_SPLIT)
        _check_trace_golden(lib, torch_cuda, h, make_batch(5, 64), doc, "cfg5-split")
        assert lib.ctqmc_last_stats(h)["path"] == lib.CTQMC_PATH_SPLIT
    finally:
        h.free()
    imp4 = impurities(4)
    for slices in (7, 8):
        h = lib.ctqmc_load_impurity(imp4, 0)
        try:
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_SPLIT_SLICES, slices)
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_SPLIT)
            good = make_batch(4, 3, start=333)
            batch = Batch.from_lists(imp4.beta, [good.config(0), ([], []), good.config(1), ([1, 1], [0.5, 0.7]), good.config(2)])
            for sched in (lib.CTQMC_SCHEDULE_THIN, lib.CTQMC_SCHEDULE_LITERAL):
                lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, sched)
                _check_trace(lib, torch_cuda, imp4, h, batch, f"cfg4-split-S{slices}-sched{sched}")
            with pytest.raises(lib.CtqmcError):
                lib.ctqmc_set_option(h, lib.CTQMC_OPT_SPLIT_SLICES, 6 if slices == 7 else 7)      # planes are built
        finally:
            h.free()
    h = lib.ctqmc_load_impurity(impurities(3), 0)
    try:
        with pytest.raises(lib.CtqmcError) as ei:
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_SPLIT)
        assert ei.value.code == lib.CTQMC_ERR_UNSUPPORTED
        assert lib.ctqmc_last_stats(h)["path"] in (lib.CTQMC_PATH_PANEL, lib.CTQMC_PATH_GROUPED, lib.CTQMC_PATH_AUTO)
    finally:
        h.free()


# --------------------------------------------------------------------------- edge cases
def test_empty_configuration_is_partition_function(lib, torch_cuda, impurities, handles):
    """L = 0 gives Z = sum_n exp(-beta E_n) (north_star pin P1), here against the closed form directly."""
    from workloads import Batch
    for cfg in (1, 2, 3):
        imp = impurities(cfg)
        batch = Batch.from_lists(imp.beta, [([], []), ([], [])])
        off, sym, tau = _dev(torch_cuda, batch)
        mant, exp2, surv, status = lib.ctqmc_trace_batch(handles(cfg), imp.beta, off, sym, tau)
        torch_cuda.cuda.synchronize()
        emin = imp.energy.min()
        z = math.fsum(np.exp(-imp.beta * (imp.energy - emin)))
        lg = -imp.beta * emin / math.log(2.0)
        k = math.floor(lg)
        zm, ze = math.frexp(z * 2.0 ** (lg - k))
        for b in range(2):
            assert status[b].item() == 0 and surv[b].all().item()
            assert rel_diff(complex(mant[b, 0].item(), mant[b, 1].item()), int(exp2[b].item()), zm, ze + k) < 1e-10


def test_empty_batch_and_null_arguments(lib, torch_cuda, impurities, handles):
    from workloads import Batch
    imp = impurities(1)
    batch = Batch.from_lists(imp.beta, [])
    off, sym, tau = _dev(torch_cuda, batch)
    mant, exp2, surv, status = lib.ctqmc_trace_batch(handles(1), imp.beta, off, sym, tau)
    assert mant.shape == (0, 2)
    with pytest.raises(lib.CtqmcError):
        lib.ctqmc_trace_batch(handles(1), -1.0, off, sym, tau)
    assert "beta" in lib.ctqmc_last_error()


def test_vanishing_invalid_and_ragged(lib, torch_cuda, impurities, handles):
    """Structurally vanishing strings (status 1, exact zero), invalid inputs (status 2, NaN) and valid ones of very
    different lengths in one batch; neighbours must be unaffected."""
    from workloads import Batch, make_batch
    imp = impurities(2)
    good = make_batch(2, 5, start=900)
    c = [good.config(b) for b in range(5)]
    beta = imp.beta
    cfgs = [
        c[0],
        ([1, 1, 1, 1], [1.0, 2.0, 3.0, 4.0]),  # c^dag_0 four times: leaves the sector table from every start sector
        ([1, 1], [1.0, 2.0]),                  # c^dag_0 twice: survives routing but q_L != q_0, contributes exactly 0
        c[1],
        ([1, 0], [3.0, 2.0]),                  # tau decreasing
        ([1, 0], [1.0, beta]),                 # tau == beta is outside [0, beta)
        ([99, 0], [1.0, 2.0]),                 # symbol out of range
        ([1, 0], [1.0, float("nan")]),
        c[2],
        ([], []),
        ([1, 0], [0.0, 0.0]),                  # equal times, tau = 0 (reading A7): legal
        ([0, 1, 3, 2], [1.0, 1.0, 7.5, 7.5]),  # ties keep input order
        c[3], c[4],
    ]
    batch = Batch.from_lists(beta, cfgs)
    _check_trace(lib, torch_cuda, imp, handles(2), batch, "edge")
    off, sym, tau = _dev(torch_cuda, batch)
    mant, exp2, surv, status = lib.ctqmc_trace_batch(handles(2), beta, off, sym, tau)
    st = status.cpu().numpy()
    assert list(st) == [0, 1, 0, 0, 2, 2, 2, 2, 0, 0, 0, 0, 0, 0]
    assert mant[1].abs().sum().item() == 0.0 and exp2[1].item() == 0 and surv[1].sum().item() == 0
    assert mant[2].abs().sum().item() == 0.0 and exp2[2].item() == 0 and surv[2].sum().item() > 0


def test_long_chain_exponent_range(lib, torch_cuda, impurities, handles):
    """A long chain (L = 2000) at large beta: the running exponent must carry ~1e4 binary orders without overflow."""
    from workloads import Batch
    from workloads.rng import Stream
    imp = impurities(2)
    rng = Stream(77)
    beta = 2000.0
    cfgs = []
    for _ in range(3):
        ops = []
        for f in range(6):
            t = np.sort(beta * rng.uniforms(334))
            first = rng.integer(2)
            ops += [(t[i], 2 * f + ((first + i) & 1)) for i in range(len(t))]
        ops.sort()
        cfgs.append(([a for _, a in ops], [t for t, _ in ops]))
    batch = Batch.from_lists(beta, cfgs)
    _check_trace(lib, torch_cuda, imp, handles(2), batch, "long")


@pytest.mark.parametrize("path", ["panel", "grouped", "large"])
def test_long_and_single_configuration_mid_size_paths(path, lib, torch_cuda, impurities, handles):
    """Chains of ~600 operators at beta = 200 on the d-shell impurity (running exponents of several 1e4 binary orders) and
    a batch of ONE configuration, through the panel, grouped and large-sector kernel families."""
    from workloads import Batch, make_batch
    from workloads.rng import Stream
    imp = impurities(3)
    h = handles(3)
    rng = Stream(991)
    beta = 200.0
    cfgs = []
    for _ in range(3):
        ops = []
        for f in range(10):
            t = np.sort(beta * rng.uniforms(60))
            first = rng.integer(2)
            ops += [(t[i], 2 * f + ((first + i) & 1)) for i in range(len(t))]
        ops.sort()
        cfgs.append(([a for _, a in ops], [t for t, _ in ops]))
    long_batch = Batch.from_lists(beta, cfgs)
    one = make_batch(3, 1, start=19000)
    lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, {"panel": lib.CTQMC_PATH_PANEL, "grouped": lib.CTQMC_PATH_GROUPED,
                                                 "large": lib.CTQMC_PATH_LARGE}[path])
    try:
        _check_trace(lib, torch_cuda, imp, h, long_batch, f"cfg3-long-{path}")
        _check_trace(lib, torch_cuda, imp, h, one, f"cfg3-one-{path}")
    finally:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)


def test_host_form_matches_device_form(lib, torch_cuda, impurities, handles):
    from workloads import make_batch
    for cfg, n in ((1, 200), (3, 5)):
        batch = make_batch(cfg, n, start=300)
        off, sym, tau = _dev(torch_cuda, batch)
        d = lib.ctqmc_trace_batch(handles(cfg), batch.beta, off, sym, tau)
        torch_cuda.cuda.synchronize()
        h = lib.ctqmc_trace_batch_host(handles(cfg), batch.beta, batch.offset, batch.symbol, batch.tau)
        for a, b in zip(d, h):
            assert np.array_equal(a.cpu().numpy(), b, equal_nan=True)


@pytest.mark.parametrize("cfg,n", [(1, 40000), (2, 300), (3, 6)])
def test_host_form_with_pinned_buffers(cfg, n, lib, torch_cuda, impurities, handles):
    """Page-locked caller buffers: direct copies (and, for the large small-sector batch, chunked copy/compute overlap) must
    give exactly the device form's results."""
    from workloads import make_batch
    torch = torch_cuda
    batch = make_batch(cfg, n, start=500)
    off, sym, tau = _dev(torch, batch)
    d = lib.ctqmc_trace_batch(handles(cfg), batch.beta, off, sym, tau)
    torch.cuda.synchronize()
    pin = [torch.from_numpy(x).pin_memory() for x in (batch.offset, batch.symbol, batch.tau)]
    Q = impurities(cfg).n_sectors
    pout = [torch.full((n, 2), -7.0, dtype=torch.float64).pin_memory(), torch.zeros(n, dtype=torch.int64).pin_memory(),
            torch.zeros((n, Q), dtype=torch.uint8).pin_memory(), torch.full((n,), -1, dtype=torch.int32).pin_memory()]
    lib.ctqmc_trace_batch_host(handles(cfg), batch.beta, *[t.numpy() for t in pin], out=tuple(t.numpy() for t in pout))
    for a, b in zip(d, pout):
        assert torch.equal(a.cpu(), b)


def test_repeatable_and_stream_ordered(lib, torch_cuda, impurities, handles):
    """Same inputs twice, on a side stream, give bit-identical outputs (fixed summation order)."""
    from workloads import make_batch
    batch = make_batch(3, 8, start=40)
    off, sym, tau = _dev(torch_cuda, batch)
    a = lib.ctqmc_trace_batch(handles(3), batch.beta, off, sym, tau)
    torch_cuda.cuda.synchronize()
    st = torch_cuda.cuda.Stream()
    with torch_cuda.cuda.stream(st):
        b = lib.ctqmc_trace_batch(handles(3), batch.beta, off, sym, tau, stream=st)
    st.synchronize()
    for x, y in zip(a, b):
        assert torch_cuda.equal(x, y)


# --------------------------------------------------------------------------- bounds
def _check_bound(lib, torch, imp, handle, batch, norm_kind, S, label, golden=None):
    """Bounds against the oracle's (1e-9), and against the traces they bound: per configuration (GPU trace) and per start
    sector (the oracle's t(q0): the lazy trace consumes per-sector bounds).  Segment products (S != 1): where a
    start sector's product vanishes by a symmetry the sector labels do not resolve, fl(G) is rounding noise on both sides and
    its norm has no digits; such a sector's bound is 2^-45 ... 2^-53 of the configuration's.  So a per-sector bound must match
    to 1e-9 relative OR to 2^-40 of the configuration's bound in absolute terms; the configuration's
    bound itself always to 1e-9.  `golden`: stored oracle traces (config 5: the oracle takes a minute per configuration)."""
    from oracle import trace_oracle as O
    off, sym, tau = _dev(torch, batch)
    bm, be, sm, se, status = lib.ctqmc_bound_batch(handle, batch.beta, off, sym, tau, norm_kind, S)
    mant, exp2, surv, tstatus = lib.ctqmc_trace_batch(handle, batch.beta, off, sym, tau)
    torch.cuda.synchronize()
    bm, be, sm, se, status = [x.cpu().numpy() for x in (bm, be, sm, se, status)]
    mant, exp2 = mant.cpu().numpy(), exp2.cpu().numpy()
    for b in range(batch.n_configs):
        s, t = batch.config(b)
        # spectral bounds of segment products: the CUDA path returns the certified estimate (oracle norm_kind 2, reading A1)
        certified = norm_kind == 1 and S != 1
        r = O.bound_config(imp, batch.beta, s, t, 2 if certified else norm_kind, S)
        assert status[b] == r["status"]
        if certified and r["status"] == 0:
            # ... which must lie between the exact spectral-norm bound (SVD of every segment product) and the Frobenius form
            rx = O.bound_config(imp, batch.beta, s, t, 1, S)
            rf = O.bound_config(imp, batch.beta, s, t, 0, S)
            dminmax = math.sqrt(max(int(d) for d in imp.dims))
            assert scaled_ge(bm[b] * (1 + 1e-9), int(be[b]), rx["mant"], rx["exp2"]), f"{label} config {b}: below the exact spectral bound"
            assert scaled_ge(rf["mant"] * dminmax * (1 + 1e-9), rf["exp2"], bm[b], int(be[b])), f"{label} config {b}: above the Frobenius bound"
        if r["status"] == 2:
            assert math.isnan(bm[b])
            continue
        d = rel_diff(bm[b], int(be[b]), r["mant"], r["exp2"])
        assert d <= TOL, f"{label} config {b}: bound rel diff {d:.3e}"
        if golden is not None:
            tsec = {q0: (complex(re, im), e) for q0, re, im, e in golden["records"][b]["sector"]}
        else:
            tsec = {q0: se_ for q0, se_ in enumerate(O.trace_config(imp, batch.beta, s, t)["sector"]) if se_ is not None}
        for q0, sec in enumerate(r["sector"]):
            if sec is None:
                assert sm[b, q0] == 0.0 and se[b, q0] == 0
                continue
            if sec[0] == 0:
                assert sm[b, q0] == 0.0
            else:
                floor_q = 0.0 if S == 1 else r["mant"] * 2.0 ** max(-300, min(300, r["exp2"] - sec[1] - 40)) / sec[0]
                dq = rel_diff(sm[b, q0], int(se[b, q0]), sec[0], sec[1])
                assert dq <= TOL + floor_q, f"{label} config {b} sector {q0}: rel diff {dq:.3e} (rounding floor {floor_q:.1e})"
            zs, es = tsec[q0]
            if S == 1:      # tables: strict
                assert scaled_ge(sm[b, q0], int(se[b, q0]), abs(zs), es), f"{label} config {b} sector {q0}: B(q0) < |t(q0)|"
            else:           # segment products: B(q0) + 2^-40 B(configuration) >= |t(q0)| (floor of fl(G))
                ok = scaled_ge(sm[b, q0], int(se[b, q0]), abs(zs), es) or scaled_ge(r["mant"], r["exp2"] - 40, abs(zs), es)
                assert ok, f"{label} config {b} sector {q0}: B(q0) + 2^-40 B < |t(q0)|"
        w = abs(complex(mant[b, 0], mant[b, 1]))
        assert scaled_ge(bm[b], int(be[b]), w, int(exp2[b])), f"{label} config {b}: bound < |trace|"


@pytest.mark.parametrize("cfg,n", [(1, 128), (2, 128), (3, 8), (4, 2)])
@pytest.mark.parametrize("norm_kind", [0, 1])
def test_bound_s1_parity(cfg, n, norm_kind, lib, torch_cuda, impurities, handles):
    from workloads import make_batch
    _check_bound(lib, torch_cuda, impurities(cfg), handles(cfg), make_batch(cfg, n, start=100), norm_kind, 1,
                 f"cfg{cfg}-nk{norm_kind}-S1")


@pytest.mark.parametrize("cfg,n", [(1, 64), (2, 64), (3, 4)])
@pytest.mark.parametrize("S", [0, 2, 8, 37])
def test_bound_segments_parity(cfg, n, S, lib, torch_cuda, impurities, handles):
    from workloads import make_batch
    _check_bound(lib, torch_cuda, impurities(cfg), handles(cfg), make_batch(cfg, n, start=200), 0, S,
                 f"cfg{cfg}-S{S}")


@pytest.mark.parametrize("cfg,n", [(1, 32), (2, 32), (3, 4), (4, 1)])
@pytest.mark.parametrize("S", [0, 3, 16])
def test_bound_segments_parity_large_path(cfg, n, S, lib, torch_cuda, impurities, handles):
    """Segment Frobenius norms through the large-sector kernel family (what config 5 uses), forced onto the small
    impurities so that the oracle can check every segment."""
    from workloads import make_batch
    h = handles(cfg)
    lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_LARGE)
    try:
        _check_bound(lib, torch_cuda, impurities(cfg), h, make_batch(cfg, n, start=250), 0, S, f"cfg{cfg}-large-S{S}")
    finally:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)


def test_bound_edge_cases(lib, torch_cuda, impurities, handles):
    from workloads import Batch, make_batch
    imp = impurities(2)
    good = make_batch(2, 2, start=77)
    cfgs = [good.config(0), ([], []), ([1, 1, 1, 1], [1.0, 2.0, 3.0, 4.0]), ([1, 0], [3.0, 2.0]), good.config(1)]
    batch = Batch.from_lists(imp.beta, cfgs)
    for nk, S in ((0, 1), (1, 1), (0, 0), (0, 3), (1, 4), (1, 0)):
        _check_bound(lib, torch_cuda, imp, handles(2), batch, nk, S, f"edge-nk{nk}-S{S}")
    off, sym, tau = _dev(torch_cuda, batch)
    with pytest.raises(lib.CtqmcError) as ei:
        lib.ctqmc_bound_batch(handles(2), imp.beta, off, sym, tau, 2, 4)
    assert ei.value.code == -1


@pytest.mark.parametrize("cfg,n,S", [(1, 32, 2), (2, 24, 4), (2, 24, 0), (3, 3, 8), (4, 1, 16)])
def test_spectral_bound_of_segment_products(cfg, n, S, lib, torch_cuda, impurities, handles):
    """norm_kind 1 with segment_len != 1: d_min prod_j min(||G_j||_F, prod sigma_max(F_i)), equal to the oracle's
    certified estimate to 1e-9, never below the exact spectral-norm bound (SVD of every segment product), never above the Frobenius
    one (up to the prefactor), and >= |trace| per configuration and per start sector."""
    from workloads import make_batch
    # config 3 from seed 3200: configuration 3300 is one of those its N-only basis leaves undetermined in fp64 on either side
    # (reading A8 (ii): the oracle's own trace moves by 100 % under an exact cyclic shift), segment norms included
    _check_bound(lib, torch_cuda, impurities(cfg), handles(cfg), make_batch(cfg, n, start=200 if cfg == 3 else 300), 1, S, f"cfg{cfg}-spectral-S{S}")


# --------------------------------------------------------------------------- generic (non c / c^dag) operators
def test_generic_operator_blocks(lib, torch_cuda, impurities):
    """The ABI takes any block-sparse operator (Bulla / worm operators): two extra symbols with seeded random
    dense blocks that route like c_0 and c^dag_0.  Trace and Frobenius bounds must match the oracle to 1e-9; the spectral
    bound uses sigma_max, which power iteration only approaches from below, so the library must fall back to a rigorous upper
    estimate: it has to dominate the oracle's exact-SVD bound (and the trace) without being pinned to it."""
    import types
    from workloads import Batch, make_batch
    from workloads.rng import Stream
    from oracle import trace_oracle as O
    base = impurities(2)
    rng = Stream(4242)
    A = base.n_symbols
    sym, src, dst, off, data = (list(base.blk_symbol), list(base.blk_src), list(base.blk_dst), list(base.blk_offset),
                                [np.asarray(base.blk_data, dtype=np.float64)])
    pos = len(data[0])
    for b in range(len(base.blk_symbol)):
        if base.blk_symbol[b] in (0, 1):
            m, n = int(base.dims[base.blk_dst[b]]), int(base.dims[base.blk_src[b]])
            blk = np.array([rng.normal() for _ in range(m * n)]) * 0.7
            sym.append(A + int(base.blk_symbol[b])); src.append(int(base.blk_src[b])); dst.append(int(base.blk_dst[b])); off.append(pos)
            data.append(blk); pos += m * n
    imp = types.SimpleNamespace(dims=base.dims, energy=base.energy, n_symbols=A + 2, is_complex=False, n_sectors=base.n_sectors,
                                beta=base.beta, blk_symbol=np.array(sym, np.int32), blk_src=np.array(src, np.int32),
                                blk_dst=np.array(dst, np.int32), blk_offset=np.array(off, np.int64), blk_data=np.concatenate(data))
    good = make_batch(2, 24, start=18000)
    cfgs = []
    for b in range(24):
        s, t = good.config(b)
        s = s.copy()
        hit = np.nonzero(s < 2)[0]
        for i in hit[::2]:
            s[i] += A          # every other c_0 / c^dag_0 becomes its generic partner (same routing)
        cfgs.append((s, t))
    batch = Batch.from_lists(base.beta, cfgs)
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        for path in (lib.CTQMC_PATH_AUTO, lib.CTQMC_PATH_PANEL, lib.CTQMC_PATH_GROUPED, lib.CTQMC_PATH_LARGE):
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, path)
            _check_trace(lib, torch_cuda, imp, h, batch, f"generic-path{path}")
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)
        for S in (1, 4, 0):
            _check_bound(lib, torch_cuda, imp, h, batch, 0, S, f"generic-frobenius-S{S}")
        offd, symd, taud = _dev(torch_cuda, batch)
        bm, be, _, _, st = lib.ctqmc_bound_batch(h, batch.beta, offd, symd, taud, 1, 1)
        mant, exp2, _, _ = lib.ctqmc_trace_batch(h, batch.beta, offd, symd, taud)
        torch_cuda.cuda.synchronize()
        looser = 0
        for b in range(24):
            s, t = batch.config(b)
            r = O.bound_config(imp, batch.beta, s, t, 1, 1)
            assert scaled_ge(bm[b].item() * (1 + 1e-12), int(be[b].item()), r["mant"], r["exp2"]), f"config {b}: spectral bound below the exact one"
            assert scaled_ge(bm[b].item(), int(be[b].item()), abs(complex(mant[b, 0].item(), mant[b, 1].item())), int(exp2[b].item()))
            looser += rel_diff(bm[b].item(), int(be[b].item()), r["mant"], r["exp2"]) > 1e-9
        print(f"generic operators: spectral bound looser than exact SVD on {looser} of 24 configurations (upper estimate in use)")
    finally:
        h.free()


# --------------------------------------------------------------------------- dynamic range inside a sector
def test_coarse_sectors_do_not_underflow(lib, torch_cuda):
    """Same inputs as the oracle pin test_P5_coarse_sectors_do_not_underflow: Delta (E_n - Emin) up to 4235 inside a
    sector.  exp() of that underflows; the (mant, exp2) result must not."""
    import numpy as np
    from workloads import Batch
    from workloads import impurity as wi
    n, beta = 3, 60.0
    eps = np.array([-2.0, 31.0, 75.0])
    Umat = np.array([[0, 3.0, 1.0], [3.0, 0, 2.0], [1.0, 2.0, 0]])
    u = np.zeros((n,) * 4)
    for a in range(n):
        for b_ in range(n):
            if a != b_:
                u[a, b_, b_, a] = Umat[a, b_]
    imp = wi.build_impurity("ising-coarse", np.diag(eps), u, [(1,)] * n, beta=beta)
    batch = Batch.from_lists(beta, [([5, 3, 2, 4], [1.0, 7.0, 19.5, 41.0]), ([5, 4], [3.0, 58.0]),
                                    ([3, 5, 4, 2, 1, 0], [2.0, 2.5, 30.0, 44.0, 50.0, 59.0])])
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        for sched in (lib.CTQMC_SCHEDULE_THIN, lib.CTQMC_SCHEDULE_LITERAL):
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_SCHEDULE, sched)
            _check_trace(lib, torch_cuda, imp, h, batch, "ising-coarse")
        for nk, S in ((0, 1), (1, 1), (0, 0), (0, 2), (1, 2)):
            _check_bound(lib, torch_cuda, imp, h, batch, nk, S, f"ising-coarse-nk{nk}-S{S}")
    finally:
        h.free()


# --------------------------------------------------------------------------- asynchrony contract and the scratch arena
def _spin(torch, stream, ms):
    """Occupy `stream` for about `ms` milliseconds (torch's spin kernel; 1.9 GHz SM clock)."""
    with torch.cuda.stream(stream):
        torch.cuda._sleep(int(ms * 1.9e6))


@pytest.mark.parametrize("cfg,n", [(2, 256), (3, 16), (3, 72), (4, 4), (4, 64)])
def test_batch_calls_only_enqueue(cfg, n, lib, torch_cuda, impurities, handles):
    """SURVEY 8(b) / PAPER.md:574 ("only asynchronous CUDA functions"): with the arena in place, ctqmc_trace_batch and
    ctqmc_bound_batch return while the stream is still busy with work enqueued BEFORE them -- small, panel, grouped (72 / 64
    configurations) and, forced, large-sector paths; the results are those of a quiet stream."""
    import time
    from workloads import make_batch
    torch = torch_cuda
    h = handles(cfg)
    batch = make_batch(cfg, n, start=21000)
    off, sym, tau = _dev(torch, batch)
    L = int(np.diff(batch.offset).max())
    paths = [lib.CTQMC_PATH_AUTO] + ([lib.CTQMC_PATH_LARGE] if cfg in (3, 4) and n <= 16 else [])
    st = torch.cuda.Stream()
    for path in paths:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, path)
        try:
            ref = lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=L)        # also brings the arena to size
            refb = lib.ctqmc_bound_batch(h, batch.beta, off, sym, tau, 0, 4, max_len=L)
            torch.cuda.synchronize()
            for which in ("trace", "bound"):
                done = torch.cuda.Event()
                _spin(torch, st, 400.0)
                t0 = time.perf_counter()
                with torch.cuda.stream(st):
                    if which == "trace":
                        got = lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, stream=st, max_len=L)
                    else:
                        got = lib.ctqmc_bound_batch(h, batch.beta, off, sym, tau, 0, 4, stream=st, max_len=L)
                    done.record(st)
                dt = time.perf_counter() - t0
                busy = not done.query()
                st.synchronize()
                assert busy, f"cfg{cfg} path {path} {which}: the call returned only after the stream had drained ({dt * 1e3:.0f} ms)"
                assert dt < 0.3, f"cfg{cfg} path {path} {which}: the call took {dt * 1e3:.0f} ms of host time behind a 400 ms spin"
                for x, y in zip(ref if which == "trace" else refb, got):
                    assert torch.equal(x, y)
        finally:
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)


@pytest.mark.parametrize("cfg,n,path", [(3, 40, "panel"), (3, 96, "grouped"), (3, 12, "large"), (4, 6, "large")])
def test_fixed_arena_runs_in_rounds_and_reports_oom_before_enqueueing(cfg, n, path, lib, torch_cuda, impurities):
    """CTQMC_OPT_ARENA_BYTES: the arena is allocated once and never grown.  A batch that does not fit is evaluated in rounds
    of configurations with identical results and summed counters; an arena too small for one configuration gives
    CTQMC_ERR_OOM and leaves the outputs untouched."""
    from workloads import make_batch
    torch = torch_cuda
    imp = impurities(cfg)
    batch = make_batch(cfg, n, start=23000)
    off, sym, tau = _dev(torch, batch)
    L = int(np.diff(batch.offset).max())
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, {"panel": lib.CTQMC_PATH_PANEL, "grouped": lib.CTQMC_PATH_GROUPED,
                                                     "large": lib.CTQMC_PATH_LARGE}[path])
        ref = lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=L)
        refb = lib.ctqmc_bound_batch(h, batch.beta, off, sym, tau, 0, 8, max_len=L)
        torch.cuda.synchronize()
        lb_full = lib.ctqmc_last_stats(h)
        lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=L)
        lt_full = lib.ctqmc_last_stats(h)
        full = lt_full["arena_bytes"]          # the larger of the two calls' needs
        assert full > 0 and lt_full["strings"] > 0
        small = max(full // 5, 1 << 16)
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_ARENA_BYTES, small)
        gotb = lib.ctqmc_bound_batch(h, batch.beta, off, sym, tau, 0, 8, max_len=L)
        lb_r = lib.ctqmc_last_stats(h)
        got = lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=L)
        lt_r = lib.ctqmc_last_stats(h)
        torch.cuda.synchronize()
        for x, y in zip(ref + refb, got + gotb):
            assert torch.equal(x, y)
        assert lt_r["arena_bytes"] == small
        assert lt_r["launches"] > lt_full["launches"] or lb_r["launches"] > lb_full["launches"]      # the larger call ran in rounds
        assert (lt_r["strings"], lt_r["alg_flops"]) == (lt_full["strings"], lt_full["alg_flops"])
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_ARENA_BYTES, 4096)
        out = (torch.full((n, 2), -7.0, dtype=torch.float64, device="cuda"), torch.zeros(n, dtype=torch.int64, device="cuda"),
               torch.zeros((n, imp.n_sectors), dtype=torch.uint8, device="cuda"), torch.full((n,), -1, dtype=torch.int32, device="cuda"))
        with pytest.raises(lib.CtqmcError) as ei:
            lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, out=out, max_len=L)
        assert ei.value.code == lib.binding.CTQMC_ERR_OOM
        torch.cuda.synchronize()
        assert (out[0] == -7.0).all().item() and (out[3] == -1).all().item()
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_ARENA_BYTES, 0)     # back to automatic growth
        got = lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=L)
        torch.cuda.synchronize()
        for x, y in zip(ref, got):
            assert torch.equal(x, y)
    finally:
        h.free()


def test_corrupt_offsets_and_understated_max_len_give_status_2(lib, torch_cuda, impurities, handles):
    """A corrupt offset array (negative, beyond n_ops, decreasing) or a configuration longer than the stated max_len must
    give status 2 / NaN for that configuration, never an out-of-bounds read, and leave the neighbours alone -- on the
    single-launch small path and on the routed paths."""
    from workloads import make_batch
    torch = torch_cuda
    for cfg, n, paths in ((2, 12, [0, 1, 4, 2]), (3, 6, [1, 4, 2])):
        h = handles(cfg)
        batch = make_batch(cfg, n, start=24000)
        L = int(np.diff(batch.offset).max())
        off, sym, tau = _dev(torch, batch)
        for path in paths:
            lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, path)
            try:
                good = lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=L)
                torch.cuda.synchronize()
                # (i) configuration 2 starts at a negative offset, configuration 4 ends beyond n_ops
                bad = batch.offset.copy()
                bad[2] = -5
                bad[5] = len(batch.symbol) + 1000
                boff = torch.from_numpy(bad).cuda()
                got = lib.ctqmc_trace_batch(h, batch.beta, boff, sym, tau, max_len=L)
                torch.cuda.synchronize()
                st = got[3].cpu().numpy()
                for b in range(n):
                    if b in (1, 2, 4, 5):      # each corrupt offset spoils the configuration before and after it
                        assert st[b] == 2 and torch.isnan(got[0][b]).all(), (cfg, path, b, st)
                    else:
                        assert st[b] == good[3][b].item() and torch.equal(got[0][b], good[0][b]) and got[1][b] == good[1][b]
                # (ii) max_len understated: longer configurations are invalid, the others unchanged
                lens = np.diff(batch.offset)
                cut = int(np.sort(lens)[n // 2])
                got = lib.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=cut)
                torch.cuda.synchronize()
                for b in range(n):
                    if lens[b] > cut:
                        assert got[3][b].item() == 2 and torch.isnan(got[0][b]).all()
                    else:
                        assert torch.equal(got[0][b], good[0][b]) and got[1][b] == good[1][b]
                bm = lib.ctqmc_bound_batch(h, batch.beta, boff, sym, tau, 0, 1, max_len=L)
                torch.cuda.synchronize()
                assert bm[4][2].item() == 2 and bm[4][0].item() == 0
            finally:
                lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_AUTO)


def test_spectral_bound_with_near_degenerate_singular_values(lib, torch_cuda):
    """sigma_max comes from a power iteration, which converges from below and stalls when the two largest singular values
    are 1 and 1 - 1e-9: the library must then fall back to its rigorous upper estimate, so that the spectral S = 1 bound still
    dominates the exact one (oracle: SVD) and the trace."""
    import types
    from oracle import trace_oracle as O
    from workloads import Batch
    from workloads.rng import Stream
    rng = Stream(515)
    d = 6

    def orth():
        m = np.array([[rng.normal() for _ in range(d)] for _ in range(d)])
        return np.linalg.qr(m)[0]

    sv = np.array([1.0, 1.0 - 1e-9, 0.7, 0.4, 0.2, 0.1])
    blocks = [orth() @ np.diag(sv) @ orth().T, orth() @ np.diag(sv[::-1].copy()) @ orth().T]
    data = np.concatenate([b.reshape(-1, order="F") for b in blocks])
    imp = types.SimpleNamespace(dims=np.array([d, d], np.int32), energy=np.array([0.1 * i for i in range(2 * d)]), n_symbols=2,
                                is_complex=False, n_sectors=2, beta=2.0, blk_symbol=np.array([0, 1], np.int32),
                                blk_src=np.array([0, 1], np.int32), blk_dst=np.array([1, 0], np.int32),
                                blk_offset=np.array([0, d * d], np.int64), blk_data=data)
    batch = Batch.from_lists(2.0, [([0, 1], [0.3, 1.1]), ([0, 1, 0, 1], [0.1, 0.5, 0.9, 1.7]), ([1, 0], [0.2, 0.4])])
    h = lib.ctqmc_load_impurity(imp, 0)
    try:
        off, sym, tau = _dev(torch_cuda, batch)
        bm, be, sm, se, st = lib.ctqmc_bound_batch(h, 2.0, off, sym, tau, 1, 1)
        mant, exp2, _, _ = lib.ctqmc_trace_batch(h, 2.0, off, sym, tau)
        torch_cuda.cuda.synchronize()
        for b in range(batch.n_configs):
            s, t = batch.config(b)
            r = O.bound_config(imp, 2.0, s, t, 1, 1)
            assert scaled_ge(bm[b].item() * (1 + 1e-12), int(be[b].item()), r["mant"], r["exp2"]), f"config {b}: spectral bound below the exact one"
            assert scaled_ge(bm[b].item(), int(be[b].item()), abs(complex(mant[b, 0].item(), mant[b, 1].item())), int(exp2[b].item()))
        _check_trace(lib, torch_cuda, imp, h, batch, "near-degenerate")
    finally:
        h.free()


def test_odd_sector_dimension_with_a_dirty_arena_and_large_exponents(lib, torch_cuda):
    """Grouped real kernel, odd sector dimensions: its 16-byte loads read one row beyond an odd-dimensional column.  With
    Delta (E - Emin) > 800 on every populated row that row is scaled by 2^(+large); whatever an earlier call left in the arena
    there must not reach the result (stale * 2^k -> inf, inf * 0 -> NaN).  A first call with 7-dimensional sectors
    dirties the arena, the second runs 5- and 3-dimensional ones over the same memory."""
    import types
    from workloads import Batch
    from workloads.rng import Stream
    rng = Stream(9091)
    torch = torch_cuda

    def make(d0, d1, spread):
        blocks = [(0, 0, 1), (1, 1, 0), (2, 0, 0)]
        dims = (d0, d1)
        data, off, pos = [], [], 0
        for _, s_, d_ in blocks:
            m, n = dims[d_], dims[s_]
            data.append(np.array([rng.normal() for _ in range(m * n)]) * (0.9 / np.sqrt(max(m, n))))
            off.append(pos); pos += m * n
        energy = np.concatenate([[0.0] + [spread * (1.0 + 0.01 * i) for i in range(1, d0)], [0.0] + [spread * (1.0 + 0.013 * i) for i in range(1, d1)]])
        return types.SimpleNamespace(dims=np.array(dims, np.int32), energy=energy, n_symbols=3, is_complex=False, n_sectors=2, name="odd",
                                     blk_symbol=np.array([b[0] for b in blocks], np.int32), blk_src=np.array([b[1] for b in blocks], np.int32),
                                     blk_dst=np.array([b[2] for b in blocks], np.int32), blk_offset=np.array(off, np.int64),
                                     blk_data=np.concatenate(data))

    beta = 10.0

    def walks(count):
        cfgs = []
        for _ in range(count):
            q, syms = 0, []
            for _ in range(4 + rng.integer(12)):
                a = (rng.integer(2) * 2) if q == 0 else 1
                syms.append(a)
                q = 1 if a == 0 else 0
            if q == 1:
                syms.append(1)
            cfgs.append((syms, np.sort(beta * rng.uniforms(len(syms)))))
        return Batch.from_lists(beta, cfgs)

    big = make(7, 7, 0.3)
    h = lib.ctqmc_load_impurity(big, 0)
    try:
        lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, lib.CTQMC_PATH_GROUPED)
        _check_trace(lib, torch, big, h, walks(70), "odd-dirty-7")
    finally:
        h.free()
    for dims in ((5, 3), (3, 5), (7, 1)):
        imp = make(dims[0], dims[1], 900.0)          # Delta (E - Emin) ~ 900 per time unit on every row but the lowest
        h = lib.ctqmc_load_impurity(imp, 0)
        try:
            for path in (lib.CTQMC_PATH_GROUPED, lib.CTQMC_PATH_LARGE, lib.CTQMC_PATH_PANEL):
                lib.ctqmc_set_option(h, lib.CTQMC_OPT_PATH, path)
                _check_trace(lib, torch, imp, h, walks(70), f"odd-{dims}-path{path}")
        finally:
            h.free()
