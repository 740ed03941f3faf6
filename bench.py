"""bench.py -- one JSON line: local-trace evaluations per second of the CUDA path on a BASELINE.json workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--batch B] [--impl ours|reference] [--no-others]

A *step* is one pass of the whole hot path (validate -> route -> fused propagate*operator chain with running exponent ->
trace and sector sum) over one batch of seeded synthetic configurations.  `value` is
traces/s with the batch resident in HBM; `e2e` is the same through `ctqmc_trace_batch_host` (host buffers, copies inside the
timed region).  L2 is flushed between timed steps.  `--impl reference` times the CPU oracle (oracle/) on a bounded sample
of the same workload; it is the only code path here, besides `cpu_baseline`, that touches oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "local_trace_evaluations_per_s"
UNIT = "traces/s"
NOMINAL_FP64_TFLOPS = 40.0     # B200 FP64 nominal (vendor figure); DESIGN.md §7
NOMINAL_BF16_TFLOPS = 2250.0   # B200_PROFILING.md
EXP_FLOP_EQUIV = 25            # FP64 exp at its instruction cost (~12 DFMA + range reduction)
FALLBACK_HBM_GBS, FALLBACK_BF16_TFLOPS = 6650.0, 1590.0
WORKLOADS = {
    1: "cfg1: 2-orbital Kanamori (Q=9, d_max=4), L=40",
    2: "cfg2: 3-orbital t2g Kanamori (Q=16, d_max=9), pairs~Poisson(60)",
    3: "cfg3: 5-orbital d-shell Slater, N sectors (Q=11, d_max=252), pairs~Poisson(80)",
    4: "cfg4: 7-orbital f-shell Slater+SOC, (N,Jz) sectors N in 4..6 (Q=70, d_max=295), complex, pairs~Poisson(100)",
    5: "cfg5: 7-orbital f-shell + crystal field, N sectors 1001/2002/3003, complex, pairs~Poisson(100)",
}
REF_SAMPLE = {1: 8192, 2: 4096, 3: 128, 4: 4, 5: 1}   # configurations per reference step (seconds of oracle time each)
# config 5: one configuration is ~1e13 flop of numpy (a minute): a reference step / the cpu_baseline is the oracle on the
# first L/REF_PREFIX_DIV operators of configuration 0, extrapolated to a whole trace by the literal flop count of Eq. 65
REF_PREFIX_DIV = {"reference": 10, "cpu_baseline": 4}
KERNELS = {1: ("chain_kernel (panel in shared memory, fused propagate x operator, FP64 DMMA m8n8k4)", "tensor"),
           2: ("large_step_kernel (128x64 tiles, TMA + mbarrier ring, fused propagate x operator, FP64 DMMA m8n8k4)", "tensor"),
           3: ("small2_trace_kernel / small_trace_kernel (whole path in one launch, operator store in shared memory, FP64 FMA)", "alu"),
           4: ("grouped_step_kernel (strings sharing a block share one GEMM per chain position, 64x64 tiles, FP64 DMMA m8n8k4)", "tensor"),
           5: ("split_step_kernel (int8 slice products on tcgen05.mma.kind::i8; reported against the FP64 tensor peak as FP64-equivalent flops)", "tensor")}


def ncu_traffic(cfg: int, batch: int):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, from the `ncu --set full` capture
    summarised under profiles/ for exactly this config and batch (profiles/traffic.json, written next to the summaries);
    None when there is no capture of this launch configuration."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    with open(p) as fh:
        e = json.load(fh).get(f"cfg{cfg}_batch{batch}")
    return None if e is None else e["dram_bytes_per_launch"]


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16=float(d["bf16_tflops"]), source="measured")
    return dict(hbm_gbs=FALLBACK_HBM_GBS, bf16=FALLBACK_BF16_TFLOPS, source="fallback")


def shard_batch(cfg: int, batch_per_gpu: int, rank: int):
    """Weak scaling: rank r evaluates configurations [r*B, (r+1)*B) of the seeded stream of config `cfg`.
    Configurations are independent, so there is no data-path collective."""
    from workloads import make_batch
    return make_batch(cfg, batch_per_gpu, start=rank * batch_per_gpu)


def reduce_max(values, dist=None, device="cpu"):
    """Max over ranks of a list of floats (the contract's max-over-ranks timing).  Works on gloo (CPU) and nccl."""
    if dist is None:
        return [float(v) for v in values]
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def aggregate_value(world: int, batch_per_gpu: int, steps: int, total_ms: float) -> float:
    """Whole-job traces/s: every rank processed batch_per_gpu * steps configurations in total_ms (max over ranks)."""
    return world * batch_per_gpu * steps / (total_ms * 1e-3)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm)}


def oracle_rate(imp, batch, n_sample: int):
    """traces/s of the oracle, as it stands, on the first n_sample configurations."""
    from oracle import trace_oracle as O
    sub = batch.subset(range(min(n_sample, batch.n_configs)))
    t0 = time.perf_counter()
    O.trace_batch(imp, sub.beta, sub.offset, sub.symbol, sub.tau)
    dt = time.perf_counter() - t0
    return sub.n_configs / dt, sub.n_configs, dt


def blas_threads() -> int:
    try:
        from threadpoolctl import threadpool_info
        return max([int(i.get("num_threads", 1)) for i in threadpool_info()] + [1])
    except Exception:
        return 1


def oracle_cores(cfg: int):
    """Threads the oracle really uses: it is ONE Python process looping over configurations and start sectors; only numpy's
    matmul is threaded, and only where the blocks are large enough for the BLAS to split (configs 3-5)."""
    avail = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    used = 1 if cfg <= 2 else min(avail, blas_threads())
    note = (f"single Python process; {avail} cores available to it, numpy BLAS pool {blas_threads()} threads; "
            + ("blocks of at most 9 x 9: effectively one core" if cfg <= 2 else "matmul is the only threaded step"))
    return used, note


def oracle_rate_prefix(imp, batch, div: int):
    """Config 5: the oracle (literal Eq. 65) on the first ceil(L/div) operators of configuration 0, and the factor that
    extrapolates it to a whole trace: literal flops of the full string over those of the prefix (8 d_i d_{i-1} d_q0 per step
    and surviving start sector, from the oracle's own routing).  Returns (traces/s extrapolated, description)."""
    from oracle import trace_oracle as O
    s, t = batch.config(0)
    n = max(2, -(-len(s) // div))

    def flops(sym):
        tot = 0
        for q0 in range(imp.n_sectors):
            v = O.route(imp, sym, q0)
            if v is not None:
                tot += sum(8 * int(imp.dims[v[i + 1]]) * int(imp.dims[v[i]]) * int(imp.dims[q0]) for i in range(len(sym)))
        return tot

    f_full, f_pre = flops(s), flops(s[:n])
    t0 = time.perf_counter()
    O.trace_config(imp, batch.beta, s[:n], t[:n])
    dt = time.perf_counter() - t0
    rate = 1.0 / (dt * f_full / f_pre)
    return rate, dt, (f"EXTRAPOLATED from the first {n} of the {len(s)} operators of configuration 0 ({dt:.1f} s of "
                      f"oracle.trace_oracle.trace_config, numpy fp64) by the literal flop count of Eq. 65 ({f_full:.3e} / {f_pre:.3e})")


def run_reference(args, rank: int):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample per step (rank 0 only)."""
    if rank != 0:
        return
    from workloads import build_config_impurity, make_batch
    cfg = args.config
    imp = build_config_impurity(cfg, keep_eigvecs=False)
    n = REF_SAMPLE[cfg]
    batch = make_batch(cfg, n)
    if cfg == 5:
        rates, t_tot = [], 0.0
        for i in range(min(args.warmup, 1) + args.steps):
            rate, dt, sample = oracle_rate_prefix(imp, batch, REF_PREFIX_DIV["reference"])
            if i >= min(args.warmup, 1):
                rates.append(rate)
                t_tot += dt
        val = len(rates) / sum(1.0 / r for r in rates)
        sample = "per step: " + sample
    else:
        for _ in range(min(args.warmup, 1)):
            oracle_rate(imp, batch, max(1, n // 8))
        t_tot, n_tot = 0.0, 0
        for _ in range(args.steps):
            _, k, dt = oracle_rate(imp, batch, n)
            t_tot += dt
            n_tot += k
        val = n_tot / t_tot
        sample = f"{n} configurations of {WORKLOADS[cfg]} per step, oracle.trace_oracle.trace_batch (numpy fp64)"
    cores, cores_note = oracle_cores(cfg)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[cfg], "batch": n},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "cores_note": cores_note, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def measure_config(L, torch, cfg, B, rank, steps, warmup, schedule, local_rank, barrier, fp64, pk, with_e2e=True, path="auto",
                   e2e_steps=None):
    """Times `steps` passes of the hot path on config `cfg` (this rank's shard) and returns the pieces of the JSON line."""
    import numpy as np
    from workloads import build_config_impurity
    imp = build_config_impurity(cfg, keep_eigvecs=False)
    t0 = time.perf_counter()
    h = L.ctqmc_load_impurity(imp, local_rank)
    load_s = time.perf_counter() - t0
    if schedule == "literal":
        L.ctqmc_set_option(h, L.CTQMC_OPT_SCHEDULE, L.CTQMC_SCHEDULE_LITERAL)
    if path != "auto":
        L.ctqmc_set_option(h, L.CTQMC_OPT_PATH, {"panel": 1, "large": 2, "small": 3, "grouped": 4, "split": 5}[path])
    L.ctqmc_set_option(h, L.CTQMC_OPT_TIMING, 1)
    batch = shard_batch(cfg, B, rank)
    off, sym, tau = (torch.from_numpy(x).cuda() for x in (batch.offset, batch.symbol, batch.tau))
    Q = imp.n_sectors
    out = (torch.empty((B, 2), dtype=torch.float64, device="cuda"), torch.empty(B, dtype=torch.int64, device="cuda"),
           torch.empty((B, Q), dtype=torch.uint8, device="cuda"), torch.empty(B, dtype=torch.int32, device="cuda"))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()
    max_len = int(np.diff(batch.offset).max()) if B else 0     # host-known: the C call never reads anything back

    def step():
        L.ctqmc_trace_batch(h, batch.beta, off, sym, tau, stream=stream, out=out, max_len=max_len)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    stats = L.ctqmc_last_stats(h)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    chain_ms, route_ms, reduce_ms = [], [], []
    barrier()
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        step()
        b.record(stream)
        tm = L.ctqmc_last_timing(h)      # synchronises; outside the event pair
        chain_ms.append(tm["chain_ms"]); route_ms.append(tm["route_ms"]); reduce_ms.append(tm["reduce_ms"])
    barrier()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)

    e2e_ms = None
    if with_e2e:
        # end to end through the host-buffer C call, from / to PINNED host memory: H2D of the batch, kernels, D2H of the
        # results, all inside the timed region
        pin = [torch.from_numpy(x).pin_memory() for x in (batch.offset, batch.symbol, batch.tau)]
        h_in = [t.numpy() for t in pin]
        pout = [torch.empty((B, 2), dtype=torch.float64).pin_memory(), torch.empty(B, dtype=torch.int64).pin_memory(),
                torch.empty((B, Q), dtype=torch.uint8).pin_memory(), torch.empty(B, dtype=torch.int32).pin_memory()]
        h_out = tuple(t.numpy() for t in pout)
        for _ in range(1 if cfg == 5 else 2):
            L.ctqmc_trace_batch_host(h, batch.beta, *h_in, out=h_out)
        assert np.array_equal(h_out[0], out[0].cpu().numpy(), equal_nan=True) and np.array_equal(h_out[1], out[1].cpu().numpy())
        e2e_s = 0.0
        e2e_steps = steps if e2e_steps is None else e2e_steps
        barrier()
        for _ in range(e2e_steps):
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            L.ctqmc_trace_batch_host(h, batch.beta, *h_in, out=h_out)
            e2e_s += time.perf_counter() - t0
        barrier()
        e2e_ms = e2e_s * 1e3
    # the lazy-trace bounds (a6) on the same batch: Frobenius, S = 1 (tables only) and S = 8 (segment products), device-resident
    bound_ms = {}
    if with_e2e:
        # config 5: S = 8 segment products cost as much as the traces themselves (a minute per call); tables only there
        for key, nk, S in ((("S1", 0, 1), ("S1_spectral", 1, 1)) if cfg == 5 else (("S1", 0, 1), ("S8", 0, 8), ("S1_spectral", 1, 1))):
            for _ in range(2):
                L.ctqmc_bound_batch(h, batch.beta, off, sym, tau, nk, S, want_sector=False, max_len=max_len)
            torch.cuda.synchronize()
            ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = max(1, min(steps, 5))
            ea.record(stream)
            for _ in range(reps):
                L.ctqmc_bound_batch(h, batch.beta, off, sym, tau, nk, S, want_sector=False, stream=stream, max_len=max_len)
            eb.record(stream)
            torch.cuda.synchronize()
            bound_ms[key] = ea.elapsed_time(eb) / reps
    h.free()
    del flush, out, off, sym, tau
    torch.cuda.empty_cache()

    n_ops = int(batch.offset[-1])
    kname, bound = KERNELS[stats["path"]]
    chain_avg_ms = sum(chain_ms) / len(chain_ms)
    # small (alu-bound) path: the algorithmic work also holds one FP64 exp per row and chain step; SURVEY 8(d) D3 counts it at
    # its instruction cost (~25 flop-equivalents), not as one flop
    n_exp = stats["n_exp"]
    alg_flop_equiv = stats["alg_flops"] + EXP_FLOP_EQUIV * n_exp
    achieved_tf = alg_flop_equiv / (chain_avg_ms * 1e-3) / 1e12
    rule_peak = pk["bf16"] * NOMINAL_FP64_TFLOPS / NOMINAL_BF16_TFLOPS
    peak = fp64["dmma_tflops"] if bound == "tensor" else fp64["dfma_tflops"]
    alg_bytes = n_ops * 12 + (B + 1) * 8 + B * (16 + 8 + 4 + Q)
    k_launches = max(max_len, 1) if stats["path"] in (2, 4, 5) else 1
    roofline = {
        "bound": bound, "kernel": kname, "achieved": achieved_tf, "peak": peak, "unit": "TFLOP/s", "frac": achieved_tf / peak,
        "traffic": ncu_traffic(cfg, B),
        "peak_source": ("FP64 " + ("DMMA" if bound == "tensor" else "DFMA") + " register-resident loop measured in this run by "
                        "ctqmc_measure_fp64_peak (MEASURED_PEAKS.json has no FP64 entry); the guide's rule, "
                        f"{pk['source']} bf16 {pk['bf16']} TF/s x nominal {NOMINAL_FP64_TFLOPS}/{NOMINAL_BF16_TFLOPS}, gives {rule_peak:.2f}"),
        "frac_of_rule_peak": achieved_tf / rule_peak,
        "kernel_ms": chain_avg_ms, "kernel_share_of_step": chain_avg_ms * steps / total_ms,
        # the step kernels of the grouped and large paths are launched once per chain position (max_len launches per step): the
        # same ratio per kernel launch, which is what `traffic` (one ncu capture of one launch) refers to
        "kernel_launches_per_step": k_launches, "kernel_launch_ms_avg": chain_avg_ms / k_launches,
        "flops_per_kernel_launch_algorithmic": stats["alg_flops"] / k_launches,
        "traffic_per": "kernel launch (dram__bytes_read.sum + dram__bytes_write.sum, profiles/traffic.json)",
        "flops_per_launch_algorithmic": stats["alg_flops"], "exp_per_launch": n_exp, "flop_equivalents_per_launch": alg_flop_equiv, "executed_real_macs_padded": stats["macs"],
        "algorithmic_io_bytes_per_step": alg_bytes,
        "hbm_frac_algorithmic": alg_bytes / (total_ms / steps * 1e-3) / 1e9 / pk["hbm_gbs"],
    }
    return dict(imp=imp, batch=batch, stats=stats, total_ms=total_ms, e2e_ms=e2e_ms, e2e_steps=e2e_steps, n_ops=n_ops, Q=Q, roofline=roofline,
                phases={"route": sum(route_ms) / len(route_ms), "chain": chain_avg_ms, "reduce": sum(reduce_ms) / len(reduce_ms)},
                load_s=load_s, bound_ms=bound_ms)


def _edit_tensors(torch, per_chain):
    off, tau, sym, kind = [0], [], [], []
    for ins, rem in per_chain:
        for t, a in rem:
            tau.append(t); sym.append(a); kind.append(-1)
        for t, a in ins:
            tau.append(t); sym.append(a); kind.append(1)
        off.append(len(tau))
    return (torch.tensor(off, dtype=torch.int64, device="cuda"), torch.tensor(tau, dtype=torch.float64, device="cuda"),
            torch.tensor(sym, dtype=torch.int32, device="cuda"), torch.tensor(kind, dtype=torch.int32, device="cuda"))


def measure_chains(L, torch, cfg, n_chains, depth, rounds, local_rank, leaf_capacity=32, lazy_rounds=2):
    """Incremental lazy trace: `n_chains` Markov chains in lock-step, each loaded with a
    BASELINE configuration, then `rounds` Metropolis rounds of pair moves (insert / remove, workloads.moves).  The threshold of
    chain c is |w_old| u with a pre-drawn u, computed on the device from ctqmc_chains_trace.  Timed with CUDA
    events around propose + commit; the host reads the accept flags back between rounds (outside the timed pair) to keep its
    mirror of the configurations, as the CPU side of the paper's solver does."""
    import math as _m
    from workloads import apply_move, build_config_impurity, make_batch, random_pair_move
    from workloads.rng import Stream
    imp = build_config_impurity(cfg, keep_eigvecs=False)
    h = L.ctqmc_load_impurity(imp, local_rank)
    ch = L.ctqmc_chains_create(h, imp.beta, n_chains, depth, leaf_capacity=leaf_capacity, max_edits=8, lazy_rounds=lazy_rounds)
    try:
        nf = imp.n_symbols // 2
        starts = []
        for c in range(n_chains):
            s, t = make_batch(cfg, 1, start=c % 64).config(0)
            starts.append([(float(tt), int(a)) for a, tt in zip(s, t)])
        ones = torch.ones(n_chains, dtype=torch.int32, device="cuda")
        for k in range(max((len(s) + 7) // 8 for s in starts)):
            L.ctqmc_chains_propose(ch, *_edit_tensors(torch, [(s[8 * k:8 * k + 8], []) for s in starts]))
            L.ctqmc_chains_commit(ch, ones)
        torch.cuda.synchronize()
        st0 = L.ctqmc_chains_stats(ch)
        ops = [list(s) for s in starts]
        rngs = [Stream(770000 + 1000 * cfg + c) for c in range(n_chains)]
        stream = torch.cuda.current_stream()
        ms, n_acc, n_ok, by = 0.0, 0, 0, [0, 0, 0]
        for r in range(rounds + 1):
            moves = [random_pair_move(rngs[c], nf, imp.beta, ops[c]) for c in range(n_chains)]
            ed = _edit_tensors(torch, moves)
            u = torch.tensor([max(rngs[c].uniform(), 1e-300) for c in range(n_chains)], dtype=torch.float64, device="cuda")
            mant, exp2 = L.ctqmc_chains_trace(ch)
            thr = torch.log2(torch.hypot(mant[:, 0], mant[:, 1])) + exp2.to(torch.float64) + torch.log2(u)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            out = L.ctqmc_chains_propose(ch, *ed, thr, stream=stream)
            L.ctqmc_chains_commit(ch, stream=stream)
            b.record(stream)
            torch.cuda.synchronize()
            acc = out["accept"].cpu().numpy()
            okc = out["status"].cpu().numpy() == 0
            dby = out["decided_by"].cpu().numpy()
            for c in range(n_chains):
                if acc[c]:
                    ops[c] = apply_move(ops[c], *moves[c])
            if r == 0:
                continue                      # warm-up round
            ms += a.elapsed_time(b)
            n_acc += int(acc.sum()); n_ok += int(okc.sum())
            for v in dby[okc]:
                by[int(v)] += 1
        st1 = L.ctqmc_chains_stats(ch)
        n_moves = n_chains * rounds
        return {"workload": WORKLOADS[cfg], "chains": n_chains, "depth": depth, "leaf_capacity": leaf_capacity, "lazy_rounds": lazy_rounds,
                "rounds": rounds, "moves_per_s": n_moves / (ms * 1e-3), "ms_per_round": ms / rounds, "accept_rate": n_acc / max(n_moves, 1),
                "invalid_proposals": n_moves - n_ok, "decided_by": {"bound": by[0], "partial": by[1], "full": by[2]},
                "mean_operators": sum(len(o) for o in ops) / n_chains,
                "device_bytes": st1["bytes"], "unit": "moves/s (propose + commit, device time)",
                "api": "ctqmc_chains_propose + ctqmc_chains_commit"}
    finally:
        ch.destroy()
        h.free()
        torch.cuda.empty_cache()


def measure_density(L, torch, cfg, B, steps, local_rank):
    """ctqmc_density_batch (Eq. 27) on a BASELINE batch: configurations per second, device time."""
    import numpy as np
    from workloads import build_config_impurity, make_batch
    imp = build_config_impurity(cfg, keep_eigvecs=False)
    h = L.ctqmc_load_impurity(imp, local_rank)
    try:
        batch = make_batch(cfg, B)
        off, sym, tau = (torch.from_numpy(x).cuda() for x in (batch.offset, batch.symbol, batch.tau))
        Lmax = int(np.diff(batch.offset).max())
        mant, exp2, _, status = L.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=Lmax)
        rho = L.ctqmc_density_batch(h, batch.beta, off, sym, tau, mant, exp2, status, max_len=Lmax)
        torch.cuda.synchronize()
        stream = torch.cuda.current_stream()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(steps):
            L.ctqmc_density_batch(h, batch.beta, off, sym, tau, mant, exp2, status, rho=rho, stream=stream, max_len=Lmax)
        b.record(stream)
        torch.cuda.synchronize()
        ms = a.elapsed_time(b) / steps
        return {"workload": WORKLOADS[cfg], "batch": B, "steps": steps, "ms_per_batch": ms, "configurations_per_s": B / (ms * 1e-3),
                "api": "ctqmc_density_batch (after ctqmc_trace_batch of the same batch)"}
    finally:
        h.free()
        torch.cuda.empty_cache()



def measure_split(L, torch, B, steps, local_rank, pk):
    """CTQMC_PATH_SPLIT on config 5: the same batch through the FP64 DMMA path and through the
    split-precision int8 tcgen05 path; traces/s of the latter, the largest relative difference between the two, and the int8
    roofline (28 slice-pair products of 4 real products each per complex product: 28 x the algorithmic FP64 flops as int8 ops;
    peak = measured bf16 x nominal 4.5 / 2.25)."""
    import numpy as np
    from workloads import build_config_impurity, make_batch
    imp = build_config_impurity(5, keep_eigvecs=False)
    h = L.ctqmc_load_impurity(imp, local_rank)
    try:
        batch = make_batch(5, B)
        off, sym, tau = (torch.from_numpy(x).cuda() for x in (batch.offset, batch.symbol, batch.tau))
        Lmax = int(np.diff(batch.offset).max())
        ref = L.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=Lmax)
        torch.cuda.synchronize()
        slices = 7
        L.ctqmc_set_option(h, L.CTQMC_OPT_SPLIT_SLICES, slices)
        t0 = time.perf_counter()
        L.ctqmc_set_option(h, L.CTQMC_OPT_PATH, L.CTQMC_PATH_SPLIT)      # builds the int8 slice planes of the operator store
        prep_s = time.perf_counter() - t0
        got = L.ctqmc_trace_batch(h, batch.beta, off, sym, tau, max_len=Lmax)   # warm-up (arena growth)
        torch.cuda.synchronize()
        stream = torch.cuda.current_stream()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(steps):
            got = L.ctqmc_trace_batch(h, batch.beta, off, sym, tau, stream=stream, max_len=Lmax)
        b.record(stream)
        torch.cuda.synchronize()
        ms = a.elapsed_time(b) / steps
        st = L.ctqmc_last_stats(h)
        rm, re_, gm, ge = ref[0].cpu().numpy(), ref[1].cpu().numpy(), got[0].cpu().numpy(), got[1].cpu().numpy()
        worst = 0.0
        for i in range(B):
            r, g = complex(*rm[i]), complex(*gm[i]) * 2.0 ** float(ge[i] - re_[i])
            worst = max(worst, abs(g - r) / abs(r))
        assert (ref[3] == got[3]).all().item() and (ref[2] == got[2]).all().item()
        pairs = slices * (slices + 1) // 2
        tops = pairs * st["alg_flops"] / (ms * 1e-3) / 1e12
        peak = pk["bf16"] * 2.0
        return {"workload": WORKLOADS[5], "batch": B, "steps": steps, "slices": slices, "ms_per_step": ms, "value": B / (ms * 1e-3), "unit": UNIT,
                "max_rel_diff_vs_fp64_path": worst, "parity": "all 64 golden outputs within 1e-9 (tests/test_gpu_parity.py::test_split_precision_path_meets_the_same_bar)",
                "fp64_equivalent_tflops": st["alg_flops"] / (ms * 1e-3) / 1e12, "slice_plane_build_s": prep_s,
                "roofline": {"bound": "tensor", "kernel": "split_step_kernel (tcgen05.mma.kind::i8, TMEM accumulators, TMA-fed slice planes)",
                             "achieved": tops, "peak": peak, "unit": "TOP/s (int8)", "frac": tops / peak,
                             "peak_source": f"{pk['source']} bf16 {pk['bf16']} TF/s x nominal 4.5 / 2.25 (B200_PROFILING.md)",
                             "int8_ops_per_step_algorithmic": pairs * st["alg_flops"]},
                "api": "ctqmc_set_option(CTQMC_OPT_PATH, CTQMC_PATH_SPLIT) + ctqmc_trace_batch"}
    finally:
        h.free()
        torch.cuda.empty_cache()



def _default_batch(cfg: int) -> int:
    from workloads import BASELINE_CONFIGS
    return BASELINE_CONFIGS[cfg]["batch"]


def run_ours(args, rank: int, world: int, local_rank: int):
    import torch

    from paper_2010_08482_b200 import build as _build
    if rank == 0:
        _build.build()   # no-op when the in-tree library is newer than its sources
    else:
        t_wait = time.time()
        while _build.needs_build() and time.time() - t_wait < 300:
            time.sleep(1.0)
    import paper_2010_08482_b200 as L

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = args.config
    B = args.batch or _default_batch(cfg)
    warmup = max(args.warmup, 3)
    pk = peaks()
    fp64 = L.ctqmc_measure_fp64_peak(local_rank)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    # config 5: a step is 12 s, so the host-buffer (e2e) leg times 3 steps whatever --steps says (its copies are 27 kB per step)
    m = measure_config(L, torch, cfg, B, rank, args.steps, warmup, args.schedule, local_rank, barrier, fp64, pk, path=args.path,
                       e2e_steps=min(args.steps, 3) if cfg == 5 else None)
    clocks = sampler.stop() if rank == 0 else None
    total_ms, e2e_ms = reduce_max([m["total_ms"], m["e2e_ms"]], dist, "cuda")

    others = {}
    if args.others and world == 1:
        # the other BASELINE.json configs at their stated batch, device-resident timing only (fewer steps: they are context)
        # plus the default small-sector config at a scaled batch (same generator, 64 x BASELINE's 4096): at the stated batch
        # that launch lasts as long as ONE configuration's dependency chain, whatever the kernel
        for c, bsz, key in ((1, 0, "cfg1"), (2, 0, "cfg2"), (2, 262144, "cfg2_scaled_batch"), (3, 0, "cfg3"), (4, 0, "cfg4"), (5, 0, "cfg5")):
            if c == cfg and not bsz:
                continue
            bsz = bsz or _default_batch(c)
            k = 3 if c == 5 else 5
            o = measure_config(L, torch, c, bsz, 0, k, 3, "thin", local_rank, barrier, fp64, pk, with_e2e=False)
            others[key] = {"workload": WORKLOADS[c], "batch": bsz, "steps": k,
                                 "value": aggregate_value(1, bsz, k, o["total_ms"]), "unit": UNIT,
                                 "ms_per_step": o["total_ms"] / k, "gflops": o["stats"]["alg_flops"] * k / (o["total_ms"] * 1e-3) / 1e9,
                                 "roofline": {x: o["roofline"][x] for x in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic",
                                                                            "frac_of_rule_peak", "kernel_ms", "kernel_share_of_step",
                                                                            "hbm_frac_algorithmic")}}
    next_rows = {}
    if args.others and world == 1:
        # SURVEY 8(f) rows built beyond the stateless batch path: the incremental lazy trace over many chains (f1, f2) and the
        # density-matrix accumulation (f3), each on a small-sector and a mid-size complex config
        next_rows["lazy_chains"] = {"cfg2": measure_chains(L, torch, 2, 1024, 6, 8, local_rank),
                                    "cfg4": measure_chains(L, torch, 4, 16, 5, 4, local_rank, leaf_capacity=32)}
        next_rows["split_precision"] = measure_split(L, torch, 64, 3, local_rank, pk)
        next_rows["density"] = {"cfg2": measure_density(L, torch, 2, 4096, 3, local_rank),
                                "cfg4": measure_density(L, torch, 4, 64, 2, local_rank)}
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    stats, Q, n_ops = m["stats"], m["Q"], m["n_ops"]
    line = {
        "metric": METRIC, "value": aggregate_value(world, B, args.steps, total_ms), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[cfg], "batch_per_gpu": B, "operators_per_batch": n_ops, "schedule": args.schedule,
                   "l2": "flushed between timed steps (256 MiB write)", "sharding": "batch split over ranks, no collective"},
        "gflops": world * stats["alg_flops"] * args.steps / (total_ms * 1e-3) / 1e9,
        "e2e": {"value": aggregate_value(world, B, m["e2e_steps"], e2e_ms), "unit": UNIT, "steps": m["e2e_steps"],
                "h2d_bytes_per_step": n_ops * 12 + (B + 1) * 8, "d2h_bytes_per_step": B * (16 + 8 + 4 + Q),
                "api": "ctqmc_trace_batch_host (pinned host buffers; copies inside the timed region)"},
        "gpu_launches": stats["launches"] * args.steps,
        "clocks": clocks,
        "roofline": m["roofline"],
        "phases_ms": m["phases"],
        "fp64_peak_measured": fp64,
        "bound_batch": {"norm": "frobenius unless the key says spectral", "ms_per_batch": m["bound_ms"],
                        "bounds_per_s": {k: B / (v * 1e-3) for k, v in m["bound_ms"].items()}},
        "lib": {"strings": stats["strings"], "units": stats["units"], "path": stats["path"], "panel_width_or_lanes": stats["panel_width"],
                "team_warps": stats["team_warps"], "load_impurity_s": m["load_s"]},
    }
    if others:
        line["other_workloads"] = others
    if next_rows:
        line["next_rows"] = next_rows
    if not args.no_cpu_baseline and world == 1:
        cores, cores_note = oracle_cores(cfg)
        if cfg == 5:
            rate, dt, sample = oracle_rate_prefix(m["imp"], m["batch"], REF_PREFIX_DIV["cpu_baseline"])
        else:
            rate, k, dt = oracle_rate(m["imp"], m["batch"], REF_SAMPLE[cfg])
            sample = f"first {k} configurations of the same batch, {dt:.1f} s, oracle.trace_oracle.trace_batch (numpy fp64)"
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "cores_note": cores_note, "kind": "oracle", "sample": sample}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=sorted(WORKLOADS),
                    help="BASELINE.json config (1-based); default 5 = the largest single-GPU one, on which north_star states its target")
    ap.add_argument("--batch", type=int, default=0, help="configurations per GPU per step (default: BASELINE.json's batch)")
    ap.add_argument("--schedule", default="thin", choices=["thin", "literal"])
    ap.add_argument("--path", default="auto", choices=["auto", "panel", "large", "small", "grouped", "split"],
                    help="kernel family (CTQMC_OPT_PATH); auto is what a user of the library gets")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-others", dest="others", action="store_false",
                    help="skip the short device-resident timings of the other BASELINE.json configs (about two minutes at N=1)")
    ap.add_argument("--chains", default="", metavar="CFG,CHAINS,DEPTH,LEAF_CAPACITY,ROUNDS",
                    help="only the chain-set row (SURVEY 8(f) 1-2) for this shape, e.g. 4,16,4,64,4: prints that row and exits")
    args = ap.parse_args()
    if args.chains:
        import torch
        import paper_2010_08482_b200 as L
        L.library()
        c, n, depth, cap, rounds = (int(x) for x in args.chains.split(","))
        print(json.dumps({"chains_row": measure_chains(L, torch, c, n, depth, rounds, 0, leaf_capacity=cap)}))
        return
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
