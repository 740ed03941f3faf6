"""Seeded CT-HYB configurations (operator strings with times) — SURVEY.md §8(d) D2.

A configuration is a time-ordered list (alpha_1, tau_1) ... (alpha_L, tau_L), 0 <= tau_1 <= ... < beta, index 1 acting
first (rightmost in PAPER.md:519 Eq. 63); alpha = 2*flavour + 1 for c^dag, 2*flavour for c.  Batches are CSR:
`offset[B+1]`, `symbol[sum L]`, `tau[sum L]`.  The paper's workloads are real Markov chains from its own input files
(PAPER.md:636-665), which are not available; these generators reproduce their *shape* (expansion order, flavour mix,
Pauli-consistent alternation, particle-number window) from a seed.  Input generation only: no routing, no traces.

Seed of configuration b of config c is 1000*c + b, so a batch of any size is a prefix of a larger one.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .rng import Stream, uniform_array

# BASELINE.json `configs` (1-based).  "order" is read as operator *pairs* (reading A11): L = 2K.
BASELINE_CONFIGS = {
    1: dict(n_flavours=4, beta=10.0, batch=1024, kind="fixed", pairs_per_flavour=5),
    2: dict(n_flavours=6, beta=50.0, batch=4096, kind="poisson", mean_pairs=60.0),
    3: dict(n_flavours=10, beta=40.0, batch=1024, kind="poisson", mean_pairs=80.0),
    4: dict(n_flavours=14, beta=1.0 / (8.617333262e-5 * 600.0), batch=256, kind="window", mean_pairs=100.0, window=(4, 6)),
    5: dict(n_flavours=14, beta=1.0 / (8.617333262e-5 * 600.0), batch=64, kind="window", mean_pairs=100.0, window=(4, 6)),
}


@dataclass
class Batch:
    beta: float
    offset: np.ndarray  # int64 [B+1]
    symbol: np.ndarray  # int32 [offset[B]]
    tau: np.ndarray     # float64 [offset[B]]

    @property
    def n_configs(self) -> int:
        return len(self.offset) - 1

    def config(self, b: int):
        lo, hi = int(self.offset[b]), int(self.offset[b + 1])
        return self.symbol[lo:hi], self.tau[lo:hi]

    def subset(self, idx) -> "Batch":
        idx = list(idx)
        syms = [self.config(b)[0] for b in idx]
        taus = [self.config(b)[1] for b in idx]
        off = np.concatenate([[0], np.cumsum([len(s) for s in syms])]).astype(np.int64)
        return Batch(self.beta, off,
                     np.concatenate(syms).astype(np.int32) if syms else np.zeros(0, np.int32),
                     np.concatenate(taus).astype(np.float64) if taus else np.zeros(0, np.float64))

    @staticmethod
    def from_lists(beta: float, configs) -> "Batch":
        """configs: iterable of (symbols, taus)."""
        configs = [(np.asarray(s, dtype=np.int32), np.asarray(t, dtype=np.float64)) for s, t in configs]
        off = np.concatenate([[0], np.cumsum([len(s) for s, _ in configs])]).astype(np.int64)
        sym = np.concatenate([s for s, _ in configs]) if configs else np.zeros(0, np.int32)
        tau = np.concatenate([t for _, t in configs]) if configs else np.zeros(0, np.float64)
        return Batch(float(beta), off, sym.astype(np.int32), tau.astype(np.float64))


# --------------------------------------------------------------------------- configs 1-3: uniform placement
def _poisson_cdf(mean: float, kmax: int) -> np.ndarray:
    k = np.arange(kmax + 1)
    logp = -mean + k * np.log(mean) - np.cumsum(np.concatenate([[0.0], np.log(np.arange(1, kmax + 1))]))
    return np.cumsum(np.exp(logp))


def _uniform_alternating(cfg: int, start: int, n: int, n_flavours: int, beta: float,
                         pairs_per_flavour: int | None, mean_pairs: float | None) -> Batch:
    """Per flavour 2 k_f times uniform in [0, beta), sorted, alternating c^dag / c starting with a fair coin;
    all flavours merged by time.  Vectorised over the batch.
    Counter layout per configuration seed: 0 = Poisson draw, 1..nf = first-type coins, then per pair j:
    (flavour, time, time)."""
    seeds = (1000 * cfg + start + np.arange(n)).astype(np.uint64)
    if pairs_per_flavour is not None:
        K = np.full(n, pairs_per_flavour * n_flavours, dtype=np.int64)
    else:
        cdf = _poisson_cdf(mean_pairs, int(mean_pairs * 4 + 50))
        K = np.searchsorted(cdf, uniform_array(seeds, np.uint64(0)), side="left").astype(np.int64)
    coin = (uniform_array(seeds[:, None], np.uint64(1) + np.arange(n_flavours, dtype=np.uint64)[None, :]) < 0.5)
    pair_cfg = np.repeat(np.arange(n), K)
    pair_j = np.arange(int(K.sum())) - np.repeat(np.cumsum(K) - K, K)
    base = (np.uint64(1 + n_flavours) + np.uint64(3) * pair_j.astype(np.uint64))
    ps = seeds[pair_cfg]
    if pairs_per_flavour is not None:
        pair_f = pair_j // pairs_per_flavour
    else:
        pair_f = np.minimum((uniform_array(ps, base) * n_flavours).astype(np.int64), n_flavours - 1)
    t1 = beta * uniform_array(ps, base + np.uint64(1))
    t2 = beta * uniform_array(ps, base + np.uint64(2))
    op_cfg = np.concatenate([pair_cfg, pair_cfg])
    op_f = np.concatenate([pair_f, pair_f])
    op_t = np.concatenate([t1, t2])
    # rank inside each (cfg, flavour) group by time decides the type
    o = np.lexsort((op_t, op_f, op_cfg))
    op_cfg, op_f, op_t = op_cfg[o], op_f[o], op_t[o]
    key = op_cfg * n_flavours + op_f
    first = np.concatenate([[True], key[1:] != key[:-1]])
    grp_start = np.maximum.accumulate(np.where(first, np.arange(len(key)), 0))
    rank = np.arange(len(key)) - grp_start
    typ = (coin[op_cfg, op_f].astype(np.int64) + rank) & 1      # 1 = creation
    o = np.lexsort((op_t, op_cfg))
    op_cfg, op_f, op_t, typ = op_cfg[o], op_f[o], op_t[o], typ[o]
    offset = np.concatenate([[0], np.cumsum(2 * K)]).astype(np.int64)
    return Batch(float(beta), offset, (2 * op_f + typ).astype(np.int32), op_t.astype(np.float64))


# --------------------------------------------------------------------------- configs 4-5: window growth
def _window_growth(seed: int, n_flavours: int, beta: float, mean_pairs: float, window: tuple):
    """Insertion growth in the Fock picture = the paper's Pauli-aware pair insertion with a flat
    weight, accepted iff N(tau) stays inside the window."""
    rng = Stream(seed)
    K = rng.poisson(mean_pairs)
    lo_w, hi_w = window
    N0 = lo_w + rng.integer(hi_w - lo_w + 1)
    occ0 = np.zeros(n_flavours, dtype=np.int64)
    pool = list(range(n_flavours))
    for _ in range(N0):
        occ0[pool.pop(rng.integer(len(pool)))] = 1
    T = np.zeros(0)
    Fl = np.zeros(0, dtype=np.int64)
    Ty = np.zeros(0, dtype=np.int64)
    pairs = 0
    tries = 0
    while pairs < K and tries < 100000:
        tries += 1
        f = rng.integer(n_flavours)
        idx = np.nonzero(Fl == f)[0]
        if idx.size == 0:
            lo, length, inside = 0.0, beta, int(occ0[f])
        else:
            i = rng.integer(idx.size)
            lo = T[idx[i]]
            hi = T[idx[(i + 1) % idx.size]]
            length = (hi - lo) % beta if idx.size > 1 else beta
            inside = int(Ty[idx[i]])
        a, b = sorted((length * rng.uniform(), length * rng.uniform()))
        ta, tb = (lo + a) % beta, (lo + b) % beta
        if a == b or ta == tb:
            continue
        dN = -1 if inside else +1
        Nseg = int(occ0.sum()) + np.concatenate([[0], np.cumsum(2 * Ty - 1)])
        ia = int(np.searchsorted(T, ta, side="right"))
        ib = int(np.searchsorted(T, tb, side="left"))
        segs = Nseg[ia:ib + 1] if tb > ta else np.concatenate([Nseg[ia:], Nseg[:ib + 1]])
        if segs.min() + dN < lo_w or segs.max() + dN > hi_w:
            continue
        for t_new, ty_new in ((ta, 0 if inside else 1), (tb, 1 if inside else 0)):
            p = int(np.searchsorted(T, t_new))
            T = np.insert(T, p, t_new)
            Fl = np.insert(Fl, p, f)
            Ty = np.insert(Ty, p, ty_new)
        if tb < ta:
            occ0[f] = 1 - occ0[f]
        pairs += 1
    return (2 * Fl + Ty).astype(np.int32), T.astype(np.float64)


def make_batch(cfg: int, n_configs: int | None = None, start: int = 0) -> Batch:
    """Configurations start .. start+n_configs-1 of BASELINE.json config `cfg` (1-based); default = its stated batch."""
    p = BASELINE_CONFIGS[cfg]
    n = p["batch"] if n_configs is None else int(n_configs)
    if p["kind"] == "fixed":
        return _uniform_alternating(cfg, start, n, p["n_flavours"], p["beta"], p["pairs_per_flavour"], None)
    if p["kind"] == "poisson":
        return _uniform_alternating(cfg, start, n, p["n_flavours"], p["beta"], None, p["mean_pairs"])
    return Batch.from_lists(p["beta"], [_window_growth(1000 * cfg + start + b, p["n_flavours"], p["beta"],
                                                       p["mean_pairs"], p["window"]) for b in range(n)])
