"""ORACLE — test infrastructure only.  Plain, slow CPU (numpy, fp64) statement of what the hot path computes.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` leg may import this.
It shares no code with the CUDA path (`paper_2010_08482_b200/`) and imports nothing from it.

What it computes (citations are PAPER.md line numbers):

  * `route`          the sector string q_0 -> q_1 = s_alpha1(q_0) -> ... of :532-534; -1 is the "zero sector".
  * `trace_config`   the sector-summed local trace, literally Eq. 65 (:529):
                       w = sum_{q0} Tr P_{beta-tau_L}(q_L) F_{alpha_L}(q_{L-1}) ... F_{alpha_1}(q_0) P_{tau_1}(q_0),
                     P_tau(q) = diag(exp(-tau E_q[n])) (:521), multiplied right to left with numpy matmul as the
                     library step.  Result returned as (mantissa, exp2), w = mant * 2**exp2.
  * `bound_config`   the lazy-trace upper bound (:542-548): product of submultiplicative norms of (segments of) the
                     factors, times a rank prefactor (readings A1, A2, A4, A9).

Scaling (paper silent, reading A5): exp(-D E_n) is written 2**x_n * 2**(-D Emin_q log2 e) with
x_n = -D (E_n - Emin_q) log2 e <= 0.  The second factor goes into a running real exponent `lg`.  Of the first, only the
mantissa 2**(x_n - floor x_n) is multiplied into row n; the integers floor(x_n) are compared across rows, the largest
(over non-zero rows) goes into a running integer exponent and the others are applied with ldexp relative to it
(`_propagate`).  Both are exact reorganisations of Eq. 65 apart from the rounding of x_n and `lg` (|x|, |lg| <~ 1e4,
i.e. ~1e-12 relative in the value), and neither can underflow: np.exp(-D (E_n - Emin)) would, for D (E_n - Emin) > 745,
which the uniformly placed operators of BASELINE config 3 reach (pin: test_P5_coarse_sectors_do_not_underflow).

Pins: tests/test_oracle_pins.py (Z closed form, cyclicity, brute force in the unblocked Fock space, gauge / shift /
time-reversal invariances, Ising closed form, atomic Green function, bound >= |trace|, S-monotonicity, S=1 closed forms).
Spectral bound with segment_len != 1 is a plain SVD here; the CUDA path does not implement it ("parity unpinned" does
not arise: it is simply not offered on the GPU side).
"""
from __future__ import annotations

import math

import numpy as np

LOG2E = 1.4426950408889634
BOUND_INFLATION = 1.0 + 2.0 ** -40   # DESIGN.md reading A9: bounds are rounded outward


# --------------------------------------------------------------------------- impurity access (duck-typed desc)
class _Imp:
    """Unpacks the ctqmc_impurity_desc-shaped object (dims, energy, blk_* arrays) into per-sector / per-block views."""

    def __init__(self, desc):
        self.dims = np.asarray(desc.dims, dtype=np.int64)
        self.Q = len(self.dims)
        self.A = int(desc.n_symbols)
        off = np.concatenate([[0], np.cumsum(self.dims)])
        en = np.asarray(desc.energy, dtype=np.float64)
        self.E = [en[off[q]:off[q + 1]] for q in range(self.Q)]
        self.Emin = np.array([e.min() for e in self.E])
        self.smap = -np.ones((self.A, self.Q), dtype=np.int64)
        self.F = {}
        data = np.asarray(desc.blk_data)
        for b in range(len(desc.blk_symbol)):
            a, s, d = int(desc.blk_symbol[b]), int(desc.blk_src[b]), int(desc.blk_dst[b])
            m, n = int(self.dims[d]), int(self.dims[s])
            o = int(desc.blk_offset[b])
            self.smap[a, s] = d
            self.F[(a, s)] = data[o:o + m * n].reshape((m, n), order="F")
        self.is_complex = bool(desc.is_complex)


def _imp(desc) -> _Imp:
    view = getattr(desc, "_oracle_view", None)
    if view is None:
        view = _Imp(desc)
        try:
            setattr(desc, "_oracle_view", view)
        except AttributeError:
            pass
    return view


# --------------------------------------------------------------------------- scaled-number helpers
def _normalize(z: complex, e: int):
    """(z, e) -> same value with max(|re|, |im|) in [1, 2); exact zero -> (0, 0)."""
    mx = max(abs(z.real), abs(z.imag))
    if mx == 0.0 or not math.isfinite(mx):
        return (z if not math.isfinite(mx) else 0j), 0
    _, ex = math.frexp(mx)
    return complex(math.ldexp(z.real, 1 - ex), math.ldexp(z.imag, 1 - ex)), e + ex - 1


def _sum_scaled(items):
    """Sum of z_s * 2**e_s, aligned to the largest exponent, each component with math.fsum."""
    items = [(z, e) for z, e in items if z != 0]
    if not items:
        return 0j, 0
    emax = max(e for _, e in items)
    re = math.fsum(math.ldexp(z.real, e - emax) for z, e in items)
    im = math.fsum(math.ldexp(z.imag, e - emax) for z, e in items)
    return _normalize(complex(re, im), emax)


def _apply_lg(z: complex, e: int, lg: float):
    """(z * 2**e) * 2**lg with lg a real number: integer part into the exponent, fraction into the mantissa."""
    k = math.floor(lg)
    return _normalize(z * (2.0 ** (lg - k)), e + int(k))


def _propagate(M: np.ndarray, delta: float, E: np.ndarray, Emin: float):
    """diag(exp(-delta (E - Emin))) @ M, returned as (M', k) with the product equal to M' * 2**k and max|component| of
    M' in [0.5, 1)  (M' = 0, k = 0 if the product vanishes).

    Row n is multiplied by 2**x_n, x_n = -delta (E_n - Emin) log2(e) <= 0, which is split into the integer floor(x_n)
    and the mantissa 2**(x_n - floor(x_n)) in [1, 2).  Only the mantissa is multiplied in; the integer parts are
    compared across rows and applied with ldexp relative to the largest row.  So a row whose factor exp(-delta (E_n -
    Emin)) is far below the smallest double keeps full precision whenever the rows with a larger factor are zero (e.g.
    by a symmetry the sector labels do not resolve) -- np.exp would underflow there, although Eq. 65's value is
    perfectly representable as mant * 2**exp2 (reading A5)."""
    x = (-float(delta) * (E - Emin)) * LOG2E
    k = np.floor(x)
    M = np.exp2(x - k)[:, None] * M
    k = k.astype(np.int64)
    rowmax = np.maximum(np.abs(M.real), np.abs(M.imag)).max(axis=1) if np.iscomplexobj(M) else np.abs(M).max(axis=1)
    nz = rowmax > 0.0
    if not nz.any():
        return M * 0.0, 0
    _, ex = np.frexp(rowmax[nz])
    kmax = int((k[nz] + ex).max())
    shift = np.clip(k - kmax, -4000, 4000).astype(np.int32)[:, None]
    if np.iscomplexobj(M):
        M = np.ldexp(M.real, shift) + 1j * np.ldexp(M.imag, shift)
    else:
        M = np.ldexp(M, shift)
    return M, kmax


# --------------------------------------------------------------------------- routing (:532-534)
def validate(desc, beta: float, symbols, taus) -> bool:
    """DESIGN.md reading A7: symbols in [0, A), taus non-decreasing in [0, beta)."""
    imp = _imp(desc)
    symbols = np.asarray(symbols)
    taus = np.asarray(taus, dtype=np.float64)
    if len(symbols) == 0:
        return True
    if symbols.min() < 0 or symbols.max() >= imp.A:
        return False
    if not np.all(np.isfinite(taus)) or taus.min() < 0.0 or taus.max() >= beta:
        return False
    return bool(np.all(np.diff(taus) >= 0.0))


def route(desc, symbols, q0: int):
    """Visited sectors [q_0, q_1, ..., q_L] or None if the string hits the zero sector (:534)."""
    imp = _imp(desc)
    q = int(q0)
    visited = [q]
    for a in symbols:
        q = int(imp.smap[int(a), q])
        if q < 0:
            return None
        visited.append(q)
    return visited


def survive_mask(desc, symbols) -> np.ndarray:
    imp = _imp(desc)
    return np.array([1 if route(desc, symbols, q0) is not None else 0 for q0 in range(imp.Q)], dtype=np.uint8)


# --------------------------------------------------------------------------- the trace, Eq. 65 (:529)
def _string_trace(imp: _Imp, beta: float, symbols, taus, visited):
    """One start sector of Eq. 65.  Returns (trace z, integer exponent e, real exponent lg, sqrt(d) ||M||_F):
    contribution = z * 2**e * 2**lg; the last item (same scaling) is the size against which rounding noise in z
    must be judged (reading A8)."""
    L = len(symbols)
    q0 = visited[0]
    tau1 = float(taus[0]) if L else float(beta)
    M = np.eye(int(imp.dims[q0]), dtype=np.complex128 if imp.is_complex else np.float64)
    M, e2 = _propagate(M, tau1, imp.E[q0], imp.Emin[q0])
    lg = -tau1 * imp.Emin[q0] * LOG2E
    for i in range(L):
        q_prev, q = visited[i], visited[i + 1]
        M = imp.F[(int(symbols[i]), q_prev)] @ M
        delta = (float(taus[i + 1]) - float(taus[i])) if i + 1 < L else (float(beta) - float(taus[i]))
        M, ex = _propagate(M, delta, imp.E[q], imp.Emin[q])
        lg += -delta * imp.Emin[q] * LOG2E
        e2 += ex
    if visited[-1] != q0:       # off-diagonal block: no trace (never happens for balanced c^dag / c strings, :532)
        return 0j, 0, 0.0, 0.0
    diag = np.diagonal(M)
    z = complex(math.fsum(diag.real), math.fsum(diag.imag))
    return z, e2, lg, math.sqrt(M.shape[0]) * float(np.linalg.norm(M))


def trace_config(desc, beta: float, symbols, taus) -> dict:
    """w_loc for one configuration.  Keys: mant (complex), exp2 (int), survive (uint8[Q]), status
    (0 ok, 1 no surviving start sector, 2 invalid input), sector (per q0: (mant, exp2) or None),
    kappa = sum_q0 sqrt(d) ||M_L(q0)||_F / |w|  (how much cancellation the value has suffered; reading A8)."""
    imp = _imp(desc)
    if not validate(desc, beta, symbols, taus):
        return dict(mant=complex(math.nan, math.nan), exp2=0, survive=np.zeros(imp.Q, np.uint8), status=2,
                    sector=[None] * imp.Q, kappa=math.nan)
    surv = np.zeros(imp.Q, dtype=np.uint8)
    sector = [None] * imp.Q
    terms, absterms = [], []
    for q0 in range(imp.Q):
        visited = route(desc, symbols, q0)
        if visited is None:
            continue
        surv[q0] = 1
        z, e, lg, absd = _string_trace(imp, beta, symbols, taus, visited)
        zs, es = _apply_lg(z, e, lg)
        sector[q0] = (zs, es)
        terms.append((zs, es))
        a, ae = _apply_lg(complex(absd, 0.0), e, lg)
        absterms.append((a, ae))
    w, ew = _sum_scaled(terms)
    aw, aew = _sum_scaled(absterms)
    kappa = math.inf if w == 0 else (aw.real / max(abs(w.real), abs(w.imag))) * 2.0 ** min(aew - ew, 1000)
    return dict(mant=w, exp2=ew, survive=surv, status=0 if surv.any() else 1, sector=sector, kappa=kappa)


def trace_batch(desc, beta: float, offset, symbol, tau):
    """Batch form with the C-ABI's output layout: mant[B,2], exp2[B], survive[B,Q], status[B]."""
    imp = _imp(desc)
    B = len(offset) - 1
    mant = np.zeros((B, 2))
    exp2 = np.zeros(B, dtype=np.int64)
    surv = np.zeros((B, imp.Q), dtype=np.uint8)
    status = np.zeros(B, dtype=np.int32)
    for b in range(B):
        lo, hi = int(offset[b]), int(offset[b + 1])
        r = trace_config(desc, beta, symbol[lo:hi], tau[lo:hi])
        mant[b] = (r["mant"].real, r["mant"].imag)
        exp2[b], surv[b], status[b] = r["exp2"], r["survive"], r["status"]
    return mant, exp2, surv, status


# --------------------------------------------------------------------------- the bound (:542-548)
def _factor_deltas(beta: float, taus):
    """Cyclic factorisation (reading A2): Tr[P_{beta-tau_L} F_L ... F_1 P_{tau_1}] = Tr[A_L ... A_1] with
    A_i = P_{Delta_i}(q_i) F_{alpha_i}(q_{i-1}), Delta_i = tau_{i+1} - tau_i, Delta_L = beta - tau_L + tau_1."""
    L = len(taus)
    return [(float(taus[i + 1]) - float(taus[i])) if i + 1 < L else (float(beta) - float(taus[i]) + float(taus[0]))
            for i in range(L)]


def _string_bound(imp: _Imp, beta: float, symbols, taus, visited, norm_kind: int, segment_len: int):
    """Bound for one start sector as (value z>=0, int exponent, real exponent lg)."""
    L = len(symbols)
    dmin = min(int(imp.dims[q]) for q in visited)
    pref = math.sqrt(dmin) if norm_kind == 0 else float(dmin)
    if norm_kind == 2 and segment_len == 1:
        norm_kind = 1          # one factor per segment: the estimate IS the factorised closed form
    if L == 0:
        q0 = visited[0]
        p = np.exp(-float(beta) * (imp.E[q0] - imp.Emin[q0]))
        nrm = math.sqrt(math.fsum(p * p)) if norm_kind == 0 else float(p.max())
        return pref * nrm, 0, -float(beta) * imp.Emin[q0] * LOG2E
    deltas = _factor_deltas(beta, taus)
    S = L if segment_len == 0 else int(segment_len)
    val, e2, lg = pref, 0, 0.0
    for start in range(0, L, S):
        stop = min(L, start + S)
        if norm_kind == 1 and S == 1:
            # factorised closed form: ||P_D(q) F||_2 <= exp(-D Emin_q) sigma_max(F)
            q_prev, q = visited[start], visited[start + 1]
            sig = float(np.linalg.svd(imp.F[(int(symbols[start]), q_prev)], compute_uv=False)[0])
            val *= sig
            lg += -deltas[start] * imp.Emin[q] * LOG2E
            continue
        M = np.eye(int(imp.dims[visited[start]]), dtype=np.complex128 if imp.is_complex else np.float64)
        ex_seg = 0
        for i in range(start, stop):
            q_prev, q = visited[i], visited[i + 1]
            M = imp.F[(int(symbols[i]), q_prev)] @ M
            M, ex = _propagate(M, deltas[i], imp.E[q], imp.Emin[q])
            lg += -deltas[i] * imp.Emin[q] * LOG2E
            e2 += ex
            ex_seg += ex
        if norm_kind == 0:
            nrm = math.sqrt(math.fsum((np.abs(M) ** 2).ravel()))
        elif norm_kind == 1:
            nrm = float(np.linalg.svd(M, compute_uv=False)[0])
        else:
            # norm_kind 2, the certified estimate of ||G_j||_2 the CUDA path returns for spectral bounds with S != 1 (DESIGN.md
            # reading A1): min(||G_j||_F, prod_i sigma_max(F_i)); M is scaled by 2**-ex_seg, the sigma product is not
            fro = math.sqrt(math.fsum((np.abs(M) ** 2).ravel()))
            sprod = 1.0
            for i in range(start, stop):
                sprod *= float(np.linalg.svd(imp.F[(int(symbols[i]), visited[i])], compute_uv=False)[0])
            if fro == 0.0 or math.log2(fro) + ex_seg <= math.log2(sprod):
                nrm = fro
            else:
                nrm, e2 = sprod, e2 - ex_seg
        val *= nrm
        if val != 0.0:
            m, ex = math.frexp(val)
            val, e2 = m, e2 + ex
    return val, e2, lg


def bound_config(desc, beta: float, symbols, taus, norm_kind: int = 0, segment_len: int = 1) -> dict:
    """Upper bound on |w_loc| (and per start sector).  norm_kind 0 Frobenius / 1 spectral (exact SVD of every segment
    product) / 2 certified spectral estimate min(||G_j||_F, prod sigma_max(F_i)) >= ||G_j||_2; segment_len S >= 1, 0 = whole
    chain.  B(q0) = prefactor(d_min) * prod_j ||G_j||, G_j = product of S consecutive cyclic factors A_i;
    prefactor sqrt(d_min) (Frobenius) or d_min (spectral), d_min = min_i dim(q_i)  (|Tr M| <= sqrt(rank)||M||_F <= rank||M||_2).
    Returned values are multiplied by BOUND_INFLATION.  Keys: mant, exp2, sector (per q0 (mant, exp2) or None), status."""
    imp = _imp(desc)
    if not validate(desc, beta, symbols, taus):
        return dict(mant=math.nan, exp2=0, sector=[None] * imp.Q, status=2)
    sector = [None] * imp.Q
    terms = []
    for q0 in range(imp.Q):
        visited = route(desc, symbols, q0)
        if visited is None:
            continue
        v, e, lg = _string_bound(imp, beta, symbols, taus, visited, norm_kind, segment_len)
        z, ez = _apply_lg(complex(v * BOUND_INFLATION, 0.0), e, lg)
        sector[q0] = (z.real, ez)
        terms.append((z, ez))
    w, ew = _sum_scaled(terms)
    return dict(mant=w.real, exp2=ew, sector=sector, status=0 if terms else 1)


def bound_batch(desc, beta: float, offset, symbol, tau, norm_kind: int = 0, segment_len: int = 1):
    """Batch form with the C-ABI's layout: bound_mant[B], bound_exp2[B], sector_mant[B,Q], sector_exp2[B,Q], status[B]."""
    imp = _imp(desc)
    B = len(offset) - 1
    bm = np.zeros(B)
    be = np.zeros(B, dtype=np.int64)
    sm = np.zeros((B, imp.Q))
    se = np.zeros((B, imp.Q), dtype=np.int64)
    status = np.zeros(B, dtype=np.int32)
    for b in range(B):
        lo, hi = int(offset[b]), int(offset[b + 1])
        r = bound_config(desc, beta, symbol[lo:hi], tau[lo:hi], norm_kind, segment_len)
        bm[b], be[b], status[b] = r["mant"], r["exp2"], r["status"]
        for q0, s in enumerate(r["sector"]):
            if s is not None:
                sm[b, q0], se[b, q0] = s
    return bm, be, sm, se, status


def to_log(mant, exp2) -> float:
    """ln|value| of a scaled number (helper for tests and reports)."""
    a = abs(mant)
    return -math.inf if a == 0 else math.log(a) + exp2 * math.log(2.0)
