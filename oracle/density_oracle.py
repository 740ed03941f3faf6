"""ORACLE -- test infrastructure only.  Plain CPU (numpy, fp64) statement of the per-configuration estimator of the reduced
density matrix of the impurity (Eq. 27),

    rho_uv(C) = (1 / beta) int_0^beta w_loc(C, P_vu(tau)) / w_loc(C) dtau,        P_vu = |v><u|,

with the tau integral done analytically ("This integration is done analytically"), u and v eigenstates of H_loc in
the same sector (P_vu must commute with the conserved charges).

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline leg may import this.  It shares no code with the CUDA
path and imports nothing from it; of `oracle/trace_oracle.py` it uses the impurity view, routing and the scaled-number helpers.

Derivation written out (nothing here is in the paper beyond Eq. 27).  With the cyclic factorisation of reading A2,
w_loc(q0) = Tr[A_L ... A_1], A_i = P_{Delta_i}(q_i) F_i, Delta_i = tau_{i+1} - tau_i, Delta_L = beta - tau_L + tau_1, put

    G_i = F_i A_{i-1} ... A_1          (dim q_i x dim q_0: everything up to, but without, the propagator of interval i),
    Y_i = A_L ... A_{i+1}              (dim q_0 x dim q_i: everything after interval i),

so that w_loc(q0) = Tr[Y_i P_{Delta_i} G_i] for every i.  Inserting P_vu at a time s after tau_i inside interval i replaces
P_{Delta_i} by P_{Delta_i - s} |v><u| P_s, i.e. the integrand becomes exp(-(Delta_i - s) E_v) exp(-s E_u) (G_i Y_i)_{uv}, and

    int_0^Delta exp(-s E_u - (Delta - s) E_v) ds = Delta exp(-Delta min(E_u, E_v)) phi(Delta |E_u - E_v|),   phi(x) = (1 - e^-x) / x.

Every interval of every surviving closed string contributes to the block rho(q_i); the interval that wraps around beta is one
interval (time-translation invariance of the trace).  L = 0: rho = diag(exp(-beta E)) / Z.

Pins: tests/test_density_oracle.py (sum_u rho_uu = 1 for every configuration; L = 0 closed form; Gauss-Legendre quadrature of
oracle.trace_oracle.trace_config with the projector inserted as one more operator symbol; hermiticity of the thermal average in
the exactly solvable one-orbital case).
"""
from __future__ import annotations

import math

import numpy as np

from . import trace_oracle as T


def _phi(x: np.ndarray) -> np.ndarray:
    """(1 - exp(-x)) / x for x >= 0, 1 at x = 0."""
    out = np.ones_like(x)
    nz = x > 0
    out[nz] = -np.expm1(-x[nz]) / x[nz]
    return out


def interval_kernel(delta: float, E: np.ndarray, Emin: float) -> np.ndarray:
    """K'[u, v] = int_0^delta exp(-s (E_u - Emin) - (delta - s) (E_v - Emin)) ds  (the factor exp(-delta Emin) is carried in the
    real exponent lg of the string, as for the propagators)."""
    d = E - Emin
    lo = np.minimum(d[:, None], d[None, :])
    return delta * np.exp(-delta * lo) * _phi(delta * np.abs(d[:, None] - d[None, :]))


def density_config(desc, beta: float, symbols, taus) -> dict:
    """rho(C) of one configuration: {"rho": [per sector q a dim_q x dim_q array, rho[q][u, v] = rho_uv], "status": as trace_config}.
    For status != 0 or w_loc = 0 every block is zero (the estimator presupposes w_loc(C) != 0)."""
    imp = T._imp(desc)
    dt = np.complex128 if imp.is_complex else np.float64
    rho = [np.zeros((int(d), int(d)), dtype=dt) for d in imp.dims]
    tr = T.trace_config(desc, beta, symbols, taus)
    if tr["status"] != 0 or tr["mant"] == 0:
        return dict(rho=rho, status=tr["status"])
    w, we = tr["mant"], tr["exp2"]
    L = len(symbols)
    if L == 0:
        for q in range(imp.Q):
            z, e = T._apply_lg(complex(1.0, 0.0), 0, -float(beta) * imp.Emin[q] * T.LOG2E)
            scale = (z / w) * 2.0 ** max(e - we, -1074)
            rho[q] += np.diag(np.exp(-float(beta) * (imp.E[q] - imp.Emin[q]))) * (scale if imp.is_complex else scale.real)
        return dict(rho=rho, status=0)
    deltas = T._factor_deltas(beta, taus)
    for q0 in range(imp.Q):
        visited = T.route(desc, symbols, q0)
        if visited is None or visited[-1] != q0:
            continue
        d0 = int(imp.dims[q0])
        # forward: G_i (stored, with its integer exponent) and X_i = P_{Delta_i} G_i
        X, ex = np.eye(d0, dtype=dt), 0
        G, eG, lg = [], [], 0.0
        for i in range(L):
            q_prev, q = visited[i], visited[i + 1]
            Gi = imp.F[(int(symbols[i]), q_prev)] @ X
            G.append(Gi)
            eG.append(ex)
            X, k = T._propagate(Gi, deltas[i], imp.E[q], imp.Emin[q])
            ex += k
            lg += -deltas[i] * imp.Emin[q] * T.LOG2E
        # backward: Y_i, starting from Y_L = 1
        Y, ey = np.eye(d0, dtype=dt), 0
        for i in range(L - 1, -1, -1):
            q_prev, q = visited[i], visited[i + 1]
            C = G[i] @ Y                                            # (dim q_i x dim q_i)
            K = interval_kernel(deltas[i], imp.E[q], imp.Emin[q])
            z, e = T._apply_lg(complex(1.0, 0.0), eG[i] + ey, lg)
            scale = (z / w) * 2.0 ** max(min(e - we, 1000), -1074) / float(beta)
            rho[q] += (K * C) * (scale if imp.is_complex else scale.real)
            # Y_{i-1} = Y_i P_{Delta_i} F_i: the propagator scales the COLUMNS of Y_i, i.e. the rows of its transpose
            Yt, k = T._propagate(np.ascontiguousarray(Y.T), deltas[i], imp.E[q], imp.Emin[q])
            Y = Yt.T @ imp.F[(int(symbols[i]), q_prev)]
            ey += k
            mx = float(np.max(np.abs(Y))) if Y.size else 0.0
            if mx > 0.0:
                _, kk = math.frexp(mx)
                Y = np.ldexp(Y.real, -kk) + 1j * np.ldexp(Y.imag, -kk) if imp.is_complex else np.ldexp(Y, -kk)
                ey += kk
    return dict(rho=rho, status=0)


def density_batch(desc, beta: float, offset, symbol, tau, weight=None):
    """sum_b weight_b rho(C_b) in the C-ABI's layout: one flat array, sector q at offset sum_{q' < q} dim_q'^2, column-major
    (element (u, v) at u + v dim_q), complex128 if the impurity is complex."""
    imp = T._imp(desc)
    dt = np.complex128 if imp.is_complex else np.float64
    out = np.zeros(int(np.sum(np.asarray(imp.dims, dtype=np.int64) ** 2)), dtype=dt)
    off2 = np.concatenate([[0], np.cumsum(np.asarray(imp.dims, dtype=np.int64) ** 2)])
    B = len(offset) - 1
    for b in range(B):
        lo, hi = int(offset[b]), int(offset[b + 1])
        r = density_config(desc, beta, symbol[lo:hi], tau[lo:hi])
        wb = 1.0 if weight is None else float(weight[b])
        for q in range(imp.Q):
            out[off2[q]:off2[q + 1]] += wb * r["rho"][q].ravel(order="F")
    return out
