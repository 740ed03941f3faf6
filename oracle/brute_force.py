"""ORACLE-B — test infrastructure only.  Brute force in the unblocked Fock space (Eq. 63).

    w_loc = Tr P_{beta-tau_L} O_L P_{tau_L - tau_{L-1}} ... O_1 P_{tau_1},     P_tau = exp(-tau H_loc)   (2^n x 2^n),

with H_loc built from Eq. 2 as dense matrix products of Jordan-Wigner c / c^dag matrices assembled from
Kronecker products, and P_tau from a scaling-and-squaring Taylor series.  No sectors, no eigen-decomposition of
sectors, no routing tables: it is independent of the input builder (`workloads/impurity.py`) and of Oracle-A
(`trace_oracle.py`), so agreement between them pins Fock signs, sector labelling, diagonalisation, basis rotation,
routing and the chain product at once.  Usable for n <= 8 flavours.  A scalar shift H -> H - e0 (e0 from a library
eigvalsh of the full matrix, used as a number only) keeps exp(-tau H) bounded; it is undone in the returned exponent.
"""
from __future__ import annotations

import math

import numpy as np

LOG2E = 1.4426950408889634


def annihilators(n: int):
    """c_f as 2^n x 2^n matrices; basis index = sum_f n_f 2^f; c_f = (prod_{g<f} (-1)^{n_g}) sigma^-_f."""
    a = np.array([[0.0, 1.0], [0.0, 0.0]])   # |0><1|
    z = np.diag([1.0, -1.0])
    one = np.eye(2)
    ops = []
    for f in range(n):
        m = np.ones((1, 1))
        for g in range(n - 1, -1, -1):        # most significant factor first
            m = np.kron(m, a if g == f else (z if g < f else one))
        ops.append(m)
    return ops


def hamiltonian(h1: np.ndarray, u: np.ndarray) -> np.ndarray:
    """Eq. 2: H = sum_ij c+_i h1_ij c_j + 1/2 sum_ijkl c+_i c+_j U_ijkl c_k c_l   (h1 = t - mu)."""
    n = h1.shape[0]
    c = annihilators(n)
    cd = [m.T.copy() for m in c]
    H = np.zeros((1 << n, 1 << n), dtype=np.complex128)
    for i in range(n):
        for j in range(n):
            if h1[i, j] != 0:
                H += h1[i, j] * (cd[i] @ c[j])
    for (i, j, k, l) in zip(*np.nonzero(u)):
        H += 0.5 * u[i, j, k, l] * (cd[i] @ cd[j] @ c[k] @ c[l])
    return H


def expm_taylor(A: np.ndarray) -> np.ndarray:
    """exp(A) by scaling and squaring with a Taylor series (no eigen-solver)."""
    nrm = np.abs(A).sum(axis=1).max()
    s = max(0, int(math.ceil(math.log2(max(nrm, 1e-300)))) + 2)
    B = A / (2.0 ** s)                        # ||B|| <= 1/4
    term = np.eye(A.shape[0], dtype=A.dtype)
    out = term.copy()
    for k in range(1, 30):
        term = term @ B / k
        out = out + term
    for _ in range(s):
        out = out @ out
    return out


def trace(h1: np.ndarray, u: np.ndarray, beta: float, symbols, taus):
    """Eq. 63 multiplied out in the full Fock space.  Returns (mant complex, exp2 int), value = mant * 2**exp2."""
    n = h1.shape[0]
    H = hamiltonian(np.asarray(h1), np.asarray(u))
    e0 = float(np.linalg.eigvalsh(H)[0])
    Hs = H - e0 * np.eye(1 << n)
    c = annihilators(n)
    ops = {}
    for f in range(n):
        ops[2 * f] = c[f].astype(np.complex128)
        ops[2 * f + 1] = c[f].T.astype(np.complex128)
    L = len(symbols)
    e2 = 0

    def rescale(M, e2):
        mx = max(np.abs(M.real).max(), np.abs(M.imag).max())
        if mx == 0:
            return M, e2
        _, ex = math.frexp(float(mx))
        return M * math.ldexp(1.0, -ex), e2 + ex

    M = expm_taylor(-(float(taus[0]) if L else float(beta)) * Hs)
    for i in range(L):
        M = ops[int(symbols[i])] @ M
        delta = (float(taus[i + 1]) - float(taus[i])) if i + 1 < L else (float(beta) - float(taus[i]))
        M = expm_taylor(-delta * Hs) @ M
        M, e2 = rescale(M, e2)
    d = np.diagonal(M)
    z = complex(math.fsum(d.real), math.fsum(d.imag))
    lg = -float(beta) * e0 * LOG2E
    k = math.floor(lg)
    z *= 2.0 ** (lg - k)
    e2 += int(k)
    mx = max(abs(z.real), abs(z.imag))
    if mx == 0:
        return 0j, 0
    _, ex = math.frexp(mx)
    return complex(math.ldexp(z.real, 1 - ex), math.ldexp(z.imag, 1 - ex)), e2 + ex - 1
