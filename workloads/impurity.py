"""Impurity-model input builder ("initialization").

Builds what `ctqmc_load_impurity` consumes: the Hilbert space of H_loc (Eq. 2)
split into sectors by Abelian quantum numbers (Eq. 64), H_loc diagonalised per
sector, and every c_f / c^dag_f rotated into that eigenbasis as dense sector-to-sector blocks
F_alpha(q).  This is *input generation*: nothing here evaluates a trace.

Conventions:
  * Fock state = integer, bit f = occupation of flavour f;  |s> = prod_{f in s, ascending}... with
    Jordan-Wigner sign  c_f|s> = (-1)^{popcount(s & (2^f - 1))} |s - f>.
  * symbol alpha = 2 f + 1 for c^dag_f and 2 f for c_f.
  * block element (m, n) = < m in dst | O_alpha | n in src >, stored column-major (dst x src).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from fractions import Fraction
from itertools import combinations

import numpy as np

from .rng import Stream

K_B_EV = 8.617333262e-5  # eV / K

_POP16 = np.array([bin(i).count("1") for i in range(1 << 16)], dtype=np.int64)


# --------------------------------------------------------------------------- interaction tensors
def spin_orbital_tensor(u_orb: np.ndarray) -> np.ndarray:
    """U_ijkl of Eq. 2 from an orbital tensor, generic/product flavour order
    (PAPER.md:754 Eq. A.4/A.5: all spin-down orbitals, then all spin-up).  i,l carry one spin and
    j,k the other (pairing fixed by PAPER.md:118 Eq. 6, reading A13)."""
    n = u_orb.shape[0]
    u = np.zeros((2 * n,) * 4, dtype=u_orb.dtype)
    for s in range(2):
        for sp in range(2):
            u[s * n:(s + 1) * n, sp * n:(sp + 1) * n, sp * n:(sp + 1) * n, s * n:(s + 1) * n] = u_orb
    return u


def kanamori_orbital_tensor(n_orb: int, U: float, J: float) -> np.ndarray:
    """Rotationally invariant Kanamori form (reading A12): U_mmmm = U, U_mm'm'm = U' = U - 2J,
    U_mm'mm' = J (exchange / spin flip), U_mmm'm' = J (pair hopping)."""
    t = np.zeros((n_orb,) * 4)
    for m in range(n_orb):
        t[m, m, m, m] = U
        for mp in range(n_orb):
            if mp != m:
                t[m, mp, mp, m] = U - 2.0 * J
                t[m, mp, m, mp] = J
                t[m, m, mp, mp] = J
    return t


def _fact(n: int) -> int:
    return math.factorial(n)


def wigner_3j(j1: int, j2: int, j3: int, m1: int, m2: int, m3: int) -> float:
    """Wigner 3j symbol for integer angular momenta by Racah's formula (exact rational sum)."""
    if m1 + m2 + m3 != 0 or abs(m1) > j1 or abs(m2) > j2 or abs(m3) > j3:
        return 0.0
    if j3 < abs(j1 - j2) or j3 > j1 + j2:
        return 0.0
    tri = Fraction(_fact(j1 + j2 - j3) * _fact(j1 - j2 + j3) * _fact(-j1 + j2 + j3), _fact(j1 + j2 + j3 + 1))
    pref = tri * _fact(j1 + m1) * _fact(j1 - m1) * _fact(j2 + m2) * _fact(j2 - m2) * _fact(j3 + m3) * _fact(j3 - m3)
    s = Fraction(0)
    for k in range(0, j1 + j2 - j3 + 1):
        a = [k, j1 + j2 - j3 - k, j1 - m1 - k, j2 + m2 - k, j3 - j2 + m1 + k, j3 - j1 - m2 + k]
        if min(a) < 0:
            continue
        den = 1
        for x in a:
            den *= _fact(x)
        s += Fraction((-1) ** k, den)
    sign = (-1) ** ((j1 - j2 - m3) % 2)
    return sign * float(s) * math.sqrt(float(pref))


def gaunt(l: int, m: int, k: int, q: int, mp: int) -> float:
    """< Y_l^m | Y_k^q | Y_l^m' >  (complex spherical harmonics; real number)."""
    return ((-1) ** (m % 2)) * (2 * l + 1) * math.sqrt((2 * k + 1) / (4.0 * math.pi)) * \
        wigner_3j(l, k, l, 0, 0, 0) * wigner_3j(l, k, l, -m, q, mp)


def slater_orbital_tensor(l: int, F: list[float]) -> np.ndarray:
    """Slater-Condon Coulomb tensor in complex Y_l^m, m = -l..l (reading A13):
    U_{m1 m2 m3 m4} = sum_k F^k 4pi/(2k+1) sum_q <m1|Y_kq|m4> conj<m3|Y_kq|m2>,  F = [F0, F2, ..., F_{2l}]."""
    n = 2 * l + 1
    u = np.zeros((n,) * 4)
    for ik, fk in enumerate(F):
        k = 2 * ik
        g = np.zeros((n, 2 * k + 1, n))
        for a in range(n):
            for q in range(-k, k + 1):
                for b in range(n):
                    g[a, q + k, b] = gaunt(l, a - l, k, q, b - l)
        # u[m1,m2,m3,m4] += F^k 4pi/(2k+1) sum_q g[m1,q,m4] g[m3,q,m2]
        u += fk * (4.0 * math.pi / (2 * k + 1)) * np.einsum("aqd,cqb->abcd", g, g)
    return u


def clebsch_gordan_l_half(l: int) -> np.ndarray:
    """T[i_product, a_coupled] = < l m ; 1/2 sigma | j m_j >  (PAPER.md:747 Eq. A.3), product order
    Eq. A.5 (m ascending, spin-down block then spin-up block), coupled order Eq. A.6
    (j = l-1/2 then j = l+1/2, m_j ascending).  Condon-Shortley phases; real."""
    n = 2 * l + 1
    T = np.zeros((2 * n, 2 * n))
    col = 0
    for twoj in (2 * l - 1, 2 * l + 1):
        for twomj in range(-twoj, twoj + 1, 2):
            mj = twomj / 2.0
            m_up, m_dn = int(round(mj - 0.5)), int(round(mj + 0.5))
            if twoj == 2 * l + 1:
                c_up = math.sqrt((l + mj + 0.5) / (2 * l + 1))
                c_dn = math.sqrt((l - mj + 0.5) / (2 * l + 1))
            else:
                c_up = -math.sqrt((l - mj + 0.5) / (2 * l + 1))
                c_dn = math.sqrt((l + mj + 0.5) / (2 * l + 1))
            if -l <= m_up <= l:
                T[n + (m_up + l), col] = c_up
            if -l <= m_dn <= l:
                T[(m_dn + l), col] = c_dn
            col += 1
    return T


def rotate_tensor(u: np.ndarray, T: np.ndarray) -> np.ndarray:
    """One-particle basis change c_a = sum_i conj(T_ia) c_i:  U'_abcd = conj(T_ia) conj(T_jb) U_ijkl T_kc T_ld."""
    Tc = T.conj()
    u = np.einsum("ia,ijkl->ajkl", Tc, u)
    u = np.einsum("jb,ajkl->abkl", Tc, u)
    u = np.einsum("kc,abkl->abcl", T, u)
    return np.einsum("ld,abcl->abcd", T, u)


# --------------------------------------------------------------------------- Fock-space machinery
def _popcount(x: np.ndarray) -> np.ndarray:
    return _POP16[x & 0xFFFF] + _POP16[(x >> 16) & 0xFFFF]


def _apply_c(states: np.ndarray, amp: np.ndarray, f: int):
    occ = (states >> f) & 1
    sign = 1 - 2 * (_popcount(states & ((1 << f) - 1)) & 1)
    return states ^ (occ << f), amp * (sign * occ)


def _apply_cdag(states: np.ndarray, amp: np.ndarray, f: int):
    emp = 1 - ((states >> f) & 1)
    sign = 1 - 2 * (_popcount(states & ((1 << f) - 1)) & 1)
    return states | (emp << f), amp * (sign * emp)


def _hamiltonian_coo(states: np.ndarray, h1: np.ndarray, u: np.ndarray):
    """H_loc over all enumerated Fock states as COO triplets (row, col, value):
    sum_ij h1_ij c+_i c_j + 1/2 sum_ijkl U_ijkl c+_i c+_j c_k c_l  (Eq. 2; h1 = t - mu).
    `states` must be sorted ascending and closed under H_loc (H conserves N)."""
    d = len(states)
    cols = np.arange(d)
    one = np.ones(d, dtype=np.int64)
    rows_l, cols_l, vals_l = [], [], []

    def scatter(new_states, amp, coef):
        nz = np.nonzero(amp)[0]
        if nz.size == 0:
            return
        pos = np.searchsorted(states, new_states[nz])
        assert np.all(pos < d) and np.all(states[pos] == new_states[nz]), "H_loc leaves the enumerated space"
        rows_l.append(pos)
        cols_l.append(cols[nz])
        vals_l.append(coef * amp[nz])

    n = h1.shape[0]
    for i in range(n):
        for j in range(n):
            if h1[i, j] != 0:
                s, a = _apply_c(states, one, j)
                s, a = _apply_cdag(s, a, i)
                scatter(s, a, h1[i, j])
    for (i, j, k, l) in zip(*np.nonzero(u)):
        s, a = _apply_c(states, one, l)
        s, a = _apply_c(s, a, k)
        s, a = _apply_cdag(s, a, j)
        s, a = _apply_cdag(s, a, i)
        scatter(s, a, 0.5 * u[i, j, k, l])
    if not rows_l:
        return np.zeros(0, np.int64), np.zeros(0, np.int64), np.zeros(0)
    return np.concatenate(rows_l), np.concatenate(cols_l), np.concatenate(vals_l)


def sector_dimensions(n: int, flavour_qn, n_window: tuple | None = None, modulo: tuple | None = None) -> dict:
    """Sector label -> dimension by counting Fock states only (no Hamiltonian).  `modulo[k]`, if non-zero, reduces
    quantum number k modulo that value (e.g. J_z mod 4 for a cubic crystal field; PAPER.md:554 block ranks)."""
    qn = np.asarray(flavour_qn, dtype=np.int64)
    states = np.arange(1 << n, dtype=np.int64)
    occ = ((states[:, None] >> np.arange(n)[None, :]) & 1)
    lab = occ @ qn
    if n_window is not None:
        keep = (lab[:, 0] >= n_window[0]) & (lab[:, 0] <= n_window[1])
        lab = lab[keep]
    if modulo is not None:
        for k, m in enumerate(modulo):
            if m:
                lab[:, k] = np.mod(lab[:, k], m)
    uniq, counts = np.unique(lab, axis=0, return_counts=True)
    return {tuple(int(x) for x in u): int(c) for u, c in zip(uniq, counts)}


# --------------------------------------------------------------------------- the impurity object
@dataclass
class Impurity:
    name: str
    n_flavours: int
    beta: float
    labels: list            # [Q] tuples of quantum numbers, sorted lexicographically
    dims: np.ndarray        # [Q] int32
    energy: np.ndarray      # [sum dims] float64, sector-major
    is_complex: bool
    blk_symbol: np.ndarray  # [n_blocks] int32
    blk_src: np.ndarray     # [n_blocks] int32
    blk_dst: np.ndarray     # [n_blocks] int32
    blk_offset: np.ndarray  # [n_blocks] int64, element offsets into blk_data
    blk_data: np.ndarray    # flat float64 / complex128, each block column-major (dst x src)
    flavour_qn: np.ndarray  # [n_flavours, n_labels] additive quantum numbers carried by each flavour
    n_window: tuple | None  # (lo, hi) particle-number window, None = full Fock space
    h1: np.ndarray          # one-body matrix t - mu (flavour basis)
    u: np.ndarray           # interaction tensor U_ijkl (flavour basis)
    sector_states: list = field(default_factory=list)  # per sector: Fock integers (row order of eigvecs)
    eigvecs: list = field(default_factory=list)        # per sector: eigenvector matrix (columns) or empty

    @property
    def n_sectors(self) -> int:
        return len(self.dims)

    @property
    def n_symbols(self) -> int:
        return 2 * self.n_flavours

    @property
    def n_blocks(self) -> int:
        return len(self.blk_symbol)

    def energy_of(self, q: int) -> np.ndarray:
        off = int(np.sum(self.dims[:q]))
        return self.energy[off:off + int(self.dims[q])]

    def block(self, b: int) -> np.ndarray:
        """Block b as a (dst x src) matrix view."""
        m, n = int(self.dims[self.blk_dst[b]]), int(self.dims[self.blk_src[b]])
        off = int(self.blk_offset[b])
        return self.blk_data[off:off + m * n].reshape((m, n), order="F")

    def sector_map(self) -> np.ndarray:
        """s_alpha(q) as an [A, Q] table, -1 = the paper's zero sector."""
        t = -np.ones((self.n_symbols, self.n_sectors), dtype=np.int32)
        t[self.blk_symbol, self.blk_src] = self.blk_dst
        return t


def build_impurity(name: str, h1: np.ndarray, u: np.ndarray, flavour_qn, beta: float,
                   n_window: tuple | None = None, phase_seed: int | None = None,
                   keep_eigvecs: bool = True) -> Impurity:
    """Sector decomposition, per-sector diagonalisation and operator blocks.

    h1 = t - mu (n x n Hermitian), u = U_ijkl (Eq. 2), flavour_qn[f] = additive quantum numbers of flavour f,
    first one must be the particle number (=1).  phase_seed: multiply each eigenvector by a seeded random
    phase (reading A17) -- makes real problems genuinely complex without changing any trace."""
    n = h1.shape[0]
    flavour_qn = np.asarray(flavour_qn, dtype=np.int64)
    assert flavour_qn.shape[0] == n and np.all(flavour_qn[:, 0] == 1)
    cplx = bool(np.iscomplexobj(h1) and np.any(np.imag(h1) != 0)) or bool(np.iscomplexobj(u) and np.any(np.imag(u) != 0))
    hdtype = np.complex128 if cplx else np.float64
    if not cplx:
        h1, u = np.real(h1), np.real(u)
    out_complex = cplx or phase_seed is not None
    odtype = np.complex128 if out_complex else np.float64

    # enumerate Fock states, group by label
    if n_window is None:
        states = np.arange(1 << n, dtype=np.int64)
    else:
        lst = []
        for N in range(n_window[0], n_window[1] + 1):
            for sub in combinations(range(n), N):
                lst.append(sum(1 << f for f in sub))
        states = np.array(sorted(lst), dtype=np.int64)
    occ = ((states[:, None] >> np.arange(n)[None, :]) & 1)
    lab = occ @ flavour_qn
    labels = sorted(set(map(tuple, lab.tolist())))
    index_of = {l: i for i, l in enumerate(labels)}
    sec_of_state = np.array([index_of[tuple(x)] for x in lab.tolist()])
    sector_states = [states[sec_of_state == q] for q in range(len(labels))]
    dims = np.array([len(s) for s in sector_states], dtype=np.int32)

    # H_loc once over the whole enumerated space, then cut into sector blocks and diagonalise each
    hr, hc, hv = _hamiltonian_coo(states, h1, u)
    sec_r, sec_c = sec_of_state[hr], sec_of_state[hc]
    assert np.all(sec_r == sec_c), "H_loc does not conserve the sector labels"
    local = np.zeros(len(states), dtype=np.int64)
    for q in range(len(labels)):
        local[sec_of_state == q] = np.arange(dims[q])
    o = np.argsort(sec_r, kind="stable")
    hr, hc, hv, sec_r = hr[o], hc[o], hv[o], sec_r[o]
    bounds = np.searchsorted(sec_r, np.arange(len(labels) + 1))
    energies, vecs = [], []
    rng = Stream(phase_seed) if phase_seed is not None else None
    for q, st in enumerate(sector_states):
        H = np.zeros((int(dims[q]), int(dims[q])), dtype=hdtype)
        sl = slice(bounds[q], bounds[q + 1])
        np.add.at(H, (local[hr[sl]], local[hc[sl]]), hv[sl])
        assert np.allclose(H, H.conj().T, atol=1e-10), "H_loc sector not Hermitian"
        e, v = np.linalg.eigh(H)
        if rng is not None:
            ph = np.exp(2j * np.pi * rng.uniforms(len(e)))
            v = v.astype(np.complex128) * ph[None, :]
        energies.append(e)
        vecs.append(v.astype(odtype))

    # operator blocks: c^dag_f from q -> q' (and its adjoint c_f from q' -> q)
    specs = []
    for f in range(n):
        for q, l in enumerate(labels):
            tl = tuple(int(a + b) for a, b in zip(l, flavour_qn[f]))
            if tl in index_of:
                specs.append((2 * f + 1, q, index_of[tl]))
                specs.append((2 * f, index_of[tl], q))
    specs.sort()
    n_blocks = len(specs)
    blk_symbol = np.array([s[0] for s in specs], dtype=np.int32)
    blk_src = np.array([s[1] for s in specs], dtype=np.int32)
    blk_dst = np.array([s[2] for s in specs], dtype=np.int32)
    sizes = dims[blk_src].astype(np.int64) * dims[blk_dst].astype(np.int64)
    blk_offset = np.concatenate([[0], np.cumsum(sizes)[:-1]]).astype(np.int64) if n_blocks else np.zeros(0, np.int64)
    blk_data = np.zeros(int(sizes.sum()), dtype=odtype)
    where = {(s[0], s[1]): b for b, s in enumerate(specs)}

    def view(b):
        m, k = int(dims[blk_dst[b]]), int(dims[blk_src[b]])
        o = int(blk_offset[b])
        return blk_data[o:o + m * k].reshape((m, k), order="F")

    for f in range(n):
        for q, l in enumerate(labels):
            b = where.get((2 * f + 1, q))
            if b is None:
                continue
            t = int(blk_dst[b])
            src = sector_states[q]
            emp = np.nonzero(((src >> f) & 1) == 0)[0]
            G = np.zeros((int(dims[t]), int(dims[q])), dtype=odtype)
            if emp.size:
                new = src[emp] | (1 << f)
                sign = 1 - 2 * (_popcount(src[emp] & ((1 << f) - 1)) & 1)
                ts = sector_states[t]
                order = np.argsort(ts)
                pos = order[np.searchsorted(ts[order], new)]
                assert np.all(ts[pos] == new)
                G[pos, :] = sign[:, None] * vecs[q][emp, :]
            Fm = vecs[t].conj().T @ G
            view(b)[:, :] = Fm
            view(where[(2 * f, t)])[:, :] = Fm.conj().T

    return Impurity(name=name, n_flavours=n, beta=float(beta), labels=labels, dims=dims,
                    energy=np.concatenate(energies), is_complex=out_complex,
                    blk_symbol=blk_symbol, blk_src=blk_src, blk_dst=blk_dst, blk_offset=blk_offset,
                    blk_data=blk_data, flavour_qn=flavour_qn, n_window=n_window,
                    h1=np.array(h1), u=np.array(u), sector_states=sector_states,
                    eigvecs=vecs if keep_eigvecs else [])


# --------------------------------------------------------------------------- BASELINE.json configs
def _kanamori(n_orb, U, J, mu):
    u = spin_orbital_tensor(kanamori_orbital_tensor(n_orb, U, J))
    h1 = -mu * np.eye(2 * n_orb)
    qn = [(1, -1)] * n_orb + [(1, +1)] * n_orb   # (N, 2 S_z); flavour order Eq. A.4: down block then up block
    return h1, u, qn


def symmetric_mu(u: np.ndarray) -> float:
    """mu = 1/2 sum_j (U_ijji - U_ijij): makes the spectrum N <-> n-N symmetric (reading A16)."""
    n = u.shape[0]
    v = [0.5 * sum(u[i, j, j, i] - u[i, j, i, j] for j in range(n)) for i in range(n)]
    assert np.allclose(v, v[0])
    return float(np.real(v[0]))


def f_shell_coupled(F, lam):
    """f-shell Slater-Condon tensor and spin-orbit term in the coupled basis (Eq. A.3/A.6; reading A15)."""
    l = 3
    u = spin_orbital_tensor(slater_orbital_tensor(l, F))
    T = clebsch_gordan_l_half(l)
    uc = rotate_tensor(u, T)
    uc[np.abs(uc) < 1e-14] = 0.0
    soc = np.array([-lam * (l + 1) / 2.0] * (2 * l) + [lam * l / 2.0] * (2 * l + 2))
    twomj = list(range(-(2 * l - 1), 2 * l, 2)) + list(range(-(2 * l + 1), 2 * l + 2, 2))
    return uc, soc, twomj


def build_config_impurity(cfg: int, keep_eigvecs: bool = True) -> Impurity:
    """The five impurities of BASELINE.json `configs` (1-based), per SURVEY.md §8(d) D1."""
    if cfg == 1:
        h1, u, qn = _kanamori(2, 4.0, 0.8, 2.0)
        return build_impurity("cfg1-kanamori2", h1, u, qn, beta=10.0, keep_eigvecs=keep_eigvecs)
    if cfg == 2:
        h1, u, qn = _kanamori(3, 3.0, 0.5, 5.0)
        return build_impurity("cfg2-kanamori3", h1, u, qn, beta=50.0, keep_eigvecs=keep_eigvecs)
    if cfg == 3:
        u = spin_orbital_tensor(slater_orbital_tensor(2, [6.0, 8.4, 5.3]))
        u[np.abs(u) < 1e-14] = 0.0
        h1 = -symmetric_mu(u) * np.eye(10)
        return build_impurity("cfg3-dshell-N", h1, u, [(1,)] * 10, beta=40.0, keep_eigvecs=keep_eigvecs)
    if cfg in (4, 5):
        uc, soc, twomj = f_shell_coupled([4.5, 6.1, 4.1, 3.0], 0.3)
        mu = 4.5 * (5 - 0.5) - 0.512 * (5 - 1) / 2.0   # reading A16: nominal double counting, N0 = 5
        beta = 1.0 / (K_B_EV * 600.0)
        h1 = np.diag(soc - mu).astype(np.complex128 if cfg == 5 else np.float64)
        if cfg == 4:
            qn = [(1, m) for m in twomj]
            return build_impurity("cfg4-fshell-NJz", h1, uc, qn, beta=beta, n_window=(4, 6),
                                  phase_seed=4, keep_eigvecs=keep_eigvecs)
        rng = Stream(5)
        cf = np.zeros((14, 14), dtype=np.complex128)
        for i in range(14):
            for j in range(i, 14):
                if i == j:
                    cf[i, i] = 0.05 * rng.normal()
                else:
                    cf[i, j] = 0.05 * (rng.normal() + 1j * rng.normal())
                    cf[j, i] = np.conj(cf[i, j])
        return build_impurity("cfg5-fshell-CF", h1 + cf, uc, [(1,)] * 14, beta=beta, n_window=(4, 6),
                              keep_eigvecs=keep_eigvecs)
    raise ValueError(f"no such config {cfg}")
