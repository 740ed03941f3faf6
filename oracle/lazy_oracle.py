"""ORACLE — test infrastructure only.  Plain CPU (numpy, fp64) statement of the INCREMENTAL, LAZY local trace
("store these subproducts in a data structure, e.g., a balanced binary tree or a skip-list ...
requiring O[log(k)] matrix multiplications rather than O(k)", PAPER.md:542-548 lazy trace: bounds from submultiplicative
norms decide a Metropolis move whose random number was drawn first).

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline leg may import this.  It shares no code with the CUDA
path and imports nothing from it; of `oracle/trace_oracle.py` it uses the impurity view and the scaled-number helpers.

Readings (the paper defers the data structure to its Ref. [9], which is not available; readings F1-F4):

  F1  The stored sub-products live in a balanced binary tree over a FIXED dyadic partition of the time axis: [0, beta) is cut
      into 2**depth equal bins; node (l, i) covers [i beta / 2**l, (i + 1) beta / 2**l) and stores, for every sector q that
      survives it, the evolution operator across its interval,
          U_node(q) = P(b - tau_n) F_n P(tau_n - tau_{n-1}) ... F_1 P(tau_1 - a)            (a, b the interval's ends),
      its target sector, and its Frobenius norm.  A parent is the plain product right * left (no propagator at the seam,
      because every node runs from boundary to boundary).  The root is the chain of Eq. 65 for every start
      sector; w_loc = sum over q0 with target(q0) = q0 of Tr U_root(q0).  This is a skip-list whose level-l towers stand at the
      multiples of beta / 2**l: deterministic, so that many chains share one launch shape on the GPU.
  F2  Inserting or removing operators dirties the leaves that contain their times and the ancestors of those leaves: at most
      2 (depth + 1) nodes for a pair, i.e. O(log k) products when 2**depth ~ k (operators are uniform in time on average).
  F3  Bound of a proposed configuration WITHOUT multiplying the dirty ancestors: the time axis is covered by the dirty
      leaves (recomputed: a leaf holds O(1) operators) and the maximal clean subtrees between them; for start sector q0
          B(q0) = sqrt(r) * prod_{nodes of the cover} ||U_node(q at that node)||_F,   r = min of the sector dimensions at
      the cover's seams (|Tr M| <= sqrt(rank M) ||M||_F, rank <= every intermediate dimension, ||XY||_F <= ||X||_F ||Y||_F),
      rounded outward by BOUND_INFLATION (reading A9).
  F4  Decision ("the random number ... is drawn first, and this number must be between the lower and upper
      bounds"): the caller passes the threshold T on |w_new| (u |w_old| / the other factors of the acceptance ratio).
      Start sectors are taken in order of decreasing bound; after each exact t(q0), with S the sum so far and R the sum of
      the remaining bounds: |S| - R > T accepts, |S| + R <= T rejects, otherwise continue.  An accepted move is completed (all
      sectors) so that the new trace is known; a rejected one stops there.

Pins: tests/test_lazy_oracle.py (root = oracle.trace_oracle.trace_config of the edited configuration on random edit sequences;
products per edit <= 2 (depth + 1) per sector + leaf work; B(q0) >= |t(q0)|; decision = exact-trace decision for thresholds
swept through and around the exact value).
"""
from __future__ import annotations

import math

import numpy as np

from . import trace_oracle as T


class _Node:
    __slots__ = ("M", "e", "lg", "tgt", "nrm")

    def __init__(self, Q):
        self.M = [None] * Q        # matrix of sector q (dim[tgt] x dim[q]) or None if the string dies inside the node
        self.e = [0] * Q           # integer exponent: value = M * 2**e * 2**lg
        self.lg = [0.0] * Q        # real exponent -sum Delta Emin log2 e
        self.tgt = [-1] * Q
        self.nrm = [0.0] * Q       # ||M||_F (same scaling as M)


def _rescale(M):
    """M -> (M', k): M = M' * 2**k with max |component| of M' in [0.5, 1) (exact power of two); zero stays zero."""
    mx = float(np.max(np.maximum(np.abs(M.real), np.abs(M.imag)))) if np.iscomplexobj(M) else float(np.max(np.abs(M)))
    if mx == 0.0:
        return M, 0
    _, k = math.frexp(mx)
    return np.ldexp(M.real, -k) + 1j * np.ldexp(M.imag, -k) if np.iscomplexobj(M) else np.ldexp(M, -k), k


class LazyChain:
    """One Markov chain's stored sub-products.  `ops` is the current configuration as a time-sorted list of (tau, symbol)."""

    def __init__(self, desc, beta: float, depth: int):
        self.imp = T._imp(desc)
        self.beta = float(beta)
        self.depth = int(depth)
        self.nleaf = 1 << self.depth
        self.ops = []
        self.n_products = 0        # matrix products performed (pin: O(log k) per edit)
        self.nodes = {}
        self._build_all()

    # ------------------------------------------------------------------ structure
    def _leaf_of(self, tau: float) -> int:
        return min(self.nleaf - 1, int(tau / self.beta * self.nleaf))

    def _leaf_interval(self, i: int):
        return i * self.beta / self.nleaf, (i + 1) * self.beta / self.nleaf

    def _leaf_ops(self, ops, i: int):
        return [(t, a) for t, a in ops if self._leaf_of(t) == i]

    def _dtype(self):
        return np.complex128 if self.imp.is_complex else np.float64

    def _make_leaf(self, ops, i: int) -> _Node:
        """U_leaf(q) for every sector: propagate from the bin's left edge through its operators to its right edge."""
        imp = self.imp
        a, b = self._leaf_interval(i)
        mine = self._leaf_ops(ops, i)
        nd = _Node(imp.Q)
        for q0 in range(imp.Q):
            q = q0
            t_prev = a
            M = np.eye(int(imp.dims[q0]), dtype=self._dtype())
            e, lg, dead = 0, 0.0, False
            for t, al in mine:
                M, k = T._propagate(M, t - t_prev, imp.E[q], imp.Emin[q])
                e += k
                lg += -(t - t_prev) * imp.Emin[q] * T.LOG2E
                qn = int(imp.smap[al, q])
                if qn < 0:
                    dead = True
                    break
                M = imp.F[(al, q)] @ M
                self.n_products += 1
                q, t_prev = qn, t
            if dead:
                continue
            M, k = T._propagate(M, b - t_prev, imp.E[q], imp.Emin[q])
            e += k
            lg += -(b - t_prev) * imp.Emin[q] * T.LOG2E
            nd.M[q0], nd.e[q0], nd.lg[q0], nd.tgt[q0] = M, e, lg, q
            nd.nrm[q0] = float(np.linalg.norm(M))
        return nd

    def _combine(self, left: _Node, right: _Node) -> _Node:
        imp = self.imp
        nd = _Node(imp.Q)
        for q in range(imp.Q):
            m = left.tgt[q]
            if m < 0 or right.tgt[m] < 0:
                continue
            M, k = _rescale(right.M[m] @ left.M[q])
            self.n_products += 1
            nd.M[q], nd.e[q], nd.lg[q], nd.tgt[q] = M, left.e[q] + right.e[m] + k, left.lg[q] + right.lg[m], right.tgt[m]
            nd.nrm[q] = float(np.linalg.norm(M))
        return nd

    def _build_all(self):
        for i in range(self.nleaf):
            self.nodes[(self.depth, i)] = self._make_leaf(self.ops, i)
        for l in range(self.depth - 1, -1, -1):
            for i in range(1 << l):
                self.nodes[(l, i)] = self._combine(self.nodes[(l + 1, 2 * i)], self.nodes[(l + 1, 2 * i + 1)])

    # ------------------------------------------------------------------ values
    def _sector_terms(self, root: _Node):
        terms = {}
        for q0 in range(self.imp.Q):
            if root.tgt[q0] < 0:
                continue
            if root.tgt[q0] != q0:
                terms[q0] = (0j, 0)
                continue
            d = np.diagonal(root.M[q0])
            z = complex(math.fsum(d.real), math.fsum(d.imag))
            terms[q0] = T._apply_lg(z, root.e[q0], root.lg[q0])
        return terms

    def trace(self):
        """(mant, exp2, per-sector dict q0 -> (mant, exp2)) of the current configuration from the stored root."""
        terms = self._sector_terms(self.nodes[(0, 0)])
        w, e = T._sum_scaled(list(terms.values()))
        return w, e, terms

    # ------------------------------------------------------------------ proposals
    def _edited(self, insert, remove):
        ops = [o for o in self.ops]
        for o in remove:
            ops.remove(o)
        ops = sorted(ops + list(insert), key=lambda o: o[0])
        return ops

    def propose(self, insert=(), remove=(), log2_threshold: float = -math.inf):
        """Lazy evaluation of the configuration with `insert` added and `remove` taken out (lists of (tau, symbol)).
        `log2_threshold` = log2 of T (reading F4).  Returns a dict: accept, decided_by ("bound" / "partial" / "full"),
        n_sectors_evaluated, bound (mant, exp2), sector_bound {q0: (mant, exp2)}, and -- when accepted -- trace (mant, exp2).
        The chain itself is not modified; `commit(result)` applies an accepted proposal."""
        imp = self.imp
        ops = self._edited(list(insert), list(remove))
        dirty_leaves = sorted({self._leaf_of(t) for t, _ in list(insert) + list(remove)})
        shadow = {(self.depth, i): self._make_leaf(ops, i) for i in dirty_leaves}
        dirty = set(shadow)
        for i in dirty_leaves:
            for l in range(self.depth - 1, -1, -1):
                dirty.add((l, i >> (self.depth - l)))

        def node(key):
            return shadow[key] if key in shadow else self.nodes[key]

        # ---- bounds from the cover: dirty leaves + maximal clean subtrees, left to right (reading F3)
        cover = []

        def walk(l, i):
            if (l, i) not in dirty or l == self.depth:
                cover.append((l, i))
            else:
                walk(l + 1, 2 * i)
                walk(l + 1, 2 * i + 1)
        walk(0, 0)
        sector_bound = {}
        for q0 in range(imp.Q):
            q, val, e, lg, dmin, alive = q0, 1.0, 0, 0.0, int(imp.dims[q0]), True
            for key in cover:
                nd = node(key)
                if nd.tgt[q] < 0:
                    alive = False
                    break
                val *= nd.nrm[q]
                e += nd.e[q]
                lg += nd.lg[q]
                q = nd.tgt[q]
                dmin = min(dmin, int(imp.dims[q]))
                if val != 0.0:
                    m, k = math.frexp(val)
                    val, e = m, e + k
            if alive:
                z, ez = T._apply_lg(complex(math.sqrt(dmin) * val * T.BOUND_INFLATION, 0.0), e, lg)
                sector_bound[q0] = (z.real, ez)
        btot, bexp = T._sum_scaled([(complex(m, 0.0), e) for m, e in sector_bound.values()])
        out = dict(sector_bound=sector_bound, bound=(btot.real, bexp), ops=ops, shadow=shadow, dirty=dirty, n_sectors_evaluated=0, trace=None)

        def log2_of(m, e):
            return -math.inf if m == 0 else math.log2(abs(m)) + e

        if log2_of(btot.real, bexp) <= log2_threshold:
            out.update(accept=False, decided_by="bound")
            return out

        # ---- exact sectors in order of decreasing bound (reading F4); a sector's value needs its path of dirty ancestors
        def root_entry(q0):
            """(M, e, lg, tgt) of the root for start sector q0, multiplying only what this sector needs."""
            def ent(l, i, q):
                key = (l, i)
                if key not in dirty or l == self.depth:
                    nd = node(key)
                    return (nd.M[q], nd.e[q], nd.lg[q], nd.tgt[q]) if nd.tgt[q] >= 0 else None
                cache = shadow.setdefault(key, _Node(imp.Q))
                if cache.tgt[q] >= 0:
                    return cache.M[q], cache.e[q], cache.lg[q], cache.tgt[q]
                le = ent(l + 1, 2 * i, q)
                if le is None:
                    return None
                re_ = ent(l + 1, 2 * i + 1, le[3])
                if re_ is None:
                    return None
                M, k = _rescale(re_[0] @ le[0])
                self.n_products += 1
                cache.M[q], cache.e[q], cache.lg[q], cache.tgt[q] = M, le[1] + re_[1] + k, le[2] + re_[2], re_[3]
                cache.nrm[q] = float(np.linalg.norm(M))
                return cache.M[q], cache.e[q], cache.lg[q], cache.tgt[q]
            return ent(0, 0, q0)

        order = sorted(sector_bound, key=lambda q0: -log2_of(*sector_bound[q0]))
        terms, decided, accept = [], None, None
        for n_done, q0 in enumerate(order):
            r = root_entry(q0)
            if r is not None and r[3] == q0:
                d = np.diagonal(r[0])
                terms.append(T._apply_lg(complex(math.fsum(d.real), math.fsum(d.imag)), r[1], r[2]))
            out["n_sectors_evaluated"] = n_done + 1
            if decided is None:
                S, eS = T._sum_scaled(terms)
                rest = [(complex(sector_bound[p][0], 0.0), sector_bound[p][1]) for p in order[n_done + 1:]]
                R, eR = T._sum_scaled(rest)
                absS = abs(S)
                lo = _scaled_sub(absS, eS, R.real, eR)          # |S| - R  (may be negative)
                hi = T._sum_scaled([(complex(absS, 0.0), eS), (R, eR)])
                if lo[0] > 0 and log2_of(*lo) > log2_threshold:
                    decided, accept = ("partial" if rest else "full"), True
                elif log2_of(hi[0].real, hi[1]) <= log2_threshold:
                    decided, accept = ("partial" if rest else "full"), False
                    break
        if decided is None:      # no sector left and still inside the bracket cannot happen: R = 0 makes lo = hi = |S|
            decided, accept = "full", False
        out.update(accept=accept, decided_by=decided)
        if accept:
            w, e = T._sum_scaled(terms)
            out["trace"] = (w, e)
        return out

    def commit(self, result):
        """Apply an ACCEPTED proposal: its operators become the configuration, its shadow nodes the stored sub-products
        (entries of dirty ancestors that the lazy evaluation never needed are completed here)."""
        assert result["accept"]
        self.ops = result["ops"]
        shadow, dirty = result["shadow"], result["dirty"]
        for key in dirty:
            if key[0] == self.depth:
                self.nodes[key] = shadow[key]
        for l in range(self.depth - 1, -1, -1):
            for i in range(1 << l):
                if (l, i) in dirty:
                    self.nodes[(l, i)] = self._combine_reusing(self.nodes[(l + 1, 2 * i)], self.nodes[(l + 1, 2 * i + 1)],
                                                               shadow.get((l, i), _Node(self.imp.Q)))

    def _combine_reusing(self, left, right, cache):
        imp = self.imp
        nd = _Node(imp.Q)
        for q in range(imp.Q):
            m = left.tgt[q]
            if m < 0 or right.tgt[m] < 0:
                continue
            if cache.tgt[q] >= 0:
                nd.M[q], nd.e[q], nd.lg[q], nd.tgt[q], nd.nrm[q] = cache.M[q], cache.e[q], cache.lg[q], cache.tgt[q], cache.nrm[q]
                continue
            M, k = _rescale(right.M[m] @ left.M[q])
            self.n_products += 1
            nd.M[q], nd.e[q], nd.lg[q], nd.tgt[q] = M, left.e[q] + right.e[m] + k, left.lg[q] + right.lg[m], right.tgt[m]
            nd.nrm[q] = float(np.linalg.norm(M))
        return nd


def _scaled_sub(a: float, ea: int, b: float, eb: int):
    """a 2**ea - b 2**eb for a, b >= 0 as (mantissa, exponent); the mantissa carries the sign."""
    if b == 0:
        return a, ea
    if a == 0:
        return -b, eb
    e = max(ea, eb)
    v = math.ldexp(a, max(ea - e, -1100)) - math.ldexp(b, max(eb - e, -1100))
    return v, e
