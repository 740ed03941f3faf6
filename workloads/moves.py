"""Seeded Monte-Carlo-like MOVES for the chain-set calls (inputs only: none of the method's arithmetic).

A move is the pair update of CT-HYB: insert c^dag_f and c_f of one flavour at two uniform times, or remove
two operators of one flavour that are adjacent in that flavour's own time-ordered sequence, so that the flavour keeps
alternating.  Whether the N window of configs 4-5 survives is for the trace to decide (a vanishing proposal is rejected).
"""
from __future__ import annotations


def random_pair_move(rng, n_flavours: int, beta: float, ops, p_remove: float = 0.4):
    """ops: the chain's current configuration as a list of (tau, symbol), symbol = 2 flavour + (1 if creation).
    Returns (insert list, remove list)."""
    f = rng.integer(n_flavours)
    mine = sorted(o for o in ops if o[1] // 2 == f)
    if len(mine) >= 2 and rng.uniform() < p_remove:
        i = rng.integer(len(mine))
        return [], [mine[i], mine[(i + 1) % len(mine)]]
    t1, t2 = sorted((beta * rng.uniform(), beta * rng.uniform()))
    before = [o for o in mine if o[0] < t1] or mine
    first = (1 - (before[-1][1] & 1)) if before else rng.integer(2)
    return [(t1, 2 * f + first), (t2, 2 * f + 1 - first)], []


def apply_move(ops, insert, remove):
    out = list(ops)
    for o in remove:
        out.remove(o)
    return sorted(out + list(insert), key=lambda o: o[0])
