"""Helpers shared by the tests (comparison of scaled numbers)."""
import math


def rel_diff(m1: complex, e1: int, m2: complex, e2: int) -> float:
    """|v1 - v2| / |v2| for v = m * 2**e, computed at a common exponent (reading A5)."""
    m1, m2 = complex(m1), complex(m2)
    if m2 == 0:
        return 0.0 if m1 == 0 else math.inf
    d = e1 - e2
    if abs(d) > 200:
        return math.inf
    return abs(m1 * 2.0 ** d - m2) / abs(m2)


def scaled_ge(m1: float, e1: int, m2: float, e2: int) -> bool:
    """m1 * 2**e1 >= m2 * 2**e2 for non-negative mantissas."""
    if m2 == 0:
        return True
    if m1 == 0:
        return False
    d = e1 - e2
    if d > 200:
        return True
    if d < -200:
        return False
    return m1 * 2.0 ** d >= m2
