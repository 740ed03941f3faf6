"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA path.

This package holds *inputs only*: impurity models (sector dimensions, eigenvalues,
operator blocks in the eigenbasis of H_loc) and Monte-Carlo-like configurations
(operator strings with times).  It contains none of the method's arithmetic — no
sector routing, no chain product, no trace, no norm bound — so that `oracle/` and
`paper_2010_08482_b200/` share nothing but what they are fed.

Recipe and readings: DESIGN.md §4 (inputs), SURVEY.md §8(d) D1–D2.
"""
from .impurity import Impurity, build_config_impurity, build_impurity  # noqa: F401
from .configs import Batch, make_batch, BASELINE_CONFIGS  # noqa: F401
from .moves import apply_move, random_pair_move  # noqa: F401
