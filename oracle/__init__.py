"""ORACLE package -- test infrastructure only.

Plain CPU restatement of the paper's hot path (PAPER.md:395 naive action algorithm; Eq. 4 / Eq. 5;
Algorithm 5; dense linking; 2D orders from coordinates).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports ``paper_1709_03013_b200``.
"""
from .oracle import (  # noqa: F401
    build,
    expand,
    counts_plain,
    counts_from_bits,
    pair_interval,
    action_local,
    f2,
    action_smeared_2d,
    f4,
    action_smeared_4d,
    alg5_counts,
    alg5_counts_rows,
    alg5_threads,
    dominance2d_counts,
    dominance2d_counts_rows,
    dominance2d_relations,
    link,
    GEOM_MINKOWSKI_2D,
    GEOM_MINKOWSKI_4D,
    GEOM_DESITTER_2D,
)
