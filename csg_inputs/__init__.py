"""Seeded synthetic inputs for the Benincasa-Dowker action hot path.

This package serves BOTH the oracle-side tests and the CUDA-side tests/bench and therefore holds none of
the method's arithmetic (no interval counts, no histogram, no action): only the seeded sprinkling, the
time sort, the relation test and the packed-matrix layout.  Recipe: DESIGN.md "Input recipe" (A17).
It imports neither ``oracle`` nor ``paper_1709_03013_b200``.
"""
from .generate import (  # noqa: F401
    CONFIGS,
    make_config,
    build,
    stride_words,
    sprinkle,
    relations_from_coords,
    make_causet,
    sprinkle_de_sitter,
    relations_de_sitter,
    make_de_sitter,
    pack_dense,
    bits_hash,
    random_poset_bits,
)
