"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds NO arithmetic of the calibration method (no coherency
prediction, no Jones corruption, no cost/gradient, no solver): it only draws
station layouts, uvw tracks, sky models, true Jones matrices and noise.
Both `oracle/` and `paper_1910_13908_b200/` consume its arrays; neither is
imported here.
"""
from .synth import (  # noqa: F401
    C0,
    CONFIGS,
    SEED_BASE,
    Problem,
    RowList,
    baseline_index,
    baseline_pairs,
    make_config,
    make_problem,
    make_rowlist,
    noise_rows,
)
