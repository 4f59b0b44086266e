"""Seeded synthetic light-curve generators (inputs only; none of the BLS arithmetic lives here).

Used by the oracle-side tests, the GPU parity tests and bench.py alike.
"""
from .lightcurves import (  # noqa: F401
    CONFIGS,
    Batch,
    Grid,
    config,
    freq_grid,
    make_batch,
    make_curve,
    make_field,
    curve_lengths,
)
