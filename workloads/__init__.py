"""Seeded synthetic workloads for the HEEPS/MARE raw-data generator hot path.

This package holds ONLY input generation (instrument / geometry / scene descriptor
arrays).  It contains none of the method's arithmetic (no delays, gains, phases or
sums), and it is the single thing shared by the CUDA path and the oracle: both
consume exactly the arrays produced here.

Recipes: SURVEY.md §8(d), BASELINE.json `configs`; restated in DESIGN.md §"Input recipe".
"""
from .generator import (  # noqa: F401
    C0,
    CONFIG_NAMES,
    MASTER_SEED,
    Workload,
    make_workload,
    make_sweep_point,
    add_wave_nodes,
    crop_rows,
    add_antenna_patterns,
    pm_spectrum,
    workload_digest,
)
