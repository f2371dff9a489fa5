"""fp64 CPU oracle of the HEEPS/MARE raw-data generator hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, `__graft_entry__.smoke()` and bench.py's `cpu_baseline` / `--impl reference`
legs may import this package.  It shares no code with `paper_2405_09938_b200/` and never
imports it.  The arithmetic lives in `heeps_oracle.c` (each step
citing PAPER.md); this file is argument marshalling over ctypes plus the parity metrics
(G19/G20) used by the tests.
"""
from .binding import (  # noqa: F401
    build_oracle,
    oracle_generate,
    oracle_facets,
    oracle_samples,
    oracle_speckle,
    oracle_philox,
    oracle_max_threads,
    rel_l2_per_vector,
    ati_phase,
    ati_phase_rms_error,
)
