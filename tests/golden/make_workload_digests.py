"""Writes tests/golden/workload_digests.txt: the frozen fingerprint of every seeded workload (reading G22:
the generator's choices "must not drift between runs").

    python tests/golden/make_workload_digests.py

Calls only `workloads/` (input generation; none of the method's arithmetic, neither oracle/ nor the CUDA path).
One line per generated array: config, key, dtype, shape, three checksums (sum, sum of squares, sum weighted by
cos(0.37 i + 0.11) over the flat index i -- sensitive to order and to any single seed / recipe change), and the
SHA-256 of its bytes.  tests/test_oracle_pins.py::test_workload_digests_match_the_committed_file asserts the
checksums (to 1e-9: libm / SIMD builds may differ in the last bit of exp, tanh, cos, the FFT) and reports a SHA
mismatch without failing.
"""
from __future__ import annotations

import hashlib
import sys
from pathlib import Path

import numpy as np

HERE = Path(__file__).resolve().parent
sys.path.insert(0, str(HERE.parent.parent))

CONFIGS = ["tiny", "ati", "hetero", "large", "sweep20", "sweep22", "sweep24", "sweep26"]


def build(name):
    from workloads import make_workload, make_sweep_point
    if name.startswith("sweep"):
        return make_sweep_point(log2_facets=int(name[5:]))
    return make_workload(name)


def fingerprint(w):
    """[(key, dtype, shape, s1, s2, s3, sha)] over every array / scalar of the three descriptor groups."""
    rows = []
    for gname, group in (("instrument", w.instrument), ("geometry", w.geometry), ("scene", w.scene)):
        for key in sorted(group):
            v = group[key]
            if v is None:
                rows.append((f"{gname}.{key}", "none", "()", 0.0, 0.0, 0.0, "-"))
                continue
            a = np.ascontiguousarray(np.asarray(v))
            sha = hashlib.sha256(str(a.dtype).encode() + str(a.shape).encode() + a.tobytes()).hexdigest()
            f = a.astype(np.float64).ravel()
            wgt = np.cos(0.37 * np.arange(f.size, dtype=np.float64) + 0.11)
            rows.append((f"{gname}.{key}", str(a.dtype), str(tuple(a.shape)).replace(" ", ""),
                         float(f.sum()), float((f * f).sum()), float((f * wgt).sum()), sha))
    return rows


def main():
    lines = ["# config key dtype shape sum sum_sq sum_cos_weighted sha256   (tests/golden/make_workload_digests.py; workloads/ only; G22)"]
    for name in CONFIGS:
        for key, dt, shape, s1, s2, s3, sha in fingerprint(build(name)):
            lines.append(f"{name} {key} {dt} {shape} {s1:.17e} {s2:.17e} {s3:.17e} {sha}")
    (HERE / "workload_digests.txt").write_text("\n".join(lines) + "\n")
    print("wrote", HERE / "workload_digests.txt", len(lines) - 1, "rows")


if __name__ == "__main__":
    main()
