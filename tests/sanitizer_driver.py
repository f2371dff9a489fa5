"""Small driver for compute-sanitizer: pushes a few tiny scenes through every kernel of the
library -- K1 (homogeneous, heterogeneous lattice), K2k (forced keyframe spacing 4, batches of 3, a stray-heavy wide
patch, tabulated patterns, AR(1) speckle), K2s, K2 / K3 / K4 (direct form), K3s (full and band transform), speckle.cu,
sim_debug_facets -- and checks each result against the oracle, so that a sanitizer run is also a parity run.

    compute-sanitizer --tool memcheck  --error-exitcode 1 python tests/sanitizer_driver.py      (likewise racecheck,
                                                                                                  initcheck, synccheck)
    HEEPS_SIM_LIBRARY=paper_2405_09938_b200/libheeps_sim_checked.so python tests/sanitizer_driver.py

The GPU pool this was developed on refuses compute-sanitizer (profiles/r2_sanitizer.md); the second form -- the library
built with device-side bounds checks that trap, `python -m paper_2405_09938_b200.build --checked` -- is what
tests/test_gpu_parity.py::test_checked_build_runs_the_driver_clean runs.

Not collected by pytest (no test_ prefix); the summaries are kept under profiles/.
"""
from __future__ import annotations

import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))
sys.path.insert(0, str(ROOT / "tests"))


def hetero_small(nx, ny, n_pulses):
    from workloads import make_workload
    w = make_workload("hetero", n_pulses=n_pulses)
    sc = w.scene
    j0, i0 = 1024 - ny // 2, 1024 - nx // 2
    for k in ("sigma0_lin", "current_mps", "xi"):
        sc[k] = np.ascontiguousarray(sc[k][j0:j0 + ny, i0:i0 + nx])
    sc["nx"], sc["ny"] = nx, ny
    return w


def main():
    import torch
    from oracle import oracle_generate, rel_l2_per_vector
    from paper_2405_09938_b200 import LIBRARY_PATH, Simulator
    from workloads import add_antenna_patterns, make_workload
    print("library:", LIBRARY_PATH, flush=True)

    cases = []
    tiny = make_workload("tiny", n_pulses=9)
    cases.append(("tiny direct", tiny, dict(accumulate_mode="direct", pulses_per_batch=4)))
    cases.append(("tiny spectral K2s", tiny, dict(accumulate_mode="spectral", geometry_keyframe=1)))
    cases.append(("tiny spectral K2k H=4 batch=3", tiny, dict(accumulate_mode="spectral", kinematics_keyframe=4, pulses_per_batch=3)))
    hs = hetero_small(96, 64, 11)
    hs.scene["choppy"] = 1
    cases.append(("hetero_small spectral K2k H=4 batch=3", hs, dict(accumulate_mode="spectral", kinematics_keyframe=4, pulses_per_batch=3)))
    cases.append(("hetero_small spectral K2k band off", hs, dict(accumulate_mode="spectral", kinematics_keyframe=4, fft_band=1)))
    cases.append(("hetero_small spectral K2s", hs, dict(accumulate_mode="spectral", geometry_keyframe=1)))
    cases.append(("hetero_small direct", hs, dict(accumulate_mode="direct")))
    wide = make_workload("tiny", n_pulses=12)
    wide.scene["spacing_m"] = 220.0                      # culling, window-clipping, fast-drifting tiles: strays, re-sorts
    wide.instrument["channel_offset_m"] = np.array([-1.5, 0.0, 1.5])
    cases.append(("wide patch spectral K2k H=4", wide, dict(accumulate_mode="spectral", kinematics_keyframe=4)))
    cases.append(("wide patch spectral K2k auto", wide, dict(accumulate_mode="spectral")))
    pat = make_workload("tiny", n_pulses=9)
    pat.scene["spacing_m"] = 120.0
    pat.instrument["channel_offset_m"] = np.array([-1.5, 0.0, 1.5])
    pat = add_antenna_patterns(pat, nu=2049, nv=257, steer_rate_deg_s=3.0)
    pat.instrument["cull_two_way_db"] = -10.0
    cases.append(("tables spectral K2k H=4", pat, dict(accumulate_mode="spectral", kinematics_keyframe=4)))
    cases.append(("tables direct", pat, dict(accumulate_mode="direct")))
    ar1 = make_workload("tiny", n_pulses=9)
    ar1.scene["speckle_tau_s"], ar1.scene["speckle_doppler_hz"], ar1.scene["seed"] = 4e-3, 35.0, 77
    cases.append(("ar1 speckle spectral K2k batch=4", ar1, dict(accumulate_mode="spectral", pulses_per_batch=4)))
    cases.append(("ar1 speckle direct", ar1, dict(accumulate_mode="direct")))

    worst, failed = 0.0, 0
    for name, w, opts in cases:
        ref = oracle_generate(w)
        with Simulator(w, 0, **opts) as sim:
            got = sim.generate().cpu().numpy()
            part = sim.generate(2, 7).cpu().numpy()
            host = sim.generate_host().numpy()
            sim.debug_facets(w.n_pulses - 1)
            torch.cuda.synchronize()
        for what, g, r in (("full", got, ref), ("range", part, ref[:, 2:7]), ("host", host, ref)):
            err = float(rel_l2_per_vector(g, r).max())
            worst = max(worst, err)
            print(f"{name:45s} {what:6s} worst rel-L2 {err:.2e}", flush=True)
            if not err <= 1e-4:
                print("PARITY FAILED", flush=True)
                failed += 1
    if failed:
        print(f"sanitizer driver: {failed} FAILED comparisons")
        return 2
    print(f"sanitizer driver ok: {len(cases)} cases, worst rel-L2 {worst:.2e}")
    return 0


if __name__ == "__main__":
    sys.exit(main())
