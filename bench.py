#!/usr/bin/env python
"""Benchmark of the raw-data generator hot path (BASELINE.json metric: facet-echoes/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload large]

One *step* is one pass of the whole hot path (K1 kinematics, K2 geometry / gains / cull / range-slice moments,
K3 echo accumulation, K4 finalize) over every pulse and channel of the workload: `sim_generate(0, P)`.
At N = 1 the workload is the largest single-GPU configuration of BASELINE.json, configs[3] "Large footprint"
(4096 x 4096 facets, 3 channels, 2048 pulses, L = 1200, Ns = 8192); the other configurations (ATI, Heterogeneous,
three points of the stress sweep) are timed in the same run and carried under `other_configs`.  Under torchrun
each rank owns its own P-pulse slab of an N*P-pulse acquisition (weak scaling, no data-path collective;
SURVEY.md 8(e)).  The timed path is the library's default (SIM_ACCUMULATE_AUTO = the spectral form where it
applies); the direct form (every chirp replica generated sample by sample) is timed on the ATI configuration
and reported under `direct_form` with K3's roofline (on Large it takes 20 s per step).

The JSON line carries, beside the base contract: `roofline` (dominant kernel of the timed path against its pipe),
`cpu_baseline` (the fp64 oracle on the host cores, bounded sample: a slab of facet rows of one pulse of the same
scene), `e2e` (through sim_update_scene + sim_generate_host with pinned HOST buffers), `clocks`, `gpu_launches`.
`--impl reference` times the oracle as it stands (this tier's reference arm), each step a slab of facet rows of one
pulse of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import re
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "facet_echoes_per_s"
UNIT = "facet-echoes/s"

# FP32-pipe roofline of K3 (DESIGN.md 4/K3): the inner loop spends 4 FP32 lane-operations per facet-sample (one
# packed FFMA2 of the three-term recurrence + one packed FADD2 into the accumulators); 148 SMs x 128 FP32 lanes.
K3_FP32_OPS_PER_FACET_SAMPLE = 4.0
SM_COUNT, FP32_LANES_PER_SM = 148, 128
# FP32-pipe roofline of the moment kernels: SURVEY.md 8(d) counts 4 Kt FFMA + ~30 setup per
# facet-echo for the moment form; Kt = 8.
MOMENT_FP32_OPS_PER_FACET_ECHO = 4.0 * 8 + 30.0
# `roofline.traffic` comes from a committed `ncu --set full` capture of the dominant kernel (dram bytes read +
# written per launch), scaled to this run's launch by the facet-echo count; the file is named in `traffic_source`.
TRAFFIC_PROFILE = {"moments": "profiles/r2_k2k_ncu_summary.txt", "accumulate": "profiles/r1_v3_k3_ncu_summary.txt"}

# oracle cost model for the bounded samples (measured: ~7e5 facet-echoes/s on the box's 16 cores at L = 1200)
ORACLE_FACET_SAMPLES_PER_S = 7.0e5 * 1200


def _peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        return json.loads(p.read_text()), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def _profile_traffic(kind, echoes_this_launch):
    """dram bytes (read + write) of the captured launch scaled to this run's launch, or (None, reason)."""
    path = ROOT / TRAFFIC_PROFILE[kind]
    if not path.exists():
        return None, f"{TRAFFIC_PROFILE[kind]} not present"
    txt = path.read_text()
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    tot = 0.0
    for name in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
        m = re.search(r"^" + re.escape(name) + r"\s+(\w+)\s+([0-9.eE+,-]+)\s*$", txt, re.M)
        if not m:
            return None, f"{name} not found in {TRAFFIC_PROFILE[kind]}"
        tot += float(m.group(2).replace(",", "")) * unit.get(m.group(1), 1.0)
    m = re.search(r"^# facet_echoes_per_launch:\s*([0-9.eE+]+)", txt, re.M)
    if not m:
        return None, f"no '# facet_echoes_per_launch' line in {TRAFFIC_PROFILE[kind]}"
    return tot * echoes_this_launch / float(m.group(1)), (
        f"{TRAFFIC_PROFILE[kind]} (ncu --set full, dram read + write of one launch of {float(m.group(1)):.4g} "
        f"facet-echoes, scaled by the facet-echo count of this run's launch)")


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML; nvidia-smi fallback)."""

    def __init__(self, index: int):
        self.index, self.samples, self.reasons = index, [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _loop(self):
        nv = self._nv
        names = {}
        if nv:
            for n in dir(nv):
                if n.startswith("nvmlClocksEventReason") or n.startswith("nvmlClocksThrottleReason"):
                    v = getattr(nv, n)
                    if isinstance(v, int) and v:
                        names.setdefault(v, n.replace("nvmlClocksEventReason", "").replace("nvmlClocksThrottleReason", ""))
        while not self._stop.is_set():
            try:
                if nv:
                    self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                    try:
                        mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                    except Exception:
                        mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                    for bit, name in names.items():
                        if mask & bit and bit & (bit - 1) == 0:
                            self.reasons.add(name)
                else:
                    import subprocess
                    out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=clocks.sm,clocks.max.sm",
                                          "--format=csv,noheader,nounits"], capture_output=True, text=True).stdout
                    a, b = out.strip().split(",")
                    self.samples.append(float(a)); self.max_mhz = float(b)
            except Exception:
                pass
            self._stop.wait(0.01)

    def __enter__(self):
        self._thread = threading.Thread(target=self._loop, daemon=True)
        self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        self._thread.join(timeout=2)

    def summary(self):
        import statistics
        s = sorted(self.samples)
        reasons = sorted(r for r in self.reasons if r not in ("None", "GpuIdle", "ApplicationsClocksSetting"))
        return {"sm_mhz": statistics.median(s) if s else None, "sm_max_mhz": self.max_mhz,
                "samples": len(s), "reasons": reasons}


_VARIANT = {"wave_node_spacing": 0.0, "speckle_tau": 0.0, "patterns": False}     # set from the command line (NEXT-1..3 modes)


def _workload(name, n_pulses=None, pulse_offset=0):
    w = _base_workload(name, n_pulses, pulse_offset)
    if _VARIANT["wave_node_spacing"] > 0:          # heterogeneous surface, uncorrelated phases per node
        from workloads import add_wave_nodes
        add_wave_nodes(w, _VARIANT["wave_node_spacing"])
    if _VARIANT["speckle_tau"] > 0:                # AR(1) intra-facet speckle (eq. (7), (10))
        w.scene["speckle_tau_s"], w.scene["speckle_doppler_hz"] = _VARIANT["speckle_tau"], 20.0
    if _VARIANT["patterns"]:                       # antenna patterns as complex u-v grids, azimuth steering
        from workloads import add_antenna_patterns
        add_antenna_patterns(w, nu=513, nv=129, steer_rate_deg_s=1.5)
    return w


def _base_workload(name, n_pulses=None, pulse_offset=0):
    """BASELINE.json configs by name, or one point of the stress sweep (configs[4], reading G23) as
    `sweep:f<log2 facets>:l<replica samples>:c<channels>`, e.g. sweep:f24:l1200:c3 (64 pulses by default)."""
    from workloads import make_workload, make_sweep_point
    if name.startswith("sweep:"):
        kv = {t[0]: int(t[1:]) for t in name.split(":")[1:]}
        return make_sweep_point(log2_facets=kv.get("f", 24), replica_samples=kv.get("l", 1200),
                                n_channels=kv.get("c", 3), n_pulses=n_pulses or 64)
    return make_workload(name, n_pulses=n_pulses, pulse_offset=pulse_offset)


def _config(w, name, world):
    """The workload as both arms state it (the same keys in the CUDA line and the reference line)."""
    F, C, P, Ns, L = w.n_facets, w.n_channels, w.n_pulses, w.n_samples, w.replica_samples
    maps = sum(int(w.scene[k].nbytes) for k in ("xi", "sigma0_lin", "current_mps") if w.scene.get(k) is not None)
    return {"workload": name, "facets": F, "channels": C, "pulses": P, "replica_samples": L, "n_samples": Ns,
            "wave_components": int(w.scene["n_waves"]), "parallelism": f"pulse-slab x{world}",
            "wave_node_spacing_m": _VARIANT["wave_node_spacing"], "speckle_tau_s": _VARIANT["speckle_tau"],
            "tabulated_patterns": _VARIANT["patterns"],
            "l2": (f"no flush: every step re-reads {maps / 1e6:.0f} MB of facet maps and {16 * F / 1e6:.0f} MB of keyframe "
                   f"surface rows per keyframe interval, zeroes and scatters into {C * P * 8 * (Ns + L) * 8 / 1e6:.0f} MB of "
                   f"range-slice moment rows and writes {C * P * Ns * 8 / 1e6:.0f} MB of output -- larger than the 126 MB L2")}


def _oracle_sample(w, pulses):
    from oracle import oracle_generate, oracle_max_threads
    t = time.perf_counter()
    oracle_generate(w, pulses)
    dt = time.perf_counter() - t
    return dt, oracle_max_threads()


def _row_slab(w, seconds):
    """A centred slab of facet rows of the scene worth about `seconds` of oracle time for one pulse (all channels);
    the whole scene when that is cheaper.  Returns (cropped workload, j0, j1)."""
    from workloads import crop_rows
    nx, ny = int(w.scene["nx"]), int(w.scene["ny"])
    per_row = nx * w.n_channels * w.replica_samples / ORACLE_FACET_SAMPLES_PER_S
    rows = int(max(1, min(ny, round(seconds / per_row))))
    if rows >= ny or w.scene.get("wave_nodes") is not None:
        return w, 0, ny
    j0 = (ny - rows) // 2
    return crop_rows(w, j0, j0 + rows), j0, j0 + rows


def run_reference(args):
    """This tier's reference arm: the fp64 oracle on the host cores; each step evaluates one pulse (all channels) of a
    centred slab of facet rows of the same workload (about 4 s of oracle time), a different pulse every step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = _workload(args.workload, args.pulses)
    F, C, P = w.n_facets, w.n_channels, w.n_pulses
    ws, j0, j1 = _row_slab(w, 4.0)
    Fs = ws.n_facets
    for _ in range(min(args.warmup, 2)):
        _oracle_sample(ws, [0])
    t_total, cores = 0.0, 1
    for k in range(args.steps):
        dt, cores = _oracle_sample(ws, [(k * 37) % P])
        t_total += dt
    value = Fs * C * args.steps / t_total
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config(w, args.workload, int(os.environ.get("WORLD_SIZE", "1"))),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"per step: facet rows [{j0}, {j1}) of {int(w.scene['ny'])} x all {int(w.scene['nx'])} columns x "
                                   f"{C} channels of one pulse of '{args.workload}' ({Fs * C} facet-echoes); {args.steps} steps, "
                                   f"pulse (37 k) mod {P} at step k"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def _time_steps(sim, out, P, steps, warmup, stream, barrier, torch, clocks_index=None):
    """W warm-ups, then K steps of sim_generate(0, P) between CUDA events on the launching stream."""
    sim.set_profiling(True)
    for _ in range(warmup):
        sim.generate(0, P, out=out)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(clocks_index) if clocks_index is not None else None
    if sampler:
        sampler.__enter__()
    barrier()
    t_wall = time.perf_counter()
    ev0.record(stream)
    for _ in range(steps):
        sim.generate(0, P, out=out)
    ev1.record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall
    if sampler:
        sampler.__exit__()
    kms = sim.kernel_ms()            # per-kernel totals of the LAST timed step (events on this stream)
    stats = sim.stats()
    stats["n_facets_x_channels"] = sim.n_facets * sim.n_channels      # pulses of the call = nominal / this
    sim.set_profiling(False)
    return ev0.elapsed_time(ev1), t_wall, kms, stats, (sampler.summary() if sampler else None)


def _n_batches(stats):
    pulses = int(stats["facet_echoes_nominal"] // max(1, stats["n_facets_x_channels"]))
    return max(1, -(-pulses // max(1, stats["pulses_per_batch"])))


def _roofline_direct(kms, stats, sm_max, pipes):
    """K3 (accumulate_kernel) against the FP32 pipe: 4 lane-ops per facet-sample (DESIGN.md 4/K3)."""
    n_batches = _n_batches(stats)
    launch_ms = kms["accumulate"] / n_batches
    fs_per_launch = stats["facet_samples"] / n_batches
    achieved = fs_per_launch / (launch_ms * 1e-3) / 1e9
    peak = SM_COUNT * FP32_LANES_PER_SM * sm_max * 1e6 / K3_FP32_OPS_PER_FACET_SAMPLE / 1e9
    pipe_peak = pipes["mix_f32x2_lane_per_s"] / K3_FP32_OPS_PER_FACET_SAMPLE / 1e9
    traffic, src = _profile_traffic("accumulate", stats["facet_echoes_kept"] / n_batches)
    return {
        "bound": "alu", "kernel": "accumulate_kernel (K3, direct form)", "achieved": achieved, "peak": peak,
        "unit": "Gfacet-samples/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": src,
        "peak_model": f"{SM_COUNT} SM x {FP32_LANES_PER_SM} FP32 lanes x {sm_max:.0f} MHz / "
                      f"{K3_FP32_OPS_PER_FACET_SAMPLE:.0f} FP32 lane-ops per facet-sample",
        "measured_pipe_peak": pipe_peak, "frac_of_measured_pipe_peak": achieved / pipe_peak,
        "launch_ms": launch_ms, "facet_samples_per_launch": fs_per_launch,
        "kernel_share_of_step": kms["accumulate"] / max(sum(kms.values()), 1e-9),
    }


def _roofline_spectral(kms, stats, sm_max, pipes):
    """K2s / K2k (moments kernels) against the FP32 pipe, on the moment form's OWN op count (SURVEY.md 8(d):
    "4 Kt FFMA + ~30 setup per facet-echo ... must be reported against its own op count"): with Kt = 8 that is
    62 FP32 lane-operations per nominal facet-echo."""
    n_batches = _n_batches(stats)
    launch_ms = kms["geometry"] / n_batches
    echoes = stats["facet_echoes_nominal"] / n_batches
    ops = echoes * MOMENT_FP32_OPS_PER_FACET_ECHO
    achieved = ops / (launch_ms * 1e-3) / 1e9
    peak = SM_COUNT * FP32_LANES_PER_SM * sm_max * 1e6 / 1e9
    keyframed = bool(stats.get("geometry_keyframed", 0))
    traffic, src = _profile_traffic("moments", echoes) if keyframed else (None, "no capture of moments_kernel (K2s) on this workload")
    out = {
        "bound": "alu", "kernel": ("moments_keyframed_kernel (K2k" if keyframed else "moments_kernel (K2s") + ", spectral form)",
        "achieved": achieved, "peak": peak, "unit": "GFP32-lane-op/s", "frac": achieved / peak,
        "traffic": traffic, "traffic_source": src,
        "peak_model": f"{SM_COUNT} SM x {FP32_LANES_PER_SM} FP32 lanes x {sm_max:.0f} MHz; algorithmic work "
                      f"{MOMENT_FP32_OPS_PER_FACET_ECHO:.0f} FP32 lane-ops per facet-echo (4 Kt + 30, Kt = 8)",
        "launch_ms": launch_ms, "launches_per_step": n_batches, "facet_echoes_per_launch": echoes,
        "kernel_share_of_step": kms["geometry"] / max(sum(kms.values()), 1e-9),
    }
    if pipes:
        out["measured_pipe_peak"] = pipes["ffma_per_s"] / 1e9
        out["frac_of_measured_pipe_peak"] = achieved / (pipes["ffma_per_s"] / 1e9)
    return out


def _side_config(name, local_rank, stream, barrier, torch, sm_max, steps=3, warmup=3):
    """One of the other configurations through the default path: value, ms per step, K2k roofline fraction, kept."""
    from paper_2405_09938_b200 import Simulator
    w = _base_workload(name)
    F, C, P, Ns = w.n_facets, w.n_channels, w.n_pulses, w.n_samples
    out = torch.empty((C, P, Ns), dtype=torch.complex64, device=f"cuda:{local_rank}")
    with Simulator(w, local_rank) as sim:
        ms, _, kms, stats, _ = _time_steps(sim, out, P, steps, warmup, stream, barrier, torch)
    del out
    roof = _roofline_spectral(kms, stats, sm_max, None) if stats["accumulate_mode"] == 2 else None
    return {"facets": F, "channels": C, "pulses": P, "replica_samples": w.replica_samples, "n_samples": Ns,
            "value": F * P * C / (ms / steps * 1e-3), "unit": UNIT, "ms_per_step": ms / steps, "ms_per_pulse": ms / steps / P,
            "steps": steps, "warmup": warmup,
            "kept": stats["facet_echoes_kept"] / max(stats["facet_echoes_nominal"], 1),
            "frac": roof["frac"] if roof else None, "kernel": roof["kernel"] if roof else None,
            "kinematics_keyframe": stats["kinematics_keyframe"], "kernel_ms_last_step": kms}


def run_cuda(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2405_09938_b200 import Simulator, sim_measure_pipe_peaks

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))

    # weak scaling: rank r simulates pulses [r P, (r+1) P) of an N*P-pulse acquisition
    w = _workload(args.workload, args.pulses, 0)
    P = w.n_pulses
    if rank > 0:
        w = _workload(args.workload, P, rank * P)
    F, C, Ns, L = w.n_facets, w.n_channels, w.n_samples, w.replica_samples
    sim = Simulator(w, local_rank, accumulate_mode=args.mode, tile_facets=args.tile)
    out = torch.empty((C, P, Ns), dtype=torch.complex64, device=f"cuda:{local_rank}")
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing (value) ----
    elapsed_ms, t_wall, kms, stats, clk = _time_steps(sim, out, P, args.steps, args.warmup, stream, barrier, torch,
                                                      clocks_index=local_rank)
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=f"cuda:{local_rank}")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_per_step = float(t.item()) / args.steps
    value = world * F * P * C / (ms_per_step * 1e-3)
    spectral = stats["accumulate_mode"] == 2
    del out

    # ---- end to end through the C ABI with HOST buffers ----
    xi_host = torch.from_numpy(np.ascontiguousarray(w.scene["xi"])).pin_memory()
    maps = {"xi": xi_host}
    h2d = xi_host.numel() * 4
    if w.scene["sigma0_lin"] is not None:
        maps["sigma0"] = torch.from_numpy(np.ascontiguousarray(w.scene["sigma0_lin"])).pin_memory()
        h2d += maps["sigma0"].numel() * 4
    if w.scene["current_mps"] is not None:
        maps["current"] = torch.from_numpy(np.ascontiguousarray(w.scene["current_mps"])).pin_memory()
        h2d += maps["current"].numel() * 4
    out_host = torch.empty((C, P, Ns), dtype=torch.complex64, pin_memory=True)
    d2h = out_host.numel() * 8
    e2e_steps = max(1, min(args.steps, 10 if ms_per_step < 200 else 5))
    sim.update_scene(**maps); sim.generate_host(0, P, out=out_host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sim.update_scene(**maps)
        sim.generate_host(0, P, out=out_host)        # returns after the samples are in host memory
    barrier()
    te = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=f"cuda:{local_rank}")
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_value = world * F * P * C * e2e_steps / float(te.item())
    sim.close()
    del out_host, maps, xi_host

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- rooflines (bound "alu"): the dominant kernel of the timed path, and K3 of the direct form ----
    peaks, peak_src = _peaks()
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    pipes = sim_measure_pipe_peaks(local_rank)          # same-run pipe microbenchmarks
    roofline = (_roofline_spectral(kms, stats, sm_max, pipes) if spectral
                else _roofline_direct(kms, stats, sm_max, pipes))
    roofline["clock_source"] = f"{peak_src} sm_max_mhz"
    roofline["kernel_ms_last_step"] = kms
    roofline["pipe_peaks_lane_ops_per_s"] = {k: v for k, v in pipes.items() if k.endswith("_per_s")}

    direct, others = None, None
    if world == 1 and not args.no_direct:
        # the direct form (every chirp replica generated sample by sample) on the ATI configuration
        wd = w if F * P * C * L <= 3e11 else _base_workload("ati")
        outd = torch.empty((wd.n_channels, wd.n_pulses, wd.n_samples), dtype=torch.complex64, device=f"cuda:{local_rank}")
        d_steps = 5
        with Simulator(wd, local_rank, accumulate_mode="direct") as sim_d:
            d_ms, _, d_kms, d_stats, _ = _time_steps(sim_d, outd, wd.n_pulses, d_steps, 3, stream, barrier, torch)
        del outd
        direct = {"workload": args.workload if wd is w else "ati", "value": wd.n_facets * wd.n_pulses * wd.n_channels / (d_ms / d_steps * 1e-3),
                  "unit": UNIT, "ms_per_step": d_ms / d_steps, "steps": d_steps,
                  "roofline": _roofline_direct(d_kms, d_stats, sm_max, pipes), "kernel_ms_last_step": d_kms}
    if world == 1 and not args.no_other_configs and args.workload == "large" and not any(_VARIANT.values()):
        others = {}
        for name in ("ati", "hetero", "sweep:f20:l1200:c3", "sweep:f24:l1200:c3", "sweep:f26:l1200:c3"):
            try:
                others[name] = _side_config(name, local_rank, stream, barrier, torch, sm_max)
            except Exception as e:                       # a side measurement must not lose the headline line
                others[name] = {"error": repr(e)}

    # ---- the oracle on the host cores, bounded sample (reported baseline, not the target) ----
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        ws, j0, j1 = _row_slab(w, 12.0)                  # about 12 s of oracle time
        pulse = P // 2
        dt, cores = _oracle_sample(ws, [pulse])
        cpu = {"value": ws.n_facets * C / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"pulse {pulse}, facet rows [{j0}, {j1}) of {int(w.scene['ny'])} x all {int(w.scene['nx'])} columns x {C} "
                         f"channels of '{args.workload}' ({ws.n_facets * C} facet-echoes, {dt:.1f} s wall)"}

    cfg = _config(w, args.workload, world)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "ms_per_pulse": ms_per_step / P, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": cfg,
        "path": {"accumulate_mode": "spectral" if spectral else "direct", "fft_size": stats["fft_size"],
                 "kinematics_keyframe": stats["kinematics_keyframe"], "geometry_keyframed": stats["geometry_keyframed"],
                 "fft_band_size": stats["fft_band_size"], "tile_facets": stats["tile_facets"],
                 "pulses_per_batch": stats["pulses_per_batch"]},
        "facet_echoes_kept_frac": stats["facet_echoes_kept"] / max(stats["facet_echoes_nominal"], 1),
        "roofline": roofline,
        "other_configs": others,
        "direct_form": direct,
        "cpu_baseline": cpu,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps},
        "gpu_launches": int(stats["kernel_launches"]) * args.steps,
        "clocks": clk,
        "wall_s_timed_region": t_wall,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="large",
                    help="tiny | ati | hetero | large | sweep:f<log2 facets>:l<replica samples>:c<channels>")
    ap.add_argument("--mode", default="auto", choices=["auto", "direct", "spectral"],
                    help="echo accumulation (include/heeps_sim.h SIM_ACCUMULATE_*)")
    ap.add_argument("--tile", type=int, default=0, help="spatial tile side in facets (0 = library default)")
    ap.add_argument("--pulses", type=int, default=None, help="override the dwell length (debugging)")
    ap.add_argument("--wave-node-spacing", type=float, default=0.0,
                    help="heterogeneous surface: lattice step L [m] of per-node wave tables (0 = homogeneous, the configs)")
    ap.add_argument("--speckle-tau", type=float, default=0.0,
                    help="time-dependent AR(1) speckle: correlation time tau_s [s] (0 = constant speckle, the configs)")
    ap.add_argument("--patterns", action="store_true",
                    help="antenna patterns as 513 x 129 complex u-v tables with 1.5 deg/s azimuth steering (default: analytic apertures)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-direct", action="store_true", help="skip the direct-form comparison leg")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the other configurations (ATI, Heterogeneous, sweep points)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    _VARIANT["wave_node_spacing"], _VARIANT["speckle_tau"] = args.wave_node_spacing, args.speckle_tau
    _VARIANT["patterns"] = args.patterns
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
