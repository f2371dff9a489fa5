"""ctypes binding of include/heeps_sim.h -- argument marshalling only.

Module-level functions carry the C names (`sim_create`, `sim_generate`, ...); `Simulator`
is a small convenience wrapper that owns the handle and hands PyTorch device memory and the
current CUDA stream to the library.  Nothing here computes anything.
"""
from __future__ import annotations

import ctypes as C
import subprocess
from pathlib import Path

import numpy as np

import os

# HEEPS_SIM_LIBRARY selects another build of the same library (the checked build, build.py --checked)
LIBRARY_PATH = Path(os.environ.get("HEEPS_SIM_LIBRARY") or Path(__file__).resolve().parent / "libheeps_sim.so").resolve()
HEADER_PATH = Path(__file__).resolve().parent.parent / "include" / "heeps_sim.h"

SIM_OK, SIM_EINVAL, SIM_ERANGE, SIM_ENOMEM, SIM_ECUDA = 0, -1, -2, -3, -4
SIM_MAX_CHANNELS = 8
SIM_ACCUMULATE_AUTO, SIM_ACCUMULATE_DIRECT, SIM_ACCUMULATE_SPECTRAL = 0, 1, 2
_MODES = {"auto": 0, "direct": 1, "spectral": 2, 0: 0, 1: 1, 2: 2}


class SimError(RuntimeError):
    def __init__(self, code: int, detail: str = ""):
        self.code = code
        msg = f"heeps_sim error {code}: {sim_error_string(code)}"
        if detail:
            msg += f" [{detail}]"
        super().__init__(msg)


class sim_instrument(C.Structure):
    _fields_ = [
        ("f0_hz", C.c_double), ("chirp_rate_hz_per_s", C.c_double), ("chirp_len_s", C.c_double),
        ("fs_hz", C.c_double), ("prf_hz", C.c_double), ("n_samples", C.c_int32),
        ("tx_aperture_m", C.c_double * 2), ("rx_aperture_m", C.c_double * 2),
        ("n_channels", C.c_int32), ("channel_offset_m", C.c_void_p), ("cull_two_way_db", C.c_double),
        ("tx_pattern", C.c_void_p), ("rx_pattern", C.c_void_p),
        ("tx_pattern_nu", C.c_int32), ("tx_pattern_nv", C.c_int32),
        ("rx_pattern_nu", C.c_int32), ("rx_pattern_nv", C.c_int32),
        ("tx_pattern_u", C.c_double * 2), ("tx_pattern_v", C.c_double * 2),
        ("rx_pattern_u", C.c_double * 2), ("rx_pattern_v", C.c_double * 2),
    ]


class sim_geometry(C.Structure):
    _fields_ = [
        ("n_pulses", C.c_int32), ("t_pulse_s", C.c_void_p),
        ("tx_pos_m", C.c_void_p), ("tx_vel_mps", C.c_void_p), ("rx_pos_m", C.c_void_p), ("rx_vel_mps", C.c_void_p),
        ("tx_frame", C.c_void_p), ("rx_frame", C.c_void_p), ("t0_s", C.c_void_p),
    ]


class sim_scene(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("spacing_m", C.c_double), ("centre_m", C.c_double * 3),
        ("n_waves", C.c_int32),
        ("kx", C.c_void_p), ("ky", C.c_void_p), ("amp", C.c_void_p), ("omega", C.c_void_p), ("phase", C.c_void_p),
        ("choppy", C.c_int32),
        ("sigma0_lin", C.c_void_p), ("sigma0_uniform", C.c_double),
        ("tilt_modulation", C.c_int32), ("look_dir", C.c_double * 2),
        ("current_mps", C.c_void_p), ("current_uniform", C.c_double * 2),
        ("xi", C.c_void_p), ("seed", C.c_uint64),
        ("speckle_tau_s", C.c_double), ("speckle_doppler_hz", C.c_double),
        ("wave_nodes_x", C.c_int32), ("wave_nodes_y", C.c_int32), ("wave_node_spacing_m", C.c_double),
        ("node_kx", C.c_void_p), ("node_ky", C.c_void_p), ("node_amp", C.c_void_p), ("node_omega", C.c_void_p),
        ("node_phase", C.c_void_p),
    ]


class sim_options(C.Structure):
    _fields_ = [("tile_facets", C.c_int32), ("pulses_per_batch", C.c_int32), ("workspace_bytes", C.c_int64),
                ("accumulate_mode", C.c_int32), ("kinematics_keyframe", C.c_int32), ("geometry_keyframe", C.c_int32),
                ("fft_band", C.c_int32), ("reserved", C.c_int32 * 4)]


class sim_stats(C.Structure):
    _fields_ = [
        ("facet_echoes_nominal", C.c_int64), ("facet_echoes_kept", C.c_int64), ("facet_samples", C.c_int64),
        ("kernel_launches", C.c_int64),
        ("tile_facets", C.c_int32), ("pulses_per_batch", C.c_int32), ("n_tiles", C.c_int32),
        ("accumulate_block_threads", C.c_int32), ("max_span_samples", C.c_int32),
        ("accumulate_mode", C.c_int32), ("fft_size", C.c_int32), ("kinematics_keyframe", C.c_int32),
        ("geometry_keyframed", C.c_int32), ("fft_band_size", C.c_int32), ("kinematics_coarse_keyframe", C.c_int32),
    ]


class sim_pipe_peaks(C.Structure):
    _fields_ = [("ffma_per_s", C.c_double), ("fadd_per_s", C.c_double), ("ffma2_lane_per_s", C.c_double),
                ("fadd2_lane_per_s", C.c_double), ("mix_f32x2_lane_per_s", C.c_double), ("mufu_per_s", C.c_double),
                ("dfma_per_s", C.c_double), ("sm_count", C.c_int32), ("reserved", C.c_int32 * 3)]


_lib = None


def load_library():
    """dlopen the in-tree CUDA library.  Fails loudly if it has not been built."""
    global _lib
    if _lib is None:
        if not LIBRARY_PATH.exists():
            raise ImportError(
                f"{LIBRARY_PATH} is missing: build it with `python -m paper_2405_09938_b200.build` "
                "(or __graft_entry__.build()).  There is no CPU fallback.")
        lib = C.CDLL(str(LIBRARY_PATH))
        vp, i32 = C.c_void_p, C.c_int32
        lib.sim_create.restype = C.c_int
        lib.sim_create.argtypes = [C.POINTER(sim_instrument), C.POINTER(sim_geometry), C.POINTER(sim_scene),
                                   C.POINTER(sim_options), C.c_int, C.POINTER(vp)]
        lib.sim_generate.restype = C.c_int
        lib.sim_generate.argtypes = [vp, i32, i32, vp, vp]
        lib.sim_generate_host.restype = C.c_int
        lib.sim_generate_host.argtypes = [vp, i32, i32, vp, vp]
        lib.sim_update_scene.restype = C.c_int
        lib.sim_update_scene.argtypes = [vp, vp, vp, vp, vp]
        lib.sim_replica.restype = C.c_int
        lib.sim_replica.argtypes = [vp, vp, C.POINTER(i32)]
        lib.sim_debug_facets.restype = C.c_int
        lib.sim_debug_facets.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp]
        lib.sim_debug_echoes.restype = C.c_int
        lib.sim_debug_echoes.argtypes = [vp, i32, vp, vp, vp, vp, C.POINTER(C.c_int64)]
        lib.sim_echoes_to_iq_static.restype = C.c_int
        lib.sim_echoes_to_iq_static.argtypes = [C.c_double, C.c_double, C.c_double, i32, vp, vp, vp, C.c_int64,
                                                C.POINTER(C.c_double * 2), vp, C.c_int, vp]
        lib.sim_get_stats.restype = C.c_int
        lib.sim_get_stats.argtypes = [vp, C.POINTER(sim_stats)]
        lib.sim_set_profiling.restype = C.c_int
        lib.sim_set_profiling.argtypes = [vp, i32]
        lib.sim_get_kernel_ms.restype = C.c_int
        lib.sim_get_kernel_ms.argtypes = [vp, C.POINTER(C.c_float * 4)]
        lib.sim_measure_pipe_peaks.restype = C.c_int
        lib.sim_measure_pipe_peaks.argtypes = [C.c_int, C.POINTER(sim_pipe_peaks)]
        lib.sim_destroy.restype = None
        lib.sim_destroy.argtypes = [vp]
        lib.sim_error_string.restype = C.c_char_p
        lib.sim_error_string.argtypes = [C.c_int]
        lib.sim_last_cuda_error.restype = C.c_char_p
        lib.sim_last_cuda_error.argtypes = [vp]
        _lib = lib
    return _lib


def exported_symbols() -> set[str]:
    """Dynamic symbols the built library exports (used by the ABI test; no compute)."""
    out = subprocess.run(["nm", "-D", "--defined-only", str(LIBRARY_PATH)], capture_output=True, text=True, check=True)
    return {line.split()[-1] for line in out.stdout.splitlines() if line.strip()}


def sim_error_string(code: int) -> str:
    try:
        return load_library().sim_error_string(int(code)).decode()
    except ImportError:
        return {0: "ok", -1: "invalid argument", -2: "pulse range out of bounds", -3: "out of memory",
                -4: "CUDA error"}.get(code, "unknown error")


def _check(rc: int, handle=None):
    if rc != SIM_OK:
        detail = ""
        if handle is not None and rc == SIM_ECUDA:
            detail = load_library().sim_last_cuda_error(handle).decode()
        raise SimError(rc, detail)


def _f64(a, shape=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if shape is not None and tuple(a.shape) != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _marshal(workload):
    """Workload dicts -> C structs (+ the numpy arrays that must outlive the call)."""
    inst, geo, sc = workload.instrument, workload.geometry, workload.scene
    keep = []

    def ptr(a):
        keep.append(a)
        return a.ctypes.data

    ci = sim_instrument()
    ci.f0_hz = inst["f0_hz"]; ci.chirp_rate_hz_per_s = inst["chirp_rate_hz_per_s"]
    ci.chirp_len_s = inst["chirp_len_s"]; ci.fs_hz = inst["fs_hz"]; ci.prf_hz = inst.get("prf_hz", 0.0)
    ci.n_samples = int(inst["n_samples"])
    ci.tx_aperture_m[:] = list(_f64(inst["tx_aperture_m"], (2,)))
    ci.rx_aperture_m[:] = list(_f64(inst["rx_aperture_m"], (2,)))
    off = _f64(inst["channel_offset_m"])
    ci.n_channels = off.size
    ci.channel_offset_m = ptr(off)
    ci.cull_two_way_db = inst["cull_two_way_db"]
    for name in ("tx_pattern", "rx_pattern"):        # dict: table complex [nv][nu], u = (first, last node), v likewise
        pat = inst.get(name)
        if pat is not None:
            tab = np.asarray(pat["table"])
            t2 = np.ascontiguousarray(np.stack([tab.real, tab.imag], axis=-1), dtype=np.float32)
            setattr(ci, name, ptr(t2))
            setattr(ci, name + "_nv", int(tab.shape[0])); setattr(ci, name + "_nu", int(tab.shape[1]))
            getattr(ci, name + "_u")[:] = [float(pat["u"][0]), float(pat["u"][1])]
            getattr(ci, name + "_v")[:] = [float(pat["v"][0]), float(pat["v"][1])]

    cg = sim_geometry()
    P = int(geo["n_pulses"]); cg.n_pulses = P
    cg.t_pulse_s = ptr(_f64(geo["t_pulse_s"], (P,)))
    for k in ("tx_pos_m", "tx_vel_mps", "rx_pos_m", "rx_vel_mps"):
        setattr(cg, k, ptr(_f64(geo[k], (P, 3))))
    cg.tx_frame = ptr(_f64(geo["tx_frame"], (P, 3, 3)))
    cg.rx_frame = ptr(_f64(geo["rx_frame"], (P, 3, 3)))
    cg.t0_s = ptr(_f64(geo["t0_s"], (P,)))

    cs = sim_scene()
    nx, ny = int(sc["nx"]), int(sc["ny"])
    cs.nx, cs.ny = nx, ny
    cs.spacing_m = sc["spacing_m"]
    cs.centre_m[:] = list(_f64(sc["centre_m"], (3,)))
    nw = int(sc["n_waves"]); cs.n_waves = nw
    for k in ("kx", "ky", "amp", "omega", "phase"):
        setattr(cs, k, ptr(_f64(sc[k], (nw,))) if nw else None)
    cs.choppy = int(sc.get("choppy", 0))
    if sc.get("sigma0_lin") is not None:
        a = np.ascontiguousarray(sc["sigma0_lin"], dtype=np.float32)
        if a.shape != (ny, nx):
            raise ValueError("sigma0_lin must be [ny][nx]")
        cs.sigma0_lin = ptr(a)
    cs.sigma0_uniform = float(sc.get("sigma0_uniform", 0.0))
    cs.tilt_modulation = int(sc.get("tilt_modulation", 0))
    cs.look_dir[:] = list(_f64(sc.get("look_dir", (0.0, 1.0)), (2,)))
    if sc.get("current_mps") is not None:
        a = np.ascontiguousarray(sc["current_mps"], dtype=np.float32)
        if a.shape != (ny, nx, 2):
            raise ValueError("current_mps must be [ny][nx][2]")
        cs.current_mps = ptr(a)
    cs.current_uniform[:] = list(_f64(sc.get("current_uniform", (0.0, 0.0)), (2,)))
    if sc.get("xi") is not None:
        a = np.ascontiguousarray(sc["xi"], dtype=np.float32)
        if a.shape != (ny, nx, 2):
            raise ValueError("xi must be [ny][nx][2]")
        cs.xi = ptr(a)
    cs.seed = int(sc.get("seed", 0))
    cs.speckle_tau_s = float(sc.get("speckle_tau_s", 0.0))
    cs.speckle_doppler_hz = float(sc.get("speckle_doppler_hz", 0.0))
    if sc.get("wave_nodes") is not None:          # heterogeneous surface: dict(spacing_m, kx/ky/amp/omega/phase [ny_n][nx_n][Nw])
        wn = sc["wave_nodes"]
        shape = np.asarray(wn["kx"]).shape
        cs.wave_nodes_y, cs.wave_nodes_x, cs.n_waves = int(shape[0]), int(shape[1]), int(shape[2])
        cs.wave_node_spacing_m = float(wn["spacing_m"])
        for k in ("kx", "ky", "amp", "omega", "phase"):
            setattr(cs, "node_" + k, ptr(_f64(wn[k], shape)))
    return ci, cg, cs, keep


# ----------------------------------------------------------------------------- C-named functions

def sim_create(workload, device: int = 0, *, tile_facets: int = 0, pulses_per_batch: int = 0,
               workspace_bytes: int = 0, accumulate_mode=0, kinematics_keyframe: int = 0,
               geometry_keyframe: int = 0, fft_band: int = 0):
    lib = load_library()
    ci, cg, cs, keep = _marshal(workload)
    opts = sim_options()
    opts.tile_facets, opts.pulses_per_batch, opts.workspace_bytes = tile_facets, pulses_per_batch, workspace_bytes
    opts.accumulate_mode = _MODES[accumulate_mode]
    opts.kinematics_keyframe = int(kinematics_keyframe)
    opts.geometry_keyframe = int(geometry_keyframe)
    opts.fft_band = int(fft_band)
    h = C.c_void_p()
    rc = lib.sim_create(C.byref(ci), C.byref(cg), C.byref(cs), C.byref(opts), int(device), C.byref(h))
    del keep
    _check(rc)
    return h


def sim_destroy(handle):
    if handle:
        load_library().sim_destroy(handle)


def sim_generate(handle, pulse_begin: int, pulse_end: int, iq_dev_ptr: int, cuda_stream: int = 0):
    _check(load_library().sim_generate(handle, pulse_begin, pulse_end, C.c_void_p(iq_dev_ptr), C.c_void_p(cuda_stream)), handle)


def sim_generate_host(handle, pulse_begin: int, pulse_end: int, iq_host_ptr: int, cuda_stream: int = 0):
    _check(load_library().sim_generate_host(handle, pulse_begin, pulse_end, C.c_void_p(iq_host_ptr), C.c_void_p(cuda_stream)), handle)


def sim_update_scene(handle, sigma0_ptr: int = 0, current_ptr: int = 0, xi_ptr: int = 0, cuda_stream: int = 0):
    _check(load_library().sim_update_scene(handle, C.c_void_p(sigma0_ptr or None), C.c_void_p(current_ptr or None),
                                           C.c_void_p(xi_ptr or None), C.c_void_p(cuda_stream)), handle)


def sim_replica(handle) -> np.ndarray:
    lib = load_library()
    n = C.c_int32(0)
    _check(lib.sim_replica(handle, None, C.byref(n)), handle)
    out = np.zeros((n.value, 2), dtype=np.float32)
    _check(lib.sim_replica(handle, out.ctypes.data, C.byref(n)), handle)
    return out[:, 0] + 1j * out[:, 1]


def sim_debug_facets(handle, pulse: int, n_facets: int, n_channels: int) -> dict:
    F, Cn = n_facets, n_channels
    res = dict(pos=np.zeros((F, 3)), slope=np.zeros((F, 2)), tau=np.zeros((Cn, F)), g_tx=np.zeros(F),
               g_rx=np.zeros((Cn, F)), amp=np.zeros((Cn, F, 2)), keep=np.zeros(F, dtype=np.int32))
    _check(load_library().sim_debug_facets(handle, pulse, *(res[k].ctypes.data for k in
                                           ("pos", "slope", "tau", "g_tx", "g_rx", "amp", "keep"))), handle)
    res["amp"] = res["amp"][..., 0] + 1j * res["amp"][..., 1]
    return res


def sim_debug_echoes(handle, pulse: int, n_facets: int, n_channels: int) -> dict:
    F, Cn = n_facets, n_channels
    res = dict(slice=np.zeros((Cn, F), dtype=np.int32), eps=np.zeros((Cn, F), dtype=np.float32),
               weight=np.zeros((Cn, F, 2), dtype=np.float32), keep=np.zeros(F, dtype=np.int32))
    n_edge = C.c_int64(0)
    _check(load_library().sim_debug_echoes(handle, pulse, res["slice"].ctypes.data, res["eps"].ctypes.data,
                                           res["weight"].ctypes.data, res["keep"].ctypes.data, C.byref(n_edge)), handle)
    res["weight"] = res["weight"][..., 0] + 1j * res["weight"][..., 1]
    res["n_edge_ambiguous"] = int(n_edge.value)
    return res


def sim_echoes_to_iq_static(chirp_rate_hz_per_s: float, chirp_len_s: float, fs_hz: float, n_samples: int,
                            slice_dev_ptr: int, eps_dev_ptr: int, weight_dev_ptr: int, n_echoes: int, phase: complex,
                            iq_dev_ptr: int, device: int = 0, cuda_stream: int = 0):
    """The entry point that allocates nothing (include/heeps_sim.h): device pointers in, complex64 [n_samples] out."""
    ph = (C.c_double * 2)(float(np.real(phase)), float(np.imag(phase)))
    _check(load_library().sim_echoes_to_iq_static(
        float(chirp_rate_hz_per_s), float(chirp_len_s), float(fs_hz), int(n_samples), C.c_void_p(slice_dev_ptr or None),
        C.c_void_p(eps_dev_ptr or None), C.c_void_p(weight_dev_ptr or None), int(n_echoes), C.byref(ph),
        C.c_void_p(iq_dev_ptr), int(device), C.c_void_p(cuda_stream or None)))


def sim_measure_pipe_peaks(device: int = 0) -> dict:
    st = sim_pipe_peaks()
    _check(load_library().sim_measure_pipe_peaks(int(device), C.byref(st)))
    return {k: getattr(st, k) for k, _ in sim_pipe_peaks._fields_ if k != "reserved"}


def sim_get_stats(handle) -> dict:
    st = sim_stats()
    _check(load_library().sim_get_stats(handle, C.byref(st)), handle)
    return {k: getattr(st, k) for k, _ in sim_stats._fields_}


# ----------------------------------------------------------------------------- convenience wrapper

class Simulator:
    """Owns a `sim_handle`; PyTorch supplies device memory and the stream."""

    def __init__(self, workload, device: int = 0, **options):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2405_09938_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self._torch = torch
        self.device = int(device)
        self.n_channels = int(len(workload.instrument["channel_offset_m"]))
        self.n_pulses = int(workload.geometry["n_pulses"])
        self.n_samples = int(workload.instrument["n_samples"])
        self.n_facets = int(workload.scene["nx"]) * int(workload.scene["ny"])
        self._h = sim_create(workload, self.device, **options)

    def close(self):
        if getattr(self, "_h", None):
            sim_destroy(self._h)
            self._h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _stream(self) -> int:
        return int(self._torch.cuda.current_stream(self.device).cuda_stream)

    def generate(self, pulse_begin: int = 0, pulse_end: int | None = None, out=None):
        """complex64 CUDA tensor [C][pulse_end-pulse_begin][Ns]; asynchronous on the current stream."""
        torch = self._torch
        pulse_end = self.n_pulses if pulse_end is None else pulse_end
        shape = (self.n_channels, max(0, pulse_end - pulse_begin), self.n_samples)
        if out is None:
            out = torch.empty(shape, dtype=torch.complex64, device=f"cuda:{self.device}")
        elif tuple(out.shape) != shape or out.dtype != torch.complex64 or not out.is_contiguous() or not out.is_cuda:
            raise ValueError(f"out must be a contiguous CUDA complex64 tensor of shape {shape}")
        sim_generate(self._h, pulse_begin, pulse_end, out.data_ptr(), self._stream())
        return out

    def generate_host(self, pulse_begin: int = 0, pulse_end: int | None = None, out=None):
        """Same through HOST memory (pinned CPU tensor); returns after the copy has completed."""
        torch = self._torch
        pulse_end = self.n_pulses if pulse_end is None else pulse_end
        shape = (self.n_channels, max(0, pulse_end - pulse_begin), self.n_samples)
        if out is None:
            out = torch.empty(shape, dtype=torch.complex64, pin_memory=True)
        sim_generate_host(self._h, pulse_begin, pulse_end, out.data_ptr(), self._stream())
        return out

    def update_scene(self, sigma0=None, current=None, xi=None):
        """Host (pinned) float32 tensors / arrays -> device maps, on the current stream."""
        def p(a):
            if a is None:
                return 0
            return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
        sim_update_scene(self._h, p(sigma0), p(current), p(xi), self._stream())

    def replica(self) -> np.ndarray:
        return sim_replica(self._h)

    def debug_facets(self, pulse: int) -> dict:
        return sim_debug_facets(self._h, pulse, self.n_facets, self.n_channels)

    def debug_echoes(self, pulse: int) -> dict:
        return sim_debug_echoes(self._h, pulse, self.n_facets, self.n_channels)

    def stats(self) -> dict:
        return sim_get_stats(self._h)

    def set_profiling(self, enable: bool):
        _check(load_library().sim_set_profiling(self._h, int(enable)), self._h)

    def kernel_ms(self) -> dict:
        ms = (C.c_float * 4)()
        _check(load_library().sim_get_kernel_ms(self._h, C.byref(ms)), self._h)
        return dict(zip(("kinematics", "geometry", "accumulate", "finalize"), [float(x) for x in ms]))
