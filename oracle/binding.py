"""ctypes marshalling for heeps_oracle.c, plus the parity metrics the tests apply.

The descriptors are the plain dicts produced by `workloads.make_workload` (instrument,
geometry, scene); any object with those three attributes works.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "heeps_oracle.c"
_LIB = _HERE / "libheeps_oracle.so"
_lib = None


def build_oracle(force: bool = False) -> Path:
    """Compile heeps_oracle.c with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _Desc(C.Structure):
    _fields_ = [
        ("f0_hz", C.c_double), ("chirp_rate", C.c_double), ("chirp_len_s", C.c_double), ("fs_hz", C.c_double),
        ("n_samples", C.c_int32), ("n_channels", C.c_int32),
        ("tx_aperture", C.c_double * 2), ("rx_aperture", C.c_double * 2),
        ("channel_offset_m", C.c_void_p),
        ("cull_two_way_db", C.c_double),
        ("n_pulses", C.c_int32),
        ("t_pulse_s", C.c_void_p),
        ("tx_pos", C.c_void_p), ("tx_vel", C.c_void_p), ("rx_pos", C.c_void_p), ("rx_vel", C.c_void_p),
        ("tx_frame", C.c_void_p), ("rx_frame", C.c_void_p),
        ("t0_s", C.c_void_p),
        ("nx", C.c_int32), ("ny", C.c_int32),
        ("spacing_m", C.c_double), ("centre_m", C.c_double * 3),
        ("n_waves", C.c_int32),
        ("kx", C.c_void_p), ("ky", C.c_void_p), ("amp", C.c_void_p), ("omega", C.c_void_p), ("phase", C.c_void_p),
        ("choppy", C.c_int32),
        ("sigma0_lin", C.c_void_p), ("sigma0_uniform", C.c_double),
        ("tilt_modulation", C.c_int32), ("look_dir", C.c_double * 2),
        ("current_mps", C.c_void_p), ("current_uniform", C.c_double * 2),
        ("xi", C.c_void_p),
        ("speckle_tau_s", C.c_double), ("speckle_doppler_hz", C.c_double), ("seed", C.c_uint64),
        ("wave_nodes_x", C.c_int32), ("wave_nodes_y", C.c_int32), ("wave_node_spacing_m", C.c_double),
        ("node_kx", C.c_void_p), ("node_ky", C.c_void_p), ("node_amp", C.c_void_p), ("node_omega", C.c_void_p),
        ("node_phase", C.c_void_p),
        ("pattern", C.c_void_p * 2), ("pattern_nu", C.c_int32 * 2), ("pattern_nv", C.c_int32 * 2),
        ("pattern_u", (C.c_double * 2) * 2), ("pattern_v", (C.c_double * 2) * 2),
    ]


class _Facets(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("pos", "slope", "vel", "tau", "g_tx", "g_rx", "amp", "keep")]


def _load():
    global _lib
    if _lib is None:
        build_oracle()
        _lib = C.CDLL(str(_LIB))
        _lib.heeps_oracle_generate.restype = C.c_int
        _lib.heeps_oracle_generate.argtypes = [C.POINTER(_Desc), C.c_void_p, C.c_int32, C.c_void_p, C.c_int32]
        _lib.heeps_oracle_facets.restype = C.c_int
        _lib.heeps_oracle_facets.argtypes = [C.POINTER(_Desc), C.c_int32, C.POINTER(_Facets)]
        _lib.heeps_oracle_max_threads.restype = C.c_int
        _lib.heeps_oracle_samples.restype = C.c_int
        _lib.heeps_oracle_samples.argtypes = [C.POINTER(_Desc), C.c_int32, C.c_void_p, C.c_int32, C.c_void_p, C.c_int32]
        _lib.heeps_oracle_speckle.restype = C.c_int
        _lib.heeps_oracle_speckle.argtypes = [C.POINTER(_Desc), C.c_int32, C.c_void_p]
        _lib.heeps_oracle_philox.restype = None
        _lib.heeps_oracle_philox.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    return _lib


def _f64(a, shape=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if shape is not None and tuple(a.shape) != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _marshal(w):
    """Fill the C descriptor; returns (desc, keepalive list)."""
    inst, geo, sc = w.instrument, w.geometry, w.scene
    keep = []

    def ptr(a):
        keep.append(a)
        return a.ctypes.data

    d = _Desc()
    d.f0_hz = inst["f0_hz"]; d.chirp_rate = inst["chirp_rate_hz_per_s"]
    d.chirp_len_s = inst["chirp_len_s"]; d.fs_hz = inst["fs_hz"]
    d.n_samples = inst["n_samples"]
    off = _f64(inst["channel_offset_m"])
    d.n_channels = off.size
    d.channel_offset_m = ptr(off)
    d.tx_aperture[:] = list(_f64(inst["tx_aperture_m"], (2,)))
    d.rx_aperture[:] = list(_f64(inst["rx_aperture_m"], (2,)))
    d.cull_two_way_db = inst["cull_two_way_db"]
    P = int(geo["n_pulses"]); d.n_pulses = P
    d.t_pulse_s = ptr(_f64(geo["t_pulse_s"], (P,)))
    for k, fld in (("tx_pos_m", "tx_pos"), ("tx_vel_mps", "tx_vel"), ("rx_pos_m", "rx_pos"), ("rx_vel_mps", "rx_vel")):
        setattr(d, fld, ptr(_f64(geo[k], (P, 3))))
    d.tx_frame = ptr(_f64(geo["tx_frame"], (P, 3, 3)))
    d.rx_frame = ptr(_f64(geo["rx_frame"], (P, 3, 3)))
    d.t0_s = ptr(_f64(geo["t0_s"], (P,)))
    nx, ny = int(sc["nx"]), int(sc["ny"])
    d.nx, d.ny = nx, ny
    d.spacing_m = sc["spacing_m"]
    d.centre_m[:] = list(_f64(sc["centre_m"], (3,)))
    nw = int(sc["n_waves"]); d.n_waves = nw
    for k in ("kx", "ky", "amp", "omega", "phase"):
        setattr(d, k, ptr(_f64(sc[k], (nw,))) if nw else None)
    d.choppy = int(sc.get("choppy", 0))
    if sc.get("sigma0_lin") is not None:
        s0 = np.ascontiguousarray(sc["sigma0_lin"], dtype=np.float32)
        assert s0.shape == (ny, nx)
        d.sigma0_lin = ptr(s0)
    d.sigma0_uniform = float(sc.get("sigma0_uniform", 0.0))
    d.tilt_modulation = int(sc.get("tilt_modulation", 0))
    d.look_dir[:] = list(_f64(sc.get("look_dir", (0.0, 1.0)), (2,)))
    if sc.get("current_mps") is not None:
        cur = np.ascontiguousarray(sc["current_mps"], dtype=np.float32)
        assert cur.shape == (ny, nx, 2)
        d.current_mps = ptr(cur)
    d.current_uniform[:] = list(_f64(sc.get("current_uniform", (0.0, 0.0)), (2,)))
    xi = np.ascontiguousarray(sc["xi"], dtype=np.float32)
    assert xi.shape == (ny, nx, 2)
    d.xi = ptr(xi)
    d.speckle_tau_s = float(sc.get("speckle_tau_s", 0.0))
    d.speckle_doppler_hz = float(sc.get("speckle_doppler_hz", 0.0))
    d.seed = int(sc.get("seed", 0))
    if sc.get("wave_nodes") is not None:                      # heterogeneous surface
        wn = sc["wave_nodes"]                                 # dict: spacing_m, kx/ky/amp/omega/phase [ny_n][nx_n][Nw]
        shape = np.asarray(wn["kx"]).shape
        d.wave_nodes_y, d.wave_nodes_x, d.n_waves = int(shape[0]), int(shape[1]), int(shape[2])
        d.wave_node_spacing_m = float(wn["spacing_m"])
        for k in ("kx", "ky", "amp", "omega", "phase"):
            setattr(d, "node_" + k, ptr(_f64(wn[k], shape)))
    for k, name in enumerate(("tx_pattern", "rx_pattern")):      # antenna patterns as complex u-v grids
        pat = inst.get(name)
        if pat is not None:                                      # dict: table complex [nv][nu], u=(u0,u1), v=(v0,v1)
            tab = np.asarray(pat["table"])
            t2 = np.ascontiguousarray(np.stack([tab.real, tab.imag], axis=-1), dtype=np.float32)
            d.pattern[k] = ptr(t2)
            d.pattern_nv[k], d.pattern_nu[k] = int(tab.shape[0]), int(tab.shape[1])
            d.pattern_u[k][0], d.pattern_u[k][1] = float(pat["u"][0]), float(pat["u"][1])
            d.pattern_v[k][0], d.pattern_v[k][1] = float(pat["v"][0]), float(pat["v"][1])
    return d, keep


def oracle_max_threads() -> int:
    return int(_load().heeps_oracle_max_threads())


def oracle_generate(w, pulses=None, n_threads: int = 0) -> np.ndarray:
    """complex128 [C][len(pulses)][Ns]: the defined sum for the listed pulses (default: all)."""
    lib = _load()
    d, keep = _marshal(w)
    if pulses is None:
        pulses = np.arange(d.n_pulses)
    pulses = np.ascontiguousarray(np.asarray(pulses, dtype=np.int32))
    out = np.zeros((d.n_channels, pulses.size, d.n_samples), dtype=np.complex128)
    rc = lib.heeps_oracle_generate(C.byref(d), pulses.ctypes.data, pulses.size, out.ctypes.data, n_threads)
    if rc != 0:
        raise ValueError(f"heeps_oracle_generate failed ({rc})")
    del keep
    return out


def oracle_samples(w, pulse: int, samples, n_threads: int = 0) -> np.ndarray:
    """complex128 [C][len(samples)]: the defined sum at the listed fast-time samples of one pulse."""
    lib = _load()
    d, keep = _marshal(w)
    samples = np.ascontiguousarray(np.asarray(samples, dtype=np.int32))
    out = np.zeros((d.n_channels, samples.size, 2), dtype=np.float64)
    rc = lib.heeps_oracle_samples(C.byref(d), int(pulse), samples.ctypes.data, samples.size, out.ctypes.data, n_threads)
    if rc != 0:
        raise ValueError(f"heeps_oracle_samples failed ({rc})")
    del keep
    return out[..., 0] + 1j * out[..., 1]


def oracle_facets(w, pulse: int) -> dict:
    """O2..O8 intermediates of one pulse, for per-kernel unit parity."""
    lib = _load()
    d, keep = _marshal(w)
    F, Cn = d.nx * d.ny, d.n_channels
    res = dict(
        pos=np.zeros((F, 3)), slope=np.zeros((F, 2)), vel=np.zeros((F, 3)), tau=np.zeros((Cn, F)),
        g_tx=np.zeros(F), g_rx=np.zeros((Cn, F)), amp=np.zeros((Cn, F, 2)), keep=np.zeros(F, dtype=np.int32),
    )
    fs = _Facets()
    for k, v in res.items():
        setattr(fs, k, v.ctypes.data)
    rc = lib.heeps_oracle_facets(C.byref(d), int(pulse), C.byref(fs))
    if rc != 0:
        raise ValueError(f"heeps_oracle_facets failed ({rc})")
    del keep
    res["amp"] = res["amp"][..., 0] + 1j * res["amp"][..., 1]
    return res


def oracle_speckle(w, pulse: int) -> np.ndarray:
    """complex128 [ny][nx]: the intra-facet speckle s_f(t_p) (eq. (7), (10)) of every facet at one pulse."""
    lib = _load()
    d, keep = _marshal(w)
    out = np.zeros((d.ny, d.nx, 2), dtype=np.float64)
    rc = lib.heeps_oracle_speckle(C.byref(d), int(pulse), out.ctypes.data)
    if rc != 0:
        raise ValueError(f"heeps_oracle_speckle failed ({rc})")
    del keep
    return out[..., 0] + 1j * out[..., 1]


def oracle_philox(counter, key) -> np.ndarray:
    """uint32[4]: one Philox4x32-10 block of the oracle's own generator (known-answer pins)."""
    lib = _load()
    c = np.ascontiguousarray(np.asarray(counter, dtype=np.uint32)); k = np.ascontiguousarray(np.asarray(key, dtype=np.uint32))
    out = np.zeros(4, dtype=np.uint32)
    lib.heeps_oracle_philox(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out


# ---------------------------------------------------------------- parity metrics

def rel_l2_per_vector(got: np.ndarray, ref: np.ndarray) -> np.ndarray:
    """||got-ref||_2 / ||ref||_2 per (channel, pulse) vector.  Where the reference vector is
    identically zero the result is 0 if `got` is exactly zero there and inf otherwise (G20)."""
    got = np.asarray(got, dtype=np.complex128)
    ref = np.asarray(ref, dtype=np.complex128)
    num = np.sqrt((np.abs(got - ref) ** 2).sum(axis=-1))
    den = np.sqrt((np.abs(ref) ** 2).sum(axis=-1))
    out = np.where(den > 0, num / np.where(den > 0, den, 1.0), np.where(num == 0, 0.0, np.inf))
    return out


def ati_phase(s: np.ndarray) -> np.ndarray:
    """Inter-channel interferometric phase arg sum_n s_a[n] conj(s_b[n]) for every channel
    pair a<b: [pairs][pulses] (G19)."""
    s = np.asarray(s, dtype=np.complex128)
    Cn = s.shape[0]
    rows = []
    for a in range(Cn):
        for b in range(a + 1, Cn):
            rows.append(np.angle((s[a] * np.conj(s[b])).sum(axis=-1)))
    return np.asarray(rows).reshape(-1, s.shape[1])


def ati_phase_rms_error(got: np.ndarray, ref: np.ndarray) -> float:
    """RMS over pulses x pairs of wrap(phi_got - phi_ref) [rad]; 0.0 with a single channel."""
    pg, pr = ati_phase(got), ati_phase(ref)
    if pg.size == 0:
        return 0.0
    dphi = np.angle(np.exp(1j * (pg - pr)))
    return float(np.sqrt(np.mean(dphi**2)))
