"""Seeded generators for the five BASELINE.json configurations.

Everything here is a *choice of inputs* (SURVEY.md §8(d), G1/G7/G12/G22): platform
tracks, antenna frames, sampling-window start, wave-component table, sigma0 / current /
speckle maps.  Nothing here evaluates the radar sum.  The arrays are laid out exactly as
`include/heeps_sim.h` expects them (C order, float64 unless noted).

The paper's real inputs (Sentinel-1/Harmony orbit files, phased-array antenna models,
sea-state descriptors) are not available; these synthetic inputs
stand in for them with the shapes and structure the paper states: metre-scale facets
(PAPER.md:51, :223), companion offset D ~ 200-300 km, up to three phase
centres, km-scale sea-state variation.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field

import numpy as np

C0 = 299_792_458.0          # m/s
G_ACC = 9.81                # m/s^2
MASTER_SEED = 20240509

ALTITUDE_M = 700e3
CROSS_TRACK_M = 300e3       # ground offset Y0 of both platforms (G22)
ALONG_TRACK_SEP_M = 250e3   # Rx ahead of Tx (BASELINE.json Tiny)
PLATFORM_SPEED = 7500.0
F0_HZ = 5.405e9
TX_APERTURE = (12.3, 0.82)  # azimuth length, elevation height [m]
RX_APERTURE = (4.0, 1.0)
WIND_SPEED = 10.0
WIND_DIR_RAD = np.pi / 4.0
CURRENT_DIR_RAD = np.pi / 4.0
PM_ALPHA = 8.1e-3
PM_BETA = 0.74

CONFIG_NAMES = ("tiny", "ati", "hetero", "large")


@dataclass
class Workload:
    """Descriptor arrays of one simulation (instrument, geometry, scene)."""

    name: str
    instrument: dict = field(default_factory=dict)
    geometry: dict = field(default_factory=dict)
    scene: dict = field(default_factory=dict)

    # -- derived sizes (counting only, no method arithmetic) -----------------
    @property
    def n_facets(self) -> int:
        return int(self.scene["nx"]) * int(self.scene["ny"])

    @property
    def n_pulses(self) -> int:
        return int(self.geometry["n_pulses"])

    @property
    def n_channels(self) -> int:
        return int(len(self.instrument["channel_offset_m"]))

    @property
    def n_samples(self) -> int:
        return int(self.instrument["n_samples"])

    @property
    def replica_samples(self) -> int:
        """L = T*fs rounded (integer in every BASELINE config)."""
        return int(round(self.instrument["chirp_len_s"] * self.instrument["fs_hz"]))

    def facet_echoes(self, n_pulses: int | None = None) -> int:
        p = self.n_pulses if n_pulses is None else n_pulses
        return self.n_facets * p * self.n_channels


def pm_spectrum(k: np.ndarray, wind: float = WIND_SPEED) -> np.ndarray:
    """Pierson-Moskowitz omnidirectional wavenumber spectrum S(k) [m^3].

    S(k) = alpha/(2 k^3) exp(-beta g^2 / (k^2 U^4)); integral over all k gives
    Hs = 2 sqrt(alpha/beta) U^2/g (closed form used as a generator pin).
    """
    k = np.asarray(k, dtype=np.float64)
    return PM_ALPHA / (2.0 * k**3) * np.exp(-PM_BETA * G_ACC**2 / (k**2 * wind**4))


def _wave_table(nk: int, ntheta: int, seed: int):
    """Nk x Ntheta component table: log-spaced k bins in [0.05, 1] rad/m, PM amplitudes,
    (2/pi) cos^2 spreading over +-90 deg about the wind, seeded uniform phases."""
    edges = np.geomspace(0.05, 1.0, nk + 1)
    kc = np.sqrt(edges[:-1] * edges[1:])
    dk = np.diff(edges)
    if ntheta == 1:
        th = np.array([0.0])
        w_th = np.array([1.0])          # unidirectional: D*dtheta = 1
    else:
        tedges = np.linspace(-np.pi / 2, np.pi / 2, ntheta + 1)
        th = 0.5 * (tedges[:-1] + tedges[1:])
        dth = np.diff(tedges)
        w_th = (2.0 / np.pi) * np.cos(th) ** 2 * dth
        w_th = w_th / w_th.sum()        # exact energy conservation on the coarse grid
    kk, tt = np.meshgrid(kc, th, indexing="ij")
    s = pm_spectrum(kk) * np.repeat(dk[:, None], len(th), 1) * w_th[None, :]
    amp = np.sqrt(2.0 * s).ravel()
    kmag = kk.ravel()
    ang = WIND_DIR_RAD + tt.ravel()
    rng = np.random.Generator(np.random.PCG64(seed))
    phase = rng.random(kmag.size) * 2.0 * np.pi
    return dict(
        n_waves=int(kmag.size),
        kx=np.ascontiguousarray(kmag * np.cos(ang)),
        ky=np.ascontiguousarray(kmag * np.sin(ang)),
        amp=np.ascontiguousarray(amp),
        omega=np.ascontiguousarray(np.sqrt(G_ACC * kmag)),
        phase=np.ascontiguousarray(phase),
    )


def _unit(v):
    v = np.asarray(v, dtype=np.float64)
    return v / np.linalg.norm(v)


def _frame(pos_mid, vel, centre):
    """Antenna frame (G7): boresight from the mid-dwell position to the scene centre;
    azimuth axis = velocity component perpendicular to boresight; elevation = b x a."""
    b = _unit(np.asarray(centre) - np.asarray(pos_mid))
    a = np.asarray(vel, dtype=np.float64)
    a = _unit(a - np.dot(a, b) * b)
    e = np.cross(b, a)
    return np.stack([b, a, e])


def _geometry(n_pulses: int, prf: float, n_samples: int, fs: float, centre, pulse_offset: int = 0):
    p = np.arange(n_pulses, dtype=np.float64) + pulse_offset
    t = p / prf
    # mid-dwell refers to the *nominal* dwell starting at pulse 0 of this workload
    t_mid = (pulse_offset + (n_pulses - 1) / 2.0) / prf
    vel = np.array([PLATFORM_SPEED, 0.0, 0.0])
    tx_pos = np.stack([PLATFORM_SPEED * (t - t_mid), np.full_like(t, -CROSS_TRACK_M),
                       np.full_like(t, ALTITUDE_M)], axis=1) + np.asarray(centre)[None, :]
    rx_pos = tx_pos + np.array([ALONG_TRACK_SEP_M, 0.0, 0.0])[None, :]
    tx_vel = np.repeat(vel[None, :], n_pulses, 0)
    rx_vel = tx_vel.copy()
    tx_mid = np.array([0.0, -CROSS_TRACK_M, ALTITUDE_M]) + np.asarray(centre)
    rx_mid = tx_mid + np.array([ALONG_TRACK_SEP_M, 0.0, 0.0])
    tx_frame = np.repeat(_frame(tx_mid, vel, centre)[None], n_pulses, 0)
    rx_frame = np.repeat(_frame(rx_mid, vel, centre)[None], n_pulses, 0)
    # G1: sample 0 is placed so that the scene-centre echo sits mid-window.
    r_c = np.linalg.norm(tx_pos - np.asarray(centre)[None, :], axis=1) + \
        np.linalg.norm(rx_pos - np.asarray(centre)[None, :], axis=1)
    t0 = r_c / C0 - (n_samples / 2.0) / fs
    # G12: look direction = horizontal part of (u_t + u_r) at the centre, mid-dwell
    look = _unit(np.asarray(centre) - tx_mid) + _unit(np.asarray(centre) - rx_mid)
    look = _unit(np.array([look[0], look[1], 0.0]))[:2]
    geo = dict(
        n_pulses=int(n_pulses),
        t_pulse_s=np.ascontiguousarray(t),
        tx_pos_m=np.ascontiguousarray(tx_pos), tx_vel_mps=np.ascontiguousarray(tx_vel),
        rx_pos_m=np.ascontiguousarray(rx_pos), rx_vel_mps=np.ascontiguousarray(rx_vel),
        tx_frame=np.ascontiguousarray(tx_frame), rx_frame=np.ascontiguousarray(rx_frame),
        t0_s=np.ascontiguousarray(t0),
    )
    return geo, look


def _xi(nx: int, ny: int, seed: int) -> np.ndarray:
    """Unit circular complex Gaussian speckle, variance 1/2 per part,
    float32 [ny][nx][2]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    z = rng.standard_normal((ny, nx, 2), dtype=np.float32)
    z *= np.float32(np.sqrt(0.5))
    return z


def _sigma0_field(nx: int, ny: int, d: float, seed: int, corr_len: float = 1000.0) -> np.ndarray:
    """Smooth Gaussian random field -> sigma0 in (-20, -10) dB (linear units, float32)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    white = rng.standard_normal((ny, nx), dtype=np.float32).astype(np.float64)
    fx = np.fft.rfftfreq(nx, d)
    fy = np.fft.fftfreq(ny, d)
    # Gaussian correlation exp(-r^2/(2 l^2)) <-> spectrum exp(-2 pi^2 l^2 f^2); filter is its sqrt
    h = np.exp(-(np.pi * corr_len) ** 2 * (fy[:, None] ** 2 + fx[None, :] ** 2))
    g = np.fft.irfft2(np.fft.rfft2(white) * h, s=(ny, nx))
    g = (g - g.mean()) / g.std()
    s_db = -15.0 + 5.0 * np.tanh(g)
    return (10.0 ** (s_db / 10.0)).astype(np.float32)


def _current_front(nx: int, ny: int, d: float, centre) -> np.ndarray:
    """0.8 tanh(y/200 m) m/s along the 45 deg direction, float32 [ny][nx][2]."""
    y = centre[1] + (np.arange(ny, dtype=np.float64) - (ny - 1) / 2.0) * d
    mag = 0.8 * np.tanh(y / 200.0)
    cur = np.empty((ny, nx, 2), dtype=np.float32)
    cur[:, :, 0] = (mag * np.cos(CURRENT_DIR_RAD)).astype(np.float32)[:, None]
    cur[:, :, 1] = (mag * np.sin(CURRENT_DIR_RAD)).astype(np.float32)[:, None]
    return cur


def _assemble(name, *, nx, ny, d, nk, ntheta, n_pulses, prf, chirp_len, bandwidth, fs, n_samples,
              offsets, sigma0_db=-15.0, hetero=False, current_uniform=(0.0, 0.0), cull_db=-30.0,
              seed=MASTER_SEED, pulse_offset=0) -> Workload:
    centre = np.zeros(3)
    geo, look = _geometry(n_pulses, prf, n_samples, fs, centre, pulse_offset)
    scene = dict(nx=int(nx), ny=int(ny), spacing_m=float(d), centre_m=centre, choppy=0)
    scene.update(_wave_table(nk, ntheta, seed + 1))
    scene["xi"] = _xi(nx, ny, seed + 2)
    scene["seed"] = int(seed)
    scene["look_dir"] = np.ascontiguousarray(look)
    if hetero:
        scene["sigma0_lin"] = _sigma0_field(nx, ny, d, seed + 3)
        scene["sigma0_uniform"] = 0.0
        scene["tilt_modulation"] = 1
        scene["current_mps"] = _current_front(nx, ny, d, centre)
        scene["current_uniform"] = np.zeros(2)
    else:
        scene["sigma0_lin"] = None
        scene["sigma0_uniform"] = float(10.0 ** (sigma0_db / 10.0))
        scene["tilt_modulation"] = 0
        scene["current_mps"] = None
        scene["current_uniform"] = np.asarray(current_uniform, dtype=np.float64)
    inst = dict(
        f0_hz=F0_HZ, chirp_rate_hz_per_s=float(bandwidth / chirp_len), chirp_len_s=float(chirp_len),
        fs_hz=float(fs), prf_hz=float(prf), n_samples=int(n_samples),
        tx_aperture_m=np.asarray(TX_APERTURE, dtype=np.float64),
        rx_aperture_m=np.asarray(RX_APERTURE, dtype=np.float64),
        channel_offset_m=np.asarray(offsets, dtype=np.float64),
        cull_two_way_db=float(cull_db),
    )
    return Workload(name=name, instrument=inst, geometry=geo, scene=scene)


def make_workload(name: str, *, n_pulses: int | None = None, pulse_offset: int = 0,
                  seed: int = MASTER_SEED) -> Workload:
    """Build one of BASELINE.json's named configurations.

    `n_pulses` overrides the dwell length (the platform track stays centred on the
    shortened dwell); `pulse_offset` shifts the pulse numbering (used to give each rank
    its own slab of a longer acquisition under multi-GPU weak scaling).
    """
    cur45 = (0.5 * np.cos(CURRENT_DIR_RAD), 0.5 * np.sin(CURRENT_DIR_RAD))
    ati_chirp = dict(prf=1700.0, chirp_len=20e-6, bandwidth=50e6, fs=60e6)
    if name == "tiny":
        return _assemble("tiny", nx=64, ny=64, d=5.0, nk=8, ntheta=1, n_pulses=n_pulses or 32,
                         prf=1000.0, chirp_len=2e-6, bandwidth=10e6, fs=12e6, n_samples=256,
                         offsets=[0.0], seed=seed, pulse_offset=pulse_offset)
    if name == "ati":
        return _assemble("ati", nx=512, ny=512, d=4.0, nk=16, ntheta=4, n_pulses=n_pulses or 256,
                         n_samples=4096, offsets=[-1.5, 0.0, 1.5], current_uniform=cur45,
                         seed=seed, pulse_offset=pulse_offset, **ati_chirp)
    if name == "hetero":
        return _assemble("hetero", nx=2048, ny=2048, d=3.0, nk=32, ntheta=8,
                         n_pulses=n_pulses or 1024, n_samples=4096, offsets=[-1.5, 0.0, 1.5],
                         hetero=True, seed=seed, pulse_offset=pulse_offset, **ati_chirp)
    if name == "large":
        return _assemble("large", nx=4096, ny=4096, d=2.0, nk=32, ntheta=8,
                         n_pulses=n_pulses or 2048, n_samples=8192, offsets=[-1.5, 0.0, 1.5],
                         hetero=True, seed=seed, pulse_offset=pulse_offset, **ati_chirp)
    raise ValueError(f"unknown workload {name!r}; known: {CONFIG_NAMES} (+ make_sweep_point)")


def make_sweep_point(*, log2_facets: int = 24, spacing_m: float | None = None,
                     replica_samples: int = 1200, n_channels: int = 3, n_pulses: int = 64,
                     seed: int = MASTER_SEED) -> Workload:
    """One point of BASELINE.json's stress sweep (reading G23).

    Facet axis: 2^20 (1024^2 @4 m), 2^22 (2048^2 @4 m), 2^24 (4096^2 @4 m), 2^26 (8192^2 @2 m);
    chirp axis: L = T*fs samples with B = 50 MHz fixed; channel axis: 1 (0), 2 (+-0.75 m),
    3 (-1.5/0/+1.5 m).  Ns = 8192 throughout.
    """
    side = 1 << (log2_facets // 2)
    if side * side != (1 << log2_facets):
        raise ValueError("log2_facets must be even")
    if spacing_m is None:
        spacing_m = 2.0 if log2_facets >= 26 else 4.0
    offsets = {1: [0.0], 2: [-0.75, 0.75], 3: [-1.5, 0.0, 1.5]}[n_channels]
    fs = 60e6
    w = _assemble(f"sweep_f{log2_facets}_l{replica_samples}_c{n_channels}", nx=side, ny=side,
                  d=spacing_m, nk=32, ntheta=8, n_pulses=n_pulses, prf=1700.0,
                  chirp_len=replica_samples / fs, bandwidth=50e6, fs=fs, n_samples=8192,
                  offsets=offsets, hetero=True, seed=seed)
    return w


def crop_rows(w: Workload, j0: int, j1: int) -> Workload:
    """A slab of facet rows [j0, j1) of the same scene as a workload of its own (input slicing only): the maps are
    sliced, the scene centre moves to the slab's centre so that every kept facet keeps its rest position, and the
    instrument, geometry and sampling window stay those of the full scene.  Used to time the oracle on a bounded
    sample of a large configuration (bench.py cpu_baseline / --impl reference)."""
    sc = dict(w.scene)
    ny = int(sc["ny"])
    if not (0 <= j0 < j1 <= ny) or sc.get("wave_nodes") is not None:
        raise ValueError("crop_rows: bad row range, or a heterogeneous-lattice workload")
    for k in ("sigma0_lin", "current_mps", "xi"):
        if sc.get(k) is not None:
            sc[k] = np.ascontiguousarray(sc[k][j0:j1])
    centre = np.array(sc["centre_m"], dtype=np.float64)
    centre[1] += (0.5 * (j0 + j1 - 1) - 0.5 * (ny - 1)) * float(sc["spacing_m"])
    sc["centre_m"] = centre
    sc["ny"] = int(j1 - j0)
    return Workload(name=f"{w.name}[rows {j0}:{j1}]", instrument=w.instrument, geometry=w.geometry, scene=sc)


def add_wave_nodes(w: Workload, spacing_m: float, seed: int = MASTER_SEED + 4) -> Workload:
    """Heterogeneous-surface variant of a workload: a lattice of wave tables of step `spacing_m`
    covering the grid, one homogeneous tile T2L per node.  Uniform sea state as the paper describes it:
    every node keeps the workload's spectrum (kx, ky, amp, omega) but draws its own phases, uncorrelated between nodes."""
    sc = w.scene
    nw = int(sc["n_waves"])
    ny_n = max(int(np.ceil((sc["ny"] - 1) * sc["spacing_m"] / spacing_m)) + 1, 2)
    nx_n = max(int(np.ceil((sc["nx"] - 1) * sc["spacing_m"] / spacing_m)) + 1, 2)
    shape = (ny_n, nx_n, nw)
    rng = np.random.Generator(np.random.PCG64(seed))
    nodes = {k: np.ascontiguousarray(np.broadcast_to(np.asarray(sc[k], dtype=np.float64), shape)) for k in ("kx", "ky", "amp", "omega")}
    nodes["phase"] = rng.uniform(0.0, 2.0 * np.pi, shape)
    nodes["spacing_m"] = float(spacing_m)
    sc["wave_nodes"] = nodes
    return w


def add_antenna_patterns(w: Workload, nu: int = 257, nv: int = 65, steer_rate_deg_s: float = 0.0,
                         margin: float = 2.5e-4) -> Workload:
    """Tabulated-antenna variant of a workload (complex Tx / Rx gains "converted into u-v grids").

    The paper's antenna-model files are not available; these synthetic tables stand in for them: on `nv` x `nu` nodes
    over the direction cosines (u along the azimuth axis, v along elevation) the scene spans during the dwell (plus
    `margin`), a uniformly illuminated aperture's field pattern with a quadratic phase error across the beam (complex,
    as a measured pattern is), stored as complex64.  `steer_rate_deg_s` != 0 adds TOPSAR-like azimuth beam steering: the
    antenna frames rotate about their elevation axis at that rate about mid-dwell (the time dependence of the gain
    enters through the per-pulse frames).  Table values are inputs; their use (lookup, interpolation) is the method's.
    """
    inst, geo, sc = w.instrument, w.geometry, w.scene
    lam = C0 / inst["f0_hz"]
    t = geo["t_pulse_s"]
    if steer_rate_deg_s:
        th = np.deg2rad(steer_rate_deg_s) * (t - 0.5 * (t[0] + t[-1]))
        c, s = np.cos(th)[:, None], np.sin(th)[:, None]
        for key in ("tx_frame", "rx_frame"):
            fr = geo[key]
            b, a = fr[:, 0].copy(), fr[:, 1].copy()
            fr[:, 0] = c * b + s * a
            fr[:, 1] = c * a - s * b
    # extent of the scene's direction cosines: the corners of the grid at the first, middle and last pulse
    hx, hy = 0.5 * (sc["nx"] - 1) * sc["spacing_m"], 0.5 * (sc["ny"] - 1) * sc["spacing_m"]
    corners = np.asarray(sc["centre_m"])[None, :] + np.array([[sx * hx, sy * hy, 0.0] for sx in (-1, 1) for sy in (-1, 1)])
    for key, ap in (("tx", inst["tx_aperture_m"]), ("rx", inst["rx_aperture_m"])):
        lo, hi = np.full(2, np.inf), np.full(2, -np.inf)
        for p in (0, len(t) // 2, len(t) - 1):
            dvec = corners - geo[key + "_pos_m"][p][None, :]
            uhat = dvec / np.linalg.norm(dvec, axis=1, keepdims=True)
            uv = np.stack([uhat @ geo[key + "_frame"][p, 1], uhat @ geo[key + "_frame"][p, 2]], axis=1)
            lo, hi = np.minimum(lo, uv.min(0)), np.maximum(hi, uv.max(0))
        ur, vr = (lo[0] - margin, hi[0] + margin), (lo[1] - margin, hi[1] + margin)
        un, vn = np.meshgrid(np.linspace(*ur, nu), np.linspace(*vr, nv))
        xa, xe = ap[0] * un / lam, ap[1] * vn / lam
        tab = np.sinc(xa) * np.sinc(xe) * np.exp(1j * (0.35 * xa**2 - 0.2 * xe))
        inst[key + "_pattern"] = dict(table=np.ascontiguousarray(tab.astype(np.complex64)), u=ur, v=vr)
    return w


def _digest_update(h, v):
    if v is None:
        h.update(b"none")
    elif isinstance(v, np.ndarray):
        h.update(str(v.dtype).encode() + str(v.shape).encode())
        h.update(np.ascontiguousarray(v).tobytes())
    elif isinstance(v, dict):
        for key in sorted(v):
            h.update(key.encode())
            _digest_update(h, v[key])
    else:
        h.update(repr(v).encode())


def workload_digest(w: Workload) -> str:
    """SHA-256 over every generated array (G22: the workload must not drift between runs)."""
    h = hashlib.sha256()
    for group in (w.instrument, w.geometry, w.scene):
        _digest_update(h, group)
    return h.hexdigest()
