"""Hand-built descriptor sets for closed-form tests (no method arithmetic here)."""
from __future__ import annotations

import numpy as np

from workloads import Workload


def custom_workload(*, nx=1, ny=1, d=1.0, centre=(0.0, 0.0, 0.0), waves=None, xi=None,
                    tx_pos, rx_pos, tx_vel=None, rx_vel=None, tx_frame=None, rx_frame=None,
                    t_pulse=None, t0, f0=5.405e9, K=5e12, T=2e-6, fs=12e6, n_samples=256,
                    tx_ap=(0.0, 0.0), rx_ap=(0.0, 0.0), offsets=(0.0,), cull_db=-400.0,
                    sigma0=1.0, sigma0_map=None, tilt=0, look=(0.0, 1.0), current=(0.0, 0.0),
                    current_map=None, choppy=0) -> Workload:
    tx_pos = np.atleast_2d(np.asarray(tx_pos, dtype=np.float64))
    rx_pos = np.atleast_2d(np.asarray(rx_pos, dtype=np.float64))
    P = tx_pos.shape[0]
    eye = np.array([[0.0, 0.0, -1.0], [1.0, 0.0, 0.0], [0.0, 1.0, 0.0]])

    def rep(a, default):
        a = default if a is None else np.asarray(a, dtype=np.float64)
        if a.ndim == np.asarray(default).ndim:
            a = np.repeat(a[None], P, 0)
        return np.ascontiguousarray(a)

    geo = dict(
        n_pulses=P,
        t_pulse_s=np.zeros(P) if t_pulse is None else np.asarray(t_pulse, dtype=np.float64),
        tx_pos_m=tx_pos, rx_pos_m=rx_pos,
        tx_vel_mps=rep(tx_vel, np.array([7500.0, 0.0, 0.0])),
        rx_vel_mps=rep(rx_vel, np.array([7500.0, 0.0, 0.0])),
        tx_frame=rep(tx_frame, eye), rx_frame=rep(rx_frame, eye),
        t0_s=np.broadcast_to(np.asarray(t0, dtype=np.float64), (P,)).copy(),
    )
    if waves is None:
        waves = dict(kx=[], ky=[], amp=[], omega=[], phase=[])
    sc = dict(nx=nx, ny=ny, spacing_m=float(d), centre_m=np.asarray(centre, dtype=np.float64),
              n_waves=len(waves["kx"]), choppy=choppy,
              sigma0_lin=sigma0_map, sigma0_uniform=float(sigma0), tilt_modulation=tilt,
              look_dir=np.asarray(look, dtype=np.float64), current_mps=current_map,
              current_uniform=np.asarray(current, dtype=np.float64), seed=0)
    for k in ("kx", "ky", "amp", "omega", "phase"):
        sc[k] = np.asarray(waves[k], dtype=np.float64)
    if xi is None:
        xi = np.zeros((ny, nx, 2), dtype=np.float32)
        xi[..., 0] = 1.0
    sc["xi"] = np.ascontiguousarray(xi, dtype=np.float32)
    inst = dict(f0_hz=f0, chirp_rate_hz_per_s=K, chirp_len_s=T, fs_hz=fs, prf_hz=1000.0,
                n_samples=n_samples, tx_aperture_m=np.asarray(tx_ap, dtype=np.float64),
                rx_aperture_m=np.asarray(rx_ap, dtype=np.float64),
                channel_offset_m=np.asarray(offsets, dtype=np.float64), cull_two_way_db=cull_db)
    return Workload(name="custom", instrument=inst, geometry=geo, scene=sc)
