"""CPU restatement of the paper's "fast mode" (section IV.B) -- TEST INFRASTRUCTURE, like everything
under oracle/: nothing in the product path imports it.

The paper: "a 'fast mode' ... consists in estimating the Doppler spectrum of each range gate at a frequency PRF/n_fast
smaller than the PRF, then generating the missing pulses through 1D IFFT and linear combination of the resulting
signals ... very similar to the method used to generate heterogeneous surfaces, but in 1D".  It gives no formulas;
the reading taken here, written out step by step and deliberately slowly:

  F1  node pulses p_i = i n_fast (and the last pulse).  At a node every facet-echo is evaluated exactly as in the
      defined sum (oracle steps O1..O8): delay tau_f, complex amplitude A~_f = a G_t G_r exp(-j 2 pi f0 tau_f).
  F2  Doppler of a facet-echo at the node: f_f = -f0 d tau_f / dt, from the exact delays one pulse apart.
  F3  Doppler spectrum: the echo goes into bin m_f = round(f_f N_d / PRF) mod N_d of N_d bins over one PRF; range gates
      are frozen at the node (delay relative to the sampling window, tau_f - t0, kept).
  F4  the 1-D inverse FFT over m of a gate's spectrum is its time series at the PRF: k pulses from the node the echo's
      phase has advanced by 2 pi m_f k / N_d.  Here the sum over facet-echoes is taken directly (an IFFT is a fast way
      to evaluate exactly this sum; nothing else changes), and each echo lays down its chirp replica at its frozen delay.
  F5  a pulse between nodes i and i + 1, a fraction s of the way: (1 - s) x node i's series + s x node i + 1's.

n_fast = 1 makes every pulse a node (k = 0, s = 0): the exact defined sum, which pins this file to heeps_oracle.c.
The error against the exact sum for n_fast > 1 is what oracle/fast_mode_table.py tabulates.
"""
from __future__ import annotations

import numpy as np

from .binding import oracle_facets


def _lay_replicas(out, tau_rel, amp, fs, T, K, n_samples):
    """out[n] += sum_f amp_f rect((n/fs - tau_rel_f)/T) exp(j pi K (n/fs - tau_rel_f)^2)   (O9, delays relative to sample 0)."""
    L = int(np.ceil(T * fs)) + 1
    nu = tau_rel * fs - 0.5 * T * fs
    first = np.ceil(nu).astype(np.int64)
    for m in range(L):
        n = first + m
        u = n / fs - tau_rel
        ok = (u >= -0.5 * T) & (u < 0.5 * T) & (n >= 0) & (n < n_samples)
        if not ok.any():
            continue
        np.add.at(out, n[ok], amp[ok] * np.exp(1j * np.pi * K * u[ok] ** 2))


def fast_mode_generate(w, n_fast: int, n_doppler: int) -> np.ndarray:
    """complex128 [C][P][Ns]: the fast-mode approximation of the defined sum (steps F1..F5 above)."""
    inst, geo = w.instrument, w.geometry
    P, C, Ns = int(geo["n_pulses"]), len(inst["channel_offset_m"]), int(inst["n_samples"])
    fs, T, K, f0 = inst["fs_hz"], inst["chirp_len_s"], inst["chirp_rate_hz_per_s"], inst["f0_hz"]
    t, t0 = np.asarray(geo["t_pulse_s"]), np.asarray(geo["t0_s"])
    pri = (t[-1] - t[0]) / max(P - 1, 1) if P > 1 else 1.0
    nodes = sorted(set(list(range(0, P, n_fast)) + [P - 1]))
    series = {}                                            # node -> (tau - t0 [C][F], amp [C][F], Doppler bin [C][F])
    for p in nodes:
        f = oracle_facets(w, p)
        q = p + 1 if p + 1 < P else p - 1                  # F2: exact delays one pulse apart
        if P == 1:
            dop = np.zeros_like(f["tau"])
        else:
            g = oracle_facets(w, q)
            dop = -f0 * (g["tau"] - f["tau"]) / (t[q] - t[p])                      # Hz
        m = np.mod(np.rint(dop * pri * n_doppler), n_doppler)                       # F3
        amp = np.where(f["keep"][None, :].astype(bool), f["amp"], 0.0)             # O7
        series[p] = (f["tau"] - t0[p], amp, m)
    out = np.zeros((C, P, Ns), dtype=np.complex128)
    for p in range(P):
        lo = max(n for n in nodes if n <= p)
        hi = min(n for n in nodes if n >= p)
        parts = [(lo, 1.0)] if lo == hi else [(lo, (hi - p) / (hi - lo)), (hi, (p - lo) / (hi - lo))]     # F5
        for node, wgt in parts:
            tau_rel, amp, m = series[node]
            k = (t[p] - t[node]) / pri                     # pulses from the node
            for c in range(C):
                a = wgt * amp[c] * np.exp(2j * np.pi * m[c] * k / n_doppler)        # F4
                _lay_replicas(out[c, p], tau_rel[c], a, fs, T, K, Ns)
    return out
