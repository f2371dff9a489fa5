"""Writes the stored expected values under tests/golden/.

    python tests/golden/make_golden.py

Two kinds of file:
  * values fixed by mathematics, evaluated with mpmath at 50 digits from the closed form the
    citation names (no code of this repository is involved): `sinc_pattern.txt`,
    `single_facet_chirp.txt`, `pierson_moskowitz.txt`;
  * values written by the fp64 oracle (`oracle/` only -- never the CUDA path) on the seeded
    Tiny workload: `tiny_oracle_samples.txt`.  They freeze the oracle: a later change to its
    arithmetic shows up as a diff of this file and must cite the passage that justifies it.
"""
from __future__ import annotations

import sys
from pathlib import Path

import mpmath as mp
import numpy as np

HERE = Path(__file__).resolve().parent
ROOT = HERE.parent.parent
sys.path.insert(0, str(ROOT))
sys.path.insert(0, str(HERE.parent))

mp.mp.dps = 50
C0 = mp.mpf(299792458)


def write_sinc_pattern():
    """Field pattern of a uniform aperture, sinc(x) = sin(pi x)/(pi x) (reading G5; PAPER.md:202
    antenna patterns; textbook values: 4/pi^2 power at x = 1/2, first side lobe -13.26 dB)."""
    lines = ["# x  sinc(x)  20log10|sinc(x)|   (mpmath, 50 digits; reading G5, PAPER.md:202)"]
    first_lobe = mp.findroot(lambda x: mp.diff(lambda t: mp.sin(mp.pi * t) / (mp.pi * t), x), 1.43)
    for x in [mp.mpf(0), mp.mpf("0.25"), mp.mpf("0.5"), mp.mpf(1), first_lobe, mp.mpf(2), mp.mpf("2.5")]:
        v = mp.mpf(1) if x == 0 else mp.sin(mp.pi * x) / (mp.pi * x)
        db = "-inf" if abs(v) < mp.mpf(10) ** -40 else mp.nstr(20 * mp.log10(abs(v)), 12)
        lines.append(f"{mp.nstr(x, 20)} {mp.nstr(v, 20)} {db}")
    (HERE / "sinc_pattern.txt").write_text("\n".join(lines) + "\n")


def write_single_facet():
    """One static facet, isotropic antennas (north_star sum; eq. (3), G1-G3):
    s[n] = a exp(-j2pi f0 tau) exp(j pi K (t_n - tau)^2) on -T/2 <= t_n - tau < T/2."""
    tx, rx, pos = (10.0, -300e3, 700e3), (250e3, -300e3, 700e3), (3.0, -7.0, 0.25)
    f0, K, T, fs, Ns = mp.mpf(5.405e9), mp.mpf(5e12), mp.mpf(2e-6), mp.mpf(12e6), 256
    dist = lambda a, b: mp.sqrt(sum((mp.mpf(x) - mp.mpf(y)) ** 2 for x, y in zip(a, b)))
    tau = (dist(pos, tx) + dist(pos, rx)) / C0
    t0 = mp.mpf(float(tau) - 100.3 / 12e6)          # the double the test passes as t0
    a = mp.sqrt(mp.mpf(4) * mp.mpf("1.5") ** 2) * mp.mpc(mp.mpf(np.float32(0.6).item()), mp.mpf(np.float32(-0.8).item()))
    lines = ["# n  Re s[n]  Im s[n]   (mpmath, 50 digits; eq. (3) PAPER.md:91; sigma0 = 4, d = 1.5, xi = (0.6, -0.8) float32)",
             f"# t0 = {mp.nstr(t0, 25)}"]
    for n in range(Ns):
        u = t0 + mp.mpf(n) / fs - tau
        if -T / 2 <= u < T / 2:
            v = a * mp.e ** (-2j * mp.pi * f0 * tau) * mp.e ** (1j * mp.pi * K * u * u)
            lines.append(f"{n} {mp.nstr(v.real, 18)} {mp.nstr(v.imag, 18)}")
    (HERE / "single_facet_chirp.txt").write_text("\n".join(lines) + "\n")


def write_pm():
    """Pierson-Moskowitz closed form Hs = 2 sqrt(alpha/beta) U^2/g (generator pin)."""
    alpha, beta, g = mp.mpf("8.1e-3"), mp.mpf("0.74"), mp.mpf("9.81")
    lines = ["# U[m/s]  Hs[m] = 2 sqrt(alpha/beta) U^2 / g   (alpha = 8.1e-3, beta = 0.74, g = 9.81)"]
    for u in (5, 10, 15):
        lines.append(f"{u} {mp.nstr(2 * mp.sqrt(alpha / beta) * mp.mpf(u) ** 2 / g, 15)}")
    (HERE / "pierson_moskowitz.txt").write_text("\n".join(lines) + "\n")


def write_tiny_oracle():
    from oracle import oracle_generate
    from workloads import make_workload
    w = make_workload("tiny")
    pulses = [0, 13, 31]
    ref = oracle_generate(w, pulses)
    lines = ["# pulse n Re Im   fp64 oracle on make_workload('tiny'), channel 0; written by make_golden.py (oracle/ only)"]
    for k, p in enumerate(pulses):
        live = np.nonzero(ref[0, k])[0]
        for n in list(live[:3]) + list(live[len(live) // 2: len(live) // 2 + 3]) + list(live[-3:]):
            lines.append(f"{p} {n} {ref[0, k, n].real:.15e} {ref[0, k, n].imag:.15e}")
        lines.append(f"# pulse {p}: support [{live[0]}, {live[-1]}], energy {np.sum(np.abs(ref[0, k]) ** 2):.15e}")
    (HERE / "tiny_oracle_samples.txt").write_text("\n".join(lines) + "\n")


if __name__ == "__main__":
    write_sinc_pattern()
    write_single_facet()
    write_pm()
    write_tiny_oracle()
    print("golden files written to", HERE)
