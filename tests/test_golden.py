"""The oracle against the stored fixtures of tests/golden/ (each file's header cites its source).

`sinc_pattern.txt`, `single_facet_chirp.txt`, `pierson_moskowitz.txt` hold values fixed by mathematics
(mpmath, 50 digits, written by tests/golden/make_golden.py without touching this repository's code);
`tiny_oracle_samples.txt` freezes the oracle itself on the seeded Tiny workload.  CPU only.
"""
from pathlib import Path

import numpy as np

from oracle import oracle_facets, oracle_generate
from workloads import C0, make_workload, pm_spectrum
from helpers import custom_workload

GOLD = Path(__file__).resolve().parent / "golden"


def _rows(name):
    return [ln.split() for ln in (GOLD / name).read_text().splitlines() if ln and not ln.startswith("#")]


def test_sinc_pattern_fixture():
    """O6 gain of one facet placed at direction cosine u = x * lambda / La against sinc(x) (G5)."""
    lam = C0 / 5.405e9
    La = 12.3
    for x_s, v_s, _ in _rows("sinc_pattern.txt"):
        x, v = float(x_s), float(v_s)
        u = x * lam / La                                  # direction cosine along the azimuth axis
        r = 700e3
        pos = (u * r, 0.0, -np.sqrt(1.0 - u * u) * r)     # boresight -z, azimuth +x (helpers' default frame)
        w = custom_workload(centre=pos, tx_pos=(0.0, 0.0, 0.0), rx_pos=(0.0, 0.0, 0.0), t0=2 * r / C0 - 1e-5,
                            tx_ap=(La, 0.0), rx_ap=(0.0, 0.0))
        g = oracle_facets(w, 0)["g_tx"][0]
        assert abs(g - v) < 2e-9, (x, g, v)


def test_single_facet_chirp_fixture():
    """Same scene as test_single_facet_is_the_delayed_chirp_mpmath, against the stored 50-digit values."""
    tx, rx, pos = (10.0, -300e3, 700e3), (250e3, -300e3, 700e3), (3.0, -7.0, 0.25)
    head = [ln for ln in (GOLD / "single_facet_chirp.txt").read_text().splitlines() if ln.startswith("# t0")][0]
    t0 = float(head.split("=")[1])
    xi = np.array([[[0.6, -0.8]]], dtype=np.float32)
    w = custom_workload(centre=pos, tx_pos=tx, rx_pos=rx, t0=t0, K=5e12, T=2e-6, fs=12e6, n_samples=256,
                        sigma0=4.0, d=1.5, xi=xi)
    s = oracle_generate(w)[0, 0]
    rows = _rows("single_facet_chirp.txt")
    ns = np.array([int(r[0]) for r in rows])
    expect = np.array([float(r[1]) + 1j * float(r[2]) for r in rows])
    assert np.array_equal(np.nonzero(s)[0], ns) and ns.size == 24
    assert np.max(np.abs(s[ns] - expect)) < 2e-7 * 3.0


def test_pierson_moskowitz_fixture():
    """Generator spectrum: integral of S(k) over all k equals Hs^2/16 with the stored closed-form Hs."""
    k = np.geomspace(1e-4, 1e3, 400001)
    for u_s, hs_s in _rows("pierson_moskowitz.txt"):
        m0 = np.trapezoid(pm_spectrum(k, float(u_s)), k)
        assert abs(4.0 * np.sqrt(m0) - float(hs_s)) < 2e-4 * float(hs_s)


def test_tiny_oracle_is_frozen():
    """The oracle's arithmetic has not drifted from the committed values (tests/golden/make_golden.py)."""
    rows = _rows("tiny_oracle_samples.txt")
    pulses = sorted({int(r[0]) for r in rows})
    ref = oracle_generate(make_workload("tiny"), pulses)
    for p_s, n_s, re_s, im_s in rows:
        got = ref[0, pulses.index(int(p_s)), int(n_s)]
        want = float(re_s) + 1j * float(im_s)
        assert abs(got - want) <= 1e-9 * max(1.0, abs(want)), (p_s, n_s, got, want)
