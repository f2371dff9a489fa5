"""Pins for the oracle's time-dependent intra-facet speckle (eq. (7), (9),
(10)) against things other than itself: the published known-answer vectors of Philox4x32-10, an independent
pure-Python restatement, the statistics the paper states, and the limiting cases.  CPU only.
"""
import numpy as np

from oracle import oracle_generate, oracle_philox, oracle_speckle
from workloads import make_workload
from helpers import custom_workload


def test_philox4x32_10_known_answers():
    """The oracle's counter-based generator (reading G27) against the known-answer vectors distributed with
    Random123 (Salmon, Moraes, Dror, Shaw, SC'11; kat_vectors, philox4x32 with 10 rounds)."""
    kat = [
        ([0, 0, 0, 0], [0, 0], [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]),
        ([0xFFFFFFFF] * 4, [0xFFFFFFFF] * 2, [0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD]),
        ([0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344], [0xA4093822, 0x299F31D0],
         [0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1]),
    ]
    for ctr, key, expect in kat:
        assert [int(x) for x in oracle_philox(ctr, key)] == expect


def _philox_py(ctr, key):
    """Third implementation with Python integers (Salmon et al., SC'11, Fig. 2: Philox-4x32 round and key bump)."""
    c, k = list(ctr), list(key)
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & 0xFFFFFFFF, p1 & 0xFFFFFFFF,
             ((p0 >> 32) ^ c[3] ^ k[1]) & 0xFFFFFFFF, p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return c


def _speckle_workload(nx=128, ny=128, P=24, tau=4e-3, fs_hz=35.0):
    w = make_workload("tiny", n_pulses=P)
    rng = np.random.default_rng(11)
    w.scene["nx"], w.scene["ny"] = nx, ny
    w.scene["xi"] = (rng.standard_normal((ny, nx, 2)) * np.sqrt(0.5)).astype(np.float32)
    w.scene["speckle_tau_s"], w.scene["speckle_doppler_hz"] = tau, fs_hz
    w.scene["seed"] = 0x1234567_89ABCDEF
    return w


def test_ar1_recursion_against_python_restatement():
    """Eq. (10) step by step with Python floats and the Python Philox for a few facets: s(t_p) of eq. (7)."""
    w = _speckle_workload(nx=7, ny=5, P=9)
    t = w.geometry["t_pulse_s"]
    tau, fd, seed = w.scene["speckle_tau_s"], w.scene["speckle_doppler_hz"], w.scene["seed"]
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for p in (0, 1, 8):
        got = oracle_speckle(w, p).reshape(-1)
        for f in (0, 3, 34):
            s = complex(*w.scene["xi"].reshape(-1, 2)[f].astype(np.float64))
            for q in range(1, p + 1):
                beta = np.exp(-(t[q] - t[q - 1]) / tau)
                w0, w1, _, _ = _philox_py([f, 0, q, 1], key)
                u1, u2 = ((w0 >> 8) + 1) / 2.0**24, (w1 >> 8) / 2.0**24
                s = beta * s + np.sqrt(1 - beta**2) * np.sqrt(-np.log(u1)) * np.exp(2j * np.pi * u2)
            s *= np.exp(2j * np.pi * fd * t[p])
            assert abs(got[f] - s) < 1e-13


def test_ar1_statistics_match_the_paper():
    """<|s|^2> = 1 at every pulse; <s(t+k dt) s*(t)> = exp(-k dt/tau_s) exp(+2 i pi f_s k dt)
    (eq. (9) with the exponential form of eq. (10)); innovations of different facets uncorrelated."""
    w = _speckle_workload()
    t = w.geometry["t_pulse_s"]
    dt, tau, fd = t[1] - t[0], w.scene["speckle_tau_s"], w.scene["speckle_doppler_hz"]
    s = np.stack([oracle_speckle(w, p).reshape(-1) for p in range(len(t))])     # [P][F]
    n = s.shape[1]
    tol = 4.0 / np.sqrt(n)
    assert np.all(np.abs((np.abs(s) ** 2).mean(axis=1) - 1.0) < 2 * tol)
    assert abs(s[-1].mean()) < tol
    for k in (1, 3, 8):
        corr = (s[k:] * np.conj(s[:-k])).mean()
        expect = np.exp(-k * dt / tau) * np.exp(2j * np.pi * fd * k * dt)
        assert abs(corr - expect) < tol, (k, corr, expect)
    inn = s[1] * np.exp(-2j * np.pi * fd * t[1]) - np.exp(-dt / tau) * s[0] * np.exp(-2j * np.pi * fd * t[0])
    assert abs((inn[1:] * np.conj(inn[:-1])).mean()) < tol * (1 - np.exp(-2 * dt / tau))


def test_ar1_limits():
    """tau_s <= 0: the speckle is the static xi; tau_s -> infinity: beta = 1, s(t) = xi exp(2 i pi f_s t)."""
    w = _speckle_workload(nx=16, ny=8, P=6)
    xi = w.scene["xi"][..., 0].astype(np.float64) + 1j * w.scene["xi"][..., 1]
    t = w.geometry["t_pulse_s"]
    w.scene["speckle_tau_s"] = 0.0
    assert np.array_equal(oracle_speckle(w, 5), xi)
    w.scene["speckle_tau_s"] = 1e30
    assert np.max(np.abs(oracle_speckle(w, 5) - xi * np.exp(2j * np.pi * w.scene["speckle_doppler_hz"] * t[5]))) < 1e-12


def test_output_is_linear_in_the_speckle():
    """The speckle multiplies the facet amplitude (eq. (5)): one facet's echo with the AR(1) speckle equals its
    static-speckle echo times s(t_p)/xi, pulse by pulse."""
    tx = np.array([[7.5 * p - 30.0, -300e3, 700e3] for p in range(8)])
    rx = tx + np.array([250e3, 0, 0])
    tp = np.arange(8) / 1000.0
    r0 = np.linalg.norm(tx[0]) + np.linalg.norm(rx[0])
    from workloads import C0
    t0 = r0 / C0 - 100.0 / 12e6
    w = custom_workload(tx_pos=tx, rx_pos=rx, t_pulse=tp, t0=t0, xi=np.array([[[0.3, -1.1]]], dtype=np.float32))
    ref = oracle_generate(w)
    w.scene["speckle_tau_s"], w.scene["speckle_doppler_hz"], w.scene["seed"] = 2.5e-3, -80.0, 77
    got = oracle_generate(w)
    xi = complex(0.3, -1.1) if False else complex(np.float32(0.3), np.float32(-1.1))
    for p in range(8):
        s = oracle_speckle(w, p)[0, 0]
        assert np.abs(ref[0, p]).max() > 0
        assert np.max(np.abs(got[0, p] - ref[0, p] * (s / xi))) < 1e-12 * np.abs(ref[0, p]).max() * max(1.0, abs(s / xi))
