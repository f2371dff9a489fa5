"""Pins for the fp64 oracle (oracle/heeps_oracle.c) against things other than itself:
closed forms evaluated with mpmath at 50 digits, textbook values, invariants, and a brute
force by an independent numpy implementation.  CPU only.

Each test names the passage it pins (PAPER.md line / SURVEY.md §8(c) step).
"""
import numpy as np
import mpmath as mp
import pytest

from oracle import oracle_generate, oracle_facets, oracle_samples
from workloads import C0, make_workload
from helpers import custom_workload

mp.mp.dps = 50
F0 = 5.405e9
LAM = C0 / F0


def _mp_norm(a, b):
    return mp.sqrt(sum((mp.mpf(float(x)) - mp.mpf(float(y))) ** 2 for x, y in zip(a, b)))


# ----------------------------------------------------------------------------- O5 + O9

def test_single_facet_is_the_delayed_chirp_mpmath():
    """One static facet, unit gains: s[n] = a exp(-j2pi f0 tau) exp(j pi K (t_n-tau)^2) on exactly
    the samples with -T/2 <= t_n - tau < T/2 (north_star sum; eq. (3); G1-G3)."""
    tx, rx, pos = (10.0, -300e3, 700e3), (250e3, -300e3, 700e3), (3.0, -7.0, 0.25)
    K, T, fs, Ns = 5e12, 2e-6, 12e6, 256
    r = _mp_norm(pos, tx) + _mp_norm(pos, rx)
    tau = r / mp.mpf(C0)
    t0 = float(tau) - 100.3 / fs
    xi = np.array([[[0.6, -0.8]]], dtype=np.float32)
    w = custom_workload(centre=pos, tx_pos=tx, rx_pos=rx, t0=t0, K=K, T=T, fs=fs, n_samples=Ns,
                        sigma0=4.0, d=1.5, xi=xi)
    s = oracle_generate(w)[0, 0]
    a = mp.sqrt(mp.mpf(4.0) * mp.mpf(1.5) ** 2) * mp.mpc(float(xi[0, 0, 0]), float(xi[0, 0, 1]))
    expect = np.zeros(Ns, dtype=np.complex128)
    support = []
    for n in range(Ns):
        u = mp.mpf(t0) + mp.mpf(n) / mp.mpf(fs) - tau
        if -mp.mpf(T) / 2 <= u < mp.mpf(T) / 2:
            support.append(n)
            val = a * mp.e ** (-2j * mp.pi * mp.mpf(F0) * tau) * mp.e ** (1j * mp.pi * mp.mpf(K) * u * u)
            expect[n] = complex(val)
    assert len(support) == 24 and support[0] == 89 and support[-1] == 112   # ceil(100.3-12) .. +L-1
    assert np.array_equal(np.nonzero(s)[0], np.array(support))
    # carrier phase: f0*tau ~ 2.8e7 cycles, the double tau itself carries ~3e-9 cycles of rounding
    assert np.max(np.abs(s - expect)) < 2e-7 * abs(complex(a))


def test_pulse_compression_peak_position_and_phase():
    """Textbook matched filter: correlating the echo with the replica peaks at (tau-t0) fs and the
    peak phase is -2 pi f0 tau (pins delay + carrier sign together)."""
    tx, rx = (0.0, -300e3, 700e3), (250e3, -300e3, 700e3)
    K, T, fs, Ns = 2.5e12, 20e-6, 60e6, 4096
    r = _mp_norm((0, 0, 0), tx) + _mp_norm((0, 0, 0), rx)
    tau = r / mp.mpf(C0)
    delay_samples = 1500.0                       # integer -> exact peak on a sample
    t0 = float(tau - mp.mpf(delay_samples) / mp.mpf(fs))
    w = custom_workload(tx_pos=tx, rx_pos=rx, t0=t0, K=K, T=T, fs=fs, n_samples=Ns)
    s = oracle_generate(w)[0, 0]
    L = int(round(T * fs))
    m = np.arange(L)
    rep = np.exp(1j * np.pi * K * (m / fs - T / 2) ** 2)
    corr = np.correlate(s, rep, mode="valid")    # sum_m s[n+m] conj(rep[m])
    peak = int(np.argmax(np.abs(corr)))
    # replica sample m sits at u = m/fs - T/2, so the echo centre is peak + L/2
    true_centre = float((tau - mp.mpf(t0)) * mp.mpf(fs))
    assert abs((peak + L / 2) - true_centre) <= 1e-6
    ph_expected = float(mp.fmod(-2 * mp.pi * mp.mpf(F0) * tau, 2 * mp.pi))
    dphi = np.angle(corr[peak] * np.exp(-1j * ph_expected))
    assert abs(dphi) < 1e-6
    assert abs(abs(corr[peak]) - L) < 1e-6 * L


def test_rect_is_half_open_and_counts_L_samples():
    """G2: rect = 1 for -1/2 <= x < 1/2.  With the echo centre exactly on a sample and L even the
    support is [centre - L/2, centre + L/2) -- the lower edge included, the upper excluded."""
    tx, rx = (0.0, 0.0, 700e3), (0.0, 0.0, 700e3)
    fs, T = 16e6, 2e-6                              # L = 32; 1/fs exactly representable scale
    tau = 2 * 700e3 / C0
    t0 = tau - 64.0 / fs
    w = custom_workload(tx_pos=tx, rx_pos=rx, t0=t0, fs=fs, T=T, n_samples=128)
    s = oracle_generate(w)[0, 0]
    nz = np.nonzero(s)[0]
    # the exact centre is 64 up to ~1e-9 samples of rounding in t0; either way 32 samples
    assert nz.size == 32 and nz[0] in (48, 49)


# ----------------------------------------------------------------------------- whole sum

def _numpy_brute(w, p):
    """Independent third implementation (vectorised numpy, complex128, different operation order):
    dense [F, Ns] evaluation of the defined sum.  Linear waves only."""
    inst, geo, sc = w.instrument, w.geometry, w.scene
    nx, ny, d = sc["nx"], sc["ny"], sc["spacing_m"]
    ii, jj = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    xb = sc["centre_m"][0] + (ii - (nx - 1) / 2) * d
    yb = sc["centre_m"][1] + (jj - (ny - 1) / 2) * d
    t = geo["t_pulse_s"][p]
    psi = (sc["kx"][:, None, None] * xb + sc["ky"][:, None, None] * yb
           - sc["omega"][:, None, None] * t + sc["phase"][:, None, None])
    z = (sc["amp"][:, None, None] * np.cos(psi)).sum(0) if sc["n_waves"] else np.zeros_like(xb)
    gz = np.stack([-(sc["amp"][:, None, None] * sc["kx"][:, None, None] * np.sin(psi)).sum(0),
                   -(sc["amp"][:, None, None] * sc["ky"][:, None, None] * np.sin(psi)).sum(0)]) \
        if sc["n_waves"] else np.zeros((2,) + xb.shape)
    cur = sc["current_mps"] if sc["current_mps"] is not None else \
        np.broadcast_to(sc["current_uniform"], (ny, nx, 2))
    pos = np.stack([xb + cur[..., 0] * t, yb + cur[..., 1] * t, sc["centre_m"][2] + z], -1).reshape(-1, 3)
    lam = C0 / inst["f0_hz"]

    def leg(ant, frame, ap):
        dv = pos - ant
        r = np.linalg.norm(dv, axis=1)
        u = dv / r[:, None]
        g = np.sinc(ap[0] * (u @ frame[1]) / lam) * np.sinc(ap[1] * (u @ frame[2]) / lam)
        return r, g

    rt, gt = leg(geo["tx_pos_m"][p], geo["tx_frame"][p], inst["tx_aperture_m"])
    vhat = geo["rx_vel_mps"][p] / np.linalg.norm(geo["rx_vel_mps"][p])
    _, gref = leg(geo["rx_pos_m"][p], geo["rx_frame"][p], inst["rx_aperture_m"])
    keep = np.ones(pos.shape[0], bool)
    if inst["cull_two_way_db"] > -300:
        keep = np.abs(gt * gref) >= 10 ** (inst["cull_two_way_db"] / 20)
    sig = sc["sigma0_lin"].astype(np.float64).ravel() if sc["sigma0_lin"] is not None else \
        np.full(pos.shape[0], sc["sigma0_uniform"])
    if sc["tilt_modulation"]:
        sig = sig * np.maximum(0.0, 1 + 2 * (gz[0].ravel() * sc["look_dir"][0] + gz[1].ravel() * sc["look_dir"][1]))
    xi = sc["xi"].astype(np.float64).reshape(-1, 2)
    a = np.sqrt(sig * d * d) * (xi[:, 0] + 1j * xi[:, 1])
    n = np.arange(inst["n_samples"])
    out = []
    for off in inst["channel_offset_m"]:
        rr, gr = leg(geo["rx_pos_m"][p] + off * vhat, geo["rx_frame"][p], inst["rx_aperture_m"])
        tau = (rt + rr) / C0
        u = geo["t0_s"][p] + n[None, :] / inst["fs_hz"] - tau[:, None]
        T = inst["chirp_len_s"]
        rect = (u >= -T / 2) & (u < T / 2) & keep[:, None]
        carrier = np.exp(-2j * np.pi * np.mod(inst["f0_hz"] * tau.astype(np.longdouble), 1.0).astype(np.float64))
        term = (a * gt * gr * carrier)[:, None] * np.exp(1j * np.pi * inst["chirp_rate_hz_per_s"] * u * u)
        out.append(np.where(rect, term, 0).sum(0))
    return np.asarray(out)


@pytest.mark.parametrize("side", [2, 4])
def test_brute_force_small_grids_independent_numpy(side):
    """Brute force on 2x2 / 4x4 grids of the Tiny recipe by an independent implementation."""
    w = make_workload("tiny", n_pulses=3)
    sc = w.scene
    sc["nx"] = sc["ny"] = side
    sc["xi"] = np.ascontiguousarray(sc["xi"][:side, :side])
    w.instrument["channel_offset_m"] = np.array([-1.5, 0.0, 1.5])
    s = oracle_generate(w)
    for p in range(3):
        ref = _numpy_brute(w, p)
        assert np.max(np.abs(s[:, p] - ref)) < 1e-7 * np.max(np.abs(ref))


def test_brute_force_with_maps_tilt_current_cull():
    """Same, exercising sigma0 map, tilt modulation, current map and the -30 dB cull (O7, O8)."""
    rng = np.random.default_rng(5)
    w = make_workload("tiny", n_pulses=2)
    sc = w.scene
    sc["nx"], sc["ny"] = 6, 5
    sc["xi"] = np.ascontiguousarray(sc["xi"][:5, :6])
    sc["sigma0_lin"] = rng.uniform(0.01, 0.1, (5, 6)).astype(np.float32)
    sc["tilt_modulation"] = 1
    sc["current_mps"] = rng.normal(0, 0.5, (5, 6, 2)).astype(np.float32)
    sc["spacing_m"] = 700.0          # spread facets across the Tx main lobe so some are culled
    w.instrument["cull_two_way_db"] = -3.0
    w.instrument["n_samples"] = 256
    f = oracle_facets(w, 1)
    assert 0 < f["keep"].sum() < 30
    s = oracle_generate(w)
    for p in range(2):
        ref = _numpy_brute(w, p)
        assert np.max(np.abs(s[:, p] - ref)) < 1e-7 * np.max(np.abs(ref))


def test_facet_velocity_is_the_time_derivative_of_the_position():
    """vel (O2: orbital + current) against a central finite difference of pos over pulse times 1 us apart:
    all three components, many components, CWM on, current map (G10)."""
    w = make_workload("tiny", n_pulses=3)
    sc = w.scene
    sc["nx"], sc["ny"] = 5, 4
    sc["xi"] = np.ascontiguousarray(sc["xi"][:4, :5])
    sc["choppy"] = 1
    sc["current_mps"] = np.random.default_rng(3).normal(0, 0.5, (4, 5, 2)).astype(np.float32)
    h = 1e-4
    w.geometry["t_pulse_s"] = np.array([0.3 - h, 0.3, 0.3 + h])
    f0, f1, f2 = (oracle_facets(w, p) for p in range(3))
    fd = (f2["pos"] - f0["pos"]) / (2 * h)
    assert np.abs(f1["vel"][:, :2]).max() > 0.3 and np.abs(f1["vel"][:, 2]).max() > 0.3
    assert np.max(np.abs(f1["vel"] - fd)) < 1e-6                  # O(h^2 w^3 A) ~ 1e-7


def test_oracle_samples_equals_oracle_generate():
    """heeps_oracle_samples (the O9 loop restricted to listed samples -- the checker of the full-size parity tests)
    against heeps_oracle_generate on Tiny with 3 channels: unsorted list, a repeated sample, samples outside every
    echo window, the first and last sample of the window; and on a culling, map-carrying scene."""
    w = make_workload("tiny", n_pulses=5)
    w.instrument["channel_offset_m"] = np.array([-1.5, 0.0, 1.5])
    full = oracle_generate(w)
    live = np.nonzero(full[1, 3])[0]
    dead = np.setdiff1d(np.arange(256), live)
    assert live.size > 30 and dead.size > 30
    ns = np.array([live[17], live[0], 255, live[-1], live[17], dead[0], 0, live[5], dead[-1], live[30]], dtype=np.int32)
    for p in (0, 3, 4):
        got = oracle_samples(w, p, ns)
        assert got.shape == (3, ns.size)
        ref = full[:, p, :][:, ns]
        assert np.max(np.abs(got - ref)) <= 1e-12 * np.abs(full).max()
        assert np.all(got[:, [2, 5, 6, 8]] == 0) and np.all(got[:, 0] == got[:, 4])
    # channels are not interchangeable here: a channel / sample stride slip would show
    assert np.abs(full[0, 3, live[17]] - full[2, 3, live[17]]) > 1e-3 * np.abs(full).max()
    # with a cull, maps and tilt: same scene as the brute-force pin
    rng = np.random.default_rng(5)
    sc = w.scene
    sc["nx"], sc["ny"] = 6, 5
    sc["xi"] = np.ascontiguousarray(sc["xi"][:5, :6])
    sc["sigma0_lin"] = rng.uniform(0.01, 0.1, (5, 6)).astype(np.float32)
    sc["tilt_modulation"] = 1
    sc["current_mps"] = rng.normal(0, 0.5, (5, 6, 2)).astype(np.float32)
    sc["spacing_m"] = 700.0
    w.instrument["cull_two_way_db"] = -3.0
    ns2 = np.arange(255, -1, -3, dtype=np.int32)
    for p in (1, 2):
        brute = _numpy_brute(w, p)
        got = oracle_samples(w, p, ns2)
        assert np.max(np.abs(got - brute[:, ns2])) < 1e-7 * np.max(np.abs(brute))


def test_oracle_samples_single_facet_mpmath_fixture():
    """heeps_oracle_samples against the stored 50-digit values of the single-facet chirp (tests/golden/
    single_facet_chirp.txt; eq. (3)): every in-window sample, listed in reverse order, plus the two
    samples just outside the half-open window."""
    from pathlib import Path
    gold = Path(__file__).resolve().parent / "golden" / "single_facet_chirp.txt"
    lines = gold.read_text().splitlines()
    t0 = float([ln for ln in lines if ln.startswith("# t0")][0].split("=")[1])
    rows = [ln.split() for ln in lines if ln and not ln.startswith("#")]
    ns = np.array([int(r[0]) for r in rows], dtype=np.int32)
    expect = np.array([float(r[1]) + 1j * float(r[2]) for r in rows])
    tx, rx, pos = (10.0, -300e3, 700e3), (250e3, -300e3, 700e3), (3.0, -7.0, 0.25)
    xi = np.array([[[0.6, -0.8]]], dtype=np.float32)
    w = custom_workload(centre=pos, tx_pos=tx, rx_pos=rx, t0=t0, K=5e12, T=2e-6, fs=12e6, n_samples=256,
                        sigma0=4.0, d=1.5, xi=xi)
    order = np.concatenate([ns[::-1], [ns[0] - 1, ns[-1] + 1]]).astype(np.int32)
    got = oracle_samples(w, 0, order)[0]
    assert np.max(np.abs(got[:ns.size] - expect[::-1])) < 2e-7 * 3.0
    assert got[-2] == 0 and got[-1] == 0


def test_linearity_and_superposition():
    """The sum is linear in a_f: scaling xi scales s; disjoint facet subsets add."""
    w = make_workload("tiny", n_pulses=2)
    xi = w.scene["xi"].copy()
    s_all = oracle_generate(w)
    mask = (np.add.outer(np.arange(64), np.arange(64)) % 3 == 0)
    w.scene["xi"] = np.where(mask[..., None], xi, 0).astype(np.float32)
    s_a = oracle_generate(w)
    w.scene["xi"] = np.where(mask[..., None], 0, xi).astype(np.float32)
    s_b = oracle_generate(w)
    scale = np.abs(s_all).max()
    assert np.max(np.abs(s_a + s_b - s_all)) < 1e-12 * scale
    w.scene["xi"] = (xi * np.float32(2.0)).astype(np.float32)      # exact in float32
    assert np.max(np.abs(oracle_generate(w) - 2 * s_all)) < 1e-12 * scale


def test_grid_reflection_invariance():
    """Permutation invariance: mirroring the grid (x -> -x with kx -> -kx, maps flipped) visits the
    same facets in another order and must give the same sum."""
    w = make_workload("tiny", n_pulses=1)
    s1 = oracle_generate(w)
    # rotate the whole world by 180 deg about z through the centre: facets, waves, platforms, frames
    R = np.diag([-1.0, -1.0, 1.0])
    g = w.geometry
    for k in ("tx_pos_m", "rx_pos_m", "tx_vel_mps", "rx_vel_mps"):
        g[k] = np.ascontiguousarray(g[k] @ R.T)
    for k in ("tx_frame", "rx_frame"):
        g[k] = np.ascontiguousarray(g[k] @ R.T)
    sc = w.scene
    sc["kx"], sc["ky"] = -sc["kx"], -sc["ky"]
    sc["xi"] = np.ascontiguousarray(sc["xi"][::-1, ::-1])
    s2 = oracle_generate(w)
    assert np.max(np.abs(s1 - s2)) < 1e-9 * np.abs(s1).max()


# ----------------------------------------------------------------------------- O6 gains

def _nadir(pos_list, ap, f0=F0):
    """Tx = Rx at 700 km straight above the origin, frame b=-z, a=+x, e=+y; one facet per call."""
    out = []
    for pos in pos_list:
        w = custom_workload(centre=pos, tx_pos=(0, 0, 700e3), rx_pos=(0, 0, 700e3), t0=0.0,
                            tx_ap=ap, rx_ap=(0.0, 0.0), f0=f0)
        out.append(oracle_facets(w, 0)["g_tx"][0])
    return np.array(out)


def test_sinc_pattern_textbook_values():
    """Uniform rectangular aperture field pattern sinc(L u / lambda) (G5):
    unit on boresight; null at u = lambda/L; sinc(1/2) = 2/pi (-3.92 dB two-... power 4/pi^2);
    first side lobe -13.26 dB with NEGATIVE field sign at L u/lambda = 1.4303."""
    La, H = 12.3, 700e3

    def x_for(arg, ap=La):     # u = x / sqrt(x^2 + H^2) = arg * lambda / ap
        u = arg * LAM / ap
        return u * H / np.sqrt(1 - u * u)

    g = _nadir([(0, 0, 0), (x_for(1.0), 0, 0), (x_for(0.5), 0, 0), (x_for(1.430297), 0, 0),
                (0.0, x_for(1.0), 0)], ap=(La, 0.0))
    assert g[0] == 1.0
    assert abs(g[1]) < 1e-9
    assert abs(g[2] - 2 / np.pi) < 1e-9 and abs(20 * np.log10(g[2] ** 2) + 7.8436) < 2e-3
    assert g[3] < 0 and abs(20 * np.log10(abs(g[3])) + 13.26) < 5e-3
    assert g[4] == 1.0                       # azimuth aperture does not see elevation offsets
    ge = _nadir([(0, x_for(1.0, 0.82), 0)], ap=(0.0, 0.82))
    assert abs(ge[0]) < 1e-9                 # elevation null of the 0.82 m aperture (u=lambda/Le)


def test_zero_gain_facet_contributes_nothing():
    """A facet sitting in a pattern null adds (numerically) nothing: removing it changes the sum by
    less than 1e-12 of the other facet's echo."""
    La, H = 12.3, 700e3
    u = LAM / La
    xnull = u * H / np.sqrt(1 - u * u)
    tau0 = 2 * H / C0
    # two facets 2*xnull/2 apart: grid 2x1 with spacing xnull centred so that facet 1 sits at x=xnull
    w = custom_workload(nx=2, ny=1, d=xnull, centre=(xnull / 2, 0, 0), tx_pos=(0, 0, H), rx_pos=(0, 0, H),
                        t0=tau0 - 50 / 12e6, tx_ap=(La, 0.0))
    both = oracle_generate(w)
    w.scene["xi"][0, 1, :] = 0
    only0 = oracle_generate(w)
    assert np.abs(only0).max() > 0.5
    assert np.max(np.abs(both - only0)) < 1e-9 * np.abs(only0).max()


# ----------------------------------------------------------------------------- O7 cull

def test_cull_threshold_changes_only_the_culled_facets():
    """O7/G6: with the cull at -X dB the output equals the no-cull output minus the culled facets'
    own contributions; and the decision is abs(G_t G_r,ref) < 10^(dB/20)."""
    w = make_workload("tiny", n_pulses=1)
    w.scene["spacing_m"] = 300.0                 # 19 km patch: reaches beyond the Tx main lobe
    w.instrument["cull_two_way_db"] = -400.0
    s_nocull = oracle_generate(w)
    f = oracle_facets(w, 0)
    w.instrument["cull_two_way_db"] = -12.0
    s_cull = oracle_generate(w)
    fk = oracle_facets(w, 0)
    # reference-channel gain == channel gain here (single channel, offset 0)
    expect_keep = np.abs(f["g_tx"] * f["g_rx"][0]) >= 10 ** (-12 / 20)
    assert np.array_equal(fk["keep"].astype(bool), expect_keep)
    assert 0.05 < expect_keep.mean() < 0.95
    xi = w.scene["xi"].copy()
    w.instrument["cull_two_way_db"] = -400.0
    w.scene["xi"] = np.where(expect_keep.reshape(64, 64)[..., None], 0, xi).astype(np.float32)
    s_culled_only = oracle_generate(w)
    assert np.max(np.abs(s_nocull - s_culled_only - s_cull)) < 1e-12 * np.abs(s_nocull).max()


# ----------------------------------------------------------------------------- O4/O5 Doppler, O3 current, channels

def _phase_history(w, c=0):
    ph = []
    for p in range(w.n_pulses):
        a = oracle_facets(w, p)["amp"][c, 0]
        ph.append(np.angle(a))
    return np.unwrap(np.array(ph))


def test_static_flat_surface_geometric_doppler():
    """Static facet, no waves/current: phi_p = -2 pi f0 tau_p exactly (mpmath geometry), and its
    finite-difference rate equals (1/lambda)(V_tx.u_t + V_rx.u_r), u = antenna->facet."""
    P, prf = 9, 1000.0
    w = make_workload("tiny", n_pulses=P)
    w.scene.update(nx=1, ny=1, n_waves=0)
    for k in ("kx", "ky", "amp", "omega", "phase"):
        w.scene[k] = np.zeros(0)
    w.scene["xi"] = np.array([[[1.0, 0.0]]], dtype=np.float32)
    w.instrument["tx_aperture_m"] = np.zeros(2)
    w.instrument["rx_aperture_m"] = np.zeros(2)
    w.scene["centre_m"] = np.array([40.0, -25.0, 0.0])
    g = w.geometry
    ph = _phase_history(w)
    pos = w.scene["centre_m"]
    exact = []
    for p in range(P):
        tau = (_mp_norm(pos, g["tx_pos_m"][p]) + _mp_norm(pos, g["rx_pos_m"][p])) / mp.mpf(C0)
        exact.append(float(mp.fmod(-2 * mp.pi * mp.mpf(F0) * tau, 2 * mp.pi)))
    d = np.angle(np.exp(1j * (ph - np.array(exact))))
    assert np.max(np.abs(d)) < 5e-7      # ulp(tau) * 2 pi f0 ~ 3e-8 rad; frac in long double
    mid = P // 2
    fd = (ph[mid + 1] - ph[mid - 1]) / (2 / prf) / (2 * np.pi)
    ut = (pos - g["tx_pos_m"][mid]); ut /= np.linalg.norm(ut)
    ur = (pos - g["rx_pos_m"][mid]); ur /= np.linalg.norm(ur)
    fd_geo = (g["tx_vel_mps"][mid] @ ut + g["rx_vel_mps"][mid] @ ur) / LAM
    # the bistatic squint Doppler (~ -42 kHz) is aliased by the PRF: compare modulo PRF
    alias = (fd - fd_geo + prf / 2) % prf - prf / 2
    assert abs(alias) < 1e-3


def test_current_adds_eq4_doppler():
    """eq. (3)-(4) PAPER.md:91-96: a facet advected at V_c adds the phase rate -K0 V_c.(r_t^ + r_r^)."""
    P, prf = 9, 1000.0
    vc = np.array([0.4, -0.7])

    def hist(cur):
        w = make_workload("tiny", n_pulses=P)
        w.scene.update(nx=1, ny=1, n_waves=0)
        for k in ("kx", "ky", "amp", "omega", "phase"):
            w.scene[k] = np.zeros(0)
        w.scene["xi"] = np.array([[[1.0, 0.0]]], dtype=np.float32)
        w.scene["current_uniform"] = np.asarray(cur, dtype=np.float64)
        return w, _phase_history(w)

    w, ph0 = hist((0.0, 0.0))
    _, ph1 = hist(vc)
    mid = P // 2
    extra = ((ph1 - ph0)[mid + 1] - (ph1 - ph0)[mid - 1]) / (2 / prf)      # rad/s
    g = w.geometry
    pos = np.array([0.0, 0.0, 0.0]) + np.array([vc[0], vc[1], 0]) * g["t_pulse_s"][mid]
    ut = pos - g["tx_pos_m"][mid]; ut /= np.linalg.norm(ut)
    ur = pos - g["rx_pos_m"][mid]; ur /= np.linalg.norm(ur)
    k0 = 2 * np.pi / LAM
    expect = -k0 * (np.array([vc[0], vc[1], 0.0]) @ (ut + ur))
    assert abs(extra - expect) < 1e-4 * abs(expect)


def test_channel_phase_difference_is_k0_path_difference():
    """Two phase centres (G8): phi_a - phi_b = -K0 (r_r,a - r_r,b) exactly (mpmath), and to first
    order K0 u_r.(P_a - P_b)."""
    w = make_workload("tiny", n_pulses=1)
    w.scene.update(nx=1, ny=1, n_waves=0)
    for k in ("kx", "ky", "amp", "omega", "phase"):
        w.scene[k] = np.zeros(0)
    w.scene["xi"] = np.array([[[1.0, 0.0]]], dtype=np.float32)
    w.scene["centre_m"] = np.array([300.0, 120.0, 0.0])
    w.instrument["tx_aperture_m"] = np.zeros(2)
    w.instrument["rx_aperture_m"] = np.zeros(2)
    w.instrument["channel_offset_m"] = np.array([-1.5, 1.5])
    # tilt the Rx velocity so the offset direction is not an axis
    w.geometry["rx_vel_mps"] = np.array([[7400.0, 900.0, -300.0]])
    f = oracle_facets(w, 0)
    dphi = np.angle(f["amp"][0, 0] * np.conj(f["amp"][1, 0]))
    vhat = w.geometry["rx_vel_mps"][0] / np.linalg.norm(w.geometry["rx_vel_mps"][0])
    pa = w.geometry["rx_pos_m"][0] - 1.5 * vhat
    pb = w.geometry["rx_pos_m"][0] + 1.5 * vhat
    pos = w.scene["centre_m"]
    dr = _mp_norm(pos, pa) - _mp_norm(pos, pb)
    exact = float(mp.fmod(-2 * mp.pi / mp.mpf(LAM) * dr, 2 * mp.pi))
    assert abs(np.angle(np.exp(1j * (dphi - exact)))) < 5e-7
    ur = pos - w.geometry["rx_pos_m"][0]; ur /= np.linalg.norm(ur)
    first = 2 * np.pi / LAM * (ur @ (pa - pb))
    assert abs(np.angle(np.exp(1j * (dphi - first)))) < 1e-3


# ----------------------------------------------------------------------------- O2 waves

def test_single_wave_component_closed_form_and_cwm_circle():
    """One component: z = A cos(k.x - w t + phi), grad z = -A k sin, dz/dt = A w sin;
    with the Choppy Wave Model flag the particle path is a circle of radius A."""
    A, kx, ky, om, phi = 0.7, 0.21, -0.13, 1.9, 0.4
    waves = dict(kx=[kx], ky=[ky], amp=[A], omega=[om], phase=[phi])
    ts = np.linspace(0.0, 2 * np.pi / om, 13)
    P = len(ts)
    tx = np.repeat([[0, -300e3, 700e3]], P, 0)
    CUR = (0.3, -0.2)
    w = custom_workload(nx=3, ny=2, d=5.0, centre=(10.0, 20.0, 1.0), waves=waves, t_pulse=ts,
                        tx_pos=tx, rx_pos=tx, t0=0.0, current=CUR)
    for choppy in (0, 1):
        w.scene["choppy"] = choppy
        path = []
        for p, t in enumerate(ts):
            f = oracle_facets(w, p)
            i, j = 2, 1
            xb, yb = 10.0 + (i - 1.0) * 5.0, 20.0 + (j - 0.5) * 5.0
            psi = kx * xb + ky * yb - om * t + phi
            fidx = j * 3 + i
            assert abs(f["pos"][fidx, 2] - (1.0 + A * np.cos(psi))) < 1e-13
            assert np.allclose(f["slope"][fidx], [-A * kx * np.sin(psi), -A * ky * np.sin(psi)], atol=1e-14)
            assert abs(f["vel"][fidx, 2] - A * om * np.sin(psi)) < 1e-13
            # horizontal facet velocity: the current, plus (CWM) the orbital velocity A w k^ cos(psi) -- the time
            # derivative of the horizontal displacement -A k^ sin(psi)
            khat_ = np.array([kx, ky]) / np.hypot(kx, ky)
            vh = np.array(CUR) + (A * om * np.cos(psi) * khat_ if choppy else 0.0)
            assert np.allclose(f["vel"][fidx, :2], vh, atol=1e-13)
            if not choppy:
                assert abs(f["pos"][fidx, 0] - (xb + CUR[0] * t)) < 1e-13 and abs(f["pos"][fidx, 1] - (yb + CUR[1] * t)) < 1e-13
            path.append(f["pos"][fidx] - np.array([xb + CUR[0] * t, yb + CUR[1] * t, 1.0]))
        if choppy:
            path = np.array(path)
            khat = np.array([kx, ky]) / np.hypot(kx, ky)
            along = path[:, :2] @ khat
            assert np.allclose(along**2 + path[:, 2] ** 2, A * A, atol=1e-13)      # circle
            assert np.allclose(path[:, :2] - np.outer(along, khat), 0, atol=1e-13)  # in the k-z plane


def test_height_variance_is_half_sum_of_squared_amplitudes():
    """Grid variance of z -> sum A_w^2 / 2 (random-phase linear surface)."""
    w = make_workload("ati", n_pulses=1)
    w.scene["nx"] = w.scene["ny"] = 256
    w.scene["xi"] = np.ascontiguousarray(w.scene["xi"][:256, :256])
    w.scene["spacing_m"] = 16.0            # 4 km patch: many wavelengths of every component
    f = oracle_facets(w, 0)
    var = f["pos"][:, 2].var()
    expect = (w.scene["amp"] ** 2).sum() / 2
    assert abs(var - expect) < 0.1 * expect


# ----------------------------------------------------------------------------- O8 amplitude / radiometry

def test_tilt_modulation_factor_and_clamp():
    """G12: sigma = sigma0 max(0, 1 + 2 grad z . n)."""
    A, k = 2.0, 0.4                                   # slope amplitude 0.8 -> factor spans [-0.6, 2.6]
    waves = dict(kx=[k], ky=[0.0], amp=[A], omega=[0.0], phase=[0.0])
    w = custom_workload(nx=16, ny=1, d=1.0, waves=waves, tx_pos=(0, 0, 700e3), rx_pos=(0, 0, 700e3),
                        t0=0.0, tilt=1, look=(1.0, 0.0), sigma0=0.25)
    f = oracle_facets(w, 0)
    x = (np.arange(16) - 7.5)
    fac = np.maximum(0.0, 1 + 2 * (-A * k * np.sin(k * x)))
    assert (fac == 0).any() and (fac > 2).any()
    assert np.allclose(np.abs(f["amp"][0]), np.sqrt(0.25 * fac), atol=1e-12)


def test_mean_power_radiometry_over_seeds():
    """E |s[n]|^2 = sum over facets covering n of sigma0 d^2 G_t^2 G_r^2 (speckle mean power)."""
    acc = 0
    K = 24
    for s in range(K):
        w = make_workload("tiny", n_pulses=1, seed=1000 + 7 * s)
        acc = acc + np.abs(oracle_generate(w)[0, 0]) ** 2
    mean_pow = acc / K
    w = make_workload("tiny", n_pulses=1)
    f = oracle_facets(w, 0)
    g2 = (f["g_tx"] * f["g_rx"][0]) ** 2 * w.scene["sigma0_uniform"] * w.scene["spacing_m"] ** 2
    # in the plateau (samples covered by every facet's replica) the expected power is the full sum
    nz = np.nonzero(mean_pow)[0]
    plateau = mean_pow[nz[0] + 14: nz[-1] - 13]
    assert plateau.size >= 8
    expect = g2.sum()
    # relative std of the estimate ~ 1/sqrt(K * plateau.size / correlation) -> generous 25 %
    assert abs(plateau.mean() - expect) < 0.25 * expect


# ----------------------------------------------------------------------------- generator pins

def test_pierson_moskowitz_closed_form_hs():
    """Hs = 2 sqrt(alpha/beta) U^2/g = 2.133 m at U = 10 m/s; the 0.05-1 rad/m band holds 2.06 m."""
    from scipy.integrate import quad
    from workloads import pm_spectrum
    m0, _ = quad(lambda k: float(pm_spectrum(np.array([k]))[0]), 1e-4, 50.0, limit=400)
    hs = 4 * np.sqrt(m0)
    assert abs(hs - 2 * np.sqrt(8.1e-3 / 0.74) * 100 / 9.81) < 2e-3
    assert abs(hs - 2.133) < 2e-3
    for name in ("tiny", "ati"):
        w = make_workload(name, n_pulses=1)
        hs_band = 4 * np.sqrt((w.scene["amp"] ** 2).sum() / 2)
        assert abs(hs_band - 2.06) < 0.03
    w = make_workload("ati", n_pulses=1)
    slope_rms = np.sqrt((w.scene["amp"] ** 2 * (w.scene["kx"] ** 2 + w.scene["ky"] ** 2)).sum() / 2)
    assert abs(slope_rms - 0.094) < 0.01


def test_workloads_are_frozen():
    """G22: the generated arrays must not drift between runs (same seed -> same bytes)."""
    from workloads import workload_digest
    a = workload_digest(make_workload("tiny"))
    b = workload_digest(make_workload("tiny"))
    assert a == b
    assert workload_digest(make_workload("tiny", seed=1)) != a
    w = make_workload("tiny")
    xi = w.scene["xi"].astype(np.float64)
    assert abs((xi ** 2).sum(-1).mean() - 1.0) < 0.05        # E|xi|^2 = 1
    assert abs(xi.mean()) < 0.02


@pytest.mark.parametrize("name", ["tiny", "ati", "hetero", "large", "sweep20", "sweep22", "sweep24", "sweep26"])
def test_workload_digests_match_the_committed_file(name):
    """G22: every seeded workload against its committed fingerprint (tests/golden/workload_digests.txt, written by
    tests/golden/make_workload_digests.py from workloads/ alone): same keys, dtypes and shapes, checksums to 1e-9
    (of the Cauchy-Schwarz scale sqrt(n sum_sq)).  A byte-level (SHA-256) difference with matching checksums is a
    last-bit libm / FFT difference of the platform and is reported, not failed."""
    import importlib.util
    import warnings
    from pathlib import Path
    gold_dir = Path(__file__).resolve().parent / "golden"
    spec = importlib.util.spec_from_file_location("make_workload_digests", gold_dir / "make_workload_digests.py")
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    want = {}
    for ln in (gold_dir / "workload_digests.txt").read_text().splitlines():
        if ln and not ln.startswith("#"):
            cfg, key, dt, shape, s1, s2, s3, sha = ln.split()
            if cfg == name:
                want[key] = (dt, shape, float(s1), float(s2), float(s3), sha)
    assert want, name
    got = mod.fingerprint(mod.build(name))
    assert sorted(k for k, *_ in got) == sorted(want)
    drift = []
    for key, dt, shape, s1, s2, s3, sha in got:
        wdt, wshape, w1, w2, w3, wsha = want[key]
        assert (dt, shape) == (wdt, wshape), key
        n = max(int(np.prod(eval(shape))) if shape != "()" else 1, 1)
        scale = np.sqrt(n * w2)
        assert abs(s2 - w2) <= 1e-9 * w2, key
        assert abs(s1 - w1) <= 1e-9 * scale and abs(s3 - w3) <= 1e-9 * scale, key
        if sha != wsha:
            drift.append(key)
    if drift:
        warnings.warn(f"{name}: byte-level differences within 1e-9 in {drift}")


# ----------------------------------------------------------------------------- NEXT-4: the paper's fast mode (CPU restatement)

def _ati_crop(n=24, n_pulses=9):
    w = make_workload("ati", n_pulses=n_pulses)
    sc = w.scene
    j0 = 256 - n // 2
    sc["xi"] = np.ascontiguousarray(sc["xi"][j0:j0 + n, j0:j0 + n])
    sc["nx"] = sc["ny"] = n
    return w


def test_fast_mode_restatement_reduces_to_the_defined_sum():
    """oracle/fast_mode.py (Doppler spectrum per range gate at PRF/n_fast, 1-D IFFT, linear combination):
    with n_fast = 1 every pulse is a node and the scheme IS the defined sum (pins the restatement to heeps_oracle.c);
    with n_fast > 1 it departs from it, the less the finer the Doppler bins; node pulses stay exact."""
    from oracle import rel_l2_per_vector
    from oracle.fast_mode import fast_mode_generate
    w = _ati_crop()
    ref = oracle_generate(w)
    exact = fast_mode_generate(w, 1, 64)
    assert np.max(np.abs(exact - ref)) <= 1e-9 * np.abs(ref).max()
    coarse = rel_l2_per_vector(fast_mode_generate(w, 4, 64), ref)
    fine = rel_l2_per_vector(fast_mode_generate(w, 4, 4096), ref)
    assert np.all(coarse[:, [0, 4, 8]] < 1e-9) and np.all(fine[:, [0, 4, 8]] < 1e-9)     # nodes
    mid = [2, 6]
    assert np.all(coarse[:, mid] > 3 * fine[:, mid]) and fine[:, mid].min() > 0
    assert fine[:, mid].max() > 1e-4            # still outside the parity bar at 1024 bins per skipped pulse
