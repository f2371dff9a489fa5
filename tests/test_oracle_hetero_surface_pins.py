"""Pins for the oracle's heterogeneous surface (eq. (1), (2)): four homogeneous
tiles T2L blended with the square-root bilinear weights.  CPU only; every expected value comes from the paper's
statements or from an independent numpy evaluation.
"""
import numpy as np

from oracle import oracle_facets
from workloads import make_workload


def _nodes(nx_n, ny_n, nw, L, seed=3, same=False):
    """One table of nw components per lattice node; `same`: every node carries the identical table."""
    rng = np.random.default_rng(seed)
    shape = (ny_n, nx_n, nw)
    k = rng.uniform(0.05, 0.6, shape)
    th = rng.uniform(-1.0, 1.0, shape)
    t = dict(spacing_m=L, kx=k * np.cos(th), ky=k * np.sin(th), amp=rng.uniform(0.02, 0.2, shape),
             omega=np.sqrt(9.81 * k), phase=rng.uniform(0, 2 * np.pi, shape))
    if same:
        for key in ("kx", "ky", "amp", "omega", "phase"):
            t[key] = np.broadcast_to(t[key][:1, :1], shape).copy()
    return t


def _workload(nx=33, ny=17, d=5.0, L=40.0, nw=6, same=False, choppy=0, P=3):
    w = make_workload("tiny", n_pulses=P)
    sc = w.scene
    sc["nx"], sc["ny"], sc["spacing_m"] = nx, ny, d
    sc["xi"] = np.ones((ny, nx, 2), dtype=np.float32)
    sc["choppy"] = choppy
    nx_n = int(np.ceil((nx - 1) * d / L)) + 1
    ny_n = int(np.ceil((ny - 1) * d / L)) + 1
    sc["wave_nodes"] = _nodes(max(nx_n, 2), max(ny_n, 2), nw, L, same=same)
    return w


def _numpy_surface(w, p):
    """Independent evaluation of eq. (1), (2): height, slope, CWM displacement of every facet at pulse p."""
    sc, t = w.scene, w.geometry["t_pulse_s"][p]
    nx, ny, d, wn = sc["nx"], sc["ny"], sc["spacing_m"], sc["wave_nodes"]
    L = wn["spacing_m"]
    i, j = np.meshgrid(np.arange(nx), np.arange(ny))
    xb = sc["centre_m"][0] + (i - (nx - 1) / 2) * d
    yb = sc["centre_m"][1] + (j - (ny - 1) / 2) * d
    ny_n, nx_n, _ = wn["kx"].shape
    a = np.minimum((i * d / L).astype(int), nx_n - 2); b = np.minimum((j * d / L).astype(int), ny_n - 2)
    z = np.zeros((ny, nx)); sx = np.zeros_like(z); sy = np.zeros_like(z); dx = np.zeros_like(z); dy = np.zeros_like(z)
    w2 = np.zeros_like(z)
    for ca in (0, 1):
        for cb in (0, 1):
            xn, yn = (a + ca) * L, (b + cb) * L                      # node position relative to facet (0, 0)
            wgt = np.sqrt((1 - np.abs(xn - i * d) / L) * (1 - np.abs(yn - j * d) / L))
            w2 += wgt**2
            tab = {k: wn[k][b + cb, a + ca] for k in ("kx", "ky", "amp", "omega", "phase")}     # [ny][nx][nw]
            psi = tab["kx"] * xb[..., None] + tab["ky"] * yb[..., None] - tab["omega"] * t + tab["phase"]
            kk = np.hypot(tab["kx"], tab["ky"])
            z += wgt * (tab["amp"] * np.cos(psi)).sum(-1)
            sx -= wgt * (tab["amp"] * tab["kx"] * np.sin(psi)).sum(-1)
            sy -= wgt * (tab["amp"] * tab["ky"] * np.sin(psi)).sum(-1)
            dx -= wgt * (tab["amp"] * tab["kx"] / kk * np.sin(psi)).sum(-1)
            dy -= wgt * (tab["amp"] * tab["ky"] / kk * np.sin(psi)).sum(-1)
    return xb, yb, z, sx, sy, dx, dy, w2


def test_blend_against_numpy_and_weight_squares_add_to_one():
    """Eq. (1) with the weights of eq. (2) by an independent numpy script, with and without the CWM displacement;
    "the squares of the weighting coefficients must add to unity"."""
    for choppy, L in ((0, 40.0), (1, 40.0), (1, 37.0)):        # L = 37 m: node lines fall between facets, and rounding
        w = _workload(choppy=choppy, L=L)                       # leaves 1 - wx - wy + wx wy = -1e-17 at some far edges
        for p in (0, 2):
            o = oracle_facets(w, p)
            xb, yb, z, sx, sy, dx, dy, w2 = _numpy_surface(w, p)
            assert np.max(np.abs(w2 - 1.0)) < 1e-14
            assert np.all(np.isfinite(o["pos"]))
            # the weight has an infinite slope at the far edge of a cell: where i d / L rounds across a node line the
            # two evaluations differ by sqrt(1e-16) times a displacement
            tol = 1e-12 if L == 40.0 else 2e-8
            assert np.max(np.abs(o["pos"][:, 2] - (w.scene["centre_m"][2] + z).reshape(-1))) < tol
            assert np.max(np.abs(o["slope"][:, 0] - sx.reshape(-1))) < tol
            assert np.max(np.abs(o["slope"][:, 1] - sy.reshape(-1))) < tol
            ex = xb + (dx if choppy else 0.0)
            assert np.max(np.abs(o["pos"][:, 0] - ex.reshape(-1))) < max(tol, 1e-10)


def test_unit_weight_at_the_corners():
    """"having one unit weight at each TL corner": a facet sitting on lattice node (a, b) sees exactly the
    homogeneous tile T2L of that node."""
    w = _workload(nx=17, ny=9, d=5.0, L=20.0)           # nodes every 4 facets
    wn, sc = w.scene["wave_nodes"], w.scene
    o = oracle_facets(w, 1)
    t = w.geometry["t_pulse_s"][1]
    for (i, j) in ((0, 0), (4, 0), (8, 4), (16, 8), (12, 4)):
        a, b = i // 4, j // 4
        xb = sc["centre_m"][0] + (i - 8.0) * 5.0; yb = sc["centre_m"][1] + (j - 4.0) * 5.0
        tab = {k: wn[k][b, a] for k in ("kx", "ky", "amp", "omega", "phase")}
        z = (tab["amp"] * np.cos(tab["kx"] * xb + tab["ky"] * yb - tab["omega"] * t + tab["phase"])).sum()
        assert abs(o["pos"][j * 17 + i, 2] - (sc["centre_m"][2] + z)) < 1e-12


def test_identical_tiles_scale_by_the_weight_sum():
    """Four IDENTICAL (fully correlated) tiles: D_TL = (sum_i W^i) D, between 1 (corners) and 2 (cell centre) -- the
    energy-preserving property needs uncorrelated tiles."""
    w = _workload(nx=9, ny=9, d=5.0, L=40.0, same=True)         # one cell; facet (4, 4) is its centre
    o = oracle_facets(w, 0)
    w_hom = _workload(nx=9, ny=9, d=5.0, L=40.0, same=True)
    wn = w_hom.scene.pop("wave_nodes")
    for k in ("kx", "ky", "amp", "omega", "phase"):
        w_hom.scene[k] = wn[k][0, 0].copy()
    w_hom.scene["n_waves"] = wn["kx"].shape[2]
    h = oracle_facets(w_hom, 0)
    zc = w.scene["centre_m"][2]
    i, j = np.meshgrid(np.arange(9), np.arange(9))
    fx, fy = i / 8.0, j / 8.0
    wsum = sum(np.sqrt((fx if ca else 1 - fx) * (fy if cb else 1 - fy)) for ca in (0, 1) for cb in (0, 1))
    assert abs(wsum[4, 4] - 2.0) < 1e-15 and abs(wsum[0, 0] - 1.0) < 1e-15
    assert np.max(np.abs((o["pos"][:, 2] - zc) - wsum.reshape(-1) * (h["pos"][:, 2] - zc))) < 1e-12


def test_uncorrelated_tiles_preserve_the_wave_energy():
    """Independent phases per node and the same spectrum everywhere: the height variance of the blended surface stays
    sum A^2 / 2, where identical tiles would give up to four times that."""
    rng = np.random.default_rng(8)
    nw, L, d, n = 24, 64.0, 4.0, 129
    k = np.geomspace(0.3, 1.2, nw); th = np.linspace(-0.6, 0.6, nw); amp = np.full(nw, 0.05)
    w = _workload(nx=n, ny=n, d=d, L=L, nw=nw)
    shape = w.scene["wave_nodes"]["kx"].shape
    w.scene["wave_nodes"] = dict(spacing_m=L, kx=np.broadcast_to(k * np.cos(th), shape).copy(),
                                 ky=np.broadcast_to(k * np.sin(th), shape).copy(), amp=np.broadcast_to(amp, shape).copy(),
                                 omega=np.broadcast_to(np.sqrt(9.81 * k), shape).copy(), phase=rng.uniform(0, 2 * np.pi, shape))
    z = oracle_facets(w, 0)["pos"][:, 2] - w.scene["centre_m"][2]
    expect = (amp**2).sum() / 2
    assert abs(z.var() / expect - 1.0) < 0.15
