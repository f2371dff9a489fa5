"""Pins for the oracle's tabulated antenna patterns (complex Tx / Rx gains,
"converted into u-v grids"): scipy's RegularGridInterpolator as the library routine, exactness on affine tables, the
analytic sinc pattern as the limit of a refined table, zero gain outside the grid.  CPU only.
"""
import numpy as np
from scipy.interpolate import RegularGridInterpolator

from oracle import oracle_facets, oracle_generate
from workloads import C0
from helpers import custom_workload

TX, RX = np.array([10.0, -300e3, 700e3]), np.array([250e3, -300e3, 700e3])
F0 = 5.405e9


def _scene(nx=9, ny=7, d=40.0, **kw):
    r0 = np.linalg.norm(TX) + np.linalg.norm(RX)
    return custom_workload(nx=nx, ny=ny, d=d, tx_pos=TX, rx_pos=RX, t0=r0 / C0 - 100.0 / 12e6,
                           xi=np.ones((ny, nx, 2), dtype=np.float32), **kw)


def _directions(w, ant):
    """(u, v) = direction cosines of antenna -> facet along the azimuth / elevation axes of helpers' default frame
    (rows boresight (0,0,-1), azimuth (1,0,0), elevation (0,1,0)), flat scene."""
    sc = w.scene
    i, j = np.meshgrid(np.arange(sc["nx"]), np.arange(sc["ny"]))
    pos = np.stack([sc["centre_m"][0] + (i - (sc["nx"] - 1) / 2) * sc["spacing_m"],
                    sc["centre_m"][1] + (j - (sc["ny"] - 1) / 2) * sc["spacing_m"],
                    np.full(i.shape, sc["centre_m"][2])], axis=-1).reshape(-1, 3)
    dvec = pos - ant
    uhat = dvec / np.linalg.norm(dvec, axis=1, keepdims=True)
    return uhat[:, 0], uhat[:, 1]


def _grid(u, v, nu=17, nv=13, margin=1e-4):
    return (u.min() - margin, u.max() + margin), (v.min() - margin, v.max() + margin), nu, nv


def _gain_ratio(w, w_iso):
    """G_t G_r of every facet = amplitude with the patterns / amplitude with isotropic antennas."""
    return (oracle_facets(w, 0)["amp"][0] / oracle_facets(w_iso, 0)["amp"][0])


def test_bilinear_lookup_against_scipy():
    """Random complex tables on both antennas: G_t G_r per facet equals the product of scipy's bilinear
    RegularGridInterpolator values at the facets' direction cosines (reading G29)."""
    rng = np.random.default_rng(2)
    w, w_iso = _scene(), _scene()
    expect = np.ones(w.scene["nx"] * w.scene["ny"], dtype=np.complex128)
    for name, ant in (("tx_pattern", TX), ("rx_pattern", RX)):
        u, v = _directions(w, ant)
        ur, vr, nu, nv = _grid(u, v)
        tab = (rng.standard_normal((nv, nu)) + 1j * rng.standard_normal((nv, nu))).astype(np.complex64)
        w.instrument[name] = dict(table=tab, u=ur, v=vr)
        un, vn = np.linspace(*ur, nu), np.linspace(*vr, nv)
        itp = RegularGridInterpolator((vn, un), tab.astype(np.complex128), method="linear")
        expect = expect * itp(np.stack([v, u], axis=-1))
    got = _gain_ratio(w, w_iso)
    assert np.max(np.abs(got - expect)) < 1e-9 * np.abs(expect).max()


def test_affine_table_is_reproduced_exactly():
    """Bilinear interpolation is exact on affine functions: a Tx table c0 + c1 u + c2 v (complex coefficients)
    gives that function of the facet's direction, whatever the grid."""
    w, w_iso = _scene(), _scene()
    u, v = _directions(w, TX)
    c0, c1, c2 = 0.7 - 0.2j, 30.0 + 55.0j, -12.0 + 4.0j
    for nu, nv in ((5, 4), (33, 21)):
        ur, vr, _, _ = _grid(u, v)
        un, vn = np.meshgrid(np.linspace(*ur, nu), np.linspace(*vr, nv))
        w.instrument["tx_pattern"] = dict(table=c0 + c1 * un + c2 * vn, u=ur, v=vr)
        got = _gain_ratio(w, w_iso)
        assert np.max(np.abs(got - (c0 + c1 * u + c2 * v))) < 2e-6          # the table itself is float32


def test_refined_table_converges_to_the_analytic_pattern():
    """A table sampled from the analytic aperture pattern sinc(La u / lambda) sinc(Le v / lambda): the lookup error is
    bounded by h_u^2/8 max|G_uu| + h_v^2/8 max|G_vv| and falls fourfold when the grid step halves."""
    lam = C0 / F0
    ap = (12.3, 0.82)
    w_ana, w_iso = _scene(nx=41, ny=5, d=100.0, tx_ap=ap), _scene(nx=41, ny=5, d=100.0)
    exact = _gain_ratio(w_ana, w_iso).real
    u, v = _directions(w_ana, TX)
    ur, vr, _, _ = _grid(u, v)
    errs = []
    for nu in (9, 17, 33):
        nv = 5
        un, vn = np.meshgrid(np.linspace(*ur, nu), np.linspace(*vr, nv))
        w = _scene(nx=41, ny=5, d=100.0)
        w.instrument["tx_pattern"] = dict(table=np.sinc(ap[0] * un / lam) * np.sinc(ap[1] * vn / lam), u=ur, v=vr)
        got = _gain_ratio(w, w_iso)
        errs.append(np.max(np.abs(got - exact)))
        hu, hv = (ur[1] - ur[0]) / (nu - 1), (vr[1] - vr[0]) / (nv - 1)
        bound = hu**2 / 8 * (np.pi * ap[0] / lam) ** 2 / 3 + hv**2 / 8 * (np.pi * ap[1] / lam) ** 2 / 3    # |sinc''| <= pi^2/3
        assert errs[-1] <= bound + 1e-6
    assert errs[0] > 1e-4                                                   # the coarse table is visibly off
    assert 3.0 < errs[0] / errs[1] < 5.0 and 3.0 < errs[1] / errs[2] < 5.0


def test_directions_outside_the_grid_have_zero_gain():
    w = _scene()
    u, v = _directions(w, RX)
    w.instrument["rx_pattern"] = dict(table=np.ones((3, 3), dtype=np.complex64), u=(u.max() + 1e-3, u.max() + 2e-3),
                                      v=(v.min(), v.max()))
    assert np.all(oracle_facets(w, 0)["amp"] == 0)
    assert np.all(oracle_generate(w) == 0)
    # half covered: the facets inside keep the table's unit gain, the others drop out
    um = 0.5 * (u.min() + u.max())
    w.instrument["rx_pattern"] = dict(table=np.ones((3, 3), dtype=np.complex64), u=(um, u.max() + 1e-6), v=(v.min() - 1e-6, v.max() + 1e-6))
    ratio = _gain_ratio(w, _scene())
    assert np.allclose(ratio[u >= um], 1.0) and np.all(ratio[u < um] == 0)
