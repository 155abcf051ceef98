"""Pins of the oracle's spherical (r, theta, phi) grid sampling, CPU only."""
import math
from dataclasses import replace

import numpy as np
import pytest

from oracle import pyoracle as po
from synth import CART3D, SPH3D, Geom, Grid, Scene, co_line, tiny_sph_scene
from tests import np_reference

KMS = 1.0e5
GM_SUN = 1.32712440018e26
AU = 1.495978707e13


@pytest.mark.parametrize("kw", [dict(seed=61), dict(seed=62, dens_ln=True, kepler_frac=True, incl_deg=0.0, az_deg=0.0),
                                dict(seed=63, incl_deg=85.0, pa_deg=-70.0, az_deg=200.0, ng=(5, 4, 3)),
                                dict(seed=64, ng=(4, 9, 16), npix=7, nstep=30)])
def test_bruteforce_numpy_spherical(kw):
    """The independent numpy transcription interpolates on explicit (ln r, theta, phi) node coordinates with the
    phi = 0 plane appended at 2 pi; the oracle works in index space with a modulo."""
    sc = tiny_sph_scene(**kw)
    a = po.render(sc)
    b = np_reference.render(sc)
    assert a.max() > 1e-3
    np.testing.assert_allclose(a, b, rtol=1e-10, atol=1e-13 * a.max())


def _blob_fields(x, y, z):
    """An analytic field without any symmetry: an off-centre, north-of-midplane density blob, a temperature gradient
    along x, Keplerian rotation about z."""
    n = 8.0 * np.exp(-((x - 110.0) ** 2 + (y - 40.0) ** 2 + (z - 25.0) ** 2) / (2.0 * 28.0 ** 2))   # far from the axis, where v_phi ~ r^-1/2 is steep
    t = 32.0 + 0.06 * x - 0.04 * z
    rc = np.maximum(np.hypot(x, y), 2.0)
    v = np.sqrt(2.0 * GM_SUN / (rc * AU))
    return n, t, v


def test_spherical_and_cartesian_grids_agree_on_an_analytic_field():
    """The Cartesian sampling path is pinned on its own; the same analytic field stored on a fine spherical grid and on
    a fine Cartesian grid must give the same cube up to interpolation error.  A swapped atan2, a polar angle measured
    from -z or a reversed phi ordering would move the blob and fail this by far more than the tolerance."""
    geom = Geom(nx=10, ny=10, fov_x=420.0, fov_y=420.0, incl=math.radians(40.0), pa=math.radians(25.0),
                az=math.radians(10.0), nstep=160)
    line = co_line(np.linspace(-4.0, 4.0, 9) * KMS, vturb_abs=0.3 * KMS)
    ns = (72, 64, 96)
    r = 12.0 * (260.0 / 12.0) ** (np.arange(ns[0]) / (ns[0] - 1.0))
    th = (0.5 * math.pi - 1.2) + 2.4 * np.arange(ns[1]) / (ns[1] - 1.0)
    ph = 2.0 * math.pi * np.arange(ns[2]) / ns[2]
    rr, tt, pp = np.meshgrid(r, th, ph, indexing="ij")
    fs = _blob_fields(rr * np.sin(tt) * np.cos(pp), rr * np.sin(tt) * np.sin(pp), rr * np.cos(tt))
    gs = Grid(kind=SPH3D, n=ns, lo=(12.0, 0.5 * math.pi - 1.2, 0.0), hi=(260.0, 0.5 * math.pi + 1.2, 2.0 * math.pi),
              dens=fs[0].astype(np.float32), temp=fs[1].astype(np.float32), vel=fs[2].astype(np.float32), mirror_z=False)
    nc = (81, 81, 81)
    ax = [np.linspace(-260.0, 260.0, nc[a]) for a in range(3)]
    xx, yy, zz = np.meshgrid(*ax, indexing="ij")
    fc = _blob_fields(xx, yy, zz)
    gc = Grid(kind=CART3D, n=nc, lo=(-260.0,) * 3, hi=(260.0,) * 3, dens=fc[0].astype(np.float32),
              temp=fc[1].astype(np.float32), vel=fc[2].astype(np.float32), mirror_z=False)
    cs = po.render(Scene(geom, line, gs))
    cc = po.render(Scene(geom, line, gc))
    assert cc.max() > 0.05
    assert np.max(np.abs(cs - cc)) < 0.03 * cc.max()
    # the cube is NOT symmetric under the flips such mistakes would cause
    assert np.max(np.abs(cc - cc[::-1])) > 0.2 * cc.max() and np.max(np.abs(cc - cc[:, ::-1])) > 0.2 * cc.max()


def test_uniform_shell_chord_closed_form():
    """Constant fields in the shell r_min < rho < r_max, face on, no motion: a ray at impact parameter b < r_min crosses
    two chords of total length L = 2 (sqrt(r_max^2 - b^2) - sqrt(r_min^2 - b^2)) and I = B (1 - exp(-kappa L)); the
    midpoint rule quantises L to the step, hence the tolerance."""
    ns = (5, 7, 4)
    lo, hi = (60.0, 0.05, 0.0), (200.0, math.pi - 0.05, 2.0 * math.pi)
    n0, T0 = 0.5, 30.0
    g = Grid(kind=SPH3D, n=ns, lo=lo, hi=hi, dens=np.full(ns, n0, np.float32), temp=np.full(ns, T0, np.float32),
             vel=np.zeros(ns, np.float32), mirror_z=False)
    geom = Geom(nx=4, ny=1, fov_x=100.0, fov_y=10.0, x0=0.0, y0=31.0, incl=math.radians(90.0), pa=0.0, nstep=6000)
    line = co_line(np.zeros(1), vturb_abs=0.0)
    sc = Scene(geom, line, g)
    cube = po.render(sc)[0, :, 0]
    X = (np.arange(4) + 0.5 - 2.0) * 25.0
    b = np.hypot(X, 31.0)
    L = 2.0 * (np.sqrt(hi[0] ** 2 - b ** 2) - np.sqrt(lo[0] ** 2 - b ** 2))
    # source function and opacity per au from one in-shell step of the first ray (they are the same everywhere);
    # edge on (i = 90 deg) the rays run in the disk's equatorial direction, far from the excluded polar cones
    tr = po.trace_ray(sc, 0)
    k = int(np.argmax(tr["inside"]))
    S, K1 = tr["S"][k], tr["K"][k] / po.ray_geometry(sc)["ds"][0]
    inside_len = tr["inside"].sum() * po.ray_geometry(sc)["ds"][0]
    assert inside_len == pytest.approx(L[0], rel=1e-3)                 # the in/out decision itself
    np.testing.assert_allclose(cube, S * (1.0 - np.exp(-K1 * L)), rtol=2e-3)
    assert 0.2 < K1 * L[0] < 5.0
