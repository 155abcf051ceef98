"""Pins of the oracle's ray geometry (O1-O3; Table 2 parameters)."""
import math
from dataclasses import replace

import numpy as np
import pytest

from oracle import pyoracle as po
from synth import slab_scene, tiny_axisym_scene, tiny_cart_scene


@pytest.mark.parametrize("incl,pa,az", [(0.0, 0.0, 0.0), (45.0, 0.0, 0.0), (47.0, 312.0, 0.0), (80.0, 33.0, 120.0)])
def test_rotation_invariants(incl, pa, az):
    """Rotations preserve lengths: |origin| = hypot(X, Y), |dir| = 1, origin . dir = 0 (s = 0 is the
    closest approach to the star)."""
    sc = tiny_axisym_scene(seed=1, npix=9, incl_deg=incl, pa_deg=pa, az_deg=az)
    geo = po.ray_geometry(sc)
    g = sc.geom
    ix, iy = np.meshgrid(np.arange(g.nx), np.arange(g.ny))
    X = (ix + 0.5 - g.nx / 2) * g.fov_x / g.nx
    Y = (iy + 0.5 - g.ny / 2) * g.fov_y / g.ny
    b = np.hypot(X, Y).ravel()
    np.testing.assert_allclose(np.linalg.norm(geo["origin"], axis=1), b, rtol=1e-13)
    assert np.linalg.norm(geo["dir"]) == pytest.approx(1.0, abs=1e-15)
    np.testing.assert_allclose(geo["origin"] @ geo["dir"], 0.0, atol=1e-10)
    # direction: inclination is the angle between the line of sight and the disk axis
    assert -geo["dir"][2] == pytest.approx(math.cos(math.radians(incl)), abs=1e-15)


def test_bounding_sphere_chord():
    """Axisymmetric grids are clipped to the sphere R_b = r_max sqrt(1 + zeta_max^2): chord = 2 sqrt(R_b^2 - b^2)."""
    sc = tiny_axisym_scene(seed=2, npix=10)
    sc = replace(sc, geom=replace(sc.geom, fov_x=900.0, fov_y=900.0))
    geo = po.ray_geometry(sc)
    g = sc.geom
    Rb = 300.0 * math.sqrt(1 + 0.6 ** 2)
    ix, iy = np.meshgrid(np.arange(g.nx), np.arange(g.ny))
    b = np.hypot((ix + 0.5 - g.nx / 2) * g.fov_x / g.nx, (iy + 0.5 - g.ny / 2) * g.fov_y / g.ny).ravel()
    hit = b < Rb
    assert hit.any() and (~hit).any()
    np.testing.assert_array_equal(geo["valid"], hit.astype(np.int32))
    np.testing.assert_allclose(geo["ds"][hit] * g.nstep, 2 * np.sqrt(Rb ** 2 - b[hit] ** 2), rtol=1e-13)
    np.testing.assert_allclose(geo["s0"][hit], -np.sqrt(Rb ** 2 - b[hit] ** 2), rtol=1e-13)
    assert np.all(geo["ds"][~hit] == 0)
    # entry and exit points lie on the sphere
    p0 = geo["origin"][hit] + geo["s0"][hit, None] * geo["dir"]
    np.testing.assert_allclose(np.linalg.norm(p0, axis=1), Rb, rtol=1e-12)


def test_box_chord_face_on_and_oblique():
    sc = slab_scene(path_au=100.0, npix=3, width_au=50.0)
    geo = po.ray_geometry(sc)
    np.testing.assert_allclose(geo["ds"] * sc.geom.nstep, 100.0, rtol=1e-14)
    np.testing.assert_allclose(geo["s0"], -50.0, rtol=1e-14)
    # oblique: both end points lie on the box surface, all interior samples lie inside
    sc = tiny_cart_scene(seed=3, npix=7)
    geo = po.ray_geometry(sc)
    lo, hi = np.array(sc.grid.lo), np.array(sc.grid.hi)
    v = geo["valid"] == 1
    assert v.any()
    for end in (0.0, float(sc.geom.nstep)):
        p = geo["origin"][v] + (geo["s0"][v] + end * geo["ds"][v])[:, None] * geo["dir"]
        on_face = np.isclose(p, lo, atol=1e-9) | np.isclose(p, hi, atol=1e-9)
        assert np.all(on_face.any(axis=1))
        assert np.all((p >= lo - 1e-9) & (p <= hi + 1e-9))
    # rays flagged invalid really miss the box: their closest points over a fine scan are outside
    for q in np.nonzero(~v)[0]:
        s = np.linspace(-2000, 2000, 4001)
        p = geo["origin"][q] + s[:, None] * geo["dir"]
        assert not np.any(np.all((p >= lo) & (p <= hi), axis=1))


def test_face_on_origin_and_pa_convention():
    """i = 0: rays run along -z through (x', y', 0).  PA = 0 puts the x' axis (line of nodes) along +Y."""
    sc = tiny_axisym_scene(seed=4, npix=4, incl_deg=0.0, pa_deg=0.0)
    geo = po.ray_geometry(sc)
    np.testing.assert_allclose(geo["dir"], [0, 0, -1], atol=1e-15)
    g = sc.geom
    org = geo["origin"].reshape(g.ny, g.nx, 3)
    Y = (np.arange(g.ny) + 0.5 - g.ny / 2) * g.fov_y / g.ny
    X = (np.arange(g.nx) + 0.5 - g.nx / 2) * g.fov_x / g.nx
    np.testing.assert_allclose(org[:, 0, 0], Y, atol=1e-12)            # x' = Y
    np.testing.assert_allclose(org[0, :, 1], -X, atol=1e-12)           # y' = -X
    np.testing.assert_allclose(org[..., 2], 0.0, atol=1e-12)


def test_pixel_grid_symmetric_about_star():
    sc = tiny_axisym_scene(seed=5, npix=6, incl_deg=30.0, pa_deg=0.0)
    org = po.ray_geometry(sc)["origin"].reshape(6, 6, 3)
    np.testing.assert_allclose(org[::-1, ::-1], -org, atol=1e-12)


def test_trace_matches_interpolated_fields_at_nodes():
    """A ray through a grid node sees exactly the stored node values (bilinear weights 0/1)."""
    sc = tiny_axisym_scene(seed=6, nr=9, nz=7, incl_deg=0.0, pa_deg=0.0, npix=1, nstep=1)
    gr = sc.grid
    r_nodes = gr.lo[0] * (gr.hi[0] / gr.lo[0]) ** (np.arange(9) / 8.0)
    # face-on single ray at sky position (X, Y) = (0, r_3); one step sampled at s = 0, i.e. z = 0 (zeta node 0)
    sc = replace(sc, geom=replace(sc.geom, fov_x=1e-9, fov_y=1e-9, y0=float(r_nodes[3])))
    tr = po.trace_ray(sc, 0)
    assert tr["inside"][0] == 1
    assert tr["n"][0] == pytest.approx(float(gr.dens[3, 0]), rel=1e-6)
    assert tr["T"][0] == pytest.approx(float(gr.temp[3, 0]), rel=1e-6)
