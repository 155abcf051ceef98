"""Pins of the oracle's adjoint (O11) against finite differences of the oracle's forward render.

The forward render is pinned by test_oracle_closed_forms.py; the adjoint must be its exact derivative
(Fig. 2 E PAPER.md:56: gradients are propagated through the ray tracer)."""
from dataclasses import replace

import numpy as np
import pytest

from oracle import pyoracle as po
from synth import slab_scene, tiny_axisym_scene, tiny_cart_scene, tiny_sph_scene

FIELDS = ("dens", "temp", "vel")


def _widen(scene):
    """FD needs perturbations below float32 resolution: the oracle reads float32 grids, so perturb in
    float32-representable steps instead (relative step 2^-10) and use a second-order central difference."""
    return scene


def _loss(scene, G):
    return float((po.render(scene) * G).sum())


def _perturbed(scene, field, delta):
    arr = getattr(scene.grid, field).astype(np.float64) + delta
    a32 = arr.astype(np.float32)
    return scene.with_fields(**{field: a32}), a32.astype(np.float64)


def _fd_directional(scene, G, field, direction, eps):
    base = getattr(scene.grid, field).astype(np.float64)
    sp, ap = _perturbed(scene, field, eps * direction)
    sm, am = _perturbed(scene, field, -eps * direction)
    # actual float32 perturbations differ slightly from eps*direction: use the realised ones
    dplus, dminus = ap - base, am - base
    return (_loss(sp, G) - _loss(sm, G)), dplus - dminus


SCENES = {
    "axisym_lin_vphi": lambda: tiny_axisym_scene(seed=31),
    "axisym_ln_kepler": lambda: tiny_axisym_scene(seed=32, dens_ln=True, kepler_frac=True, vsys=0.3e5, vturb_mach=0.3,
                                                  mirror=False, az_deg=20.0),
    "cart_ln_kepler": lambda: tiny_cart_scene(seed=33),
    "cart_lin_vphi": lambda: tiny_cart_scene(seed=34, dens_ln=False, kepler_frac=False),
    "sph_lin_vphi": lambda: tiny_sph_scene(seed=35),
    "sph_ln_kepler": lambda: tiny_sph_scene(seed=36, dens_ln=True, kepler_frac=True),
}


@pytest.mark.parametrize("name", list(SCENES))
def test_gradient_elementwise_vs_central_differences(name):
    sc = SCENES[name]()
    rng = np.random.default_rng(5)
    G = rng.standard_normal(sc.cube_shape)
    grads = dict(zip(FIELDS, po.render_bwd(sc, G)))
    for field in FIELDS:
        base = getattr(sc.grid, field).astype(np.float64)
        g = grads[field]
        flat = np.argsort(-np.abs(g).ravel())
        # the 12 largest entries plus 12 random ones
        pick = np.unique(np.concatenate([flat[:12], rng.choice(g.size, 12, replace=False)]))
        scale = np.abs(g).max()
        assert scale > 0
        for p in pick:
            idx = np.unravel_index(p, g.shape)
            h = max(abs(base[idx]), 1e-2) * 2.0 ** -9
            d = np.zeros_like(base); d[idx] = 1.0
            dL, dd = _fd_directional(sc, G, field, d, h)
            fd = dL / dd[idx]
            assert fd == pytest.approx(g[idx], rel=2e-4, abs=2e-5 * scale), (field, idx)


@pytest.mark.parametrize("name", list(SCENES))
def test_gradient_directional(name):
    sc = SCENES[name]()
    rng = np.random.default_rng(6)
    G = rng.standard_normal(sc.cube_shape)
    grads = dict(zip(FIELDS, po.render_bwd(sc, G)))
    for field in FIELDS:
        base = getattr(sc.grid, field).astype(np.float64)
        for _ in range(3):
            d = rng.standard_normal(base.shape) * np.maximum(np.abs(base), 1e-2)
            dL, dd = _fd_directional(sc, G, field, d, 2.0 ** -11)
            assert dL == pytest.approx(float((grads[field] * dd).sum()), rel=5e-4), field


def test_adjoint_is_linear_in_G_and_dot_product():
    """<J d, G> = <d, J^T G> with J d from central differences; J^T(aG1 + bG2) = a J^T G1 + b J^T G2."""
    sc = tiny_axisym_scene(seed=35)
    rng = np.random.default_rng(7)
    G1, G2 = rng.standard_normal(sc.cube_shape), rng.standard_normal(sc.cube_shape)
    g1 = po.render_bwd(sc, G1); g2 = po.render_bwd(sc, G2); g12 = po.render_bwd(sc, 2.0 * G1 - 0.5 * G2)
    for a, b, c in zip(g1, g2, g12):
        np.testing.assert_allclose(c, 2.0 * a - 0.5 * b, rtol=1e-10, atol=1e-12 * np.abs(c).max())
    base = sc.grid.temp.astype(np.float64)
    d = rng.standard_normal(base.shape) * base
    eps = 2.0 ** -11
    sp, ap = _perturbed(sc, "temp", eps * d); sm, am = _perturbed(sc, "temp", -eps * d)
    Jd = (po.render(sp) - po.render(sm))
    assert float((Jd * G1).sum()) == pytest.approx(float((g1[1] * (ap - am)).sum()), rel=5e-4)


def test_gradient_zero_through_temperature_clamp_and_outside():
    sc = slab_scene(temp=0.5, n_co=1e-2, vchan_cms=[0.0, 0.05e5], nstep=6)
    gd, gt, gv = po.render_bwd(sc, np.ones(sc.cube_shape))
    assert np.all(gt == 0.0)            # T < 1 K is clamped: zero gradient through the clamp
    assert np.abs(gd).max() > 0
    # rays that miss carry no gradient
    sc = tiny_axisym_scene(seed=36, npix=4)
    far = replace(sc, geom=replace(sc.geom, x0=5000.0))
    for g in po.render_bwd(far, np.ones(far.cube_shape)):
        assert np.all(g == 0.0)


def test_density_gradient_nonzero_where_density_is_zero():
    """dL/dn = A0 K / n must be evaluated as A0 C F ds / alpha: finite and non-zero at n = 0
    (SURVEY.md section 8(a) row i)."""
    sc = slab_scene(n_co=0.0, temp=30.0, vchan_cms=[0.0], nstep=4, npix=1)
    sc = replace(sc, geom=replace(sc.geom, x0=3.0))
    gd, gt, gv = po.render_bwd(sc, np.ones(sc.cube_shape))
    assert gd.sum() > 0 and np.all(gt == 0) and np.all(gv == 0)
    # equals d/dn of S * tau(n) at n -> 0
    sc1 = slab_scene(n_co=1e-6, temp=30.0, vchan_cms=[0.0], nstep=4, npix=1)
    sc1 = replace(sc1, geom=replace(sc1.geom, x0=3.0))
    assert gd.sum() == pytest.approx(po.render(sc1)[0, 0, 0] / 1e-6, rel=1e-5)


def test_subset_rays_gradient_matches_masked_G():
    sc = tiny_axisym_scene(seed=37, npix=6)
    rng = np.random.default_rng(8)
    G = rng.standard_normal(sc.cube_shape)
    idx = np.array([3, 8, 20, 33])
    Gm = np.zeros_like(G).reshape(-1, G.shape[-1]); Gm[idx] = G.reshape(-1, G.shape[-1])[idx]
    a = po.render_bwd(sc, Gm.reshape(G.shape))
    b = po.render_bwd(sc, G.reshape(-1, G.shape[-1])[idx], rays=idx)
    for x, y in zip(a, b):
        np.testing.assert_allclose(x, y, rtol=1e-12, atol=1e-300)
