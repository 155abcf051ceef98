"""Pins of the fp64 oracle's forward render against closed forms, invariants and brute force.

None of these re-types the oracle's formula: each compares against something the paper and the
mathematics fix independently (SURVEY.md section 8(c) "What pins the oracle").
"""
import math
from dataclasses import replace

import numpy as np
import pytest

from oracle import pyoracle as po
from synth import (AXISYM, CART3D, DENS_LINEAR, DENS_LN, UNIT_CGS, UNIT_JY_PIXEL, UNIT_S0, VEL_VPHI, Geom, Grid,
                   Scene, co_line, make_config, slab_scene, tiny_axisym_scene, tiny_cart_scene)
from tests import np_reference

H, KB, CL = 6.62607015e-27, 1.380649e-16, 2.99792458e10
AU = 1.495978707e13
S0 = 2 * H * 230.538e9 ** 3 / CL ** 2


# ------------------------------------------------------------------ pin 1: isothermal slab
def test_slab_worked_values(slab_golden):
    """Values printed in SURVEY.md:287-288, computed independently of this oracle."""
    g = slab_golden
    sc = slab_scene(vchan_cms=[0.0, 0.1e5, 0.3e5])
    cube = po.render(sc)[0, 0]
    assert cube[0] == pytest.approx(g["I_v0_over_S0"], rel=2e-7)
    assert cube[0] * S0 == pytest.approx(g["I_v0_cgs"], rel=2e-7)
    assert cube[1] * S0 == pytest.approx(g["I_v0p1kms_cgs"], rel=2e-7)
    assert cube[2] * S0 == pytest.approx(g["I_v0p3kms_cgs"], rel=2e-7)
    assert S0 == pytest.approx(g["S0_cgs"], rel=1e-7)
    tr = po.trace_ray(sc, 0)
    assert tr["alpha"][0] == pytest.approx(g["alpha_cms_T30"], rel=1e-8)
    assert tr["K"].sum() == pytest.approx(g["tau_center_T30"], rel=2e-7)
    assert tr["S"][0] == pytest.approx(g["B_nu0_T30_over_S0"], rel=1e-5)
    assert po.partition(sc, 30.0) == pytest.approx(g["Q_T30"], rel=1e-7)
    sc = slab_scene(vchan_cms=[0.1e5], vturb_abs=0.05e5)
    assert po.render(sc)[0, 0, 0] * S0 == pytest.approx(g["I_v0p1kms_vturb0p05_cgs"], rel=2e-7)
    assert po.trace_ray(sc, 0)["alpha"][0] == pytest.approx(g["alpha_cms_T30_vturb0p05"], rel=1e-8)
    # Planck values and per-molecule cross-sections at other temperatures
    for T, kB, ksig in ((20.0, "B_nu0_T20_cgs", "sigma_center_T20_cm2"), (60.0, "B_nu0_T60_cgs", "sigma_center_T60_cm2"),
                        (30.0, "B_nu0_T30_cgs", "sigma_center_T30_cm2")):
        sc = slab_scene(temp=T, vchan_cms=[0.0])
        tr = po.trace_ray(sc, 0)
        assert tr["S"][0] * S0 == pytest.approx(g[kB], rel=2e-7)
        sigma = tr["K"].sum() / (1.0 * 100.0 * AU)      # tau / (n L)
        assert sigma == pytest.approx(g[ksig], rel=1e-4)
    # optically thin slab
    sc = slab_scene(n_co=1e-4, vchan_cms=[0.0])
    assert po.render(sc)[0, 0, 0] * S0 == pytest.approx(g["I_thin_n1e-4_cgs"], rel=2e-7)


def _tau_einstein_B(line, n, T, L_cm, v):
    """Line optical depth from Eq. 14 as printed: Einstein B coefficients and Boltzmann
    populations of BOTH levels -- a route the oracle does not take (it uses the LTE identity)."""
    nu = line.nu0
    B_ul = line.a_ul * CL ** 2 / (2 * H * nu ** 3)
    j_up = int(round((line.g_u - 1) / 2))
    g_l, e_l = line.g_lev[j_up - 1], line.e_lev_K[j_up - 1]
    B_lu = line.g_u / g_l * B_ul
    Q = sum(gj * math.exp(-ej / T) for gj, ej in zip(line.g_lev, line.e_lev_K))
    n_u = n * line.g_u * math.exp(-line.e_u_K / T) / Q
    n_l = n * g_l * math.exp(-e_l / T) / Q
    alpha = math.sqrt(2 * KB * T / line.m_line + line.vturb_abs ** 2)
    phi = CL / (nu * alpha * math.sqrt(math.pi)) * math.exp(-(v / alpha) ** 2)
    return H * nu / (4 * math.pi) * (n_l * B_lu - n_u * B_ul) * phi * L_cm


@pytest.mark.parametrize("T,n,v", [(30.0, 1.0, 0.0), (20.0, 3.0, 0.1e5), (60.0, 50.0, 0.2e5), (150.0, 400.0, 0.0)])
def test_slab_planck_closed_form(T, n, v):
    """I = B_nu0(T) (1 - exp(-tau)), exact for the discretised sum (it telescopes).

    tau comes from Eq. 14 as printed; the rigid-rotor table gives E_u - E_l = 11.06436 K against
    h nu0 / k = 11.06408 K, so the two routes differ by ~3e-5 (reading 9)."""
    sc = slab_scene(n_co=n, temp=T, vchan_cms=[v], nstep=7)
    tau = _tau_einstein_B(sc.line, n, T, 100.0 * AU, v)
    x = H * sc.line.nu0 / (KB * T)
    expect = (1.0 / math.expm1(x)) * (-math.expm1(-tau))
    got = po.render(sc)[0, 0, 0]
    assert got == pytest.approx(expect, rel=1e-4)


def test_slab_independent_of_step_count():
    """Telescoping: sum_k S(1-e^{-dtau}) e^{-k dtau} = S(1-e^{-N dtau}) for any N."""
    ref = None
    for nstep in (1, 2, 5, 64, 333):
        sc = slab_scene(n_co=7.0, temp=45.0, vchan_cms=[0.0, 0.05e5, 0.2e5], nstep=nstep)
        cube = po.render(sc)
        assert np.all(np.abs(cube - cube[0, 0]) <= 1e-13 * np.abs(cube[0, 0]))   # all pixels identical
        if ref is None:
            ref = cube[0, 0]
        np.testing.assert_allclose(cube[0, 0], ref, rtol=2e-13)


def test_slab_optically_thick_saturates():
    sc = slab_scene(n_co=1e6, temp=40.0, vchan_cms=[0.0])
    x = H * sc.line.nu0 / (KB * 40.0)
    assert po.render(sc)[0, 0, 0] == pytest.approx(1.0 / math.expm1(x), rel=1e-12)


def test_ln_density_equals_linear_for_uniform_field():
    a = po.render(slab_scene(n_co=3.0, vchan_cms=[0.0, 0.1e5], dens_ln=False))
    b = po.render(slab_scene(n_co=3.0, vchan_cms=[0.0, 0.1e5], dens_ln=True))
    np.testing.assert_allclose(a, b, rtol=1e-6)   # float32 storage of ln 3


# ------------------------------------------------------------------ pin 2: optically thin limit
def test_thin_limit_uniform():
    """I -> int j ds = S tau; the first correction is -tau/2 relative (SURVEY.md:288)."""
    sc = slab_scene(n_co=1e-4, temp=30.0, vchan_cms=[0.0], nstep=1)
    tr = po.trace_ray(sc, 0)
    tau, S = tr["K"].sum(), tr["S"][0]
    got = po.render(sc)[0, 0, 0]
    assert got == pytest.approx(S * tau, rel=tau)            # thin limit
    assert got == pytest.approx(S * tau * (1 - tau / 2), rel=tau * tau)


def _gaussian_column_scene(nz, nstep, h=20.0, n0=1e-3, T=35.0):
    zmax = 8.0 * h
    shape = (2, 2, nz)
    z = np.linspace(-zmax, zmax, nz)
    dens = np.broadcast_to(n0 * np.exp(-0.5 * (z / h) ** 2), shape).astype(np.float32)
    grid = Grid(kind=CART3D, n=shape, lo=(-10.0, -10.0, -zmax), hi=(10.0, 10.0, zmax), dens=np.ascontiguousarray(dens),
                temp=np.full(shape, T, np.float32), vel=np.zeros(shape, np.float32), mirror_z=False)
    geom = Geom(nx=1, ny=1, fov_x=5.0, fov_y=5.0, incl=0.0, nstep=nstep, x0=3.0)   # off-axis: r = 0 is skipped
    return Scene(geom, co_line(np.zeros(1)), grid)


def test_thin_limit_gaussian_column():
    """int j ds along a Gaussian density has the closed form sqrt(2 pi) h j0.  The midpoint sum of a
    Gaussian converges faster than any power of ds, so a modest resolution already matches to 1e-6
    (float32 storage of the nodes bounds it); a coarse one does not."""
    h, n0 = 20.0, 1e-8          # tau ~ 1e-9: self-absorption is negligible
    errs = []
    for nz, nstep in ((17, 20), (65, 80), (129, 160)):
        sc = _gaussian_column_scene(nz, nstep, h=h, n0=n0)
        unit = slab_scene(n_co=n0, temp=35.0, path_au=1.0, vchan_cms=[0.0], nstep=1)
        tr = po.trace_ray(unit, 0)
        tau_per_au, S = tr["K"][0], tr["S"][0]                 # line-centre dtau of 1 au at n0 (uniform-slab pin)
        expect = S * tau_per_au * math.sqrt(2 * math.pi) * h
        errs.append(abs(po.render(sc)[0, 0, 0] / expect - 1.0))
    assert errs[0] > 1e-3
    assert errs[1] < 1e-6 and errs[2] < 1e-6


# ------------------------------------------------------------------ pin 3: line normalisation
@pytest.mark.parametrize("vturb_abs,vturb_mach,vsys", [(0.0, 0.0, 0.0), (0.2e5, 0.0, 0.35e5), (0.0, 0.5, -0.2e5)])
def test_line_profile_normalisation(vturb_abs, vturb_mach, vsys):
    """Thin limit: sum_c I_c dv = (h nu0 / 4 pi) A_ul N_u (c / nu0), whatever alpha, v_sys, turbulence
    (Eq. 13 and 15): the Gaussian of Eq. 15 integrates to one."""
    T, n, L = 40.0, 1e-5, 100.0
    dv = 0.02e5
    vch = (np.arange(241) - 120) * dv + vsys
    sc = slab_scene(n_co=n, temp=T, path_au=L, vchan_cms=vch, nstep=4, vturb_abs=vturb_abs, vturb_mach=vturb_mach,
                    unit=UNIT_CGS)
    sc = replace(sc, geom=replace(sc.geom, vsys=vsys))
    ln = sc.line
    Q = sum(g * math.exp(-e / T) for g, e in zip(ln.g_lev, ln.e_lev_K))
    N_u = n * ln.g_u * math.exp(-ln.e_u_K / T) / Q * L * AU
    expect = H * ln.nu0 / (4 * math.pi) * ln.a_ul * N_u * (CL / ln.nu0)
    got = po.render(sc)[0, 0].sum() * dv
    assert got == pytest.approx(expect, rel=2e-5)   # residual = tau/2 self-absorption


def test_line_width_eq16_eq17():
    """alpha^2 = 2kT/m_CO + v_turb^2 * 2kT/m_mol (Eq. 16-17 as printed)."""
    T = 50.0
    sc = slab_scene(temp=T, vturb_mach=0.3, vturb_abs=0.1e5)
    ln = sc.line
    expect = math.sqrt(2 * KB * T / ln.m_line + 0.09 * 2 * KB * T / ln.m_gas + 1e8)
    assert po.trace_ray(sc, 0)["alpha"][0] == pytest.approx(expect, rel=1e-14)
    # FWHM of the rendered thin line = 2 sqrt(ln 2) alpha
    vch = np.linspace(-1.5e5, 1.5e5, 3001)
    sc = slab_scene(n_co=1e-6, temp=T, vturb_mach=0.3, vturb_abs=0.1e5, vchan_cms=vch, nstep=1)
    prof = po.render(sc)[0, 0]
    above = vch[prof >= 0.5 * prof.max()]
    assert above.max() - above.min() == pytest.approx(2 * math.sqrt(math.log(2)) * expect, rel=2e-3)


# ------------------------------------------------------------------ pin 4: symmetries
def test_face_on_velocity_symmetry():
    """i = 0, pure rotation: v_los = 0 everywhere, so I(+v) = I(-v) (SURVEY.md:290)."""
    sc = tiny_axisym_scene(seed=3, incl_deg=0.0, pa_deg=0.0, nchan=7, npix=8, nstep=24)
    cube = po.render(sc)
    assert cube.max() > 0
    np.testing.assert_allclose(cube, cube[:, :, ::-1], rtol=1e-12, atol=1e-300)


def test_minor_axis_mirror_with_velocity_flip():
    """Any inclination, axisymmetric (r, zeta) grid, PA = 0, symmetric channels, v_sys = 0:
    cube[iy][ix][c] = cube[ny-1-iy][ix][C-1-c] (x_d -> -x_d flips v_los only)."""
    sc = make_config(1, npix=24)
    cube = po.render(sc)
    assert cube.max() > 0.1
    np.testing.assert_allclose(cube, cube[::-1, :, ::-1], rtol=1e-9, atol=1e-12 * cube.max())
    # and it is NOT symmetric without the velocity flip (the test has teeth)
    assert np.abs(cube - cube[::-1, :, :]).max() > 0.05 * cube.max()


def test_azimuth_invariance_axisym():
    a = po.render(tiny_axisym_scene(seed=4, az_deg=0.0))
    b = po.render(tiny_axisym_scene(seed=4, az_deg=77.0))
    np.testing.assert_allclose(a, b, rtol=1e-10, atol=1e-14 * a.max())


def test_receding_side_is_the_pa_direction():
    """Counter-clockwise rotation, PA = 0: the +Y (north) half of the major axis recedes, so its
    spectrum peaks at positive velocity (readings 5-6; Eq. 15 nu0(1 - delta_nu))."""
    sc = make_config(1, npix=16)
    cube = po.render(sc)
    v = sc.line.vchan
    top = cube[12, 8]       # Y > 0 on the major axis (x' = Y for PA = 0)
    bot = cube[3, 8]
    assert top.sum() > 0 and bot.sum() > 0
    assert (top * v).sum() / top.sum() > 0.3e5
    assert (bot * v).sum() / bot.sum() < -0.3e5


# ------------------------------------------------------------------ pin 5: step refinement
def test_step_refinement_second_order():
    base = tiny_axisym_scene(seed=5, nr=33, nz=25, npix=4, nchan=3, nstep=64, incl_deg=30.0)
    cubes = []
    for nstep in (128, 256, 512, 1024):
        cubes.append(po.render(replace(base, geom=replace(base.geom, nstep=nstep))))
    d1 = np.abs(cubes[1] - cubes[0]).max()
    d2 = np.abs(cubes[2] - cubes[1]).max()
    d3 = np.abs(cubes[3] - cubes[2]).max()
    assert d2 < d1 and d3 < d2
    assert d3 < 2e-3 * cubes[3].max()


# ------------------------------------------------------------------ pin 7: textbook reductions
@pytest.mark.parametrize("T,tol", [(5.0, 5e-4), (20.0, 3e-6), (60.0, 5e-8)])
def test_partition_function_asymptotic(T, tol):
    """Rigid rotor: Q = kT/hB + 1/3 + (1/15)(hB/kT) + (4/315)(hB/kT)^2 + ... (SURVEY.md:293)."""
    line = co_line(np.zeros(1))
    y = 2.766090 / T
    expect = 1 / y + 1 / 3 + y / 15 + 4 * y * y / 315
    assert po.partition(line, T) == pytest.approx(expect, rel=tol)


def test_source_function_rayleigh_jeans():
    """S/S0 = 1/(e^x - 1) -> 1/x - 1/2 + x/12 for x = h nu0 / kT << 1."""
    T = 5000.0
    sc = slab_scene(temp=T)
    x = H * sc.line.nu0 / (KB * T)
    assert po.trace_ray(sc, 0)["S"][0] == pytest.approx(1 / x - 0.5 + x / 12, rel=1e-9)


def test_intensity_units():
    base = slab_scene(n_co=2.0, vchan_cms=[0.0, 0.1e5])
    c_s0 = po.render(base)
    c_cgs = po.render(replace(base, line=replace(base.line, unit=UNIT_CGS)))
    c_jy = po.render(replace(base, line=replace(base.line, unit=UNIT_JY_PIXEL)))
    np.testing.assert_allclose(c_cgs, c_s0 * S0, rtol=1e-13)
    g = base.geom
    pix_rad = (g.fov_x / g.nx) / (g.dist_pc * 3.0856775814913673e18 / AU)
    np.testing.assert_allclose(c_jy, c_cgs * pix_rad ** 2 * 1e23, rtol=1e-12)
    assert po.source_unit(base) == 1.0


def test_temperature_clamp():
    a = slab_scene(temp=0.2, n_co=1e-3, vchan_cms=[0.0])
    b = slab_scene(temp=1.0, n_co=1e-3, vchan_cms=[0.0])
    np.testing.assert_allclose(po.render(a), po.render(b), rtol=0, atol=0)


# ------------------------------------------------------------------ ordering along the ray
def test_two_layer_front_to_back_order():
    """Cold layer in FRONT (+z, nearer the face-on observer) of a hot layer: I = S_f(1-e^{-tau_f}) +
    e^{-tau_f} S_b (1-e^{-tau_b}).  Swapping the layers changes the answer; checks k = 0 is nearest."""
    nz = 9
    z = np.linspace(-80.0, 80.0, nz)
    Tf, Tb = 15.0, 70.0
    temp_z = np.where(z > 0, Tf, Tb)
    dens_z = np.where(np.abs(z) >= 39.0, 2.0, 0.0)     # zero at the nodes next to the interface (z = -20, 0, 20)
    shape = (2, 2, nz)
    for flip in (False, True):
        tz = temp_z[::-1] if flip else temp_z
        grid = Grid(kind=CART3D, n=shape, lo=(-5.0, -5.0, -80.0), hi=(5.0, 5.0, 80.0),
                    dens=np.ascontiguousarray(np.broadcast_to(dens_z, shape), np.float32),
                    temp=np.ascontiguousarray(np.broadcast_to(tz, shape), np.float32),
                    vel=np.zeros(shape, np.float32), mirror_z=False)
        sc = Scene(Geom(nx=1, ny=1, fov_x=1.0, fov_y=1.0, incl=0.0, nstep=160, x0=2.0), co_line(np.zeros(1)), grid)
        tr = po.trace_ray(sc, 0)
        front = slice(0, 80)       # s increases away from the observer: first half is z > 0
        back = slice(80, 160)
        tau_f, tau_b = tr["K"][front].sum(), tr["K"][back].sum()
        S_f, S_b = tr["S"][front][tr["K"][front] > 0][0], tr["S"][back][tr["K"][back] > 0][0]
        assert S_f == pytest.approx(1 / math.expm1(H * 230.538e9 / KB / (Tb if flip else Tf)), rel=1e-12)
        expect = S_f * -math.expm1(-tau_f) + math.exp(-tau_f) * S_b * -math.expm1(-tau_b)
        assert min(tau_f, tau_b) > 0.05 and max(tau_f, tau_b) > 1.0
        assert po.render(sc)[0, 0, 0] == pytest.approx(expect, rel=1e-12)


def test_rays_that_miss_are_zero():
    sc = tiny_axisym_scene(seed=6, npix=6)
    sc = replace(sc, geom=replace(sc.geom, fov_x=2000.0, fov_y=2000.0))
    cube = po.render(sc)
    geo = po.ray_geometry(sc)
    miss = geo["valid"].reshape(6, 6) == 0
    assert miss.any() and not miss.all()
    assert np.all(cube[miss] == 0.0)
    assert cube[~miss].max() > 0


# ------------------------------------------------------------------ pin 8: brute force
@pytest.mark.parametrize("kw", [
    dict(seed=11),
    dict(seed=12, mirror=False, incl_deg=63.0, pa_deg=200.0, az_deg=31.0),
    dict(seed=13, dens_ln=True, kepler_frac=True, vsys=0.4e5, vturb_mach=0.4),
    dict(seed=14, incl_deg=0.0, pa_deg=0.0),
    dict(seed=15, incl_deg=90.0, pa_deg=312.0, npix=5, npix_y=3),
])
def test_bruteforce_numpy_axisym(kw):
    sc = tiny_axisym_scene(**kw)
    a = po.render(sc)
    b = np_reference.render(sc)
    assert a.max() > 1e-3
    np.testing.assert_allclose(a, b, rtol=1e-10, atol=1e-13 * a.max())


@pytest.mark.parametrize("kw", [dict(seed=21), dict(seed=22, dens_ln=False, kepler_frac=False, az_deg=0.0, incl_deg=0.0),
                                dict(seed=23, incl_deg=80.0, pa_deg=-40.0)])
def test_bruteforce_numpy_cart(kw):
    sc = tiny_cart_scene(**kw)
    a = po.render(sc)
    b = np_reference.render(sc)
    assert a.max() > 1e-3
    np.testing.assert_allclose(a, b, rtol=1e-10, atol=1e-13 * a.max())


def test_bruteforce_numpy_units():
    sc = tiny_cart_scene(seed=24)
    sc = replace(sc, line=replace(sc.line, unit=UNIT_JY_PIXEL))
    np.testing.assert_allclose(po.render(sc), np_reference.render(sc), rtol=1e-10)


def test_ray_subset_matches_full():
    sc = tiny_axisym_scene(seed=7, npix=7)
    full = po.render(sc).reshape(-1, len(sc.line.vchan))
    idx = np.array([0, 5, 13, 24, 48])
    np.testing.assert_array_equal(po.render(sc, rays=idx), full[idx])


# ---------------------------------------------------------------------------------------------
# chi^2 data term: pins of oracle.pyoracle.chi2_loss_grad
# ---------------------------------------------------------------------------------------------
def test_chi2_constant_residual_and_zero():
    rng = np.random.default_rng(5)
    D = rng.normal(size=(3, 4, 5))
    L, g = po.chi2_loss_grad(D + 0.3, D, 0.3)          # every residual is one sigma: chi^2/n = 1, L = 1/2
    assert L == pytest.approx(0.5, rel=1e-12)
    np.testing.assert_allclose(g, 1.0 / (0.3 * D.size), rtol=1e-12)
    L0, g0 = po.chi2_loss_grad(D, D, 2.0)
    assert L0 == 0.0 and not g0.any()


def test_chi2_gradient_matches_finite_differences_and_scaling():
    rng = np.random.default_rng(6)
    I, D = rng.normal(size=(2, 3, 4)), rng.normal(size=(2, 3, 4))
    L, g = po.chi2_loss_grad(I, D, 0.7)
    for idx in [(0, 0, 0), (1, 2, 3), (0, 1, 2)]:
        e = np.zeros_like(I)
        e[idx] = 1e-6
        fd = (po.chi2_loss_grad(I + e, D, 0.7)[0] - po.chi2_loss_grad(I - e, D, 0.7)[0]) / 2e-6
        assert g[idx] == pytest.approx(fd, rel=1e-7)
    # quadratic in the residual, inverse quadratic in sigma
    assert po.chi2_loss_grad(D + 2 * (I - D), D, 0.7)[0] == pytest.approx(4 * L, rel=1e-12)
    assert po.chi2_loss_grad(I, D, 1.4)[0] == pytest.approx(L / 4, rel=1e-12)
