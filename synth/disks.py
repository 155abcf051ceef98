"""Seeded synthetic disks shaped like the paper's workloads (BASELINE.json `configs`).

The paper renders HD 163296 ALMA cubes (222x222x115 and 502x502) and a hydro
simulation; none of those data exist offline.  These generators are the stand-ins:
the analytic disk family of BASELINE.json configs (power-law surface density with Gaussian vertical
structure, two-layer temperature blended as PAPER.md:178 Eq. 5, CO mask shaped like PAPER.md:200
Eq. 9, Keplerian rotation PAPER.md:185 Eq. 6 without the pressure term), plus seeded noise.
Everything is produced in float64 and cast to float32.  No render arithmetic lives here.

Config numbering follows SURVEY.md §8: config k (1..5) is BASELINE.json `configs[k-1]`.
"""
from __future__ import annotations

import math

import numpy as np
from scipy.special import erfc

from .lines import co_line, channels_centered
from .scene import SPH3D
from .scene import (AXISYM, CART3D, DENS_LINEAR, DENS_LN, VEL_KEPLER_FRAC, VEL_VPHI, Geom, Grid, Scene,
                    UNIT_S0)

AU_CM = 1.495978707e13
GM_SUN = 1.32712440018e26      # cm^3 s^-2
KMS = 1.0e5                    # cm/s
X_CO = 1.0e-4
T_FREEZE = 20.0                # K   (BASELINE.json configs[0])
N_DISSOC = 1.0e21              # cm^-2
N0_H2 = 1.0e9                  # cm^-3 at 100 au midplane (BASELINE.json is silent)
LN_MASKED = -60.0              # stored ln n for masked cells (SURVEY.md §8(c) reading 12)


def _seed(cfg: int) -> int:
    return 3623 * 10 + cfg


def _hscale_none(r):
    return np.ones_like(r)


def _hscale_taper(r):
    """Emission surface narrowing beyond 400 au: h scaled to 0.6 (BASELINE.json configs[2])."""
    return 1.0 - 0.4 * 0.5 * (1.0 + np.tanh((r - 400.0) / 20.0))


def disk_family(r, z, mstar_msun=2.0, h0=8.0, hscale=_hscale_none):
    """Noise-free fields of the analytic disk family at cylindrical (r, z) [au].

    Returns n_CO [cm^-3], T [K], v_phi [cm/s].
    """
    r = np.asarray(r, np.float64)
    z = np.abs(np.asarray(z, np.float64))
    h = h0 * (r / 100.0) ** 1.25 * hscale(r)
    n_mid = N0_H2 * (r / 100.0) ** -1.0
    n_h2 = n_mid * np.exp(-0.5 * (z / h) ** 2)
    t_mid = 20.0 * (r / 100.0) ** -0.5
    t_atm = 60.0
    zq = 2.0 * h
    blend = np.cos(0.5 * np.pi * np.minimum(z, zq) / zq) ** 2
    temp = t_atm + (t_mid - t_atm) * blend
    col = n_mid * (h * AU_CM) * math.sqrt(0.5 * math.pi) * erfc(z / (math.sqrt(2.0) * h))
    mask = (temp >= T_FREEZE) & (col >= N_DISSOC)
    n_co = np.where(mask, X_CO * n_h2, 0.0)
    gm = mstar_msun * GM_SUN
    rho = np.sqrt(r * r + z * z)
    vphi = np.sqrt(gm * (r * AU_CM) ** 2 / (rho * AU_CM) ** 3)
    return n_co, temp, vphi


def _axisym_nodes(nr, nz, rmin=10.0, rmax=600.0, zeta_max=0.5):
    r = rmin * (rmax / rmin) ** (np.arange(nr, dtype=np.float64) / (nr - 1))
    zeta = zeta_max * np.arange(nz, dtype=np.float64) / (nz - 1)
    rr, zz = np.meshgrid(r, zeta, indexing="ij")
    return rr, rr * zz


def _axisym_grid(nr, nz, rng, mstar=2.0, h0=8.0, hscale=_hscale_none, noise=0.1):
    rr, zz = _axisym_nodes(nr, nz)
    n_co, temp, vphi = disk_family(rr, zz, mstar, h0, hscale)
    if noise > 0.0:
        n_co = n_co * np.exp(noise * rng.standard_normal(n_co.shape))
        temp = temp * np.exp(noise * rng.standard_normal(temp.shape))
    return Grid(kind=AXISYM, n=(nr, nz), lo=(10.0, 0.0), hi=(600.0, 0.5),
                dens=np.ascontiguousarray(n_co, np.float32), temp=np.ascontiguousarray(temp, np.float32),
                vel=np.ascontiguousarray(vphi, np.float32), mirror_z=True,
                dens_mode=DENS_LINEAR, vel_mode=VEL_VPHI)


def _grf(shape, spacing_au, corr_au, rms, rng):
    """Gaussian random field: white noise filtered by exp(-k^2 l^2 / 2), normalised to `rms`."""
    white = rng.standard_normal(shape)
    fk = np.fft.rfftn(white, axes=(0, 1, 2))
    ks = [2.0 * np.pi * np.fft.fftfreq(shape[0], d=spacing_au[0]),
          2.0 * np.pi * np.fft.fftfreq(shape[1], d=spacing_au[1]),
          2.0 * np.pi * np.fft.rfftfreq(shape[2], d=spacing_au[2])]
    k2 = ks[0][:, None, None] ** 2 + ks[1][None, :, None] ** 2 + ks[2][None, None, :] ** 2
    fk *= np.exp(-0.5 * k2 * corr_au * corr_au)
    out = np.fft.irfftn(fk, s=shape, axes=(0, 1, 2))
    out *= rms / out.std()
    return out


def config_names():
    return {1: "cfg1_axisym_64x32_img64_c15_n64", 2: "cfg2_axisym_256x128_img256_c64_n256",
            3: "cfg3_alma_512x256_img512_c128_n512", 4: "cfg4_cart256_img512_c64_n512",
            5: "cfg5_batch16_256x128_img512_c128_n512"}


def make_config(cfg: int, npix: int | None = None, ngrid3d: int | None = None, batch: int | None = None):
    """Scene(s) of SURVEY.md §8(d) config `cfg` (1..5).

    Returns one Scene for configs 1-4 and a list of Scenes (one per batch item) for config 5.
    `npix` / `ngrid3d` / `batch` override the image size, the 3-D grid size and the batch count so
    that parity tests can run reduced variants of the same recipe; the default is the full size.
    """
    rng = np.random.default_rng(np.random.PCG64(_seed(cfg)))
    name = config_names()[cfg]
    if cfg == 1:
        grid = _axisym_grid(64, 32, rng)
        px = npix or 64
        geom = Geom(nx=px, ny=px, fov_x=1200.0, fov_y=1200.0, incl=math.radians(45.0), pa=0.0,
                    dist_pc=100.0, nstep=64)
        line = co_line(np.linspace(-3.0, 3.0, 15) * KMS, vturb_abs=0.05 * KMS)
        return Scene(geom, line, grid, name)
    if cfg == 2:
        grid = _axisym_grid(256, 128, rng)
        px = npix or 256
        geom = Geom(nx=px, ny=px, fov_x=1200.0, fov_y=1200.0, incl=math.radians(45.0), pa=0.0,
                    dist_pc=100.0, nstep=256)
        line = co_line(channels_centered(64, 0.1 * KMS), vturb_abs=0.05 * KMS)
        return Scene(geom, line, grid, name)
    if cfg == 3:
        grid = _axisym_grid(512, 256, rng, hscale=_hscale_taper)
        px = npix or 512
        geom = Geom(nx=px, ny=px, fov_x=1200.0, fov_y=1200.0, incl=math.radians(47.0),
                    pa=math.radians(312.0), dist_pc=101.0, nstep=512)
        line = co_line(channels_centered(128, 0.08 * KMS), vturb_abs=0.05 * KMS)
        return Scene(geom, line, grid, name)
    if cfg == 4:
        ng = ngrid3d or 256
        lo, hi = (-600.0, -600.0, -300.0), (600.0, 600.0, 300.0)
        ax = [np.linspace(lo[a], hi[a], ng) for a in range(3)]
        spacing = [(hi[a] - lo[a]) / (ng - 1) for a in range(3)]
        xx, yy, zz = np.meshgrid(ax[0], ax[1], ax[2], indexing="ij", sparse=True)
        rr = np.maximum(np.sqrt(xx * xx + yy * yy), 1.0) + 0.0 * zz
        n_co, temp, _ = disk_family(rr, zz + 0.0 * rr)
        n_co = np.where((rr < 10.0) | (rr > 600.0), 0.0, n_co)
        g1 = _grf((ng, ng, ng), spacing, 20.0, 0.1, rng)
        g2 = _grf((ng, ng, ng), spacing, 20.0, 0.1, rng)
        g3 = _grf((ng, ng, ng), spacing, 20.0, 0.1, rng)
        with np.errstate(divide="ignore"):
            ln_n = np.where(n_co > 0.0, np.log(np.where(n_co > 0.0, n_co, 1.0)) + g1, LN_MASKED)
        temp = temp * (1.0 + g2)
        grid = Grid(kind=CART3D, n=(ng, ng, ng), lo=lo, hi=hi,
                    dens=np.ascontiguousarray(ln_n, np.float32), temp=np.ascontiguousarray(temp, np.float32),
                    vel=np.ascontiguousarray(g3, np.float32), mirror_z=False,
                    dens_mode=DENS_LN, vel_mode=VEL_KEPLER_FRAC)
        px = npix or 512
        geom = Geom(nx=px, ny=px, fov_x=1200.0, fov_y=1200.0, incl=math.radians(45.0), pa=0.0,
                    dist_pc=100.0, nstep=512, gm_star=2.0 * GM_SUN)
        line = co_line(channels_centered(64, 0.1 * KMS), vturb_abs=0.05 * KMS)
        return Scene(geom, line, grid, name)
    if cfg == 5:
        nb = batch or 16
        px = npix or 512
        scenes = []
        incl = rng.uniform(30.0, 60.0, size=16)
        mass = rng.uniform(1.5, 2.5, size=16)
        h0 = rng.uniform(6.0, 10.0, size=16)
        for b in range(nb):
            grid = _axisym_grid(256, 128, rng, mstar=float(mass[b]), h0=float(h0[b]))
            geom = Geom(nx=px, ny=px, fov_x=1200.0, fov_y=1200.0, incl=math.radians(float(incl[b])),
                        pa=0.0, dist_pc=100.0, nstep=512)
            line = co_line(channels_centered(128, 0.08 * KMS), vturb_abs=0.05 * KMS)
            scenes.append(Scene(geom, line, grid, f"{name}[{b}]",
                                meta={"incl_deg": float(incl[b]), "mstar": float(mass[b]), "h0": float(h0[b])}))
        return scenes
    raise ValueError(f"unknown config {cfg}")


def l2_target(cube: np.ndarray, seed: int):
    """Seed-generated target cube and noise level for the L2 loss (cfg 2).

    D = cube (1 + 0.05 xi) + sigma eta with sigma = 0.015 max(cube)  (noise level of PAPER.md:252).
    The loss is L = (1 / 2 N_vox) sum ((I - D) / sigma)^2, so dL/dI = (I - D) / (sigma^2 N_vox).
    """
    rng = np.random.default_rng(np.random.PCG64(seed))
    cube = np.asarray(cube, np.float64)
    sigma = 0.015 * float(cube.max())
    target = cube * (1.0 + 0.05 * rng.standard_normal(cube.shape)) + sigma * rng.standard_normal(cube.shape)
    return target, sigma


# ----------------------------------------------------------------------------------------------
# Small analytic scenes for closed-form pins and edge cases
# ----------------------------------------------------------------------------------------------

def slab_scene(n_co=1.0, temp=30.0, path_au=100.0, vchan_cms=(0.0,), nstep=16, vturb_abs=0.0,
               vturb_mach=0.0, npix=2, width_au=50.0, unit=UNIT_S0, dens_ln=False, ngrid=3) -> Scene:
    """Uniform isothermal static slab seen face-on: a CART3D box of constant fields.

    The ray path through the box is exactly `path_au` (box z-extent), so the render has the
    closed form I = B_nu0(T) (1 - exp(-tau)) (SURVEY.md §8(c) pin 1).
    """
    shape = (ngrid, ngrid, ngrid)
    lo = (-width_au, -width_au, -0.5 * path_au)
    hi = (width_au, width_au, 0.5 * path_au)
    dens = np.full(shape, math.log(n_co) if dens_ln else n_co, np.float32)
    grid = Grid(kind=CART3D, n=shape, lo=lo, hi=hi, dens=dens,
                temp=np.full(shape, temp, np.float32), vel=np.zeros(shape, np.float32), mirror_z=False,
                dens_mode=DENS_LN if dens_ln else DENS_LINEAR, vel_mode=VEL_VPHI)
    geom = Geom(nx=npix, ny=npix, fov_x=width_au, fov_y=width_au, incl=0.0, pa=0.0, nstep=nstep)
    line = co_line(np.asarray(vchan_cms, np.float64), vturb_abs=vturb_abs, vturb_mach=vturb_mach, unit=unit)
    return Scene(geom, line, grid, "slab")


def tiny_axisym_scene(seed=1, nr=9, nz=7, npix=6, nchan=5, nstep=12, incl_deg=40.0, pa_deg=25.0,
                      az_deg=0.0, mirror=True, dens_ln=False, kepler_frac=False, vsys=0.0,
                      vturb_mach=0.0, npix_y=None) -> Scene:
    """Small random axisymmetric scene (smooth positive fields, optical depth of order one)."""
    rng = np.random.default_rng(np.random.PCG64(1000 + seed))
    rmin, rmax, zmax = 20.0, 300.0, 0.6
    r = rmin * (rmax / rmin) ** (np.arange(nr) / (nr - 1.0))
    zlo = 0.0 if mirror else -zmax
    zeta = zlo + (zmax - zlo) * np.arange(nz) / (nz - 1.0)
    rr, zz = np.meshgrid(r, zeta, indexing="ij")
    n = 40.0 * (rr / 100.0) ** -1.5 * np.exp(-0.5 * (zz / 0.25) ** 2) * np.exp(0.3 * rng.standard_normal(rr.shape))
    t = (25.0 + 40.0 * np.abs(zz)) * (rr / 100.0) ** -0.3 * np.exp(0.1 * rng.standard_normal(rr.shape))
    gm = 2.0 * GM_SUN
    if kepler_frac:
        v = 0.05 * rng.standard_normal(rr.shape)
    else:
        v = np.sqrt(gm / (rr * AU_CM)) * (1.0 + 0.05 * rng.standard_normal(rr.shape))
    dens = np.log(n) if dens_ln else n
    grid = Grid(kind=AXISYM, n=(nr, nz), lo=(rmin, zlo), hi=(rmax, zmax),
                dens=np.ascontiguousarray(dens, np.float32), temp=np.ascontiguousarray(t, np.float32),
                vel=np.ascontiguousarray(v, np.float32), mirror_z=mirror,
                dens_mode=DENS_LN if dens_ln else DENS_LINEAR,
                vel_mode=VEL_KEPLER_FRAC if kepler_frac else VEL_VPHI)
    geom = Geom(nx=npix, ny=npix_y or npix, fov_x=500.0, fov_y=500.0, incl=math.radians(incl_deg),
                pa=math.radians(pa_deg), az=math.radians(az_deg), nstep=nstep, vsys=vsys, gm_star=gm)
    line = co_line(np.linspace(-4.0, 4.0, nchan) * KMS if nchan > 1 else np.zeros(1),
                   vturb_abs=0.3 * KMS, vturb_mach=vturb_mach)
    return Scene(geom, line, grid, "tiny_axisym")


def tiny_cart_scene(seed=2, ng=(7, 6, 5), npix=5, nchan=5, nstep=10, incl_deg=35.0, pa_deg=70.0,
                    az_deg=15.0, dens_ln=True, kepler_frac=True, vsys=0.2e5) -> Scene:
    """Small random 3-D Cartesian scene."""
    rng = np.random.default_rng(np.random.PCG64(2000 + seed))
    lo, hi = (-200.0, -180.0, -90.0), (200.0, 180.0, 90.0)
    ax = [np.linspace(lo[a], hi[a], ng[a]) for a in range(3)]
    xx, yy, zz = np.meshgrid(*ax, indexing="ij")
    rr = np.maximum(np.hypot(xx, yy), 5.0)
    n = 30.0 * (rr / 100.0) ** -1.0 * np.exp(-0.5 * (zz / 40.0) ** 2) * np.exp(0.3 * rng.standard_normal(rr.shape))
    t = (25.0 + 0.3 * np.abs(zz)) * np.exp(0.1 * rng.standard_normal(rr.shape))
    gm = 2.0 * GM_SUN
    if kepler_frac:
        v = 0.1 * rng.standard_normal(rr.shape)
    else:
        v = np.sqrt(gm / (rr * AU_CM)) * (1.0 + 0.05 * rng.standard_normal(rr.shape))
    dens = np.log(n) if dens_ln else n
    grid = Grid(kind=CART3D, n=tuple(ng), lo=lo, hi=hi,
                dens=np.ascontiguousarray(dens, np.float32), temp=np.ascontiguousarray(t, np.float32),
                vel=np.ascontiguousarray(v, np.float32), mirror_z=False,
                dens_mode=DENS_LN if dens_ln else DENS_LINEAR,
                vel_mode=VEL_KEPLER_FRAC if kepler_frac else VEL_VPHI)
    geom = Geom(nx=npix, ny=npix, fov_x=420.0, fov_y=420.0, incl=math.radians(incl_deg),
                pa=math.radians(pa_deg), az=math.radians(az_deg), nstep=nstep, vsys=vsys, gm_star=gm)
    line = co_line(np.linspace(-5.0, 5.0, nchan) * KMS, vturb_abs=0.4 * KMS)
    return Scene(geom, line, grid, "tiny_cart")


def _sph_nodes(n, rmin, rmax, th_half):
    r = rmin * (rmax / rmin) ** (np.arange(n[0]) / (n[0] - 1.0))
    th = (0.5 * math.pi - th_half) + 2.0 * th_half * np.arange(n[1]) / (n[1] - 1.0)
    ph = 2.0 * math.pi * np.arange(n[2]) / n[2]
    return r, th, ph


def tiny_sph_scene(seed=3, ng=(7, 6, 8), npix=6, nchan=5, nstep=14, incl_deg=50.0, pa_deg=40.0, az_deg=20.0,
                   dens_ln=False, kepler_frac=False, vsys=-0.1e5) -> Scene:
    """Small random spherical (r, theta, phi) scene; theta spans +-0.7 rad about the equator."""
    rng = np.random.default_rng(np.random.PCG64(3000 + seed))
    lo, hi = (30.0, 0.5 * math.pi - 0.7, 0.0), (220.0, 0.5 * math.pi + 0.7, 2.0 * math.pi)
    r, th, ph = _sph_nodes(ng, lo[0], hi[0], 0.7)
    rr, tt, pp = np.meshgrid(r, th, ph, indexing="ij")
    rc, zz = rr * np.sin(tt), rr * np.cos(tt)
    n = 40.0 * (rc / 100.0) ** -1.0 * np.exp(-0.5 * (zz / 35.0) ** 2) * np.exp(0.3 * rng.standard_normal(rr.shape))
    t = (25.0 + 0.3 * np.abs(zz)) * np.exp(0.1 * rng.standard_normal(rr.shape))
    gm = 2.0 * GM_SUN
    if kepler_frac:
        v = 0.1 * rng.standard_normal(rr.shape)
    else:
        v = np.sqrt(gm / (rc * AU_CM)) * (1.0 + 0.05 * rng.standard_normal(rr.shape))
    dens = np.log(n) if dens_ln else n
    grid = Grid(kind=SPH3D, n=tuple(ng), lo=lo, hi=hi,
                dens=np.ascontiguousarray(dens, np.float32), temp=np.ascontiguousarray(t, np.float32),
                vel=np.ascontiguousarray(v, np.float32), mirror_z=False,
                dens_mode=DENS_LN if dens_ln else DENS_LINEAR,
                vel_mode=VEL_KEPLER_FRAC if kepler_frac else VEL_VPHI)
    geom = Geom(nx=npix, ny=npix, fov_x=460.0, fov_y=460.0, incl=math.radians(incl_deg),
                pa=math.radians(pa_deg), az=math.radians(az_deg), nstep=nstep, vsys=vsys, gm_star=gm)
    line = co_line(np.linspace(-5.0, 5.0, nchan) * KMS, vturb_abs=0.4 * KMS)
    return Scene(geom, line, grid, "tiny_sph")


def sph_benchmark_scene(ng=(512, 96, 256), npix=256, nchan=64, nstep=256, seed=36236) -> Scene:
    """Stand-in for the workload of the paper's only timing benchmark (hydro-simulation fields on a
    512 x 96 x 256 spherical grid rendered at 256 x 256 px; the simulation of ref. [3] is not available): the config-2
    disk family evaluated on a spherical grid (r in [10, 600] au, theta within +-0.46 rad of the equator, all phi) with a
    two-armed logarithmic spiral (15 % in density, 5 % in temperature, 2 % in rotation speed) and 5 % log-normal
    noise, so that the fields depend on all three coordinates as hydro fields do."""
    rng = np.random.default_rng(np.random.PCG64(seed))
    th_half = 0.46
    lo, hi = (10.0, 0.5 * math.pi - th_half, 0.0), (600.0, 0.5 * math.pi + th_half, 2.0 * math.pi)
    r, th, ph = _sph_nodes(ng, lo[0], hi[0], th_half)
    rc, zz = np.outer(r, np.sin(th)), np.outer(r, np.cos(th))                      # [nr][nt]
    n_co, temp, vphi = disk_family(rc, np.abs(zz))
    arm = np.cos(2.0 * ph[None, None, :] - 6.0 * np.log(r / 100.0)[:, None, None])   # [nr][1][np]
    dens = n_co[:, :, None] * (1.0 + 0.15 * arm) * np.exp(0.05 * rng.standard_normal(tuple(ng)))
    tt = temp[:, :, None] * (1.0 + 0.05 * arm) * np.exp(0.05 * rng.standard_normal(tuple(ng)))
    vv = vphi[:, :, None] * (1.0 + 0.02 * arm)
    grid = Grid(kind=SPH3D, n=tuple(ng), lo=lo, hi=hi, dens=np.ascontiguousarray(dens, np.float32),
                temp=np.ascontiguousarray(tt, np.float32), vel=np.ascontiguousarray(vv, np.float32), mirror_z=False)
    geom = Geom(nx=npix, ny=npix, fov_x=1200.0, fov_y=1200.0, incl=math.radians(45.0), pa=0.0, dist_pc=100.0, nstep=nstep)
    line = co_line(channels_centered(nchan, 0.1 * KMS), vturb_abs=0.05 * KMS)
    return Scene(geom, line, grid, f"sph{ng[0]}x{ng[1]}x{ng[2]}_img{npix}_c{nchan}_n{nstep}")
