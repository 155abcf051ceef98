"""Plain containers describing one render problem (geometry, line, grid).

They mirror the problem statement of the paper (Eq. 11-17; geometry parameters
Table 2) and carry data only.  Units: lengths in au, velocities in cm/s,
number densities in cm^-3, temperatures in K, angles in rad, frequencies in Hz, masses in g.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

# grid kinds
AXISYM = 0   # (r, zeta=z/r) grid, r log-spaced, zeta uniform
CART3D = 1   # uniform Cartesian box in the disk frame
SPH3D = 2    # spherical (r, theta, phi): r log-spaced, theta (polar angle from +z) uniform, phi periodic over 2 pi
# density storage
DENS_LINEAR = 0  # grid stores n [cm^-3], interpolated linearly
DENS_LN = 1      # grid stores ln n, interpolated then exponentiated
# velocity storage
VEL_VPHI = 0         # grid stores v_phi [cm/s]
VEL_KEPLER_FRAC = 1  # grid stores delta, v_phi = v_Kepler(r,z) * (1 + delta)
# intensity units of the output cube
UNIT_S0 = 0        # cube = I_nu / (2 h nu0^3 / c^2)
UNIT_CGS = 1       # cube = I_nu [erg s^-1 cm^-2 Hz^-1 sr^-1]
UNIT_JY_PIXEL = 2  # cube = I_nu * pixel solid angle [Jy / pixel] (uses the distance)


@dataclass
class Geom:
    """Image plane and viewing geometry (Table 2 'Ray-tracing Geometry')."""
    nx: int
    ny: int
    fov_x: float          # au, full width of the image
    fov_y: float          # au
    incl: float           # rad
    pa: float = 0.0       # rad
    az: float = 0.0       # rad
    dist_pc: float = 100.0
    nstep: int = 64
    x0: float = 0.0       # au, image centre offset
    y0: float = 0.0
    vsys: float = 0.0     # cm/s
    gm_star: float = 0.0  # cm^3 s^-2 (only used by VEL_KEPLER_FRAC)


@dataclass
class Line:
    """One molecular line in LTE plus the channel grid (Eq. 13-17)."""
    nu0: float                 # Hz
    a_ul: float                # s^-1
    g_u: float
    e_u_K: float               # E_u / k  [K]
    e_lev_K: np.ndarray        # level energies / k [K], for the partition function
    g_lev: np.ndarray          # level degeneracies
    m_line: float              # g, mass of the emitting molecule
    m_gas: float               # g, mean molecular mass (Eq. 17)
    vchan: np.ndarray          # channel-centre velocities, cm/s (radio convention)
    vturb_abs: float = 0.0     # cm/s, absolute micro-turbulence added in quadrature
    vturb_mach: float = 0.0    # dimensionless (Eq. 16)
    unit: int = UNIT_S0


@dataclass
class Grid:
    """Field grids. AXISYM: arrays [nr][nzeta]; CART3D: arrays [nx][ny][nz]; SPH3D: arrays [nr][ntheta][nphi] (last index fastest)."""
    kind: int
    n: tuple                   # (nr, nzeta) or (nx, ny, nz)
    lo: tuple                  # AXISYM: (r_min, zeta_lo); CART3D: box lower corner, au
    hi: tuple                  # AXISYM: (r_max, zeta_hi); CART3D: box upper corner, au
    dens: np.ndarray           # float32
    temp: np.ndarray           # float32
    vel: np.ndarray            # float32
    mirror_z: bool = True      # AXISYM only: sample at zeta = |z|/r
    dens_mode: int = DENS_LINEAR
    vel_mode: int = VEL_VPHI


@dataclass
class Scene:
    geom: Geom
    line: Line
    grid: Grid
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def cube_shape(self):
        return (self.geom.ny, self.geom.nx, len(self.line.vchan))

    @property
    def nrays(self):
        return self.geom.nx * self.geom.ny

    @property
    def nominal_samples(self):
        return self.nrays * len(self.line.vchan) * self.geom.nstep

    def with_fields(self, dens=None, temp=None, vel=None) -> "Scene":
        g = replace(self.grid,
                    dens=self.grid.dens if dens is None else np.ascontiguousarray(dens, np.float32),
                    temp=self.grid.temp if temp is None else np.ascontiguousarray(temp, np.float32),
                    vel=self.grid.vel if vel is None else np.ascontiguousarray(vel, np.float32))
        return replace(self, grid=g)
