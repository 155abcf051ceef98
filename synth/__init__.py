"""Seeded synthetic inputs for the line-RT render (shared by the oracle tests and the CUDA path).

This package holds *only* input descriptions and generators: scene containers, the CO rigid-rotor
line table used by the configs, the analytic disk family of BASELINE.json `configs[0..4]`, and small
analytic scenes (slabs) for the closed-form pins.  It holds none of the render's arithmetic
(no ray geometry, no profile, no transfer) and imports neither `oracle/` nor the CUDA package.
"""
from .scene import Geom, Line, Grid, Scene, AXISYM, CART3D, SPH3D, DENS_LINEAR, DENS_LN, VEL_VPHI, VEL_KEPLER_FRAC
from .scene import UNIT_S0, UNIT_CGS, UNIT_JY_PIXEL
from .lines import co_line
from .disks import make_config, config_names, slab_scene, tiny_axisym_scene, tiny_cart_scene, l2_target
from .disks import tiny_sph_scene, sph_benchmark_scene

__all__ = [
    "Geom", "Line", "Grid", "Scene", "AXISYM", "CART3D", "SPH3D", "DENS_LINEAR", "DENS_LN", "VEL_VPHI",
    "VEL_KEPLER_FRAC", "UNIT_S0", "UNIT_CGS", "UNIT_JY_PIXEL", "co_line", "make_config",
    "config_names", "slab_scene", "tiny_axisym_scene", "tiny_cart_scene", "l2_target", "tiny_sph_scene", "sph_benchmark_scene",
]
