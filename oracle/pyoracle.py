"""ctypes binding of the fp64 CPU oracle (TEST INFRASTRUCTURE).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It marshals `synth.Scene` containers into the oracle's own C structs and never touches
the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


class _Geom(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nstep", C.c_int32), ("pad_", C.c_int32),
                ("fov_x", C.c_double), ("fov_y", C.c_double), ("x0", C.c_double), ("y0", C.c_double),
                ("incl", C.c_double), ("pa", C.c_double), ("az", C.c_double), ("dist_pc", C.c_double),
                ("vsys", C.c_double), ("gm_star", C.c_double)]


class _Line(C.Structure):
    _fields_ = [("nu0", C.c_double), ("a_ul", C.c_double), ("g_u", C.c_double), ("e_u_K", C.c_double),
                ("nlev", C.c_int32), ("nchan", C.c_int32),
                ("e_lev_K", C.POINTER(C.c_double)), ("g_lev", C.POINTER(C.c_double)),
                ("m_line", C.c_double), ("m_gas", C.c_double), ("vturb_abs", C.c_double),
                ("vturb_mach", C.c_double), ("vchan", C.POINTER(C.c_double)),
                ("unit", C.c_int32), ("pad_", C.c_int32)]


class _Grid(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n", C.c_int32 * 3), ("lo", C.c_double * 3), ("hi", C.c_double * 3),
                ("mirror_z", C.c_int32), ("dens_mode", C.c_int32), ("vel_mode", C.c_int32), ("pad_", C.c_int32),
                ("dens", C.POINTER(C.c_float)), ("temp", C.POINTER(C.c_float)), ("vel", C.POINTER(C.c_float))]


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        _lib = C.CDLL(path)
        i64p = C.POINTER(C.c_int64)
        dp = C.POINTER(C.c_double)
        _lib.orc_ray_geometry.argtypes = [C.POINTER(_Geom), C.POINTER(_Grid), C.c_int64, i64p, dp, dp, dp, dp,
                                          C.POINTER(C.c_int32)]
        _lib.orc_render.argtypes = [C.POINTER(_Geom), C.POINTER(_Line), C.POINTER(_Grid), C.c_int64, i64p, dp]
        _lib.orc_render_bwd.argtypes = [C.POINTER(_Geom), C.POINTER(_Line), C.POINTER(_Grid), C.c_int64, i64p,
                                        dp, dp, dp, dp]
        _lib.orc_trace_ray.argtypes = [C.POINTER(_Geom), C.POINTER(_Line), C.POINTER(_Grid), C.c_int64,
                                       C.POINTER(C.c_int32), dp, dp, dp, dp, dp, dp]
        _lib.orc_partition.argtypes = [C.POINTER(_Line), C.c_double]
        _lib.orc_partition.restype = C.c_double
        _lib.orc_source_unit.argtypes = [C.POINTER(_Line), C.POINTER(_Geom)]
        _lib.orc_source_unit.restype = C.c_double
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_set_num_threads.argtypes = [C.c_int]
        _lib.orc_set_num_threads.restype = None
    return _lib


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class _Marshalled:
    """Keeps the numpy buffers alive next to the C structs that point into them."""

    def __init__(self, scene):
        g, ln, gr = scene.geom, scene.line, scene.grid
        self.geom = _Geom(nx=g.nx, ny=g.ny, nstep=g.nstep, pad_=0, fov_x=g.fov_x, fov_y=g.fov_y, x0=g.x0, y0=g.y0,
                          incl=g.incl, pa=g.pa, az=g.az, dist_pc=g.dist_pc, vsys=g.vsys, gm_star=g.gm_star)
        self.e_lev = np.ascontiguousarray(ln.e_lev_K, np.float64)
        self.g_lev = np.ascontiguousarray(ln.g_lev, np.float64)
        self.vchan = np.ascontiguousarray(ln.vchan, np.float64)
        self.line = _Line(nu0=ln.nu0, a_ul=ln.a_ul, g_u=ln.g_u, e_u_K=ln.e_u_K, nlev=len(self.e_lev),
                          nchan=len(self.vchan), e_lev_K=_dptr(self.e_lev), g_lev=_dptr(self.g_lev),
                          m_line=ln.m_line, m_gas=ln.m_gas, vturb_abs=ln.vturb_abs, vturb_mach=ln.vturb_mach,
                          vchan=_dptr(self.vchan), unit=ln.unit, pad_=0)
        self.dens = np.ascontiguousarray(gr.dens, np.float32)
        self.temp = np.ascontiguousarray(gr.temp, np.float32)
        self.vel = np.ascontiguousarray(gr.vel, np.float32)
        n3 = tuple(gr.n) + (1,) * (3 - len(gr.n))
        lo3 = tuple(gr.lo) + (0.0,) * (3 - len(gr.lo))
        hi3 = tuple(gr.hi) + (0.0,) * (3 - len(gr.hi))
        fp = C.POINTER(C.c_float)
        self.grid = _Grid(kind=gr.kind, n=(C.c_int32 * 3)(*n3), lo=(C.c_double * 3)(*lo3),
                          hi=(C.c_double * 3)(*hi3), mirror_z=int(gr.mirror_z), dens_mode=gr.dens_mode,
                          vel_mode=gr.vel_mode, pad_=0, dens=self.dens.ctypes.data_as(fp),
                          temp=self.temp.ctypes.data_as(fp), vel=self.vel.ctypes.data_as(fp))
        self.nchan = len(self.vchan)
        self.nrays_all = g.nx * g.ny
        self.grid_shape = self.dens.shape


def _rays(m, rays):
    if rays is None:
        return m.nrays_all, None, None
    idx = np.ascontiguousarray(rays, np.int64)
    return len(idx), idx, idx.ctypes.data_as(C.POINTER(C.c_int64))


def render(scene, rays=None) -> np.ndarray:
    """Forward cube, fp64.  rays=None -> array [ny][nx][nchan]; else [len(rays)][nchan]."""
    m = _Marshalled(scene)
    n, idx, ip = _rays(m, rays)
    out = np.zeros((n, m.nchan), np.float64)
    rc = lib().orc_render(C.byref(m.geom), C.byref(m.line), C.byref(m.grid), n, ip, _dptr(out))
    assert rc == 0
    if rays is None:
        return out.reshape(scene.geom.ny, scene.geom.nx, m.nchan)
    return out


def render_bwd(scene, G, rays=None):
    """Adjoint: returns (g_dens, g_temp, g_vel), fp64, grid-shaped, for G = dL/dcube."""
    m = _Marshalled(scene)
    n, idx, ip = _rays(m, rays)
    Gc = np.ascontiguousarray(np.asarray(G, np.float64).reshape(n, m.nchan))
    gd = np.zeros(m.grid_shape, np.float64)
    gt = np.zeros(m.grid_shape, np.float64)
    gv = np.zeros(m.grid_shape, np.float64)
    rc = lib().orc_render_bwd(C.byref(m.geom), C.byref(m.line), C.byref(m.grid), n, ip, _dptr(Gc),
                              _dptr(gd), _dptr(gt), _dptr(gv))
    assert rc == 0
    return gd, gt, gv


def ray_geometry(scene, rays=None):
    """Returns dict(origin [n,3], dir [3], s0 [n], ds [n], valid [n])."""
    m = _Marshalled(scene)
    n, idx, ip = _rays(m, rays)
    org = np.zeros((n, 3)); d = np.zeros(3); s0 = np.zeros(n); ds = np.zeros(n)
    valid = np.zeros(n, np.int32)
    lib().orc_ray_geometry(C.byref(m.geom), C.byref(m.grid), n, ip, _dptr(org), _dptr(d), _dptr(s0), _dptr(ds),
                           valid.ctypes.data_as(C.POINTER(C.c_int32)))
    return {"origin": org, "dir": d, "s0": s0, "ds": ds, "valid": valid}


def trace_ray(scene, ray: int):
    """Per-step diagnostics of one ray: dict of arrays of length nstep."""
    m = _Marshalled(scene)
    N = scene.geom.nstep
    inside = np.zeros(N, np.int32)
    arrs = {k: np.zeros(N) for k in ("n", "T", "vlos", "alpha", "K", "S")}
    valid = lib().orc_trace_ray(C.byref(m.geom), C.byref(m.line), C.byref(m.grid), int(ray),
                                inside.ctypes.data_as(C.POINTER(C.c_int32)),
                                *[_dptr(arrs[k]) for k in ("n", "T", "vlos", "alpha", "K", "S")])
    arrs["inside"] = inside
    arrs["valid"] = valid
    return arrs


def partition(scene_or_line, T: float) -> float:
    line = getattr(scene_or_line, "line", scene_or_line)

    class _S:  # minimal scene shim
        pass
    from synth.scene import Geom, Grid, Scene
    dummy = Scene(Geom(1, 1, 1.0, 1.0, 0.0), line,
                  Grid(0, (2, 2), (1.0, 0.0), (2.0, 1.0), np.zeros((2, 2), np.float32),
                       np.ones((2, 2), np.float32), np.zeros((2, 2), np.float32)))
    m = _Marshalled(dummy)
    return float(lib().orc_partition(C.byref(m.line), float(T)))


def source_unit(scene) -> float:
    m = _Marshalled(scene)
    return float(lib().orc_source_unit(C.byref(m.line), C.byref(m.geom)))


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int):
    """Threads for the following oracle calls (timing only)."""
    lib().orc_set_num_threads(int(n))


def chi2_loss_grad(cube, target, sigma: float):
    """Pixel-wise chi^2 data term of the fit ("chi^2 ... averaged over pixels"; the L2 loss of
    BASELINE.json configs 2-5), plain numpy in fp64:
        L = 1/(2 n) sum_i ((I_i - D_i)/sigma)^2,    dL/dI_i = (I_i - D_i) / (sigma^2 n),    n = number of voxels.
    Returns (L, dL/dI).  Pinned in tests/test_oracle_closed_forms.py (constant residual, finite differences)."""
    I = np.asarray(cube, dtype=np.float64)
    D = np.asarray(target, dtype=np.float64)
    n = I.size
    r = I - D
    return float(np.sum((r / sigma) ** 2) / (2.0 * n)), r / (sigma * sigma * n)
