"""Thin ctypes binding of libradt.so (include/radt.h): argument marshalling only.

Every step of the render runs in the CUDA kernels of csrc/; this module converts `synth.Scene`
containers and torch tensors (device memory + streams) into the C structs and pointers of the ABI.
There is no CPU path: if the shared library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("RADT_LIB") or os.path.join(_HERE, "libradt.so")      # (RADT_LIB: another build of the same ABI)

PASS_FWD, PASS_BWD = 0, 1

EXPORTS = ["radt_version", "radt_last_error", "radt_options_default", "radt_workspace_bytes",
           "radt_ray_geometry", "radt_render", "radt_render_bwd", "radt_grad_layout", "radt_unpack_grad",
           "radt_l2_loss_grad", "radt_render_host",
           "radt_render_loss", "radt_disk_workspace_bytes", "radt_disk_fields", "radt_disk_fields_bwd",
           "radt_disk_fields_static",
           "radt_mlp_num_params", "radt_mlp_temperature", "radt_mlp_temperature_bwd",
           "radt_fit_step_host", "radt_render_bwd_host", "radt_pipe_peak", "radt_read_counters", "radt_read_lane_counters",
           "radt_last_launch_count", "radt_forget", "radt_debug_host_split"]


class RadtError(RuntimeError):
    pass


class radt_geom(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("nx", C.c_int32), ("ny", C.c_int32), ("nstep", C.c_int32),
                ("fov_x", C.c_double), ("fov_y", C.c_double), ("x0", C.c_double), ("y0", C.c_double),
                ("incl", C.c_double), ("pa", C.c_double), ("az", C.c_double), ("dist_pc", C.c_double),
                ("vsys", C.c_double), ("gm_star", C.c_double)]


class radt_line(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("nlev", C.c_int32), ("nchan", C.c_int32), ("unit", C.c_int32),
                ("nu0", C.c_double), ("a_ul", C.c_double), ("g_u", C.c_double), ("e_u_K", C.c_double),
                ("e_lev_K", C.POINTER(C.c_double)), ("g_lev", C.POINTER(C.c_double)),
                ("m_line", C.c_double), ("m_gas", C.c_double), ("vturb_abs", C.c_double), ("vturb_mach", C.c_double),
                ("vchan", C.POINTER(C.c_double))]


class radt_grid(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("kind", C.c_int32), ("n", C.c_int32 * 3), ("mirror_z", C.c_int32),
                ("dens_mode", C.c_int32), ("vel_mode", C.c_int32), ("lo", C.c_double * 3), ("hi", C.c_double * 3),
                ("batch_stride", C.c_int64), ("dens", C.c_void_p), ("temp", C.c_void_p), ("vel", C.c_void_p)]


class radt_options(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("window", C.c_int32), ("skip_empty", C.c_int32), ("win_path", C.c_int32),
                ("zero_dens_grad", C.c_int32), ("reuse_setup", C.c_int32)]


_lib = None


def make_options(**kw):
    """radt_options with the library's defaults (radt_options_default), fields overridden by keyword."""
    o = radt_options()
    lib().radt_options_default(C.byref(o))
    for k, v in kw.items():
        if k not in ("window", "skip_empty", "win_path", "zero_dens_grad", "reuse_setup"):
            raise KeyError(f"unknown radt_options field {k!r}")
        setattr(o, k, int(v))
    return o


def _optp(opt):
    return C.byref(opt) if opt is not None else None


class radt_disk(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("pad_", C.c_uint32), ("gm_star", C.c_double), ("m_gas", C.c_double),
                ("sigma0", C.c_double), ("r_c", C.c_double), ("gamma", C.c_double), ("x_co", C.c_double),
                ("t_freeze", C.c_double), ("n_dissoc", C.c_double), ("f_col", C.c_double)]


class radt_mlp(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("L", C.c_int32), ("width", C.c_int32), ("nhidden", C.c_int32),
                ("t_lo", C.c_double), ("t_hi", C.c_double)]


def make_mlp(L=4, t_lo=5.0, t_hi=400.0, width=64, nhidden=4):
    return radt_mlp(C.sizeof(radt_mlp), L, width, nhidden, t_lo, t_hi)


def make_disks(params):
    """ctypes array of radt_disk from objects with the fields of radt_disk (gm_star, m_gas | m_mol, sigma0, ...)."""
    params = _as_list(params)
    arr = (radt_disk * len(params))()
    for b, p in enumerate(params):
        arr[b] = radt_disk(C.sizeof(radt_disk), 0, p.gm_star, getattr(p, "m_gas", None) or p.m_mol, p.sigma0, p.r_c,
                           p.gamma, p.x_co, p.t_freeze, p.n_dissoc, p.f_col)
    return arr


def lib():
    """Load libradt.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RadtError(f"{LIB_PATH} not found: build it with `python -m paper_2509_03623_b200.build` "
                            "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        gp, lp, rp = C.POINTER(radt_geom), C.POINTER(radt_line), C.POINTER(radt_grid)
        L.radt_version.restype = C.c_int
        L.radt_last_error.restype = C.c_char_p
        op = C.POINTER(radt_options)
        L.radt_options_default.argtypes = [op]
        L.radt_options_default.restype = None
        L.radt_workspace_bytes.argtypes = [gp, lp, rp, i32, i32, C.POINTER(C.c_size_t)]
        L.radt_ray_geometry.argtypes = [gp, rp, i32, vp, vp]
        L.radt_render.argtypes = [gp, lp, rp, i32, op, vp, vp, vp, C.c_size_t, vp]
        L.radt_render_bwd.argtypes = [gp, lp, rp, i32, op, vp, vp, vp, vp, vp, vp, vp, C.c_size_t, vp]
        L.radt_grad_layout.argtypes = [gp, lp, rp, i32, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
        L.radt_unpack_grad.argtypes = [gp, lp, rp, i32, vp, C.c_size_t, vp, vp, vp, vp]
        L.radt_l2_loss_grad.argtypes = [vp, vp, dbl, i64, vp, vp, vp]
        L.radt_render_loss.argtypes = [gp, lp, rp, i32, op, vp, dbl, vp, vp, vp, vp, vp, C.c_size_t, vp]
        L.radt_render_host.argtypes = [gp, lp, rp, i32, op, vp, vp]
        L.radt_mlp_num_params.argtypes = [C.POINTER(radt_mlp), C.POINTER(C.c_int64)]
        L.radt_mlp_temperature.argtypes = [C.POINTER(radt_mlp), rp, vp, vp, vp]
        L.radt_mlp_temperature_bwd.argtypes = [C.POINTER(radt_mlp), rp, vp, vp, vp, vp]
        L.radt_disk_workspace_bytes.argtypes = [rp, i32, C.POINTER(C.c_size_t)]
        L.radt_disk_fields.argtypes = [C.POINTER(radt_disk), rp, i32, vp, vp, vp, vp, C.c_size_t, vp]
        L.radt_disk_fields_bwd.argtypes = [C.POINTER(radt_disk), rp, i32, vp, vp, vp, vp, vp, C.c_size_t, vp]
        L.radt_disk_fields_static.argtypes = [C.POINTER(radt_disk), rp, i32, vp, vp, vp, vp]
        L.radt_fit_step_host.argtypes = [gp, lp, rp, i32, op, vp, dbl, vp, C.POINTER(dbl), vp, vp, vp]
        L.radt_render_bwd_host.argtypes = [gp, lp, rp, i32, op, vp, vp, vp, vp, vp, vp]
        L.radt_pipe_peak.argtypes = [i32, C.POINTER(dbl), C.POINTER(dbl)]
        L.radt_read_counters.argtypes = [vp, C.POINTER(C.c_uint64), vp]
        L.radt_read_lane_counters.argtypes = [vp, C.POINTER(C.c_uint64), vp]
        L.radt_last_launch_count.restype = C.c_int
        L.radt_forget.argtypes = [vp]
        L.radt_debug_host_split.argtypes = [i32, i32]
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise RadtError(f"radt error {rc}: {lib().radt_last_error().decode()}")


def _as_list(scenes):
    return list(scenes) if isinstance(scenes, (list, tuple)) else [scenes]


class Descriptors:
    """C descriptors of a batch of scenes that share line, grid geometry and image size."""

    def __init__(self, scenes):
        scenes = _as_list(scenes)
        s0 = scenes[0]
        self.batch = len(scenes)
        self.geom = (radt_geom * self.batch)()
        for b, sc in enumerate(scenes):
            g = sc.geom
            self.geom[b] = radt_geom(C.sizeof(radt_geom), g.nx, g.ny, g.nstep, g.fov_x, g.fov_y, g.x0, g.y0, g.incl,
                                     g.pa, g.az, g.dist_pc, g.vsys, g.gm_star)
        ln = s0.line
        self._e = np.ascontiguousarray(ln.e_lev_K, np.float64)
        self._g = np.ascontiguousarray(ln.g_lev, np.float64)
        self._v = np.ascontiguousarray(ln.vchan, np.float64)
        dp = C.POINTER(C.c_double)
        self.line = radt_line(C.sizeof(radt_line), len(self._e), len(self._v), ln.unit, ln.nu0, ln.a_ul, ln.g_u,
                              ln.e_u_K, self._e.ctypes.data_as(dp), self._g.ctypes.data_as(dp), ln.m_line, ln.m_gas,
                              ln.vturb_abs, ln.vturb_mach, self._v.ctypes.data_as(dp))
        gr = s0.grid
        n3 = tuple(gr.n) + (1,) * (3 - len(gr.n))
        lo3 = tuple(gr.lo) + (0.0,) * (3 - len(gr.lo))
        hi3 = tuple(gr.hi) + (0.0,) * (3 - len(gr.hi))
        self.cells = int(np.prod(gr.n))
        self.grid_shape = tuple(gr.n)
        self.grid = radt_grid(C.sizeof(radt_grid), gr.kind, (C.c_int32 * 3)(*n3), int(gr.mirror_z), gr.dens_mode,
                              gr.vel_mode, (C.c_double * 3)(*lo3), (C.c_double * 3)(*hi3), self.cells, None, None, None)
        self.nx, self.ny, self.nchan, self.nstep = s0.geom.nx, s0.geom.ny, len(self._v), s0.geom.nstep
        self.cube_shape = (self.batch, self.ny, self.nx, self.nchan)

    def with_fields(self, dens_ptr, temp_ptr, vel_ptr):
        self.grid.dens, self.grid.temp, self.grid.vel = dens_ptr, temp_ptr, vel_ptr
        return self


def stack_fields(scenes):
    """Host float32 arrays [batch, *grid] of the three fields."""
    scenes = _as_list(scenes)
    return tuple(np.ascontiguousarray(np.stack([np.asarray(getattr(sc.grid, f), np.float32) for sc in scenes]))
                 for f in ("dens", "temp", "vel"))


class _on:
    """Make the tensor's device current for the duration of a C-ABI call: the library launches on the CURRENT device,
    so a Renderer on cuda:1 must not run its kernels on cuda:0 against cuda:1 pointers."""

    def __init__(self, t):
        import torch
        self._ctx = torch.cuda.device(t.device)

    def __enter__(self):
        return self._ctx.__enter__()

    def __exit__(self, *a):
        return self._ctx.__exit__(*a)


def _stream_ptr(stream, like=None):
    """Pointer of `stream`, or of the current stream of the device that holds tensor `like`."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream(like.device if like is not None else None)
    return C.c_void_p(stream.cuda_stream)


def _p(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


# ------------------------------------------------------------------------------------------------
# same names as the C ABI
# ------------------------------------------------------------------------------------------------
def radt_version() -> int:
    return lib().radt_version()


def radt_workspace_bytes(desc: Descriptors, pass_: int) -> int:
    out = C.c_size_t(0)
    _check(lib().radt_workspace_bytes(desc.geom, C.byref(desc.line), C.byref(desc.grid), desc.batch, pass_, C.byref(out)))
    return out.value


def radt_ray_geometry(desc: Descriptors, rays_out, stream=None):
    """rays_out: CUDA float64 tensor [batch, ny, nx, 2]."""
    with _on(rays_out):
        _check(lib().radt_ray_geometry(desc.geom, C.byref(desc.grid), desc.batch, _p(rays_out), _stream_ptr(stream, rays_out)))


def radt_render(desc: Descriptors, dens, temp, vel, cube, ws, stream=None, opt=None, cube_lo=None):
    """dens/temp/vel: CUDA float32 tensors [batch, *grid]; cube (and cube_lo, optional): CUDA float32 [batch, ny, nx, nchan];
    ws: CUDA uint8; opt: radt_options or None (defaults)."""
    desc.with_fields(dens.data_ptr(), temp.data_ptr(), vel.data_ptr())
    with _on(cube):
        _check(lib().radt_render(desc.geom, C.byref(desc.line), C.byref(desc.grid), desc.batch, _optp(opt), _p(cube),
                                 _p(cube_lo), _p(ws), ws.numel(), _stream_ptr(stream, cube)))


def radt_render_bwd(desc: Descriptors, dens, temp, vel, cube, dl_dcube, g_dens, g_temp, g_vel, ws, stream=None, opt=None,
                    cube_lo=None):
    desc.with_fields(dens.data_ptr(), temp.data_ptr(), vel.data_ptr())
    with _on(cube):
        _check(lib().radt_render_bwd(desc.geom, C.byref(desc.line), C.byref(desc.grid), desc.batch, _optp(opt), _p(cube),
                                     _p(cube_lo), _p(dl_dcube), _p(g_dens), _p(g_temp), _p(g_vel), _p(ws), ws.numel(),
                                     _stream_ptr(stream, cube)))


def radt_grad_layout(desc: Descriptors):
    """(byte offset, number of floats) of the packed gradient cells inside a PASS_BWD workspace."""
    off, n = C.c_size_t(0), C.c_size_t(0)
    _check(lib().radt_grad_layout(desc.geom, C.byref(desc.line), C.byref(desc.grid), desc.batch, C.byref(off), C.byref(n)))
    return off.value, n.value


def radt_unpack_grad(desc: Descriptors, ws, g_dens, g_temp, g_vel, stream=None):
    with _on(ws):
        _check(lib().radt_unpack_grad(desc.geom, C.byref(desc.line), C.byref(desc.grid), desc.batch, _p(ws), ws.numel(),
                                      _p(g_dens), _p(g_temp), _p(g_vel), _stream_ptr(stream, ws)))


def radt_l2_loss_grad(cube, target, sigma: float, dl_dcube, loss_out, stream=None):
    """loss_out: CUDA float64 tensor [1]."""
    with _on(cube):
        _check(lib().radt_l2_loss_grad(_p(cube), _p(target), float(sigma), cube.numel(), _p(dl_dcube), _p(loss_out),
                                       _stream_ptr(stream, cube)))


def radt_render_loss(desc: Descriptors, dens, temp, vel, target, sigma: float, cube, dl_dcube, loss_out, ws, stream=None,
                     opt=None, cube_lo=None):
    """Forward render with the fused chi^2 data term: cube, dl_dcube, loss_out (CUDA float64 [1]) in one pass."""
    desc.with_fields(dens.data_ptr(), temp.data_ptr(), vel.data_ptr())
    with _on(cube):
        _check(lib().radt_render_loss(desc.geom, C.byref(desc.line), C.byref(desc.grid), desc.batch, _optp(opt), _p(target),
                                      C.c_double(float(sigma)), _p(cube), _p(cube_lo), _p(dl_dcube), _p(loss_out), _p(ws),
                                      C.c_size_t(ws.numel()), _stream_ptr(stream, cube)))


def radt_forget(tensor_or_ptr) -> None:
    """Drop what the library remembers about a device buffer (a cube's forward options, a workspace's setup)."""
    ptr = tensor_or_ptr.data_ptr() if hasattr(tensor_or_ptr, "data_ptr") else int(tensor_or_ptr)
    _check(lib().radt_forget(C.c_void_p(ptr)))


def radt_debug_host_split(chunk_items: int = 0, band_rows: int = 0) -> None:
    """Test hook of the HOST entry points (this thread): forced chunk / band sizes, 0 = the library's policy."""
    _check(lib().radt_debug_host_split(int(chunk_items), int(band_rows)))


def radt_disk_workspace_bytes(desc: Descriptors) -> int:
    out = C.c_size_t(0)
    _check(lib().radt_disk_workspace_bytes(C.byref(desc.grid), desc.batch, C.byref(out)))
    return out.value


def radt_disk_fields(disks, desc: Descriptors, temp, dens_out, vel_out, ws, stream=None):
    """Physics pre-pass: temp -> n_CO, v_phi (CUDA float32 tensors [batch, nr, nzeta]); disks from make_disks()."""
    with _on(temp):
        _check(lib().radt_disk_fields(disks, C.byref(desc.grid), desc.batch, _p(temp), _p(dens_out), _p(vel_out), _p(ws),
                                      C.c_size_t(ws.numel()), _stream_ptr(stream, temp)))


DISK_STATIC_MAX_CELLS = 262144          # RADT_DISK_STATIC_MAX_CELLS of include/radt.h


def radt_disk_fields_static(disks, desc: Descriptors, temp, dens_out, vel_out, stream=None):
    """radt_disk_fields for callers that cannot allocate a workspace (all device memory belongs to someone else, or
    cudaMalloc's device-wide synchronisation is not acceptable): the scratch is a fixed array inside libradt.so, at most
    DISK_STATIC_MAX_CELLS cells per call.  One array per GPU: do not overlap two calls on the same GPU; make the first
    call on a device before any stream capture (include/radt.h)."""
    with _on(temp):
        _check(lib().radt_disk_fields_static(disks, C.byref(desc.grid), desc.batch, _p(temp), _p(dens_out), _p(vel_out),
                                             _stream_ptr(stream, temp)))


def radt_disk_fields_bwd(disks, desc: Descriptors, temp, g_dens, g_vel, g_temp, ws, stream=None):
    """g_temp += (d n_CO/d temp)^T g_dens + (d v_phi/d temp)^T g_vel."""
    with _on(temp):
        _check(lib().radt_disk_fields_bwd(disks, C.byref(desc.grid), desc.batch, _p(temp), _p(g_dens), _p(g_vel), _p(g_temp),
                                          _p(ws), C.c_size_t(ws.numel()), _stream_ptr(stream, temp)))


def radt_mlp_num_params(mlp) -> int:
    out = C.c_int64(0)
    _check(lib().radt_mlp_num_params(C.byref(mlp), C.byref(out)))
    return out.value


def radt_mlp_temperature(mlp, desc: Descriptors, params, temp_out, stream=None):
    """MLP temperature field on the grid nodes: params CUDA float32 [num_params] -> temp_out CUDA float32 [nr, nzeta]."""
    with _on(params):
        _check(lib().radt_mlp_temperature(C.byref(mlp), C.byref(desc.grid), _p(params), _p(temp_out),
                                          _stream_ptr(stream, params)))


def radt_mlp_temperature_bwd(mlp, desc: Descriptors, params, g_temp, g_params, stream=None):
    with _on(params):
        _check(lib().radt_mlp_temperature_bwd(C.byref(mlp), C.byref(desc.grid), _p(params), _p(g_temp), _p(g_params),
                                              _stream_ptr(stream, params)))


def radt_read_counters(ws, stream=None):
    out = (C.c_uint64 * 4)()
    with _on(ws):
        _check(lib().radt_read_counters(_p(ws), out, _stream_ptr(stream, ws)))
    return [int(x) for x in out]


def radt_read_lane_counters(ws, stream=None):
    """(samples inside their line window, samples executed) of the last forward march on `ws`."""
    out = (C.c_uint64 * 2)()
    with _on(ws):
        _check(lib().radt_read_lane_counters(_p(ws), out, _stream_ptr(stream, ws)))
    return int(out[0]), int(out[1])


def radt_last_launch_count() -> int:
    return lib().radt_last_launch_count()


def _hptr(a):
    return C.c_void_p(a.ctypes.data) if a is not None else None


def radt_render_host(desc: Descriptors, dens, temp, vel, cube, opt=None, cube_lo=None):
    """HOST numpy float32 arrays in, HOST cube (and optionally its low-order words) out (copies inside the call)."""
    desc.with_fields(dens.ctypes.data, temp.ctypes.data, vel.ctypes.data)
    _check(lib().radt_render_host(desc.geom, C.byref(desc.line), C.byref(desc.grid), desc.batch, _optp(opt), _hptr(cube),
                                  _hptr(cube_lo)))


def radt_fit_step_host(desc: Descriptors, dens, temp, vel, target, sigma, cube, g_dens, g_temp, g_vel, opt=None) -> float:
    desc.with_fields(dens.ctypes.data, temp.ctypes.data, vel.ctypes.data)
    loss = C.c_double(0.0)
    _check(lib().radt_fit_step_host(desc.geom, C.byref(desc.line), C.byref(desc.grid), desc.batch, _optp(opt), _hptr(target),
                                    float(sigma), _hptr(cube), C.byref(loss), _hptr(g_dens), _hptr(g_temp), _hptr(g_vel)))
    return loss.value


def radt_render_bwd_host(desc: Descriptors, dens, temp, vel, cube, dl_dcube, g_dens, g_temp, g_vel, opt=None, cube_lo=None):
    desc.with_fields(dens.ctypes.data, temp.ctypes.data, vel.ctypes.data)
    _check(lib().radt_render_bwd_host(desc.geom, C.byref(desc.line), C.byref(desc.grid), desc.batch, _optp(opt), _hptr(cube),
                                      _hptr(cube_lo), _hptr(dl_dcube), _hptr(g_dens), _hptr(g_temp), _hptr(g_vel)))


def radt_pipe_peak(kind: int):
    """Returns (lane-ops per second, SM clock in MHz) of pipe `kind` (0 MUFU.EX2, 1 FFMA, 2 DFMA, 3 FFMA2)."""
    ops, clk = C.c_double(0.0), C.c_double(0.0)
    _check(lib().radt_pipe_peak(kind, C.byref(ops), C.byref(clk)))
    return ops.value, clk.value
