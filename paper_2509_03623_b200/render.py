"""Device-buffer plumbing around the C ABI: owns the torch tensors a render needs and forwards pointers."""
from __future__ import annotations

import numpy as np

from . import binding as B


class Renderer:
    """Holds fields, workspace, cube and gradient buffers on one CUDA device for a batch of scenes.

    options: radt_options fields (window, skip_empty, win_path, zero_dens_grad) for every call of this object;
    compensated: keep the low-order words of the cube (cube_lo) so that the adjoint is free of cancellation noise on
    optically thick rays (the default; include/radt.h radt_render)."""

    def __init__(self, scenes, device="cuda:0", need_bwd=True, options=None, compensated=True):
        import torch
        if not torch.cuda.is_available():
            raise B.RadtError("no CUDA device: the render has no CPU fallback")
        B.lib()
        self.torch = torch
        self.device = torch.device(device)
        self.desc = B.Descriptors(scenes)
        self.options = dict(options or {})
        self.opt = B.make_options(**self.options)
        self.opt_reuse = B.make_options(**self.options, reuse_setup=1)
        d = self.desc
        host = B.stack_fields(scenes)
        self.dens, self.temp, self.vel = (torch.from_numpy(h).to(self.device) for h in host)
        self.cube = torch.empty(d.cube_shape, dtype=torch.float32, device=self.device)
        self.cube_lo = torch.empty_like(self.cube) if (compensated and need_bwd) else None
        nbytes = B.radt_workspace_bytes(d, B.PASS_BWD if need_bwd else B.PASS_FWD)
        self.ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.need_bwd = need_bwd
        if need_bwd:
            self.dl_dcube = torch.empty_like(self.cube)
            self.g_dens = torch.empty_like(self.dens)
            self.g_temp = torch.empty_like(self.temp)
            self.g_vel = torch.empty_like(self.vel)
            self.loss = torch.zeros(1, dtype=torch.float64, device=self.device)
        self.target = None
        self.sigma = None
        # True while the workspace holds the setup (packed cells, occupancy words, T_max) of this object's last forward of the
        # CURRENT field values and options.  The library can only compare descriptors and pointers; set_fields copies in place,
        # so the pointers stay the same when the values change: that part of the reuse_setup contract is checked here.
        self._setup_valid = False

    def __del__(self):
        # The library remembers cubes and workspaces by raw device pointer and knows nothing of torch's allocator, which may hand
        # these addresses to the next tensor: drop that memory with the buffers (include/radt.h radt_forget).
        try:
            for t in (getattr(self, "cube", None), getattr(self, "ws", None)):
                if t is not None:
                    B.radt_forget(t)
        except Exception:      # noqa: BLE001  (interpreter shutdown: the binding may already be gone)
            pass

    def set_options(self, **kw):
        """Change this object's radt_options for the calls that follow (a forward and its adjoint must share them)."""
        self.options.update(kw)
        self.opt = B.make_options(**self.options)
        self.opt_reuse = B.make_options(**self.options, reuse_setup=1)
        self._setup_valid = False

    # ---- hot path: every call below is one C-ABI entry point ----
    def render(self, stream=None):
        B.radt_render(self.desc, self.dens, self.temp, self.vel, self.cube, self.ws, stream, self.opt, self.cube_lo)
        self._setup_valid = True
        return self.cube

    def render_bwd(self, dl_dcube=None, stream=None, reuse_setup=False, unpack=True):
        """reuse_setup: the workspace still holds what this object's last render()/render_loss() of the same fields left
        there; refused (RadtError) when the fields or options changed since, or an adjoint rebuilt the workspace for itself.
        unpack=False leaves the gradient as packed cells in the workspace (grad_packed())."""
        if reuse_setup and not self._setup_valid:
            raise B.RadtError("-1 (RADT_E_INVALID): reuse_setup, but the workspace does not hold the setup of a forward of the "
                              "current fields and options (set_fields / set_options / an adjoint with its own setup came after it)")
        if not reuse_setup:
            self._setup_valid = False          # the adjoint's own setup replaces the forward's
        g = self.dl_dcube if dl_dcube is None else dl_dcube
        outs = (self.g_dens, self.g_temp, self.g_vel) if unpack else (None, None, None)
        B.radt_render_bwd(self.desc, self.dens, self.temp, self.vel, self.cube, g, *outs, self.ws, stream,
                          self.opt_reuse if reuse_setup else self.opt, self.cube_lo)
        return self.g_dens, self.g_temp, self.g_vel

    def grad_packed(self):
        """View of the packed float4 gradient cells inside the workspace (what ONE all-reduce over ranks sums)."""
        off, n = B.radt_grad_layout(self.desc)
        return self.ws[off:off + 4 * n].view(self.torch.float32)

    def unpack_grad(self, stream=None):
        B.radt_unpack_grad(self.desc, self.ws, self.g_dens, self.g_temp, self.g_vel, stream)
        return self.g_dens, self.g_temp, self.g_vel

    def set_target(self, target, sigma):
        t = self.torch.as_tensor(np.ascontiguousarray(target, np.float32)) if not self.torch.is_tensor(target) else target
        self.target = t.to(self.device, dtype=self.torch.float32).reshape(self.cube.shape).contiguous()
        self.sigma = float(sigma)

    def l2_loss_grad(self, stream=None):
        B.radt_l2_loss_grad(self.cube, self.target, self.sigma, self.dl_dcube, self.loss, stream)
        return self.loss

    def render_loss(self, stream=None):
        """forward with the chi^2 data term fused into its epilogue: cube, dl_dcube and loss in one pass."""
        B.radt_render_loss(self.desc, self.dens, self.temp, self.vel, self.target, self.sigma, self.cube, self.dl_dcube,
                           self.loss, self.ws, stream, self.opt, self.cube_lo)
        self._setup_valid = True
        return self.loss

    def fit_step(self, stream=None, fused=True):
        """forward -> L2 data term -> adjoint (one pass of the whole hot path); the adjoint reuses the forward's setup."""
        if fused:
            self.render_loss(stream)
        else:
            self.render(stream)
            self.l2_loss_grad(stream)
        self.render_bwd(stream=stream, reuse_setup=True)

    def set_fields(self, dens=None, temp=None, vel=None):
        self._setup_valid = False
        for name, val in (("dens", dens), ("temp", temp), ("vel", vel)):
            if val is not None:
                getattr(self, name).copy_(self.torch.as_tensor(np.ascontiguousarray(val, np.float32)).reshape(
                    getattr(self, name).shape))

    def counters(self):
        return B.radt_read_counters(self.ws)

    def lane_counters(self):
        return B.radt_read_lane_counters(self.ws)

    def ray_table(self):
        d = self.desc
        rays = self.torch.empty((d.batch, d.ny, d.nx, 2), dtype=self.torch.float64, device=self.device)
        B.radt_ray_geometry(d, rays)
        return rays
