"""Host-side sharding of ONE image across ranks: rays are independent.

A slab of image rows [r0, r1) is itself a valid image description, so sharding needs no kernel support:
    ny' = r1 - r0,   fov_y' = fov_y * ny' / ny,   y0' = y0 + ((r0 + r1)/2 - ny/2) * fov_y / ny
The forward needs no collective (each rank owns its cube rows); the adjoint needs one all-reduce(sum) of
the three gradient buffers, because every rank's rays scatter into the same grid.

The `engine` does the rendering: on GPUs it is `CudaEngine` (the C-ABI path, NCCL for the reduction);
tests inject a CPU engine and the gloo backend to cover this plumbing without a GPU.
"""
from __future__ import annotations

from dataclasses import replace

import numpy as np


def plan_rows(ny: int, world: int):
    """Contiguous, balanced row slabs [(r0, r1)] covering 0..ny exactly once; empty slabs if world > ny."""
    base, rem = divmod(ny, world)
    out, r0 = [], 0
    for k in range(world):
        r1 = r0 + base + (1 if k < rem else 0)
        out.append((r0, r1))
        r0 = r1
    return out


def row_slab_scene(scene, r0: int, r1: int):
    """The sub-image made of rows r0..r1-1 of `scene` (same pixel centres, same pixel size)."""
    g = scene.geom
    if not (0 <= r0 < r1 <= g.ny):
        raise ValueError("need 0 <= r0 < r1 <= ny")
    pix = g.fov_y / g.ny
    sub = replace(g, ny=r1 - r0, fov_y=pix * (r1 - r0), y0=g.y0 + (0.5 * (r0 + r1) - 0.5 * g.ny) * pix)
    return replace(scene, geom=sub)


class CudaEngine:
    """Product engine: the CUDA render through the C ABI."""

    def __init__(self, scene, device):
        from .render import Renderer
        self.R = Renderer([scene], device=device)

    def render(self):
        return self.R.render()[0]

    def render_bwd(self, dl_dcube):
        self.R.dl_dcube.copy_(dl_dcube.reshape(self.R.dl_dcube.shape))
        return [g[0] for g in self.R.render_bwd()]


class ShardedImage:
    """One image split by rows over the ranks of a torch.distributed process group."""

    def __init__(self, scene, engine_factory, rank=None, world=None, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank = dist.get_rank(group) if rank is None else rank
        self.world = dist.get_world_size(group) if world is None else world
        self.scene = scene
        self.rows = plan_rows(scene.geom.ny, self.world)
        r0, r1 = self.rows[self.rank]
        self.r0, self.r1 = r0, r1
        self.engine = engine_factory(row_slab_scene(scene, r0, r1)) if r1 > r0 else None

    def render(self):
        """This rank's rows of the cube, [r1 - r0, nx, nchan] (no communication)."""
        return self.engine.render() if self.engine is not None else None

    def gather_cube(self, slab):
        """All ranks' slabs concatenated along rows (all_gather; only when one rank needs the whole cube)."""
        import torch
        nx, nchan = self.scene.geom.nx, len(self.scene.line.vchan)
        parts = [torch.empty((b - a, nx, nchan), dtype=slab.dtype if slab is not None else torch.float32,
                             device=slab.device if slab is not None else "cpu") for a, b in self.rows]
        mine = slab if slab is not None else parts[self.rank]
        # all_gather needs equal shapes: pad to the largest slab
        hmax = max(b - a for a, b in self.rows)
        pad = torch.zeros((hmax, nx, nchan), dtype=mine.dtype, device=mine.device)
        pad[: mine.shape[0]] = mine
        bufs = [torch.empty_like(pad) for _ in range(self.world)]
        self.dist.all_gather(bufs, pad, group=self.group)
        return torch.cat([bufs[k][: b - a] for k, (a, b) in enumerate(self.rows)], dim=0)

    def render_bwd(self, dl_dcube_slab):
        """Gradients w.r.t. the (replicated) grid: local adjoint of this rank's rows, then all_reduce(sum)."""
        import torch
        if self.engine is not None:
            grads = [g.clone() for g in self.engine.render_bwd(dl_dcube_slab)]
        else:
            shape = tuple(self.scene.grid.n)
            grads = [torch.zeros(shape, dtype=torch.float32) for _ in range(3)]
        for g in grads:
            self.dist.all_reduce(g, op=self.dist.ReduceOp.SUM, group=self.group)
        return grads
