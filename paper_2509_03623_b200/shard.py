"""Host-side sharding of one render call across ranks: rays are independent
(PAPER.md:272), so the work splits by BATCH ITEMS first and by IMAGE ROWS second.

A slab of image rows [r0, r1) of one item is itself a valid image description, so sharding needs no kernel support:
    ny' = r1 - r0,   fov_y' = fov_y * ny' / ny,   y0' = y0 + ((r0 + r1)/2 - ny/2) * fov_y / ny
The forward needs no collective (each rank owns its cube rows).  The adjoint ends with ONE collective over the packed float4
gradient cells [item][cells][4] -- the buffer the adjoint march accumulates into, before it is unpacked into the three planes:
  - whole items per rank (world <= batch): every item's gradient is complete on the rank that owns it, so the ranks only
    exchange what they own: an ALL-GATHER of the owned items' cells (an all-reduce would move and add a [batch, cells * 4]
    buffer that is zero for every item a rank does not own: 268 MB per rank on config 4's shape);
  - rows of an item split over ranks (world > batch): the ranks hold partial sums of the same cells: an ALL-REDUCE.
`ShardedRender.collective` names which one a plan uses; `n_collectives` counts the calls.

The `engine` does the rendering: on GPUs it is `CudaEngine` (the C-ABI path; the all-reduce then runs over NCCL); tests inject
a CPU engine and the gloo backend to cover this plumbing without a GPU.
"""
from __future__ import annotations

from dataclasses import replace


def plan_rows(ny: int, world: int):
    """Contiguous, balanced row slabs [(r0, r1)] covering 0..ny exactly once; empty slabs if world > ny."""
    base, rem = divmod(ny, world)
    out, r0 = [], 0
    for k in range(world):
        r1 = r0 + base + (1 if k < rem else 0)
        out.append((r0, r1))
        r0 = r1
    return out


def plan_units(batch: int, ny: int, world: int):
    """Work units [(item, r0, r1)] per rank: batch items first, image rows second.

    world <= batch: every rank gets whole items (contiguous, balanced; no item is split).
    world >  batch: the ranks are dealt to the items (contiguous, balanced) and each item's rows are split among its ranks.
    Every (item, row) is covered exactly once; a rank may be left without work only if an item has fewer rows than ranks."""
    if batch < 1 or ny < 1 or world < 1:
        raise ValueError("need batch, ny, world >= 1")
    if world <= batch:
        return [[(b, 0, ny) for b in range(a, e)] for a, e in plan_rows(batch, world)]
    out = []
    for b, (k0, k1) in enumerate(plan_rows(world, batch)):      # ranks k0..k1-1 serve item b
        for r0, r1 in plan_rows(ny, k1 - k0):
            out.append([(b, r0, r1)] if r1 > r0 else [])
    return out


def row_slab_scene(scene, r0: int, r1: int):
    """The sub-image made of rows r0..r1-1 of `scene` (same pixel centres, same pixel size)."""
    g = scene.geom
    if not (0 <= r0 < r1 <= g.ny):
        raise ValueError("need 0 <= r0 < r1 <= ny")
    if r0 == 0 and r1 == g.ny:
        return scene
    pix = g.fov_y / g.ny
    sub = replace(g, ny=r1 - r0, fov_y=pix * (r1 - r0), y0=g.y0 + (0.5 * (r0 + r1) - 0.5 * g.ny) * pix)
    return replace(scene, geom=sub)


class CudaEngine:
    """Product engine: the CUDA render of a list of same-shaped scenes (one batched call) through the C ABI."""

    def __init__(self, scenes, device):
        from .render import Renderer
        self.R = Renderer(list(scenes), device=device)

    def render(self):
        return self.R.render()

    def render_bwd_packed(self, dl_dcube):
        """Adjoint without unpacking: returns the packed cells [n, cells * 4] as a VIEW into the workspace."""
        R = self.R
        R.dl_dcube.copy_(dl_dcube.reshape(R.dl_dcube.shape))
        R.render_bwd(unpack=False)
        return R.grad_packed().view(R.desc.batch, -1)

    def unpack(self):
        """k_unpack_grad on the workspace's own cells (after they were all-reduced in place)."""
        return self.R.unpack_grad()

    def set_target(self, target, sigma):
        self.R.set_target(target, sigma)

    def fit_step_packed(self):
        """Forward with the fused chi^2 term + adjoint (setup reused), gradient left packed: (cells [n, cells * 4], loss [1])."""
        R = self.R
        R.render_loss()
        R.render_bwd(unpack=False, reuse_setup=True)
        return R.grad_packed().view(R.desc.batch, -1), R.loss


class ShardedRender:
    """One render call (a batch of scenes that share line, grid layout and image size) split over the ranks of a
    torch.distributed process group.  `engine_factory(scenes)` builds an engine for a list of same-shaped scenes with
    render() -> [n, ny', nx, nchan] and render_bwd_packed(dl) -> [n, cells * 4]."""

    def __init__(self, scenes, engine_factory, rank=None, world=None, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank = dist.get_rank(group) if rank is None else rank
        self.world = dist.get_world_size(group) if world is None else world
        self.scenes = list(scenes) if isinstance(scenes, (list, tuple)) else [scenes]
        s0 = self.scenes[0]
        self.batch, self.ny, self.nx, self.nchan = len(self.scenes), s0.geom.ny, s0.geom.nx, len(s0.line.vchan)
        self.grid_shape = tuple(s0.grid.n)
        self.cells = 1
        for n in self.grid_shape:
            self.cells *= int(n)
        self.plan = plan_units(self.batch, self.ny, self.world)
        self.units = self.plan[self.rank]
        # which collective ends the adjoint (module docstring): whole items per rank -> all-gather, split rows -> all-reduce
        self.collective = "all_gather" if (self.world <= self.batch and self.world > 1) else "all_reduce"
        self.n_collectives = 0
        # one engine per slab height (all units of a rank have the same height unless rows do not divide evenly)
        self.groups = {}
        for u in self.units:
            self.groups.setdefault(u[2] - u[1], []).append(u)
        self.engines = {h: engine_factory([row_slab_scene(self.scenes[b], r0, r1) for b, r0, r1 in us])
                        for h, us in self.groups.items()}

    # ---- forward: no communication
    def render(self):
        """This rank's cube slabs: {(item, r0, r1): tensor [r1 - r0, nx, nchan]}."""
        out = {}
        for h, us in self.groups.items():
            cube = self.engines[h].render()
            for k, u in enumerate(us):
                out[u] = cube[k]
        return out

    def gather_cube(self, slabs):
        """The whole cube [batch, ny, nx, nchan] on every rank (all_gather of padded slabs; only when one rank needs it)."""
        import torch
        any_slab = next(iter(slabs.values())) if slabs else None
        dev = any_slab.device if any_slab is not None else "cpu"
        nmax = max(sum(r1 - r0 for _, r0, r1 in us) for us in self.plan)
        pad = torch.zeros((max(nmax, 1), self.nx, self.nchan), dtype=torch.float32, device=dev)
        row = 0
        for u in self.units:
            pad[row:row + u[2] - u[1]] = slabs[u]
            row += u[2] - u[1]
        bufs = [torch.empty_like(pad) for _ in range(self.world)]
        self.dist.all_gather(bufs, pad, group=self.group)
        cube = torch.empty((self.batch, self.ny, self.nx, self.nchan), dtype=torch.float32, device=dev)
        for k, us in enumerate(self.plan):
            row = 0
            for b, r0, r1 in us:
                cube[b, r0:r1] = bufs[k][row:row + r1 - r0]
                row += r1 - r0
        return cube

    # ---- adjoint: ONE collective over the packed gradient cells
    def render_bwd(self, dl_slabs):
        """dl_slabs: {(item, r0, r1): dL/dcube of that slab}.  Returns (g_dens, g_temp, g_vel), each [batch, *grid], the
        same on every rank (the grids are replicated)."""
        import torch
        packed = {}
        for h, us in self.groups.items():
            dl = torch.stack([dl_slabs[u] for u in us])
            packed[h] = self.engines[h].render_bwd_packed(dl)        # [n, cells * 4]
        return self._combine(packed)

    # ---- fit step: forward + chi^2 + adjoint per rank, then the same ONE collective
    def set_targets(self, target_slabs, sigma):
        """target_slabs: {(item, r0, r1): data cube rows of that slab}.  The chi^2 term is normalised by the voxel count of the
        WHOLE job, L = sum (I - D)^2 / (2 sigma^2 n_job): an engine normalises by the voxels of its own call, so it is given
        sigma sqrt(n_job / n_call), which yields exactly dL/dcube = (I - D) / (sigma^2 n_job) and this rank's share of L."""
        import torch
        n_job = self.batch * self.ny * self.nx * self.nchan
        for h, us in self.groups.items():
            n_call = len(us) * h * self.nx * self.nchan
            self.engines[h].set_target(torch.stack([target_slabs[u] for u in us]), float(sigma) * (n_job / n_call) ** 0.5)

    def fit_step(self):
        """One pass of the hot path over this rank's units and the collective.  Returns ((g_dens, g_temp, g_vel), loss_share):
        the gradients of the whole batch on every rank; loss_share is THIS rank's part of L (a tensor; summing it over ranks is
        left to the caller so that the step keeps its single collective)."""
        packed, loss = {}, None
        for h in self.groups:
            packed[h], l = self.engines[h].fit_step_packed()
            loss = l.clone() if loss is None else loss + l
        return self._combine(packed), loss

    def _combine(self, packed):
        """packed: {slab height: [n, cells * 4] of that engine's units} -> gradients of the whole batch on every rank."""
        import torch
        width = self.cells * 4
        if self.collective == "all_gather":
            # whole items per rank, contiguous and balanced (plan_units): rank k owns items plan[k][0][0] .. + len(plan[k])
            counts = [len(us) for us in self.plan]
            nmax = max(counts)
            (h, mine), = packed.items()                              # world <= batch: one group (full-height items) per rank
            if counts[self.rank] < nmax:
                pad = torch.zeros((nmax, width), dtype=torch.float32, device=mine.device)
                pad[:counts[self.rank]] = mine
                mine = pad
            out = torch.empty((self.world, nmax, width), dtype=torch.float32, device=mine.device)
            self.dist.all_gather([out[k] for k in range(self.world)], mine.contiguous(), group=self.group)      # the ONE collective
            self.n_collectives += 1
            if min(counts) == nmax:
                acc = out.view(self.batch, width)
            else:
                acc = torch.cat([out[k, :counts[k]] for k in range(self.world)])
        else:
            acc, inplace = None, None
            for h, us in self.groups.items():
                if acc is None and len(self.groups) == 1 and [u[0] for u in us] == list(range(self.batch)):
                    acc, inplace = packed[h], self.engines[h]        # this rank's cells already span the whole batch
                    continue
                if acc is None:
                    acc = torch.zeros((self.batch, width), dtype=torch.float32, device=packed[h].device)
                for k, (b, _, _) in enumerate(us):
                    acc[b] += packed[h][k]
            if acc is None:                                          # a rank without work still joins the collective
                dev = "cuda" if self.dist.get_backend(self.group) == "nccl" else "cpu"
                acc = torch.zeros((self.batch, width), dtype=torch.float32, device=dev)
            self.dist.all_reduce(acc, op=self.dist.ReduceOp.SUM, group=self.group)          # the ONE collective
            self.n_collectives += 1
            if inplace is not None and hasattr(inplace, "unpack"):
                return inplace.unpack()
        cells = acc.view(self.batch, self.cells, 4)
        return tuple(cells[:, :, k].reshape((self.batch,) + self.grid_shape).contiguous() for k in range(3))
