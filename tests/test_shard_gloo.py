"""World-size-2 gloo test (CPU) of the multi-GPU host logic: row-slab geometry, cube gather, gradient all-reduce.
The render engine injected here is the CPU oracle; on GPUs the same plumbing drives the CUDA engine over NCCL."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import pyoracle as po
from paper_2509_03623_b200.shard import ShardedImage, plan_rows, row_slab_scene
from synth import tiny_axisym_scene


def test_plan_rows_covers_every_row_once():
    for ny, world in ((7, 2), (8, 3), (2, 4), (512, 8), (1, 1)):
        plan = plan_rows(ny, world)
        assert len(plan) == world and plan[0][0] == 0 and plan[-1][1] == ny
        assert all(a[1] == b[0] for a, b in zip(plan, plan[1:]))
        sizes = [b - a for a, b in plan]
        assert max(sizes) - min(sizes) <= 1


def test_row_slab_is_the_same_pixels():
    sc = tiny_axisym_scene(seed=71, npix=6, npix_y=7)
    full = po.render(sc)
    for r0, r1 in ((0, 3), (3, 7), (2, 5), (6, 7)):
        np.testing.assert_allclose(po.render(row_slab_scene(sc, r0, r1)), full[r0:r1], rtol=1e-11, atol=1e-300)
    with pytest.raises(ValueError):
        row_slab_scene(sc, 3, 3)


class _OracleEngine:
    def __init__(self, scene):
        self.scene = scene

    def render(self):
        return torch.from_numpy(po.render(self.scene).astype(np.float32))

    def render_bwd(self, g):
        return [torch.from_numpy(x.astype(np.float32)) for x in po.render_bwd(self.scene, g.numpy().astype(np.float64))]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        sc = tiny_axisym_scene(seed=72, npix=6, npix_y=7)
        sh = ShardedImage(sc, _OracleEngine)
        slab = sh.render()
        cube = sh.gather_cube(slab)
        G = torch.from_numpy(np.random.default_rng(5).standard_normal(sc.cube_shape).astype(np.float32))
        grads = sh.render_bwd(G[sh.r0:sh.r1])
        if rank == 0:
            torch.save({"cube": cube, "grads": grads, "G": G}, out)
    finally:
        dist.destroy_process_group()


def test_two_rank_sharded_image_matches_single_process(tmp_path):
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    out = str(tmp_path / "res.pt")
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    res = torch.load(out)
    sc = tiny_axisym_scene(seed=72, npix=6, npix_y=7)
    np.testing.assert_allclose(res["cube"].numpy(), po.render(sc), rtol=1e-6, atol=1e-30)
    ref = po.render_bwd(sc, res["G"].numpy().astype(np.float64))
    for got, want in zip(res["grads"], ref):
        np.testing.assert_allclose(got.numpy(), want, rtol=1e-5, atol=1e-6 * np.abs(want).max())
