"""World-size-2 gloo tests (CPU) of the multi-GPU host logic: batch-first / rows-second work plan,
row-slab geometry, cube gather, ONE all-reduce over the packed gradient cells, and bench.py's rank / aggregation logic.
The render engine injected here is the CPU oracle; on GPUs the same plumbing drives the CUDA engine over NCCL."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import pyoracle as po
from paper_2509_03623_b200.shard import ShardedRender, plan_rows, plan_units, row_slab_scene
from synth import tiny_axisym_scene

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_plan_rows_covers_every_row_once():
    for ny, world in ((7, 2), (8, 3), (2, 4), (512, 8), (1, 1)):
        plan = plan_rows(ny, world)
        assert len(plan) == world and plan[0][0] == 0 and plan[-1][1] == ny
        assert all(a[1] == b[0] for a, b in zip(plan, plan[1:]))
        sizes = [b - a for a, b in plan]
        assert max(sizes) - min(sizes) <= 1


@pytest.mark.parametrize("batch,ny,world", [(16, 512, 1), (16, 512, 2), (16, 512, 8), (16, 512, 16), (16, 512, 32), (3, 7, 2),
                                            (1, 7, 2), (1, 512, 8), (2, 5, 8), (5, 9, 3), (3, 4, 7)])
def test_plan_units_batch_items_first_then_rows(batch, ny, world):
    plan = plan_units(batch, ny, world)
    assert len(plan) == world
    seen = np.zeros((batch, ny), int)
    for us in plan:
        for b, r0, r1 in us:
            assert 0 <= r0 < r1 <= ny
            seen[b, r0:r1] += 1
    assert np.all(seen == 1)                                   # every (item, row) exactly once
    if world <= batch:
        assert all(r0 == 0 and r1 == ny for us in plan for _, r0, r1 in us)      # items are never split
        n = [len(us) for us in plan]
        assert max(n) - min(n) <= 1
    else:
        assert all(len(us) <= 1 for us in plan)                # one slab of one item per rank
        per_item = [sum(1 for us in plan for u in us if u[0] == b) for b in range(batch)]
        assert max(per_item) - min(per_item) <= 1 or ny < max(per_item)


def test_row_slab_is_the_same_pixels():
    sc = tiny_axisym_scene(seed=71, npix=6, npix_y=7)
    full = po.render(sc)
    for r0, r1 in ((0, 3), (3, 7), (2, 5), (6, 7), (0, 7)):
        np.testing.assert_allclose(po.render(row_slab_scene(sc, r0, r1)), full[r0:r1], rtol=1e-11, atol=1e-300)
    with pytest.raises(ValueError):
        row_slab_scene(sc, 3, 3)


class _OracleEngine:
    """CPU stand-in for shard.CudaEngine: a list of same-shaped scenes, packed float4 gradient cells out."""

    def __init__(self, scenes):
        self.scenes = scenes

    def render(self):
        return torch.from_numpy(np.stack([po.render(s) for s in self.scenes]).astype(np.float32))

    def render_bwd_packed(self, g):
        out = []
        for s, gi in zip(self.scenes, g):
            gd, gt, gv = po.render_bwd(s, gi.numpy().astype(np.float64))
            out.append(np.stack([gd, gt, gv, np.zeros_like(gd)], axis=-1).reshape(-1))
        return torch.from_numpy(np.stack(out).astype(np.float32))

    def set_target(self, target, sigma):
        self.target, self.sigma = target.numpy().astype(np.float64), float(sigma)

    def fit_step_packed(self):
        """As CudaEngine.fit_step_packed: the chi^2 term normalised by the voxels of THIS call."""
        cube = np.stack([po.render(s) for s in self.scenes])
        res = cube - self.target
        dl = res / (self.sigma ** 2 * res.size)
        loss = 0.5 * np.sum(res ** 2) / (self.sigma ** 2 * res.size)
        return self.render_bwd_packed(torch.from_numpy(dl)), torch.tensor([loss], dtype=torch.float64)


def _scenes(batch):
    return [tiny_axisym_scene(seed=72 + b, npix=6, npix_y=7, incl_deg=30.0 + 10 * b) for b in range(batch)]


def _worker(rank, world, port, out, batch):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        scs = _scenes(batch)
        sh = ShardedRender(scs, _OracleEngine)
        calls, gathers = [], []
        orig, orig_g = dist.all_reduce, dist.all_gather
        dist.all_reduce = lambda *a, **k: (calls.append(1), orig(*a, **k))[1]
        slabs = sh.render()
        cube = sh.gather_cube(slabs)
        dist.all_gather = lambda *a, **k: (gathers.append(1), orig_g(*a, **k))[1]
        G = torch.from_numpy(np.random.default_rng(5).standard_normal((batch,) + scs[0].cube_shape).astype(np.float32))
        grads = sh.render_bwd({u: G[u[0], u[1]:u[2]] for u in sh.units})
        n_ar, n_ag = len(calls), len(gathers)
        # fit step: chi^2 against a target, normalised over the WHOLE job; one more collective of the same kind
        D = torch.from_numpy(np.random.default_rng(6).random((batch,) + scs[0].cube_shape).astype(np.float32)) * float(cube.max())
        sh.set_targets({u: D[u[0], u[1]:u[2]] for u in sh.units}, 0.3)
        fit_grads, share = sh.fit_step()
        dist.all_reduce, dist.all_gather = orig, orig_g
        n_fit = len(calls) + len(gathers) - n_ar - n_ag
        dist.all_reduce(share)                                   # (outside the step: the test wants the whole loss)
        if rank == 0:
            torch.save({"cube": cube, "grads": grads, "G": G, "units": sh.plan, "n_allreduce": n_ar, "n_allgather": n_ag,
                        "collective": sh.collective, "n_collectives": sh.n_collectives, "n_fit": n_fit, "D": D,
                        "fit_grads": fit_grads, "loss": float(share)}, out)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("batch", [1, 3])
def test_two_rank_sharded_render_matches_single_process(tmp_path, batch):
    """batch 1: one image split by rows over the two ranks: the adjoint issues exactly ONE all-reduce (partial sums of the same
    cells); batch 3: whole items per rank (2 + 1): exactly ONE all-gather of the owned items' cells (uneven counts: padded) and
    no all-reduce.  Either way every rank ends with the full gradient; a fit step (chi^2 normalised over the whole job) costs
    the same single collective and its loss shares add up to the job's loss."""
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    out = str(tmp_path / "res.pt")
    mp.spawn(_worker, args=(2, port, out, batch), nprocs=2, join=True)
    res = torch.load(out)
    assert res["n_fit"] == 1 and res["n_collectives"] == 2
    if batch == 1:
        assert res["units"] == [[(0, 0, 4)], [(0, 4, 7)]]
        assert (res["collective"], res["n_allreduce"], res["n_allgather"]) == ("all_reduce", 1, 0)
    else:
        assert res["units"] == [[(0, 0, 7), (1, 0, 7)], [(2, 0, 7)]]
        assert (res["collective"], res["n_allreduce"], res["n_allgather"]) == ("all_gather", 0, 1)
    scs = _scenes(batch)
    for b, sc in enumerate(scs):
        np.testing.assert_allclose(res["cube"][b].numpy(), po.render(sc), rtol=1e-6, atol=1e-30)
        ref = po.render_bwd(sc, res["G"][b].numpy().astype(np.float64))
        for got, want in zip(res["grads"], ref):
            assert got.shape[0] == batch
            np.testing.assert_allclose(got[b].numpy(), want, rtol=1e-5, atol=1e-6 * np.abs(want).max())
    # the fit step against a single-process evaluation: L = sum (I - D)^2 / (2 sigma^2 n_job)
    cubes = np.stack([po.render(sc) for sc in scs])
    resid = cubes - res["D"].numpy().astype(np.float64)
    assert res["loss"] == pytest.approx(0.5 * np.sum(resid ** 2) / (0.3 ** 2 * resid.size), rel=1e-6)
    for b, sc in enumerate(scs):
        ref = po.render_bwd(sc, resid[b] / (0.3 ** 2 * resid.size))
        for got, want in zip(res["fit_grads"], ref):
            np.testing.assert_allclose(got[b].numpy(), want, rtol=1e-4, atol=1e-5 * np.abs(want).max())


def test_bench_multi_rank_logic_dry_run():
    """bench.py --gpus 2 --dry-run under torch.distributed.run (gloo, no GPU): one JSON line from rank 0 only, the step time is
    the MAX over ranks (rank r 'takes' (1 + r) ms per step) and `value` the whole-job aggregate of both ranks."""
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "4", "--warmup", "1", "--dry-run"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT, env={**os.environ, "OMP_NUM_THREADS": "1"})
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                       # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["steps"] == 4 and d["scaling"] == "weak" and d["dry_run"] is True
    assert d["ms_per_step"] == pytest.approx(2.0)                # max over ranks of (1 + rank) ms
    assert d["config"]["workload"].startswith("cfg5")
    assert d["value"] == pytest.approx(2 * 274877906944 * 4 / (8.0e-3))
    assert [k for k in d["per_config_ms"] if k != "columns"] == ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "cfg6"]
    assert len(lines[0]) < 3000                                  # the driver reads one short line (tests/test_bench_line.py)


def test_bench_shard_mode_dry_run_two_ranks():
    """bench.py --gpus 2 --shard --dry-run (gloo): ONE job, config 5's 16 items, 8 whole items per rank through ShardedRender with
    a stub engine; every step ends with exactly one collective, an all-gather of the owned items' packed cells; strong scaling:
    `value` = the job's samples (not twice them) / max-over-ranks time."""
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3", "--warmup", "1", "--dry-run",
           "--shard"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT, env={**os.environ, "OMP_NUM_THREADS": "1"})
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1 and len(lines[0]) < 3000
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "strong" and d["config"]["workload"].startswith("cfg5")
    assert d["shard"] == {"collective": "all_gather", "collectives_per_step": 1.0, "units_per_rank": [8, 8]}
    assert d["ms_per_step"] == pytest.approx(2.0)
    assert d["value"] == pytest.approx(274877906944 * 3 / 6.0e-3)
