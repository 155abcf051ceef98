"""GPU parity of the physics pre-pass (radt_disk_fields / radt_disk_fields_bwd) against oracle/disk_physics.py."""
from dataclasses import replace

import numpy as np
import pytest

from oracle import disk_physics as dp
from synth import make_config
from tests.tolerances import check_grad

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

GM_SUN = 1.32712440018e26
AMU = 1.66053906660e-24


def _params(k=0):
    return dp.DiskParams(gm_star=(2.0 + 0.2 * k) * GM_SUN, m_mol=2.37 * AMU, sigma0=30.0 + 5.0 * k, r_c=150.0 - 10.0 * k,
                         gamma=1.0 - 0.1 * k, t_freeze=19.0 + k, n_dissoc=1e21)


def _setup(scenes):
    from paper_2509_03623_b200 import binding as B
    B.lib()
    desc = B.Descriptors(scenes)
    params = [_params(k) for k in range(len(scenes))]
    temp = torch.from_numpy(B.stack_fields(scenes)[1]).cuda()
    ws = torch.empty(B.radt_disk_workspace_bytes(desc), dtype=torch.uint8, device="cuda")
    return B, desc, params, temp, ws


@pytest.mark.parametrize("make", [lambda: [make_config(1)], lambda: [make_config(2)],
                                  lambda: make_config(5, npix=8, batch=3)])
def test_disk_fields_match_oracle(make):
    scenes = make()
    B, desc, params, temp, ws = _setup(scenes)
    dens, vel = torch.empty_like(temp), torch.empty_like(temp)
    B.radt_disk_fields(B.make_disks(params), desc, temp, dens, vel, ws)
    gr = scenes[0].grid
    r, zeta = dp.nodes(gr.n[0], gr.n[1], gr.lo[0], gr.hi[0], gr.hi[1])
    for b in range(len(scenes)):
        fw = dp.forward(params[b], temp[b].cpu().numpy(), r, zeta)
        got_n, got_v = dens[b].cpu().numpy(), vel[b].cpu().numpy()
        # fp64 kernels rounded once to fp32; a node that sits within rounding of a mask threshold may differ
        same = (got_n > 0) == fw["mask"]
        edge = (np.abs(params[b].f_col * fw["N"] / params[b].n_dissoc - 1.0) < 1e-9) | (np.abs(fw["T"] / params[b].t_freeze - 1.0) < 1e-9)
        assert np.all(same | edge)
        np.testing.assert_allclose(got_n[same], fw["n_co"][same], rtol=2e-7)
        np.testing.assert_allclose(got_v, fw["v_phi"], rtol=2e-7, atol=1e-3)
        assert fw["mask"].any() and (~fw["mask"]).any()


@pytest.mark.parametrize("make", [lambda: [make_config(1)], lambda: make_config(5, npix=8, batch=2)])
def test_disk_fields_adjoint_matches_oracle(make):
    scenes = make()
    B, desc, params, temp, ws = _setup(scenes)
    rng = np.random.default_rng(17)
    gn = (rng.standard_normal(tuple(temp.shape)) * 1e-8).astype(np.float32)
    gv = (rng.standard_normal(tuple(temp.shape)) * 1e-6).astype(np.float32)
    g0 = (rng.standard_normal(tuple(temp.shape)) * 1e-3).astype(np.float32)
    gT = torch.from_numpy(g0.copy()).cuda()
    B.radt_disk_fields_bwd(B.make_disks(params), desc, temp, torch.from_numpy(gn).cuda(), torch.from_numpy(gv).cuda(), gT, ws)
    gr = scenes[0].grid
    r, zeta = dp.nodes(gr.n[0], gr.n[1], gr.lo[0], gr.hi[0], gr.hi[1])
    for b in range(len(scenes)):
        fw = dp.forward(params[b], temp[b].cpu().numpy(), r, zeta)
        want = dp.adjoint(params[b], fw, gn[b], gv[b], r, zeta)
        got = gT[b].cpu().numpy().astype(np.float64) - g0[b]          # the call ADDS to g_temp
        scale = np.abs(want).max()
        assert np.max(np.abs(got - want)) <= 1e-3 * scale               # BASELINE.json gradient tolerance
        assert np.linalg.norm(got - want) <= 1e-5 * np.linalg.norm(want) + 1e-7 * np.abs(g0[b]).max() * want.size ** 0.5
    # element by element (tests/tolerances.py, as the render's gradients), on a call that adds to zeros so that the fp32
    # rounding of `g0 + .` is not part of the comparison
    gZ = torch.zeros_like(gT)
    B.radt_disk_fields_bwd(B.make_disks(params), desc, temp, torch.from_numpy(gn).cuda(), torch.from_numpy(gv).cuda(), gZ, ws)
    for b in range(len(scenes)):
        fw = dp.forward(params[b], temp[b].cpu().numpy(), r, zeta)
        check_grad(f"pre-pass dL/dT item {b}", gZ[b].cpu().numpy(), dp.adjoint(params[b], fw, gn[b], gv[b], r, zeta))


def test_disk_fields_feed_the_render_end_to_end():
    """T grid -> pre-pass -> render -> chi^2 -> render adjoint -> pre-pass adjoint: dL/dT of the whole chain against a
    directional finite difference of the same chain run through the oracles in fp64."""
    from oracle import pyoracle as po
    from paper_2509_03623_b200 import Renderer
    from synth import l2_target
    sc = make_config(1, npix=24)
    B, desc, params, temp, ws = _setup([sc])
    p = params[0]
    gr = sc.grid
    r, zeta = dp.nodes(gr.n[0], gr.n[1], gr.lo[0], gr.hi[0], gr.hi[1])
    T0 = temp[0].cpu().numpy().astype(np.float64)

    def oracle_loss(T, target=None, sigma=None, mask=None):
        fw = dp.forward(p, T, r, zeta)
        nco = fw["n_co"] if mask is None else np.where(mask, p.x_co * fw["n_h2"], 0.0)
        s2 = sc.with_fields(dens=nco.astype(np.float32), temp=T.astype(np.float32), vel=fw["v_phi"].astype(np.float32))
        cube = po.render(s2)
        if target is None:
            return cube, fw
        return po.chi2_loss_grad(cube, target, sigma)[0]

    cube0, fw0 = oracle_loss(T0)
    target, sigma = l2_target(cube0, 99)
    # GPU chain
    R = Renderer([sc])
    B.radt_disk_fields(B.make_disks(params), desc, temp, R.dens, R.vel, ws)
    R.temp.copy_(temp)
    R.set_target(target[None], sigma)
    R.fit_step()
    gT = R.g_temp.clone()
    B.radt_disk_fields_bwd(B.make_disks(params), desc, temp, R.g_dens, R.g_vel, gT, ws)
    gT = gT[0].cpu().numpy().astype(np.float64)
    # smooth multiplicative direction; fp32 field storage limits the step from below
    d = T0 * 0.02 * np.cos(np.linspace(0, 3, T0.shape[0]))[:, None] * np.ones((1, T0.shape[1]))
    eps = 0.25
    fd = (oracle_loss(T0 + eps * d, target, sigma, fw0["mask"]) - oracle_loss(T0 - eps * d, target, sigma, fw0["mask"])) / (2 * eps)
    assert np.sum(gT * d) == pytest.approx(fd, rel=2e-2)


@pytest.mark.parametrize("nr,nz", [(9, 7), (37, 45), (20, 200), (33, 33), (130, 3)])
def test_disk_fields_on_ragged_grid_sizes(nr, nz):
    """Column lengths that are not a multiple of the 32 lanes a column is split over (7, 45, 200, 33, 3 nodes) and column counts
    that leave the last block partly empty: forward fields and the adjoint against the oracle."""
    from synth import tiny_axisym_scene
    scenes = [tiny_axisym_scene(seed=3, nr=nr, nz=nz), tiny_axisym_scene(seed=4, nr=nr, nz=nz)]
    B, desc, params, temp, ws = _setup(scenes)
    dens, vel = torch.empty_like(temp), torch.empty_like(temp)
    B.radt_disk_fields(B.make_disks(params), desc, temp, dens, vel, ws)
    gr = scenes[0].grid
    r, zeta = dp.nodes(gr.n[0], gr.n[1], gr.lo[0], gr.hi[0], gr.hi[1])
    rng = np.random.default_rng(nr * 1000 + nz)
    gn = (rng.standard_normal(tuple(temp.shape)) * 1e-8).astype(np.float32)
    gv = (rng.standard_normal(tuple(temp.shape)) * 1e-6).astype(np.float32)
    gT = torch.zeros_like(temp)
    B.radt_disk_fields_bwd(B.make_disks(params), desc, temp, torch.from_numpy(gn).cuda(), torch.from_numpy(gv).cuda(), gT, ws)
    for b in range(len(scenes)):
        fw = dp.forward(params[b], temp[b].cpu().numpy(), r, zeta)
        got_n, got_v = dens[b].cpu().numpy(), vel[b].cpu().numpy()
        same = (got_n > 0) == fw["mask"]
        edge = (np.abs(params[b].f_col * fw["N"] / params[b].n_dissoc - 1.0) < 1e-9) | (np.abs(fw["T"] / params[b].t_freeze - 1.0) < 1e-9)
        assert np.all(same | edge)
        np.testing.assert_allclose(got_n[same], fw["n_co"][same], rtol=2e-7)
        np.testing.assert_allclose(got_v, fw["v_phi"], rtol=2e-7, atol=1e-3)
        want = dp.adjoint(params[b], fw, gn[b], gv[b], r, zeta)
        got = gT[b].cpu().numpy().astype(np.float64)
        scale = np.abs(want).max()
        if scale > 0:
            assert np.max(np.abs(got - want)) <= 1e-3 * scale
