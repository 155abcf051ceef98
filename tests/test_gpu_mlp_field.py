"""GPU parity of the MLP temperature field (radt_mlp_temperature / _bwd) against oracle/mlp_field.py."""
import numpy as np
import pytest

from oracle import mlp_field as mf
from synth import make_config
from tests.tolerances import check_grad

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _desc(cfg):
    from paper_2509_03623_b200 import binding as B
    B.lib()
    return B, B.Descriptors([make_config(cfg, npix=8)])


@pytest.mark.parametrize("cfg,L,seed", [(1, 4, 1), (2, 4, 2), (1, 2, 3), (1, 8, 4), (1, 0, 5)])
def test_mlp_temperature_matches_oracle(cfg, L, seed):
    B, desc = _desc(cfg)
    nr, nz = desc.grid_shape
    mlp = B.make_mlp(L=L)
    assert B.radt_mlp_num_params(mlp) == mf.n_params(L)
    p = 3.0 * mf.init_params(L, seed)                       # scaled up so that the output leaves the sigmoid's middle
    T = torch.empty((nr, nz), dtype=torch.float32, device="cuda")
    B.radt_mlp_temperature(mlp, desc, torch.from_numpy(p).cuda(), T)
    want = mf.forward(p, nr, nz, L)
    # fp32 accumulation over 64-term dot products, four layers deep: 1e-5 of the 395 K range
    assert np.max(np.abs(T.cpu().numpy() - want)) <= 1e-5 * 395.0
    assert want.max() - want.min() > 0.1


@pytest.mark.parametrize("cfg,L,seed", [(1, 4, 11), (2, 4, 12), (1, 1, 13)])
def test_mlp_adjoint_matches_oracle(cfg, L, seed):
    B, desc = _desc(cfg)
    nr, nz = desc.grid_shape
    mlp = B.make_mlp(L=L)
    p = 3.0 * mf.init_params(L, seed)
    gT = np.random.default_rng(seed).standard_normal((nr, nz)).astype(np.float32)
    kink = mf.near_kink(p, nr, nz, L)          # ReLU subgradients: both branches are correct there
    assert kink.mean() < 0.2
    gT[kink] = 0.0
    gp = torch.full((mf.n_params(L),), 7.0, dtype=torch.float32, device="cuda")      # must be overwritten
    B.radt_mlp_temperature_bwd(mlp, desc, torch.from_numpy(p).cuda(), torch.from_numpy(gT).cuda(), gp)
    want = mf.adjoint(p, gT, nr, nz, L)
    got = gp.cpu().numpy().astype(np.float64)
    # BASELINE.json gradient tolerance (1e-3 of the maximum); measured far below
    assert np.max(np.abs(got - want)) <= 1e-3 * np.abs(want).max()
    assert np.linalg.norm(got - want) <= 1e-4 * np.linalg.norm(want)
    check_grad("mlp g_params", got, want)      # and element by element, as the render's gradients (tests/tolerances.py)


@pytest.mark.parametrize("nr,nz,L", [(9, 7, 4), (37, 11, 4), (50, 30, 8), (129, 2, 0)])
def test_mlp_ragged_node_counts(nr, nz, L):
    """Node counts that are not a multiple of the 128-node tensor-core tile (63, 407, 1500, 258 nodes): the last tile of the
    forward and of the adjoint is partly empty; its padding rows must neither show in T nor reach the parameter gradients."""
    from paper_2509_03623_b200 import binding as B
    from synth import tiny_axisym_scene
    B.lib()
    desc = B.Descriptors([tiny_axisym_scene(seed=5, nr=nr, nz=nz)])
    assert desc.grid_shape == (nr, nz)
    mlp = B.make_mlp(L=L)
    p = 3.0 * mf.init_params(L, 100 + nr)
    T = torch.full((nr, nz), -1.0, dtype=torch.float32, device="cuda")
    B.radt_mlp_temperature(mlp, desc, torch.from_numpy(p).cuda(), T)
    want = mf.forward(p, nr, nz, L)
    assert np.max(np.abs(T.cpu().numpy() - want)) <= 1e-5 * 395.0
    gT = np.random.default_rng(nr).standard_normal((nr, nz)).astype(np.float32)
    gT[mf.near_kink(p, nr, nz, L)] = 0.0
    gp = torch.full((mf.n_params(L),), 7.0, dtype=torch.float32, device="cuda")
    B.radt_mlp_temperature_bwd(mlp, desc, torch.from_numpy(p).cuda(), torch.from_numpy(gT).cuda(), gp)
    wantg = mf.adjoint(p, gT, nr, nz, L)
    got = gp.cpu().numpy().astype(np.float64)
    assert np.max(np.abs(got - wantg)) <= 1e-3 * np.abs(wantg).max()
    assert np.linalg.norm(got - wantg) <= 1e-4 * np.linalg.norm(wantg)
    check_grad(f"mlp g_params {nr}x{nz}", got, wantg)


def test_mlp_adjoint_without_masking_the_relu_kinks():
    """include/radt.h radt_mlp_temperature_bwd: the adjoint recomputes the activations with two-term bf16 products (about
    2^-16 per product) while the forward uses the three-product split (about fp32), so relu' of a unit whose pre-activation
    lies within ~1e-4 of zero may be taken on the other branch than the oracle's.  Either branch is a valid subgradient, but
    the parameter gradient then leaves the 1e-3 tolerance: a KNOWN LIMIT, stated in the header with the figures measured
    here (max 6.0e-3, L2 4.0e-3 on this harsh case: three times the initialisation scale, NO node masked; the other tests
    zero g_T at near-kink nodes and meet 1e-3 / 1e-4 and the element-wise criterion).  The bound below keeps it from growing."""
    from paper_2509_03623_b200 import binding as B
    B.lib()
    desc = B.Descriptors([make_config(2)])
    nr, nz = desc.grid_shape
    L = 4
    mlp = B.make_mlp(L=L)
    p = 3.0 * mf.init_params(L, 77)
    assert mf.near_kink(p, nr, nz, L).any()
    gT = np.random.default_rng(78).standard_normal((nr, nz)).astype(np.float32)
    gp = torch.full((mf.n_params(L),), 7.0, dtype=torch.float32, device="cuda")
    B.radt_mlp_temperature_bwd(mlp, desc, torch.from_numpy(p).cuda(), torch.from_numpy(gT).cuda(), gp)
    want = mf.adjoint(p, gT, nr, nz, L)
    got = gp.cpu().numpy().astype(np.float64)
    err_max = np.max(np.abs(got - want)) / np.abs(want).max()
    err_l2 = np.linalg.norm(got - want) / np.linalg.norm(want)
    print(f"unmasked MLP adjoint: max {err_max:.3e}, L2 {err_l2:.3e}")
    assert err_max <= 1e-2 and err_l2 <= 1e-2


def test_neural_field_fit_reduces_the_loss():
    """The paper's chain end to end on the GPU (Fig. 2): parameters -> MLP T grid -> physics pre-pass -> render ->
    chi^2 -> adjoints back to the parameters; a few plain gradient steps towards a target cube rendered from a known
    temperature grid lower the loss, and the chain's gradient matches a finite difference of the GPU loss."""
    from types import SimpleNamespace
    from paper_2509_03623_b200 import Renderer, binding as B
    sc = make_config(1, npix=32)
    R = Renderer([sc])
    desc = R.desc
    nr, nz = desc.grid_shape
    disks = B.make_disks([SimpleNamespace(gm_star=2.0 * 1.32712440018e26, m_gas=2.37 * 1.66053906660e-24, sigma0=30.0,
                                          r_c=150.0, gamma=1.0, x_co=1e-4, t_freeze=19.0, n_dissoc=1e21, f_col=0.706)])
    pws = torch.empty(B.radt_disk_workspace_bytes(desc), dtype=torch.uint8, device="cuda")
    mlp = B.make_mlp(L=4)

    def chain(params, need_grad):
        B.radt_mlp_temperature(mlp, desc, params, R.temp[0])
        B.radt_disk_fields(disks, desc, R.temp, R.dens, R.vel, pws)
        if not need_grad:
            R.render_loss()
            return float(R.loss.cpu()), None
        R.fit_step()
        gT = R.g_temp.clone()
        B.radt_disk_fields_bwd(disks, desc, R.temp, R.g_dens, R.g_vel, gT, pws)
        gp = torch.empty_like(params)
        B.radt_mlp_temperature_bwd(mlp, desc, params, gT[0], gp)
        return float(R.loss.cpu()), gp

    # target: the cube of the config's own (noisy, parametric) temperature grid pushed through the same pre-pass
    B.radt_disk_fields(disks, desc, R.temp, R.dens, R.vel, pws)
    R.render()
    target = R.cube.clone()
    R.set_target(target, 0.015 * float(target.max()))
    params = torch.from_numpy(mf.init_params(4, 21)).cuda()
    loss0, g = chain(params, True)
    # directional finite difference of the GPU chain along the gradient
    d = g / g.norm()
    eps = 2e-3
    lp, _ = chain(params + eps * d, False)
    lm, _ = chain(params - eps * d, False)
    assert float((g * d).sum()) == pytest.approx((lp - lm) / (2 * eps), rel=5e-2)
    # normalised gradient descent with a decaying step
    loss = loss0
    for it in range(40):
        loss, g = chain(params, True)
        params = params - 0.05 * (0.95 ** it) * g / g.norm()
    loss_end, _ = chain(params, False)
    assert loss_end < 0.7 * loss0
