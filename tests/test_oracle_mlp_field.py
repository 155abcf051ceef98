"""Pins of oracle/mlp_field.py (CPU only): Eq. 10."""
import numpy as np
import pytest

from oracle import mlp_field as mf


def test_sizes_and_encoding_values():
    assert mf.n_inputs(4) == 18 and mf.n_params(4) == 64 * 18 + 64 + 3 * (64 * 64 + 64) + 64 + 1
    g = mf.encode(5, 3, 4)
    assert g.shape == (15, 18)
    # node (0, 0): p = 0 -> every sine 0, every cosine 1; node (4, 2): p = 1 -> sin(2^k pi) = 0, cos = -1 for k = 0, +1 above
    np.testing.assert_allclose(g[0], [0, 0] + [0, 1, 0, 1] * 4, atol=1e-15)
    np.testing.assert_allclose(g[-1], [1, 1] + [0, -1, 0, -1] + [0, 1, 0, 1] * 3, atol=1e-14)
    # node (2, 1): p = (1/2, 1/2): k = 0 -> sin = 1, cos = 0; k = 1 -> sin(pi) = 0, cos = -1; frequencies double with k
    np.testing.assert_allclose(g[2 * 3 + 1][:10], [0.5, 0.5, 1, 0, 1, 0, 0, -1, 0, -1], atol=1e-14)
    p0 = np.arange(5) / 4.0
    np.testing.assert_allclose(g[::3, 2 + 4 * 3], np.sin(8 * np.pi * p0), atol=1e-14)      # k = 3, coordinate 0


def test_output_range_and_hand_evaluated_network():
    L = 1
    p = np.zeros(mf.n_params(L))
    # all-zero network: o = 0 -> sigmoid 1/2 -> the middle of [5, 400] K everywhere
    np.testing.assert_allclose(mf.forward(p, 4, 3, L), 202.5, rtol=1e-15)
    # one path: h_1[0] = relu(2 p_0 - 0.5), copied through layers 2-4, o = 3 h_4[0] - 1
    lay = mf.split(p, L)
    lay[0][0][0, 0] = 2.0; lay[0][1][0] = -0.5
    for l in (1, 2, 3):
        lay[l][0][0, 0] = 1.0
    lay[4][0][0, 0] = 3.0; lay[4][1][0] = -1.0
    T = mf.forward(p, 5, 2, L)
    h = np.maximum(2.0 * np.arange(5) / 4.0 - 0.5, 0.0)
    np.testing.assert_allclose(T[:, 0], 5.0 + 395.0 / (1.0 + np.exp(-(3.0 * h - 1.0))), rtol=1e-14)
    np.testing.assert_allclose(T[:, 1], T[:, 0], rtol=1e-15)                 # no dependence on p_1 in this network
    # saturation: the range is [t_lo, t_hi]
    lay[4][1][0] = 60.0
    assert np.all(mf.forward(p, 5, 2, L) <= 400.0) and mf.forward(p, 5, 2, L).max() == pytest.approx(400.0, rel=1e-12)
    lay[4][0][0, 0] = 0.0; lay[4][1][0] = -60.0
    assert mf.forward(p, 5, 2, L).min() == pytest.approx(5.0, rel=1e-12)


def test_against_torch_autograd():
    """An independent library evaluates the same network (torch.nn.functional on CPU, fp64) and differentiates it."""
    torch = pytest.importorskip("torch")
    L, nr, nz = 4, 7, 5
    p = mf.init_params(L, 3).astype(np.float64)
    rng = np.random.default_rng(4)
    gT = rng.standard_normal((nr, nz))
    tp = torch.tensor(p, dtype=torch.float64, requires_grad=True)
    x = torch.tensor(mf.encode(nr, nz, L), dtype=torch.float64)
    off = 0
    for fan_in, fan_out in [(18, 64), (64, 64), (64, 64), (64, 64), (64, 1)]:
        W = tp[off:off + fan_in * fan_out].reshape(fan_out, fan_in); off += fan_in * fan_out
        b = tp[off:off + fan_out]; off += fan_out
        x = torch.nn.functional.linear(x, W, b)
        if fan_out != 1:
            x = torch.relu(x)
    T = 5.0 + 395.0 * torch.sigmoid(x[:, 0])
    (T * torch.tensor(gT.ravel())).sum().backward()
    np.testing.assert_allclose(mf.forward(p, nr, nz, L), T.detach().numpy().reshape(nr, nz), rtol=1e-13)
    np.testing.assert_allclose(mf.adjoint(p, gT, nr, nz, L), tp.grad.numpy(), rtol=1e-10, atol=1e-12)


def test_adjoint_finite_differences():
    L, nr, nz = 2, 6, 4
    p = mf.init_params(L, 5).astype(np.float64)
    rng = np.random.default_rng(6)
    gT = rng.standard_normal((nr, nz))
    g = mf.adjoint(p, gT, nr, nz, L)
    for idx in rng.integers(0, p.size, 12):
        e = np.zeros_like(p)
        e[idx] = 1e-6
        fd = np.sum((mf.forward(p + e, nr, nz, L) - mf.forward(p - e, nr, nz, L)) * gT) / 2e-6
        assert g[idx] == pytest.approx(fd, rel=1e-5, abs=1e-8)
