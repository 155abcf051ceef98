"""fp64 CPU oracle of the symmetric MLP temperature field (TEST INFRASTRUCTURE).

PAPER.md:209-215, Eq. 10:  T(r, |z|) = MLP_w(gamma(r, |z|)); four fully connected layers of
64 hidden units with ReLU, a sigmoid output scaled to [5, 400] K, sinusoidal positional encoding of degree L = 4
("a set of sinusoids with exponentially increasing frequencies" [27]).

Algorithm (M1-M4), evaluated on the nodes of the render's (r, zeta) grid:
  M1  p = (i/(nr-1), j/(nz-1)) in [0, 1]^2: the node's normalised grid coordinates (ln r and zeta = |z|/r; the grid is
      mirror symmetric, so the field is a function of |z|)
  M2  gamma(p) = (p_0, p_1, sin(2^k pi p_0), cos(2^k pi p_0), sin(2^k pi p_1), cos(2^k pi p_1))_{k = 0..L-1}      (2 + 4L values)
  M3  h_1 = relu(W_1 gamma + b_1), h_l = relu(W_l h_{l-1} + b_l), l = 2..4;  o = w_5 . h_4 + b_5
  M4  T = T_lo + (T_hi - T_lo) sigmoid(o)
and the adjoint: dL/d(parameters) from dL/dT on the grid.

Readings (the paper gives the layer count, width, activations, range and L only): four hidden layers plus a linear
output unit; the encoding's input is the normalised grid coordinate, its ordering as in M2; parameters are one flat
float32 vector [W_1 (64 x D) | b_1 | W_2 (64 x 64) | b_2 | W_3 | b_3 | W_4 | b_4 | w_5 (64) | b_5], row-major, D = 2 + 4L.
Plain numpy, shares nothing with the CUDA path.  Pinned in tests/test_oracle_mlp_field.py (encoding values, output
range, a hand-evaluated tiny network, torch autograd as an independent library, finite differences).
"""
from __future__ import annotations

import numpy as np

WIDTH = 64
NHIDDEN = 4


def n_inputs(L: int) -> int:
    return 2 + 4 * L


def n_params(L: int) -> int:
    D = n_inputs(L)
    return WIDTH * D + WIDTH + (NHIDDEN - 1) * (WIDTH * WIDTH + WIDTH) + WIDTH + 1


def split(params, L: int):
    """Views (W_l, b_l) of the flat parameter vector, l = 1..5 (w_5 as a 1 x 64 matrix)."""
    p = np.asarray(params, dtype=np.float64)
    D = n_inputs(L)
    out, off = [], 0
    for fan_in, fan_out in [(D, WIDTH)] + [(WIDTH, WIDTH)] * (NHIDDEN - 1) + [(WIDTH, 1)]:
        W = p[off:off + fan_out * fan_in].reshape(fan_out, fan_in)
        off += fan_out * fan_in
        b = p[off:off + fan_out]
        off += fan_out
        out.append((W, b))
    assert off == p.size == n_params(L)
    return out


def encode(nr: int, nz: int, L: int):
    """M1-M2: gamma of every node, [nr*nz][2 + 4L]."""
    i, j = np.meshgrid(np.arange(nr), np.arange(nz), indexing="ij")
    p = np.stack([i.ravel() / (nr - 1.0), j.ravel() / (nz - 1.0)], axis=1)
    cols = [p[:, 0], p[:, 1]]
    for k in range(L):
        for c in (0, 1):
            cols.append(np.sin(2.0 ** k * np.pi * p[:, c]))
            cols.append(np.cos(2.0 ** k * np.pi * p[:, c]))
    return np.stack(cols, axis=1)


def forward(params, nr: int, nz: int, L: int = 4, t_lo: float = 5.0, t_hi: float = 400.0, keep=False):
    """T [nr][nz] (M1-M4)."""
    layers = split(params, L)
    a = encode(nr, nz, L)
    acts = [a]
    for W, b in layers[:-1]:
        a = np.maximum(a @ W.T + b, 0.0)
        acts.append(a)
    W5, b5 = layers[-1]
    o = (a @ W5.T + b5)[:, 0]
    s = 1.0 / (1.0 + np.exp(-o))
    T = (t_lo + (t_hi - t_lo) * s).reshape(nr, nz)
    return (T, acts, s) if keep else T


def near_kink(params, nr: int, nz: int, L: int = 4, tol: float = 1e-4):
    """Nodes [nr][nz] where some hidden pre-activation lies within `tol` of the ReLU kink: there the derivative is a
    subgradient (any value between the two one-sided ones is valid) and lower-precision arithmetic may take the other
    branch, so parity tests give such nodes no incoming gradient."""
    layers = split(params, L)
    a = encode(nr, nz, L)
    bad = np.zeros(a.shape[0], dtype=bool)
    for W, b in layers[:-1]:
        x = a @ W.T + b
        bad |= np.any(np.abs(x) < tol * np.maximum(1.0, np.abs(a).max()), axis=1)
        a = np.maximum(x, 0.0)
    return bad.reshape(nr, nz)


def adjoint(params, g_temp, nr: int, nz: int, L: int = 4, t_lo: float = 5.0, t_hi: float = 400.0):
    """dL/d(parameters) (flat, same layout) from dL/dT [nr][nz]: reverse of M4..M3."""
    layers = split(params, L)
    _, acts, s = forward(params, nr, nz, L, t_lo, t_hi, keep=True)
    g_o = np.asarray(g_temp, dtype=np.float64).ravel() * (t_hi - t_lo) * s * (1.0 - s)
    grads = []
    W5, _ = layers[-1]
    grads.append((np.outer(g_o, np.ones(1)).T @ acts[-1], np.array([g_o.sum()])))
    delta = np.outer(g_o, W5[0]) * (acts[-1] > 0.0)
    for l in range(NHIDDEN - 1, -1, -1):
        W, _ = layers[l]
        grads.append((delta.T @ acts[l], delta.sum(axis=0)))
        if l > 0:
            delta = (delta @ W) * (acts[l] > 0.0)
    flat = []
    for gW, gb in reversed(grads):
        flat += [gW.ravel(), gb.ravel()]
    return np.concatenate(flat)


def init_params(L: int, seed: int):
    """Seeded test parameters (uniform +-1/sqrt(fan_in), the usual default of linear layers), float32."""
    rng = np.random.default_rng(seed)
    D = n_inputs(L)
    parts = []
    for fan_in, fan_out in [(D, WIDTH)] + [(WIDTH, WIDTH)] * (NHIDDEN - 1) + [(WIDTH, 1)]:
        k = 1.0 / np.sqrt(fan_in)
        parts += [rng.uniform(-k, k, fan_out * fan_in), rng.uniform(-k, k, fan_out)]
    return np.concatenate(parts).astype(np.float32)
