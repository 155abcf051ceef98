"""Parity criteria (from BASELINE.json north_star: cube 1e-4, gradients 1e-3).

A result passes when ALL three hold against the fp64 oracle `ref`:
  max-norm   max|d|  <= rel * max|ref|
  L2         ||d||_2 <= rel * ||ref||_2
  element    |d_i|   <= rel * |ref_i| + floor * max|ref|
with (rel, floor) = (1e-4, 1e-6) for the cube and (1e-3, 1e-5) for each gradient field.
"""
import numpy as np

CUBE = (1e-4, 1e-6)
GRAD = (1e-3, 1e-5)


def check(name, got, ref, rel, floor):
    got = np.asarray(got, np.float64)
    ref = np.asarray(ref, np.float64)
    assert got.shape == ref.shape, (name, got.shape, ref.shape)
    assert np.all(np.isfinite(got)), f"{name}: non-finite values"
    d = np.abs(got - ref)
    m = float(np.abs(ref).max())
    if m == 0.0:
        assert float(d.max()) == 0.0, f"{name}: reference is identically zero but got max {d.max():.3e}"
        return 0.0
    tol = rel * np.abs(ref) + floor * m
    worst = float((d / tol).max())
    nrm = float(np.linalg.norm(d) / np.linalg.norm(ref))
    msg = (f"{name}: max|d|/max|ref| = {d.max() / m:.3e}, L2 = {nrm:.3e}, worst element/tol = {worst:.3f}, "
           f"failing = {int((d > tol).sum())} of {d.size}")
    assert d.max() <= rel * m, msg
    assert nrm <= rel, msg
    assert worst <= 1.0, msg
    return worst


def check_cube(name, got, ref):
    return check(name, got, ref, *CUBE)


def check_grad(name, got, ref):
    return check(name, got, ref, *GRAD)
