"""fp64 CPU oracle of the physics pre-pass that turns a temperature grid into the render's fields (TEST INFRASTRUCTURE).

What it computes (Eq. 1-2, 6-9; "Physics-Informed Constraints"):
on the render's axisymmetric grid (nodes r_i log-spaced, zeta_j = z/r uniform from 0, mirror symmetric) and for every
radius r = r_i with heights z_j = zeta_j r, in the paper's order:

  P1  f_j = z_j / (T_j (r^2 + z_j^2)^{3/2})                              gravity term of Eq. 1 without G M m/k
  P2  A_0 = 0,  A_j = A_{j-1} + (f_{j-1} + f_j)(z_j - z_{j-1})/2           "integrated numerically": trapezoid rule
  P3  rho~_j = (T_0/T_j) exp(-(G M m_mol/k) A_j)                         Eq. 1; the -dlnT/dz term integrates exactly
  P4  H = sum_j (rho~_{j-1} + rho~_j)(z_j - z_{j-1})/2,  rho_j = rho~_j Sigma(r)/(2 H)     Eq. 2, both sides of the disk
      Sigma(r) = Sigma_0 (r/r_c)^-gamma exp[-(r/r_c)^(2-gamma)]
  P5  n_j = rho_j/m_mol,  N_j = sum_{l>j} (n_{l-1} + n_l)(z_l - z_{l-1})/2                Eq. 8, z_max = the top node
  P6  n_CO = X_CO n  where T > T_freeze and f_col N > N_dissoc, else 0                   Eq. 7, 9 (f_col = 0.706)
  P7  P = rho k T/m_mol;  dP/dr at fixed z = (1/r)[dP/dln r at fixed zeta - zeta dP/dzeta], central differences in index
      space, one-sided at the edges;  v_phi^2 = G M r^2/(r^2+z^2)^{3/2} + (r/rho) dP/dr,  v_phi = sqrt(max(., 0))   Eq. 6

and the adjoint: given dL/dn_CO and dL/dv_phi on the grid, dL/dT with the CO mask held fixed (it is piecewise constant)
and zero gradient through the clamp of P7.  Readings of the paper (all silent there): the trapezoid rule, the mirror
factor 2, n_H2 = rho/m_mol, z_max = top node of the grid, centred differences; DESIGN.md lists them.

Plain numpy, loops over the vertical index, nothing shared with the CUDA path.  Pinned in tests/test_oracle_disk_physics.py
(isothermal closed form, thin-disk Gaussian, column and surface-density identities, Keplerian limit, analytic pressure
field, finite differences of the adjoint).  Parity with RadJAX's own pre-pass is unpinned (no code, no printed values).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

K_B = 1.380649e-16
AU = 1.495978707e13


@dataclass(frozen=True)
class DiskParams:
    gm_star: float          # cm^3 s^-2
    m_mol: float            # g, mean molecular mass (Eq. 1)
    sigma0: float           # g cm^-2 (Eq. 2)
    r_c: float              # au
    gamma: float
    x_co: float = 1e-4      # Eq. 7
    t_freeze: float = 19.0  # K
    n_dissoc: float = 1e21  # cm^-2
    f_col: float = 0.706    # Eq. 9


def nodes(nr, nz, rmin, rmax, zeta_max):
    r = rmin * (rmax / rmin) ** (np.arange(nr) / (nr - 1.0))
    zeta = zeta_max * np.arange(nz) / (nz - 1.0)
    return r, zeta


def surface_density(p: DiskParams, r_au):
    x = np.asarray(r_au, dtype=np.float64) / p.r_c
    return p.sigma0 * x ** (-p.gamma) * np.exp(-x ** (2.0 - p.gamma))


def _diff_index(P, axis, h):
    """Central differences in index space along `axis` with spacing h, one-sided at both ends (P7)."""
    D = np.empty_like(P)
    Pm = np.moveaxis(P, axis, 0)
    Dm = np.moveaxis(D, axis, 0)
    Dm[1:-1] = (Pm[2:] - Pm[:-2]) / (2.0 * h)
    Dm[0] = (Pm[1] - Pm[0]) / h
    Dm[-1] = (Pm[-1] - Pm[-2]) / h
    return D


def _diff_index_adjoint(gD, axis, h):
    """Transpose of _diff_index."""
    gP = np.zeros_like(gD)
    gm = np.moveaxis(gD, axis, 0)
    pm = np.moveaxis(gP, axis, 0)
    pm[2:] += gm[1:-1] / (2.0 * h)
    pm[:-2] -= gm[1:-1] / (2.0 * h)
    pm[1] += gm[0] / h
    pm[0] -= gm[0] / h
    pm[-1] += gm[-1] / h
    pm[-2] -= gm[-1] / h
    return gP


def pressure_gradient_r(P, r_au, zeta):
    """dP/dr [per cm] at fixed z on the (ln r, zeta) grid (P7)."""
    r = np.asarray(r_au, dtype=np.float64)[:, None] * AU
    dl = np.log(r_au[-1] / r_au[0]) / (len(r_au) - 1.0)
    dz = (zeta[-1] - zeta[0]) / (len(zeta) - 1.0)
    return (_diff_index(P, 0, dl) - zeta[None, :] * _diff_index(P, 1, dz)) / r


def forward(p: DiskParams, temp, r_au, zeta):
    """P1-P7.  temp [nr][nz] (K).  Returns a dict with n_co [cm^-3], v_phi [cm/s], n_h2, rho, column N, mask and the
    intermediates the adjoint needs."""
    T = np.asarray(temp, dtype=np.float64)
    r_au = np.asarray(r_au, dtype=np.float64)
    zeta = np.asarray(zeta, dtype=np.float64)
    nr, nz = T.shape
    r = r_au[:, None] * AU
    z = zeta[None, :] * r
    dzv = np.diff(z, axis=1)                                   # z_j - z_{j-1}, [nr][nz-1]
    f = z / (T * (r * r + z * z) ** 1.5)                       # P1
    A = np.zeros_like(T)
    for j in range(1, nz):                                     # P2
        A[:, j] = A[:, j - 1] + 0.5 * (f[:, j - 1] + f[:, j]) * dzv[:, j - 1]
    c = p.gm_star * p.m_mol / K_B
    rt = T[:, :1] / T * np.exp(-c * A)                         # P3
    H = np.zeros(nr)
    for j in range(1, nz):                                     # P4
        H += 0.5 * (rt[:, j - 1] + rt[:, j]) * dzv[:, j - 1]
    sig = surface_density(p, r_au)
    rho = rt * (sig / (2.0 * H))[:, None]
    n = rho / p.m_mol                                          # P5
    N = np.zeros_like(T)
    for j in range(nz - 2, -1, -1):
        N[:, j] = N[:, j + 1] + 0.5 * (n[:, j] + n[:, j + 1]) * dzv[:, j]
    mask = (T > p.t_freeze) & (p.f_col * N > p.n_dissoc)       # P6
    n_co = np.where(mask, p.x_co * n, 0.0)
    P = rho * K_B * T / p.m_mol                                # P7
    dPdr = pressure_gradient_r(P, r_au, zeta)
    kep = p.gm_star * r * r / (r * r + z * z) ** 1.5
    with np.errstate(divide="ignore", invalid="ignore"):
        press = np.where(rho > 0.0, r / rho * dPdr, 0.0)
    v2 = kep + press
    v = np.sqrt(np.maximum(v2, 0.0))
    return dict(n_co=n_co, v_phi=v, n_h2=n, rho=rho, N=N, mask=mask, T=T, f=f, A=A, rt=rt, H=H, sig=sig, P=P,
                dPdr=dPdr, v2=v2, r=r, z=z, dzv=dzv, c=c)


def adjoint(p: DiskParams, fw, g_nco, g_v, r_au, zeta):
    """dL/dT [nr][nz] from dL/dn_CO and dL/dv_phi (reverse of P7..P1; CO mask fixed, zero gradient through the clamp)."""
    T, rho, rt, H, f, r, dzv = fw["T"], fw["rho"], fw["rt"], fw["H"], fw["f"], fw["r"], fw["dzv"]
    r_au = np.asarray(r_au, dtype=np.float64)
    zeta = np.asarray(zeta, dtype=np.float64)
    nr, nz = T.shape
    g_nco = np.asarray(g_nco, dtype=np.float64)
    g_v = np.asarray(g_v, dtype=np.float64)
    gT = np.zeros_like(T)
    # P7
    pos = (fw["v2"] > 0.0) & (rho > 0.0)
    with np.errstate(divide="ignore", invalid="ignore"):
        g_v2 = np.where(fw["v2"] > 0.0, g_v / (2.0 * fw["v_phi"]), 0.0)
        g_dPdr = np.where(pos, g_v2 * r / rho, 0.0)
        g_rho = np.where(pos, -g_v2 * r * fw["dPdr"] / (rho * rho), 0.0)
    dl = np.log(r_au[-1] / r_au[0]) / (nr - 1.0)
    dz = (zeta[-1] - zeta[0]) / (nz - 1.0)
    gP = _diff_index_adjoint(g_dPdr / r, 0, dl) + _diff_index_adjoint(-zeta[None, :] * g_dPdr / r, 1, dz)
    g_rho += gP * K_B * T / p.m_mol
    gT += gP * rho * K_B / p.m_mol
    # P6, P5
    g_rho += np.where(fw["mask"], p.x_co * g_nco, 0.0) / p.m_mol
    # P4
    scale = (fw["sig"] / (2.0 * H))[:, None]
    g_rt = g_rho * scale
    gH = -np.sum(g_rho * rho, axis=1) / H
    w = np.zeros_like(T)
    w[:, :-1] += 0.5 * dzv
    w[:, 1:] += 0.5 * dzv
    g_rt += gH[:, None] * w
    # P3
    t = g_rt * rt
    gT[:, 0] += np.sum(t, axis=1) / T[:, 0]
    gT -= t / T
    gA = -fw["c"] * t
    # P2
    gf = np.zeros_like(T)
    for j in range(nz - 1, 0, -1):
        gf[:, j] += 0.5 * dzv[:, j - 1] * gA[:, j]
        gf[:, j - 1] += 0.5 * dzv[:, j - 1] * gA[:, j]
        gA[:, j - 1] += gA[:, j]
    # P1
    gT -= gf * f / T
    return gT
