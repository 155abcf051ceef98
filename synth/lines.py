"""Line data used by the synthetic configs (input data, not method arithmetic).

The paper takes level energies from the LAMDA tables (ref. [26]); that file is not
available offline, so the configs use the rigid-rotor CO ladder stated in SURVEY.md §8(c):
E_J/k = (hB/k) J(J+1) with B = 57.635968 GHz, g_J = 2J+1, J <= 40, A_21 = 6.910e-7 s^-1,
nu0 = 230.538 GHz (BASELINE.json configs[0]).  Parity never depends on these values: both the
oracle and the CUDA path take them as inputs.
"""
from __future__ import annotations

import numpy as np

from .scene import Line, UNIT_S0

AMU_G = 1.66053906660e-24
HB_OVER_K_CO = 2.766090          # K  (h * 57.635968 GHz / k)
NU0_CO21 = 230.538e9             # Hz
A21_CO = 6.910e-7                # s^-1
M_CO = 28.0101 * AMU_G
M_GAS = 2.37 * AMU_G


def co_line(vchan_cms, j_up: int = 2, nlev: int = 41, vturb_abs: float = 0.0, vturb_mach: float = 0.0,
            unit: int = UNIT_S0) -> Line:
    """CO J_up -> J_up-1 with a rigid-rotor partition table of `nlev` levels."""
    J = np.arange(nlev, dtype=np.float64)
    e_lev = HB_OVER_K_CO * J * (J + 1.0)
    g_lev = 2.0 * J + 1.0
    if j_up != 2:
        raise ValueError("only CO J=2-1 line constants are tabulated here")
    return Line(nu0=NU0_CO21, a_ul=A21_CO, g_u=float(g_lev[j_up]), e_u_K=float(e_lev[j_up]),
                e_lev_K=e_lev, g_lev=g_lev, m_line=M_CO, m_gas=M_GAS,
                vchan=np.ascontiguousarray(vchan_cms, dtype=np.float64),
                vturb_abs=vturb_abs, vturb_mach=vturb_mach, unit=unit)


def channels_centered(nchan: int, dv_cms: float) -> np.ndarray:
    """v_c = (c - (C-1)/2) dv  (SURVEY.md §8(c) reading 16)."""
    return (np.arange(nchan, dtype=np.float64) - 0.5 * (nchan - 1)) * dv_cms
