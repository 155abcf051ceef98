"""A second, independent transcription of the render algorithm O1-O10 in numpy.

Brute force for tiny scenes only (pure-Python loops over rays and steps).  It exists to pin the C
oracle: the two were written separately from the same algorithm statement, with different code
structure (rotation matrices instead of expanded formulas, searchsorted on explicit node arrays
instead of index arithmetic, cumulative optical depth instead of a running transmittance product),
so a wrong sign, index or transposed operand in either shows up as a disagreement.
Cites: PAPER.md:262-294 (Eq. 11-17), PAPER.md:241-248 (Table 2), PAPER.md:296 (grids).
"""
import numpy as np

H, KB, CL = 6.62607015e-27, 1.380649e-16, 2.99792458e10
AU, PC = 1.495978707e13, 3.0856775814913673e18


def _rot_sky_to_disk(incl, pa, az):
    """3x3 matrix M with p_disk = M @ (X, Y, zeta)."""
    th = pa + np.pi / 2
    Rz_pa = np.array([[np.cos(th), np.sin(th), 0], [-np.sin(th), np.cos(th), 0], [0, 0, 1.0]])
    Rx_i = np.array([[1.0, 0, 0], [0, np.cos(incl), -np.sin(incl)], [0, np.sin(incl), np.cos(incl)]])
    Rz_az = np.array([[np.cos(az), np.sin(az), 0], [-np.sin(az), np.cos(az), 0], [0, 0, 1.0]])
    return Rz_az @ Rx_i @ Rz_pa


def _interp_weights(nodes, t):
    """Linear interpolation on explicit, increasing node coordinates: (i, i+1, w_i, w_i+1) or None."""
    if t < nodes[0] or t > nodes[-1]:
        return None
    i = int(np.searchsorted(nodes, t, side="right") - 1)
    i = min(max(i, 0), len(nodes) - 2)
    f = (t - nodes[i]) / (nodes[i + 1] - nodes[i])
    return i, 1.0 - f, f


def render(scene):
    g, ln, gr = scene.geom, scene.line, scene.grid
    M = _rot_sky_to_disk(g.incl, g.pa, g.az)
    w_dir = M @ np.array([0.0, 0.0, -1.0])          # direction of increasing s (away from the observer)
    vch = np.asarray(ln.vchan, float)
    C = len(vch)
    T0 = H * ln.nu0 / KB
    S0 = 2 * H * ln.nu0 ** 3 / CL ** 2
    if ln.unit == 0:
        unit = S0
    elif ln.unit == 1:
        unit = 1.0
    else:
        d_au = g.dist_pc * PC / AU
        unit = 1.0 / ((g.fov_x / g.nx) * (g.fov_y / g.ny) / d_au ** 2 * 1e23)
    dens = np.asarray(gr.dens, float); temp = np.asarray(gr.temp, float); vel = np.asarray(gr.vel, float)
    if gr.kind == 0:
        nr, nz = gr.n
        lnr_nodes = np.log(gr.lo[0]) + (np.log(gr.hi[0]) - np.log(gr.lo[0])) * np.arange(nr) / (nr - 1)
        zeta_nodes = gr.lo[1] + (gr.hi[1] - gr.lo[1]) * np.arange(nz) / (nz - 1)
    elif gr.kind == 2:
        lnr_nodes = np.log(gr.lo[0]) + (np.log(gr.hi[0]) - np.log(gr.lo[0])) * np.arange(gr.n[0]) / (gr.n[0] - 1)
        th_nodes = gr.lo[1] + (gr.hi[1] - gr.lo[1]) * np.arange(gr.n[1]) / (gr.n[1] - 1)
        ph_nodes = 2 * np.pi * np.arange(gr.n[2] + 1) / gr.n[2]          # one extra node: 2 pi is node 0 again
        wrap = lambda f: np.concatenate([f, f[:, :, :1]], axis=2)        # noqa: E731
        dens, temp, vel = wrap(dens), wrap(temp), wrap(vel)
    else:
        axes = [np.linspace(gr.lo[a], gr.hi[a], gr.n[a]) for a in range(3)]
    cube = np.zeros((g.ny, g.nx, C))
    for iy in range(g.ny):
        for ix in range(g.nx):
            X = g.x0 + (ix + 0.5 - g.nx / 2) * g.fov_x / g.nx
            Y = g.y0 + (iy + 0.5 - g.ny / 2) * g.fov_y / g.ny
            org = M @ np.array([X, Y, 0.0])
            if gr.kind in (0, 2):
                zm = max(abs(gr.lo[1]), abs(gr.hi[1])) if gr.kind == 0 else 0.0
                Rb = gr.hi[0] * np.sqrt(1 + zm ** 2)
                b2 = X * X + Y * Y
                if b2 >= Rb * Rb:
                    continue
                s_in, s_out = -np.sqrt(Rb * Rb - b2), np.sqrt(Rb * Rb - b2)
            else:
                s_in, s_out = -np.inf, np.inf
                ok = True
                for a in range(3):
                    if w_dir[a] == 0:
                        ok &= gr.lo[a] <= org[a] <= gr.hi[a]
                        continue
                    ta, tb = sorted(((gr.lo[a] - org[a]) / w_dir[a], (gr.hi[a] - org[a]) / w_dir[a]))
                    s_in, s_out = max(s_in, ta), min(s_out, tb)
                if not ok or s_out <= s_in:
                    continue
            ds = (s_out - s_in) / g.nstep
            tau = np.zeros(C)          # optical depth in front of the current step
            I = np.zeros(C)
            for k in range(g.nstep):
                p = org + (s_in + (k + 0.5) * ds) * w_dir
                r = np.hypot(p[0], p[1])
                if r == 0:
                    continue
                if gr.kind == 0:
                    zeta = (abs(p[2]) if gr.mirror_z else p[2]) / r
                    if r < gr.lo[0] or r > gr.hi[0]:
                        continue
                    a = _interp_weights(lnr_nodes, min(max(np.log(r), lnr_nodes[0]), lnr_nodes[-1]))
                    b = _interp_weights(zeta_nodes, zeta)
                    if a is None or b is None:
                        continue
                    (i, wa0, wa1), (j, wb0, wb1) = a, b

                    def samp(f):
                        return (wa0 * (wb0 * f[i, j] + wb1 * f[i, j + 1]) + wa1 * (wb0 * f[i + 1, j] + wb1 * f[i + 1, j + 1]))
                else:
                    if gr.kind == 2:
                        rho_ = np.linalg.norm(p)
                        phi_ = np.arctan2(p[1], p[0]) % (2 * np.pi)
                        ws = [_interp_weights(lnr_nodes, np.log(rho_)), _interp_weights(th_nodes, np.arccos(p[2] / rho_)),
                              _interp_weights(ph_nodes, phi_)]
                    else:
                        ws = [_interp_weights(axes[a], p[a]) for a in range(3)]
                    if any(w is None for w in ws):
                        continue
                    (i, wx0, wx1), (j, wy0, wy1), (l, wz0, wz1) = ws

                    def samp(f):
                        acc = 0.0
                        for di, wx in ((0, wx0), (1, wx1)):
                            for dj, wy in ((0, wy0), (1, wy1)):
                                for dl, wz in ((0, wz0), (1, wz1)):
                                    acc += wx * wy * wz * f[i + di, j + dj, l + dl]
                        return acc
                n = samp(dens)
                if gr.dens_mode == 1:
                    n = np.exp(n)
                T = max(samp(temp), 1.0)
                v = samp(vel)
                if gr.vel_mode == 1:
                    rho = np.linalg.norm(p)
                    v = np.sqrt(g.gm_star * (r * AU) ** 2 / (rho * AU) ** 3) * (1 + v)
                vvec = v * np.array([-p[1], p[0], 0.0]) / r
                vlos = float(w_dir @ vvec)
                alpha = np.sqrt(2 * KB * T / ln.m_line + ln.vturb_mach ** 2 * 2 * KB * T / ln.m_gas + ln.vturb_abs ** 2)
                Q = np.sum(np.asarray(ln.g_lev) * np.exp(-np.asarray(ln.e_lev_K) / T))
                n_u = n * ln.g_u * np.exp(-ln.e_u_K / T) / Q
                x = T0 / T
                phi_nu = CL / (ln.nu0 * alpha * np.sqrt(np.pi)) * np.exp(-((vch - g.vsys - vlos) / alpha) ** 2)
                beta = CL ** 2 / (8 * np.pi * ln.nu0 ** 2) * ln.a_ul * n_u * np.expm1(x) * phi_nu
                dtau = beta * ds * AU
                Bnu = S0 / np.expm1(x)
                I += Bnu * (-np.expm1(-dtau)) * np.exp(-tau)
                tau += dtau
            cube[iy, ix] = I / unit
    return cube
