"""Pins of oracle/disk_physics.py (CPU only): closed forms and invariants of PAPER.md Eq. 1-2, 6-9."""
import numpy as np
import pytest

from oracle import disk_physics as dp

GM_SUN = 1.32712440018e26
AMU = 1.66053906660e-24
P0 = dp.DiskParams(gm_star=2.0 * GM_SUN, m_mol=2.37 * AMU, sigma0=30.0, r_c=150.0, gamma=1.0, t_freeze=19.0, n_dissoc=1e21)


def _noisy_T(r, zeta, seed=0):
    rng = np.random.default_rng(seed)
    return 20.0 * (r[:, None] / 100.0) ** -0.5 * (1.0 + 2.0 * zeta[None, :]) * np.exp(0.05 * rng.standard_normal((r.size, zeta.size)))


def test_surface_density_eq2_values():
    # Eq. 2 at r = r_c is Sigma_0 / e for any gamma; far inside it is the power law
    for g in (0.5, 1.0, 1.5):
        p = dp.DiskParams(gm_star=1.0, m_mol=1.0, sigma0=7.0, r_c=120.0, gamma=g)
        assert dp.surface_density(p, 120.0) == pytest.approx(7.0 / np.e, rel=1e-14)
        assert dp.surface_density(p, 1.2e-8) == pytest.approx(7.0 * 1e-10 ** -g, rel=1e-4)


@pytest.mark.parametrize("T0", [15.0, 40.0])
def test_isothermal_column_closed_form_and_second_order(T0):
    """T = const: Eq. 1 integrates to rho(z)/rho(0) = exp[-(G M m/k T)(1/r - 1/sqrt(r^2 + z^2))]; the trapezoid rule
    converges to it at second order."""
    errs = []
    for nz in (65, 129, 257):
        r, zeta = dp.nodes(3, nz, 50.0, 400.0, 0.5)
        fw = dp.forward(P0, np.full((3, nz), T0), r, zeta)
        rr, z = fw["r"], fw["z"]
        exact = np.exp(-(P0.gm_star * P0.m_mol / (dp.K_B * T0)) * (1.0 / rr - 1.0 / np.sqrt(rr * rr + z * z)))
        ratio = fw["rho"] / fw["rho"][:, :1]
        sel = exact > 1e-12
        errs.append(np.max(np.abs(ratio[sel] / exact[sel] - 1.0)))
    assert errs[2] < 2e-3
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.15) and errs[1] / errs[2] == pytest.approx(4.0, rel=0.15)


def test_thin_disk_gaussian_limit():
    """z << r: rho ~ exp(-z^2 / 2 h^2) with h^2 = k T r^3 / (G M m) (the textbook scale height)."""
    r, zeta = dp.nodes(2, 401, 100.0, 200.0, 0.02)
    T0 = 25.0
    fw = dp.forward(P0, np.full((2, 401), T0), r, zeta)
    h2 = dp.K_B * T0 * fw["r"] ** 3 / (P0.gm_star * P0.m_mol)
    np.testing.assert_allclose(np.log(fw["rho"] / fw["rho"][:, :1]), -fw["z"] ** 2 / (2.0 * h2), rtol=1e-3, atol=1e-9)


def test_normalisation_column_and_mask():
    r, zeta = dp.nodes(17, 33, 10.0, 600.0, 0.5)
    T = _noisy_T(r, zeta, 3)
    fw = dp.forward(P0, T, r, zeta)
    # Eq. 2: both sides of the mirror-symmetric disk integrate to Sigma(r) (numpy's own trapezoid routine)
    trapz = getattr(np, "trapezoid", None) or np.trapz
    np.testing.assert_allclose(2.0 * trapz(fw["rho"], fw["z"], axis=1), dp.surface_density(P0, r), rtol=1e-13)
    # Eq. 8: the column above the midplane is half the surface density; it falls to zero at the top node
    np.testing.assert_allclose(fw["N"][:, 0], dp.surface_density(P0, r) / (2.0 * P0.m_mol), rtol=1e-13)
    assert np.all(np.diff(fw["N"], axis=1) < 0) and np.all(fw["N"][:, -1] == 0.0)
    # Eq. 9: CO only where it is warm enough and shielded; the abundance there is exactly X_CO (Eq. 7)
    m = (T > P0.t_freeze) & (P0.f_col * fw["N"] > P0.n_dissoc)
    assert m.any() and (~m).any()
    np.testing.assert_array_equal(fw["n_co"][~m], 0.0)
    np.testing.assert_allclose(fw["n_co"][m], 1e-4 * fw["n_h2"][m], rtol=1e-15)
    # a hotter freeze-out threshold or a thicker shielding column can only shrink the layer
    m2 = dp.forward(dp.DiskParams(**{**P0.__dict__, "t_freeze": 30.0, "n_dissoc": 1e22}), T, r, zeta)["mask"]
    assert not np.any(m2 & ~m) and m2.sum() < m.sum()


def test_pressure_gradient_operator_on_an_analytic_field():
    """P = r^a exp(-b z): dP/dr at FIXED z is a P / r.  On the (ln r, zeta) grid this needs the -zeta d/dzeta term; the
    centred differences converge at second order."""
    a, b = -2.5, 1.0e-15
    errs = []
    for n in (33, 65, 129):
        r, zeta = dp.nodes(n, n, 20.0, 300.0, 0.4)
        rr = r[:, None] * dp.AU
        z = zeta[None, :] * rr
        P = rr ** a * np.exp(-b * z)
        got = dp.pressure_gradient_r(P, r, zeta)
        errs.append(np.max(np.abs(got[2:-2, 2:-2] / (a * P / rr)[2:-2, 2:-2] - 1.0)))
    assert errs[2] < 2e-3 and errs[0] / errs[1] == pytest.approx(4.0, rel=0.2) and errs[1] / errs[2] == pytest.approx(4.0, rel=0.2)


def test_velocity_eq6_kepler_term_and_sub_keplerian_midplane():
    r, zeta = dp.nodes(33, 17, 10.0, 600.0, 0.5)
    fw = dp.forward(P0, 20.0 * (r[:, None] / 100.0) ** -0.5 * np.ones((1, 17)), r, zeta)
    rr, z = fw["r"], fw["z"]
    kep2 = P0.gm_star * rr ** 2 / (rr ** 2 + z ** 2) ** 1.5
    np.testing.assert_allclose(fw["v_phi"] ** 2, kep2 + rr / fw["rho"] * fw["dPdr"], rtol=1e-12)
    # Keplerian speed at the midplane of a 2 Msun star at 100 au: sqrt(G M / r) = 4.21 km/s
    assert np.sqrt(kep2[np.argmin(np.abs(r - 100.0)), 0]) == pytest.approx(np.sqrt(P0.gm_star / (r[np.argmin(np.abs(r - 100.0))] * dp.AU)), rel=1e-14)
    assert np.sqrt(2.0 * GM_SUN / (100.0 * dp.AU)) == pytest.approx(4.212e5, rel=1e-3)
    # pressure falls outwards in the midplane of the tapered disk: the gas is sub-Keplerian there by O((h/r)^2)
    mid = fw["v_phi"][2:-2, 0] / np.sqrt(kep2[2:-2, 0])
    assert np.all(mid < 1.0) and np.all(mid > 0.95)


def test_adjoint_matches_finite_differences_and_dot_product():
    r, zeta = dp.nodes(13, 11, 10.0, 600.0, 0.5)
    T = _noisy_T(r, zeta, 8)
    fw = dp.forward(P0, T, r, zeta)
    rng = np.random.default_rng(9)
    gn, gv = rng.standard_normal(T.shape) * 1e-8, rng.standard_normal(T.shape) * 1e-6
    gT = dp.adjoint(P0, fw, gn, gv, r, zeta)

    def loss(Tx):
        f = dp.forward(P0, Tx, r, zeta)
        return np.sum(np.where(fw["mask"], P0.x_co * f["n_h2"], 0.0) * gn) + np.sum(f["v_phi"] * gv)

    for idx in [(0, 0), (3, 0), (6, 5), (12, 10), (0, 7), (12, 0), (7, 10)]:
        e = np.zeros_like(T)
        e[idx] = 1e-5 * T[idx]
        fd = (loss(T + e) - loss(T - e)) / (2.0 * e[idx])
        assert gT[idx] == pytest.approx(fd, rel=2e-6, abs=1e-12 * np.abs(gT).max())
    d = rng.standard_normal(T.shape) * T * 1e-2
    eps = 1e-5
    fdd = (loss(T + eps * d) - loss(T - eps * d)) / (2.0 * eps)
    assert np.sum(gT * d) == pytest.approx(fdd, rel=1e-6)
    # linear in the incoming gradients
    np.testing.assert_allclose(dp.adjoint(P0, fw, 3.0 * gn, 3.0 * gv, r, zeta), 3.0 * gT, rtol=1e-12, atol=1e-14 * np.abs(gT).max())
