"""-m "not gpu": pins of the hydrostatic-equilibrium oracle (oracle/hydro_oracle.c)
against what the paper and the mathematics fix."""
import numpy as np
from scipy.integrate import quad

import oracle as orc
from paper_2402_18471_b200 import synth_disc as sd

GM = sd.G_GRAV * sd.M_SUN


def _grid(n_r, n_z, r_in=5.0, r_out=100.0, tmax=0.3):
    R_e = r_in * sd.AU * (r_out / r_in) ** (np.arange(n_r + 1) / n_r)
    R_c = np.sqrt(R_e[:-1] * R_e[1:])
    tan_e = tmax * np.arange(n_z + 1) / n_z
    tan_c = 0.5 * (tan_e[:-1] + tan_e[1:])
    return R_e, tan_e, R_c, tan_c


def test_isothermal_column_is_the_closed_form_and_the_thin_disc_gaussian():
    """Eq. 33 integrates exactly for constant c_s: P / P_0 = exp[GM / c_s^2 (1/r - 1/r_0)] -- the product
    of Eq. 36 telescopes to it -- and for Z << R this is the Gaussian exp(-(Z^2 - Z_0^2) / 2 H^2), H = c_s / Omega_K."""
    n_r, n_z = 7, 64
    R_e, tan_e, R_c, tan_c = _grid(n_r, n_z, tmax=0.08)
    T = 150.0 * (R_c / sd.AU) ** -0.5
    cs2 = np.repeat((sd.K_B * T / (2.4 * sd.M_H))[:, None], n_z, axis=1)
    Sigma = 1000.0 * (R_c / sd.AU) ** -1.0
    rho = orc.hydrostatic(R_e, tan_e, R_c, tan_c, cs2, Sigma, GM)
    r = R_c[:, None] * np.sqrt(1.0 + tan_c[None, :] ** 2)
    exact = np.exp(GM / cs2 * (1.0 / r - 1.0 / r[:, :1]))
    np.testing.assert_allclose(rho / rho[:, :1], exact, rtol=1e-13)
    Z = R_c[:, None] * tan_c[None, :]
    H2 = cs2 * R_c[:, None] ** 3 / GM
    gauss = np.exp(-(Z ** 2 - Z[:, :1] ** 2) / (2.0 * H2))
    # the Gaussian is the O((Z/R)^2) approximation of the closed form
    np.testing.assert_allclose(rho / rho[:, :1], gauss, rtol=0.75 * (Z ** 4 / (H2 * R_c[:, None] ** 2)).max() + 1e-12)
    assert np.all(rho > 0) and np.all(np.diff(rho, axis=1) < 0)          # positive, falling with height


def test_column_mass_equals_surface_density_exactly():
    """Eq. 37: sum_k rho V = Sigma_g (R dR) for every column, any temperature structure."""
    n_r, n_z = 9, 40
    R_e, tan_e, R_c, tan_c = _grid(n_r, n_z)
    rng = np.random.default_rng(3)
    cs2 = 1e9 * np.exp(rng.uniform(-0.5, 0.5, (n_r, n_z)))
    Sigma = 10 ** rng.uniform(0, 3, n_r)
    rho = orc.hydrostatic(R_e, tan_e, R_c, tan_c, cs2, Sigma, GM)
    V = (np.diff(R_e ** 3)[:, None] * np.diff(tan_e)[None, :]) / 3.0          # Eq. 1
    RdR = 0.5 * np.diff(R_e ** 2)
    np.testing.assert_allclose((rho * V).sum(axis=1), Sigma * RdR, rtol=1e-14)
    # scaling: doubling Sigma doubles rho, to the bit
    assert np.array_equal(orc.hydrostatic(R_e, tan_e, R_c, tan_c, cs2, 2.0 * Sigma, GM), 2.0 * rho)


def test_stratified_column_converges_to_the_integral_of_eq33_at_second_order():
    """c_s^2 rising with height (a warm surface layer): d log P = GM / c_s^2 d(1/r) integrated by adaptive
    quadrature; the trapezoidal average of Eq. 35 converges to it at second order in the cell size."""
    R0 = 20.0 * sd.AU
    cs2_of = lambda tan: 4.0e8 * (1.0 + 30.0 * tan ** 2 + 200.0 * tan ** 3)
    r_of = lambda tan: R0 * np.sqrt(1.0 + tan ** 2)
    # d(1/r)/d tan = -tan / (R0 (1 + tan^2)^(3/2))
    integrand = lambda tan: GM / cs2_of(tan) * (-tan / (R0 * (1.0 + tan ** 2) ** 1.5))
    errs = []
    for n_z in (32, 64, 128):
        tan_e = 0.3 * np.arange(n_z + 1) / n_z
        tan_c = 0.5 * (tan_e[:-1] + tan_e[1:])
        R_e = np.array([0.98 * R0, R0 / 0.98]); R_c = np.array([R0])
        cs2 = cs2_of(tan_c)[None, :]
        rho = orc.hydrostatic(R_e, tan_e, R_c, tan_c, cs2, np.array([100.0]), GM)
        P = rho[0] * cs2[0]
        ref = np.array([np.exp(quad(integrand, tan_c[0], t, epsabs=0, epsrel=1e-12)[0]) for t in tan_c])
        errs.append(np.max(np.abs(P / P[0] / ref - 1.0)))
    assert errs[0] < 2e-2 and errs[1] < errs[0] / 3.5 and errs[2] < errs[1] / 3.5, errs


def test_single_cell_and_two_cell_columns_by_hand():
    R_e = np.array([1.0, 2.0]) * sd.AU; R_c = np.array([np.sqrt(2.0)]) * sd.AU
    rho = orc.hydrostatic(R_e, np.array([0.0, 0.1]), R_c, np.array([0.05]), np.array([[1e9]]), np.array([50.0]), GM)
    V = (R_e[1] ** 3 - R_e[0] ** 3) * 0.1 / 3.0
    assert rho[0, 0] == 50.0 * 0.5 * (R_e[1] ** 2 - R_e[0] ** 2) / V or abs(rho[0, 0] * V / (50.0 * 0.5 * (R_e[1] ** 2 - R_e[0] ** 2)) - 1) < 1e-15
    tan_e = np.array([0.0, 0.1, 0.3]); tan_c = np.array([0.05, 0.2]); cs2 = np.array([[1e9, 2e9]])
    rho = orc.hydrostatic(R_e, tan_e, R_c, tan_c, cs2, np.array([50.0]), GM)
    r = R_c[0] * np.sqrt(1.0 + tan_c ** 2)
    ratio = np.exp(GM * 0.5 * (1 / 1e9 + 1 / 2e9) * (1 / r[1] - 1 / r[0]))       # Eqs. 34, 35 typed out
    assert abs(rho[0, 1] / rho[0, 0] - ratio * 1e9 / 2e9) < 1e-15 * ratio
