"""The oracle against the closed-form solutions of the Smoluchowski equation (the
authors' constant-kernel runs were 'consistent with the analytic solutions') and the integrator
 against its textbook properties.

Initial condition n(m,0) = (N0/mbar) exp(-m/mbar).
  constant K:          n(m,t) = N0/(mbar (1+tau)^2) exp(-m/(mbar (1+tau))),  tau = K N0 t / 2,
                       M0(t) = N0/(1+tau)
  additive K=b(m+m'):  M0(t) = N0 exp(-tau), tau = b N0 mbar t;
                       n = (N0/mbar) (1-f)/(x sqrt f) exp(-(1+f) x) I1(2 x sqrt f), x = m/mbar, f = 1-e^-tau
On a log grid with the two-bin split these are approximate (numerical diffusion): total mass is
exact, M0(t) is close, and the error falls as the grid is refined.
"""
import numpy as np
import pytest
from scipy.special import ive

import oracle as orc

RHO_M = 1.0
MBAR = 4.0 * np.pi / 3.0 * RHO_M * (1e-3) ** 3     # mean mass: a 10 um grain


def _grid(N):
    # 15 mass decades: a from 1e-5 to 1 cm
    return orc.mass_grid(N, 1e-5, 1.0, RHO_M)


def _initial(g, N0=1.0):
    x = g.m_e / MBAR
    F = (1.0 + x) * np.exp(-x)
    return N0 * MBAR * (F[:-1] - F[1:])              # mass density per bin, integral of m n dm


def _planes(g, kind, beta=1.0):
    N = g.N
    if kind == "const":
        K = np.full((N, N), beta)
    else:
        K = beta * (g.m_c[:, None] + g.m_c[None, :])
    return orc.pack_planes(K, np.zeros((N, N)))


def _run(g, Kp, rho0, t_end, nsteps):
    rho = rho0[None, :].copy()
    k1 = None
    dt = t_end / nsteps
    emax = 0.0
    for _ in range(nsteps):
        rho, k1, err = orc.step_cells_planes(g.N, g.a_min, g.a_max, g.rho_m, Kp, rho, dt, k1=k1)
        emax = max(emax, err[0])
    return rho[0], emax


def _m2n_exact_const(g, tau, N0=1.0):
    mb = MBAR * (1 + tau)
    m = g.m_c
    return m * m * N0 / (MBAR * (1 + tau) ** 2) * np.exp(-m / mb)


def _m2n_exact_add(g, tau, N0=1.0):
    f = 1.0 - np.exp(-tau)
    x = g.m_c / MBAR
    z = 2.0 * x * np.sqrt(f)
    # I1(z) exp(-(1+f)x) = ive(1,z) exp(z - (1+f) x)
    # scipy's ive() returns nan beyond z ~ 1e9; there exp(z - (1+f)x) has long underflowed to 0
    expo = z - (1 + f) * x
    live = expo > -700.0
    n = np.zeros_like(x)
    n[live] = (N0 / MBAR) * (1 - f) / (x[live] * np.sqrt(f)) * ive(1, z[live]) * np.exp(expo[live])
    return g.m_c ** 2 * n


def _m2n_numeric(g, rho):
    # rho_k = integral m n dm over the bin ~ m^2 n dln m  ->  m^2 n ~ rho_k / dln m
    return rho / np.log(g.m_e[1:] / g.m_e[:-1])


@pytest.mark.parametrize("kind,tau_end", [("const", 50.0), ("add", 3.0)])
def test_closed_form_moments_and_convergence(kind, tau_end):
    errs = []
    for N in (40, 80, 160):
        g = _grid(N)
        rho0 = _initial(g)
        Kp = _planes(g, kind)
        t_end = 2.0 * tau_end if kind == "const" else tau_end / MBAR
        rho, emax = _run(g, Kp, rho0, t_end, 400)
        # first moment: exact conservation
        assert rho.sum() == pytest.approx(rho0.sum(), rel=1e-12)
        assert rho.min() > -1e-12 * rho.sum()
        M0 = (rho / g.m_c).sum()
        M0_exact = 1.0 / (1 + tau_end) if kind == "const" else np.exp(-tau_end)
        M0_0 = (rho0 / g.m_c).sum()
        relM0 = abs(M0 / M0_0 / M0_exact - 1)
        exact = _m2n_exact_const(g, tau_end) if kind == "const" else _m2n_exact_add(g, tau_end)
        num = _m2n_numeric(g, rho)
        dl = np.log(g.m_e[1:] / g.m_e[:-1])
        l1 = np.sum(np.abs(num - exact) * dl) / np.sum(exact * dl)
        errs.append((N, relM0, l1, emax))
    # >= 7 bins per mass decade (N = 160 -> 10.7; N = 80 -> 5.3): zeroth moment within a few %
    assert errs[2][1] < 0.05, errs
    # the shape error falls monotonically under refinement
    assert errs[0][2] > errs[1][2] > errs[2][2], errs
    assert errs[2][2] < 0.35, errs


def test_constant_kernel_short_time_is_accurate():
    """Early times (tau = 0.5), fine grid: number density within 1 %."""
    g = _grid(160)
    rho0 = _initial(g)
    rho, _ = _run(g, _planes(g, "const"), rho0, 1.0, 100)
    M0 = (rho / g.m_c).sum() / (rho0 / g.m_c).sum()
    assert M0 == pytest.approx(1.0 / 1.5, rel=1e-2)


def test_monodisperse_constant_kernel_first_step_by_hand():
    """All mass in one bin, K = 1: dn/dt = -n^2/2 * 2 + ... by hand for the first evaluation:
    bin i loses m n^2 K (Eq. 54) and the doubled grains are split between l(2m) and l(2m)+1."""
    g = _grid(80)
    i = 30
    rho = np.zeros(g.N); rho[i] = 2.5 * g.m_c[i]
    d, ga, lo = orc.rates_cells_planes(g.N, g.a_min, g.a_max, g.rho_m, _planes(g, "const", 3.0), rho[None, :])
    M = 2 * g.m_c[i]
    l = int(np.searchsorted(g.m_c, M, side="right") - 1)
    eps = (g.m_c[l + 1] - M) / (g.m_c[l + 1] - g.m_c[l])
    R = 0.5 * 2.5 * 2.5 * 3.0
    exp = np.zeros(g.N)
    exp[i] -= g.m_c[i] * 2.5 * 2.5 * 3.0
    exp[l] += R * M * eps
    exp[l + 1] += R * M * (1 - eps)
    assert np.allclose(d[0], exp, rtol=1e-13, atol=1e-14 * np.abs(exp).max())


# ------------------------------------------------------------------------------------------ BS3(2)
def _ref_problem():
    g = orc.mass_grid(48, 1e-5, 1e-1, 1.67)
    St = 1e-4 * (g.a_c / g.a_c[0])
    vR = -300.0 * St / (1 + St * St); vZ = -200.0 * St / (1 + St * St)
    K, pf, *_ = orc.cell_kernel(g, 50.0, 1e-13, 4e-9, 1e-3, vR, vZ, orc.Params(v_frag=100.0))
    rho = 1e-15 * np.exp(-0.5 * ((np.log10(g.a_c) + 3.2) / 0.5) ** 2)
    return g, K, pf, rho


def _integrate(g, K, pf, rho, t, n):
    y = rho.copy(); k = None
    for _ in range(n):
        y, k, E = orc.bs32_step(g, K, pf, y, t / n, k1=k)
    return y


def test_bs32_third_order_convergence_and_error_estimate():
    g, K, pf, rho = _ref_problem()
    d0, ga, lo, _ = orc.rates_flux(g, K, pf, rho)
    tscale = (rho[rho > 1e-3 * rho.max()] / np.abs(d0[rho > 1e-3 * rho.max()])).min()
    t = 0.5 * tscale
    ref = _integrate(g, K, pf, rho, t, 256)
    e = []
    for n in (2, 4, 8):
        e.append(np.abs(_integrate(g, K, pf, rho, t, n) - ref).max())
    # global error of a 3rd-order method falls ~8x per halving
    assert 5.5 < e[0] / e[1] < 11 and 5.5 < e[1] / e[2] < 11, e
    # embedded estimate: E ~ h^3 (difference between the 3rd- and 2nd-order solutions)
    _, _, E1 = orc.bs32_step(g, K, pf, rho, t / 4, rtol=1e-2, atol_factor=1e-10)
    _, _, E2 = orc.bs32_step(g, K, pf, rho, t / 8, rtol=1e-2, atol_factor=1e-10)
    assert 5.5 < E1 / E2 < 11


def test_bs32_tableau_against_independent_implementation():
    """The same step assembled here from rates_flux() calls with the textbook Bogacki-Shampine
    coefficients (c = 0, 1/2, 3/4, 1; b = 2/9, 1/3, 4/9; b* = 7/24, 1/4, 1/3, 1/8)."""
    g, K, pf, rho = _ref_problem()
    h = 3e9
    f = lambda y: orc.rates_flux(g, K, pf, y)[0]
    k1 = f(rho); k2 = f(rho + 0.5 * h * k1); k3 = f(rho + 0.75 * h * k2)
    y3 = rho + h * (2 / 9 * k1 + 1 / 3 * k2 + 4 / 9 * k3)
    k4 = f(y3)
    y2 = rho + h * (7 / 24 * k1 + 1 / 4 * k2 + 1 / 3 * k3 + 1 / 8 * k4)
    sc = 1e-10 * rho.sum() + 1e-2 * np.maximum(np.abs(rho), np.abs(y3))
    E_exp = np.max(np.abs(y3 - y2) / sc)
    y, k, E = orc.bs32_step(g, K, pf, rho, h)
    assert np.allclose(y, y3, rtol=1e-14, atol=0)
    assert np.array_equal(k, k4)                       # FSAL: returned slope is f(y_new)
    assert E == pytest.approx(E_exp, rel=1e-9)
    # FSAL reuse gives the same second step as recomputing k1
    ya, ka, _ = orc.bs32_step(g, K, pf, y, h, k1=k)
    yb, kb, _ = orc.bs32_step(g, K, pf, y, h)
    assert np.array_equal(ya, yb)


def test_step_conserves_mass_to_1e13():
    g, K, pf, rho = _ref_problem()
    y = rho.copy(); k = None
    m0 = float(np.sum(rho.astype(np.longdouble)))
    for _ in range(20):
        y, k, E = orc.bs32_step(g, K, pf, y, 2e9, k1=k)
        m1 = float(np.sum(y.astype(np.longdouble)))
        assert abs(m1 / m0 - 1) < 1e-13
        m0 = m1
