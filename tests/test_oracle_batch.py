"""-m "not gpu": pins of the oracle's batch drivers (the functions every multi-step GPU parity test
trusts) against the single-cell functions that test_oracle_pins / test_oracle_rates /
test_oracle_closed_forms pin.  orc_step_cells must be exactly cell_kernel -> (vint_scale) ->
Eq. 55 -> bs32_step per cell, with the FSAL derivative carried from step to step."""
import numpy as np

import oracle as orc


def _inputs(C, N, seed):
    rng = np.random.default_rng(seed)
    T = rng.uniform(20, 100, C); rg = 10 ** rng.uniform(-14, -11, C); Om = 10 ** rng.uniform(-9, -8, C)
    al = 10 ** rng.uniform(-4, -2, C)
    vR = rng.standard_normal((C, N)) * 50; vZ = rng.standard_normal((C, N)) * 50
    rho = 10 ** rng.uniform(-18, -15, (C, N))
    return T, rg, Om, al, vR, vZ, rho


def _step_cell_by_cell(g, p, inp, dt, k1, hd=None, vphi=None):
    T, rg, Om, al, vR, vZ, rho = inp
    C, N = rho.shape
    out = np.empty_like(rho); k4 = np.empty_like(rho); E = np.empty(C)
    for c in range(C):
        K, pf, *_ = orc.cell_kernel(g, T[c], rg[c], Om[c], al[c], vR[c], vZ[c], p,
                                    vphi=None if vphi is None else vphi[c])
        if hd is not None:
            K = orc.vint_scale(hd[c], K)
        out[c], k4[c], E[c] = orc.bs32_step(g, K, pf, rho[c], dt, k1=None if k1 is None else k1[c],
                                            eta=p.eta, chi=p.chi_im, rtol=p.rtol, atol_factor=p.atol_factor)
    return out, k4, E


def test_step_cells_is_cell_kernel_then_bs32_step_bit_for_bit():
    N, C = 24, 7
    g = orc.mass_grid(N, 1e-5, 1.0, 1.67)
    p = orc.Params(v_frag=300.0, chi_im=1.0, rtol=3e-2, atol_factor=1e-9)
    inp = _inputs(C, N, 3)
    T, rg, Om, al, vR, vZ, rho = inp
    dt = 2.0e7
    # step 1: no FSAL derivative; step 2: k1 = k4 of step 1
    r1, k1, e1 = orc.step_cells(N, 1e-5, 1.0, 1.67, T, rg, Om, al, vR, vZ, p, rho, dt)
    s1, q1, f1 = _step_cell_by_cell(g, p, inp, dt, None)
    assert np.array_equal(r1, s1) and np.array_equal(k1, q1) and np.array_equal(e1, f1)
    assert not np.array_equal(r1, rho)                       # the step moved the state
    r2, k2, e2 = orc.step_cells(N, 1e-5, 1.0, 1.67, T, rg, Om, al, vR, vZ, p, r1, dt, k1=k1)
    s2, q2, f2 = _step_cell_by_cell(g, p, (T, rg, Om, al, vR, vZ, s1), dt, q1)
    assert np.array_equal(r2, s2) and np.array_equal(k2, q2) and np.array_equal(e2, f2)
    # have_k1 is honoured: a wrong derivative changes the result; a recomputed one does not
    r2b, _, _ = orc.step_cells(N, 1e-5, 1.0, 1.67, T, rg, Om, al, vR, vZ, p, r1, dt, k1=None)
    np.testing.assert_allclose(r2b, r2, rtol=1e-12)
    r2c, _, _ = orc.step_cells(N, 1e-5, 1.0, 1.67, T, rg, Om, al, vR, vZ, p, r1, dt, k1=2.0 * k1)
    assert np.max(np.abs(r2c - r2) / r2) > 1e-6
    # the inputs are not modified
    assert np.array_equal(inp[6], rho)


def test_step_cells_vphi_and_h_dust_branches_bit_for_bit():
    N, C = 16, 4
    g = orc.mass_grid(N, 1e-5, 1.0, 1.67)
    p = orc.Params()
    inp = _inputs(C, N, 11)
    T, rg, Om, al, vR, vZ, rho = inp
    rng = np.random.default_rng(12)
    vphi = rng.standard_normal((C, N)) * 40
    hd = 10 ** rng.uniform(10, 12, (C, N))
    dt = 1.0e18                                             # rates carry 1/h ~ 1e-11
    r, k, e = orc.step_cells(N, 1e-5, 1.0, 1.67, T, rg, Om, al, vR, vZ, p, rho, dt, vphi=vphi)
    s, q, f = _step_cell_by_cell(g, p, inp, dt, None, vphi=vphi)
    assert np.array_equal(r, s) and np.array_equal(k, q) and np.array_equal(e, f)
    r, k, e = orc.step_cells(N, 1e-5, 1.0, 1.67, T, rg, Om, al, vR, vZ, p, rho, dt, h_dust=hd)
    s, q, f = _step_cell_by_cell(g, p, inp, dt, None, hd=hd)
    assert np.array_equal(r, s) and np.array_equal(k, q) and np.array_equal(e, f)
    r0, _, _ = orc.step_cells(N, 1e-5, 1.0, 1.67, T, rg, Om, al, vR, vZ, p, rho, dt)
    assert not np.array_equal(r, r0)                        # h_dust really entered


def test_step_cells_planes_is_bs32_step_per_cell():
    N, C = 20, 3
    g = orc.mass_grid(N, 1e-5, 1.0, 1.67)
    rng = np.random.default_rng(5)
    K = rng.uniform(0.5, 2.0, (N, N)); K = 0.5 * (K + K.T)
    pf = rng.uniform(0.0, 1.0, (N, N)); pf = 0.5 * (pf + pf.T)
    rho = 10 ** rng.uniform(-3, 0, (C, N))
    Kp = orc.pack_planes(K, pf)
    dt = 1e-3 / (K.max() * (rho / g.m_c).sum(axis=1).max())
    r, k, e = orc.step_cells_planes(N, 1e-5, 1.0, 1.67, Kp, rho, dt)
    r2, k2, e2 = orc.step_cells_planes(N, 1e-5, 1.0, 1.67, Kp, r, dt, k1=k)
    y, kk = rho.copy(), [None] * C
    for c in range(C):
        y1, k1, E1 = orc.bs32_step(g, K, pf, rho[c], dt)
        assert np.array_equal(y1, r[c]) and np.array_equal(k1, k[c]) and E1 == e[c]
        y2, k2c, E2 = orc.bs32_step(g, K, pf, y1, dt, k1=k1)
        assert np.array_equal(y2, r2[c]) and np.array_equal(k2c, k2[c]) and E2 == e2[c]


def test_error_norm_of_an_empty_cell_is_zero():
    """DESIGN.md R10: a bin whose error estimate is exactly 0 contributes 0 to the norm, so a cell with
    no dust (atol = 0 and max(|y|, |y'|) = 0: 0/0 in the plain formula) has E = 0 and stays empty."""
    N = 12
    g = orc.mass_grid(N, 1e-5, 1.0, 1.67)
    K = np.ones((N, N)); pf = np.full((N, N), 0.3)
    y, k, E = orc.bs32_step(g, K, pf, np.zeros(N), 1.0)
    assert E == 0.0 and np.all(y == 0.0) and np.all(k == 0.0)
    # a populated cell is unaffected by the rule, and a single populated bin gives a finite norm
    y0 = np.zeros(N); y0[3] = 1e-3
    _, _, E1 = orc.bs32_step(g, K, pf, y0, 10.0)
    assert np.isfinite(E1) and E1 > 0.0
