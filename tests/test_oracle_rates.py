"""Pins of the oracle's rate evaluation (Eqs. 53, 54, 61-68).

The independent references here are: (a) the paper's LITERAL triple-loop definition evaluated in
exact rational arithmetic (python Fractions) inside this file, with explicit C_ijk, R_ijk, F_ijk
tensors; (b) exact invariants (mass conservation, pure-sticking support, fragment bookkeeping).
The oracle's production form is the algebraically rearranged pair-flux form (R9) -- a
different formula, so agreement with (a) is a real check, and a dropped term / wrong sign / wrong
bin index anywhere fails it.
"""
from fractions import Fraction as Fr

import numpy as np
import pytest

import oracle as orc


# ------------------------------------------------------------------------------------------
# (a) the paper's definition in exact arithmetic
# ------------------------------------------------------------------------------------------
def literal_exact(m_c, m_e, K, pf, rho, eta_int, chi, variant=0):
    """Eq. 53 with Eq. 54 (loss), Eq. 61 (gain), Eqs. 63-65 (C, R), Eq. 67 (F = N_k(m^e_{l+1})),
    Eq. 68 (m_rem), in Fractions.  eta_int: integer eta so that (.)^(2-eta) stays rational.
    Readings: R1 (1/2 on the diagonal in the gain only), R2, R5 (j <= i), R7, R8."""
    N = len(m_c)
    m = [Fr(x) for x in m_c]
    me = [Fr(x) for x in m_e]
    n = [Fr(r) / mk for r, mk in zip(rho, m)]
    chi = Fr(chi)
    ex = 2 - eta_int

    def lower(mass):        # largest index with m_l <= mass, or -1
        ls = [k for k in range(N) if m[k] <= mass]
        return max(ls) if ls else -1

    def split_weights(mass):
        w = [Fr(0)] * N
        l = lower(mass)
        if l == -1:
            w[0] = Fr(1)
        elif l == N - 1:
            w[N - 1] = Fr(1)
        else:
            eps = (m[l + 1] - mass) / (m[l + 1] - m[l])       # Eq. 65
            w[l] = eps
            w[l + 1] = 1 - eps
            if variant & 1:     # G11: eps is the NUMBER fraction; the mass fractions are eps m_l / m, (1 - eps) m_u / m
                w[l] = eps * m[l] / mass
                w[l + 1] = (1 - eps) * m[l + 1] / mass
        return w

    out = [Fr(0)] * N
    for i in range(N):
        for j in range(i + 1):
            Kij = Fr(K[i][j]) * (Fr(1, 2) if i == j else 1)
            pfr = Fr(pf[i][j])
            pco = 1 - pfr
            x = chi * m[j]
            m_rem = m[i] - x if x < m[i] else Fr(0)            # Eq. 68
            m_ft = m[i] + m[j] - m_rem
            m_lf = min(x, m[i])
            if variant & 2:     # G2: look the largest fragment's bin up with the total fragment mass
                m_lf = m_ft
            Cw = split_weights(m[i] + m[j])
            Rw = split_weights(m_rem) if m_rem > 0 else [Fr(0)] * N
            l = min((k for k in range(N) if me[k + 1] > m_lf), default=N - 1)    # PAPER.md:469 (R8: clamped to the last bin)
            mmax = me[l + 1]
            Fw = [(me[k + 1] ** ex - me[k] ** ex) / (mmax ** ex - me[0] ** ex) if k <= l else Fr(0)
                  for k in range(N)]                            # Eq. 67
            for k in range(N):
                out[k] += n[i] * n[j] * Kij * (pco * (m[i] + m[j]) * Cw[k]
                                               + pfr * (m_rem * Rw[k] + m_ft * Fw[k]))
    for k in range(N):
        for i in range(N):
            out[k] -= m[k] * n[i] * n[k] * Fr(K[i][k])          # Eq. 54 (p_c + p_f = 1)
    return out


def _random_problem(N, q, seed, span_lo=1e-9):
    rng = np.random.default_rng(seed)
    m_e = span_lo * q ** np.arange(N + 1)
    m_c = np.sqrt(m_e[:-1] * m_e[1:])
    K = rng.uniform(0.1, 2.0, size=(N, N)); K = 0.5 * (K + K.T)
    pf = rng.uniform(0.0, 1.0, size=(N, N)); pf = 0.5 * (pf + pf.T)
    rho = rng.uniform(0.1, 1.0, size=N) * m_c * 10 ** rng.uniform(-2, 2, size=N)
    return orc.grid_from_masses(m_c, m_e), K, pf, rho


@pytest.mark.parametrize("q", [1.3, 1.4, 1.7, 2.0, 2.4, 3.1])
@pytest.mark.parametrize("chi", [0.5, 1.0, 2.0])
def test_flux_form_equals_literal_definition_exactly(q, chi):
    """8-bin brute force: pair-flux form (double) and literal form (__float128) against the exact
    rational value of the paper's definition."""
    N = 8
    for eta_int, seed in ((1, 11), (0, 12)):
        g, K, pf, rho = _random_problem(N, q, seed + int(q * 10))
        exact = literal_exact(g.m_c, g.m_e, K, pf, rho, eta_int, chi)
        # exact arithmetic conserves mass exactly: checks the reading R1/R2/R7/R8 bundle itself
        assert sum(exact) == 0
        d, gain, loss, S = orc.rates_flux(g, K, pf, rho, eta=float(eta_int), chi=chi)
        lit = orc.rates_literal(g, K, pf, rho, eta=float(eta_int), chi=chi)
        scale = gain + loss
        for k in range(N):
            assert abs(d[k] - float(exact[k])) <= 2e-14 * scale[k]
            assert abs(lit[k] - float(exact[k])) <= 2e-15 * scale[k] + 1e-300
        # gain/loss bookkeeping is consistent with the net rate
        assert np.allclose(gain - loss, d, rtol=0, atol=1e-14 * scale.max())


def test_literal_and_flux_agree_with_physical_eta():
    """eta = 11/6 (irrational exponents): literal definition in __float128 vs pair-flux in double."""
    for q in (1.318, 1.514, 2.371):
        g, K, pf, rho = _random_problem(10, q, 5)
        d, gain, loss, _ = orc.rates_flux(g, K, pf, rho)
        lit = orc.rates_literal(g, K, pf, rho)
        assert np.all(np.abs(d - lit) <= 5e-14 * (gain + loss))


def test_literal_form_loses_swept_mass_on_wide_grids_flux_form_does_not():
    """DESIGN.md R9: with mass ratios beyond 1e16 the literal gain-loss form (even in double) cannot
    conserve mass; the pair-flux form conserves it to rounding."""
    g = orc.mass_grid(100, 1e-5, 10.0, 1.67)
    rng = np.random.default_rng(2)
    K = rng.uniform(0.5, 1.5, size=(100, 100)); K = 0.5 * (K + K.T)
    K *= 1e-2
    pf = np.full((100, 100), 0.3)
    rho = np.zeros(100); rho[:12] = 1e-14; rho[80:92] = 1e-14
    d, gain, loss, _ = orc.rates_flux(g, K, pf, rho)
    assert abs(d.sum()) <= 1e-15 * (gain.sum() + loss.sum())
    assert abs(np.sum(d.astype(np.longdouble))) <= 2e-16 * float(np.sum(np.abs(d)))  * 50


# ------------------------------------------------------------------------------------------
# (b) invariants
# ------------------------------------------------------------------------------------------
def _disc_cell(N=60, seed=0):
    g = orc.mass_grid(N, 1e-5, 10.0, 1.67)
    rng = np.random.default_rng(seed)
    St = 1e-4 * (g.a_c / g.a_c[0])
    vR = -300.0 * St / (1 + St * St); vZ = -500.0 * St / (1 + St * St)
    p = orc.Params(v_frag=100.0)
    K, pf, *_ = orc.cell_kernel(g, 40.0, 1e-13, 5e-9, 1e-3, vR, vZ, p)
    rho = 1e-15 * np.exp(-0.5 * ((np.log10(g.a_c) + 2.5) / 0.8) ** 2) * np.exp(0.1 * rng.standard_normal(N))
    return g, K, pf, rho


def test_mass_conservation_of_rates():
    """sum_k drho_k = 0 (PAPER.md: Eq. 61 moves mass, never creates it)."""
    for seed in range(4):
        g, K, pf, rho = _disc_cell(seed=seed)
        d, gain, loss, S = orc.rates_flux(g, K, pf, rho)
        tot = float(np.sum(d.astype(np.longdouble)))
        assert abs(tot) <= 1e-15 * (gain.sum() + loss.sum())
        assert gain.min() >= 0 and loss.min() >= 0


def test_pure_sticking_never_populates_lower_bins():
    """p_frag = 0: nothing ever appears below the lowest initially populated bin, and
    those bins' rates are exactly zero (l(m_i+m_j) >= i)."""
    g, K, pf, rho = _disc_cell()
    rho[:17] = 0.0
    d, gain, loss, S = orc.rates_flux(g, K, 0.0 * pf, rho)
    assert np.all(d[:17] == 0.0) and np.all(S == 0.0)
    assert d[17] < 0 and d.sum() == pytest.approx(0.0, abs=1e-15 * loss.sum())
    # and over a step
    y, k4, E = orc.bs32_step(g, K, 0.0 * pf, rho, 1e3)
    assert np.all(y[:17] == 0.0)


def test_all_fragmenting_with_huge_chi_sends_everything_to_the_power_law():
    """p_frag = 1 and chi -> inf (m_rem = 0): total fragment input = sum_pairs R (m_i + m_j), every
    bin's own mass is lost at rate rho_k sum_i n_i K_ik, fragments only go to bins <= l."""
    g, K, pf, rho = _disc_cell(N=30)
    N = g.N
    d, gain, loss, S = orc.rates_flux(g, K, np.ones_like(pf), rho, chi=1e40)
    n = rho / g.m_c
    tot = 0.0
    for i in range(N):
        for j in range(i + 1):
            tot += n[i] * n[j] * K[i, j] * (0.5 if i == j else 1.0) * (g.m_c[i] + g.m_c[j])
    assert S.sum() == pytest.approx(tot, rel=1e-13)
    # m_lf = min(chi m_j, m_i) = m_i: fragments of pair (i, j) enter at l-bin i
    expect_loss = rho * (K @ n)
    assert np.allclose(loss, expect_loss, rtol=1e-13)
    assert d.sum() == pytest.approx(0.0, abs=1e-14 * loss.sum())


def test_fragment_redistribution_against_eq67_directly():
    """Two-stage l-bin algorithm == sum_l S_l N_k(m^e_{l+1}) with Eq. 67 written out;
    N_k sums to one over k <= l (telescoping)."""
    g = orc.mass_grid(25, 1e-5, 1e-1, 1.67)
    rng = np.random.default_rng(8)
    S = rng.uniform(0, 1, g.N)
    for eta in (11.0 / 6.0, 1.5, 1.0, 0.3):
        ex = 2.0 - eta
        Nk = np.zeros((g.N, g.N))          # [l, k]
        for l in range(g.N):
            for k in range(l + 1):
                Nk[l, k] = (g.m_e[k + 1] ** ex - g.m_e[k] ** ex) / (g.m_e[l + 1] ** ex - g.m_e[0] ** ex)
        assert np.allclose(Nk.sum(axis=1), 1.0, rtol=1e-13)
        direct = S @ Nk
        d = orc.frag_redistribute(g, S, eta=eta)
        assert np.allclose(d, direct, rtol=1e-12)
        assert d.sum() == pytest.approx(S.sum(), rel=1e-13)


def test_single_pair_outcomes_by_hand():
    """One populated pair, every product placed by hand from Eqs. 63-68 (chi = 1, eta = 11/6)."""
    g = orc.mass_grid(12, 1e-4, 1e-2, 1.0)
    N = g.N
    m = g.m_c
    i, j = 7, 5
    K = np.zeros((N, N)); K[i, j] = K[j, i] = 2.0
    pf = np.full((N, N), 0.25)
    rho = np.zeros(N); rho[i] = 3.0 * m[i]; rho[j] = 5.0 * m[j]      # n_i = 3, n_j = 5
    R = 3.0 * 5.0 * 2.0
    d, gain, loss, S = orc.rates_flux(g, K, pf, rho)
    exp = np.zeros(N)
    # coagulation (prob 0.75): product m_i + m_j split between l and l+1
    M = m[i] + m[j]
    l = max(k for k in range(N) if m[k] <= M)
    eps = (m[l + 1] - M) / (m[l + 1] - m[l])
    exp[i] -= 0.75 * R * m[i]; exp[j] -= 0.75 * R * m[j]
    exp[l] += 0.75 * R * M * eps; exp[l + 1] += 0.75 * R * M * (1 - eps)
    # fragmentation (prob 0.25): remnant m_i - m_j, fragments 2 m_j with largest fragment m_j -> l-bin j
    mr = m[i] - m[j]
    lr = max(k for k in range(N) if m[k] <= mr)
    er = (m[lr + 1] - mr) / (m[lr + 1] - m[lr])
    exp[i] -= 0.25 * R * m[i]; exp[j] -= 0.25 * R * m[j]
    exp[lr] += 0.25 * R * mr * er; exp[lr + 1] += 0.25 * R * mr * (1 - er)
    ex = 1.0 / 6.0
    for k in range(j + 1):
        exp[k] += 0.25 * R * 2 * m[j] * (g.m_e[k + 1] ** ex - g.m_e[k] ** ex) / (g.m_e[j + 1] ** ex - g.m_e[0] ** ex)
    assert np.allclose(d, exp, rtol=1e-12, atol=1e-13 * np.abs(exp).max())
    assert S[j] == pytest.approx(0.25 * R * 2 * m[j], rel=1e-14) and np.count_nonzero(S) == 1


def test_diagonal_half_rule():
    """PAPER.md:436 with reading R1: i = j collisions at rate n_i^2 K_ii / 2, each removing two grains:
    bin i loses m_i n_i^2 K_ii, and 2 m_i per collision reappears as product."""
    g = orc.mass_grid(12, 1e-4, 1e-2, 1.0)
    N = g.N
    K = np.zeros((N, N)); K[4, 4] = 7.0
    rho = np.zeros(N); rho[4] = 2.0 * g.m_c[4]
    d, gain, loss, S = orc.rates_flux(g, K, np.zeros((N, N)), rho)
    m = g.m_c
    Rh = 0.5 * 2.0 * 2.0 * 7.0                      # n_i^2 K_ii / 2
    assert 2 * m[4] < m[5]                          # product lands between bins 4 and 5 on this grid
    eps = (m[5] - 2 * m[4]) / (m[5] - m[4])
    # literal: bin 4 loses m_4 n^2 K (full K, two grains per collision) and regains Rh 2 m_4 eps
    assert d[4] == pytest.approx(-m[4] * 4.0 * 7.0 + Rh * 2 * m[4] * eps, rel=1e-13)
    assert d[5] == pytest.approx(Rh * 2 * m[4] * (1 - eps), rel=1e-13)
    assert d.sum() == pytest.approx(0.0, abs=1e-14 * abs(d[5]))
    # halving the loss too (the other reading of PAPER.md:436) would create mass:
    assert -0.5 * m[4] * 4.0 * 7.0 + Rh * 2 * m[4] * eps + d[5] > 0.4 * abs(d[5])


def test_rates_scale_quadratically_in_density():
    g, K, pf, rho = _disc_cell()
    d1, *_ = orc.rates_flux(g, K, pf, rho)
    d2, *_ = orc.rates_flux(g, K, pf, 3.0 * rho)
    assert np.allclose(d2, 9.0 * d1, rtol=1e-12, atol=1e-30)


def test_cells_batch_matches_single_cell_and_planes_roundtrip():
    N = 20
    g = orc.mass_grid(N, 1e-5, 1.0, 1.67)
    rng = np.random.default_rng(0)
    C = 5
    T = rng.uniform(20, 100, C); rg = 10 ** rng.uniform(-14, -11, C); Om = 10 ** rng.uniform(-9, -8, C)
    al = np.full(C, 1e-3)
    vR = rng.standard_normal((C, N)) * 50; vZ = rng.standard_normal((C, N)) * 50
    rho = 10 ** rng.uniform(-18, -15, (C, N))
    p = orc.Params()
    d, ga, lo = orc.rates_cells(N, 1e-5, 1.0, 1.67, T, rg, Om, al, vR, vZ, p, rho)
    Kp = orc.kernel_cells(N, 1e-5, 1.0, 1.67, T, rg, Om, al, vR, vZ, p)
    d2, ga2, lo2 = orc.rates_cells_planes(N, 1e-5, 1.0, 1.67, Kp, rho)
    assert np.array_equal(d, d2)
    for c in range(C):
        K, pf, *_ = orc.cell_kernel(g, T[c], rg[c], Om[c], al[c], vR[c], vZ[c], p)
        ds, gs, ls, _ = orc.rates_flux(g, K, pf, rho[c])
        assert np.array_equal(ds, d[c])
        assert np.array_equal(orc.pack_planes(K, pf), Kp[c])


# ------------------------------------------------------------------------------------------
# (e) the two switched readings (R2 / R11)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [1, 2, 3])
@pytest.mark.parametrize("q,chi", [(1.3, 1.0), (1.7, 0.5), (2.0, 2.0), (2.4, 1.0)])
def test_variants_flux_form_equals_their_exact_definition_and_conserve_mass(variant, q, chi):
    N = 8
    try:
        orc.set_variant(variant)
        for eta_int, seed in ((1, 21), (0, 22)):
            g, K, pf, rho = _random_problem(N, q, seed + int(q * 10))
            exact = literal_exact(g.m_c, g.m_e, K, pf, rho, eta_int, chi, variant=variant)
            assert sum(exact) == 0                                   # mass is conserved exactly by either reading
            d, gain, loss, S = orc.rates_flux(g, K, pf, rho, eta=float(eta_int), chi=chi)
            lit = orc.rates_literal(g, K, pf, rho, eta=float(eta_int), chi=chi)
            scale = gain + loss
            for k in range(N):
                assert abs(d[k] - float(exact[k])) <= 2e-14 * scale[k]
                assert abs(lit[k] - float(exact[k])) <= 2e-15 * scale[k] + 1e-300
            # the variant is not the default reading
            base = literal_exact(g.m_c, g.m_e, K, pf, rho, eta_int, chi, variant=0)
            assert any(a != b for a, b in zip(exact, base))
    finally:
        orc.set_variant(0)


def test_number_conserving_split_removes_exactly_one_particle_per_collision():
    """G11 pin: with sticking only and every product on the grid, each collision turns two particles into one,
    so d/dt sum_k n_k = - sum_{i >= j} R_ij EXACTLY for the number-weighted split -- and not for the
    mass-weighted one (which creates or destroys particles when it splits a product over two bins)."""
    N, q = 10, 1.6
    g, K, pf, rho = _random_problem(N, q, 77)
    pf[:] = 0.0
    rho[N - 3:] = 0.0                                 # nothing can leave the top of the grid (q^3 > 2)
    m = [Fr(x) for x in g.m_c]
    n = [Fr(r) / mk for r, mk in zip(rho, m)]
    collisions = sum(n[i] * n[j] * Fr(K[i][j]) * (Fr(1, 2) if i == j else 1) for i in range(N) for j in range(i + 1))
    for variant, exact_number in ((1, True), (0, False)):
        ex = literal_exact(g.m_c, g.m_e, K, pf, rho, 1, 1.0, variant=variant)
        dN = sum(e / mk for e, mk in zip(ex, m))
        assert (dN == -collisions) == exact_number
        try:
            orc.set_variant(variant)
            d, gain, loss, _ = orc.rates_flux(g, K, pf, rho, eta=1.0, chi=1.0)
        finally:
            orc.set_variant(0)
        dN_f = float(np.sum(d / g.m_c))
        assert abs(dN_f - float(dN)) <= 1e-13 * float(collisions)
