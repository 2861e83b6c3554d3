"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by
element, on the same seeded inputs.  Tolerances: tests/gpu_common.py (BASELINE.json north_star)."""
import numpy as np
import pytest

import oracle as orc
import paper_2402_18471_b200 as cd
from paper_2402_18471_b200 import synth_disc

from gpu_common import (TOL_K, TOL_MASS, TOL_RHO_1, TOL_RHO_100, GpuDisc, assert_rates_close,
                        assert_rho_close, dt_of, oracle_args, params_pair, split_free_magnitudes)

pytestmark = pytest.mark.gpu


def _disc(index, n_cells=None):
    cfg = synth_disc.CONFIGS[index]
    cells = None if n_cells is None else synth_disc.sample_cells(cfg, n_cells)
    return cfg, synth_disc.make_disc(index, cells=cells)


# ------------------------------------------------------------------------------------------ kernel
@pytest.mark.parametrize("index,n_cells", [(1, None), (2, 24), (3, 24), (4, 12), (5, 8)])
def test_kernel_matches_oracle(index, n_cells):
    cfg, d = _disc(index, n_cells)
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc)
    K = g.kernel().cpu().numpy()
    Kref = orc.kernel_cells(*oracle_args(d), po)
    Ktot = Kref[:, 0] + Kref[:, 1]
    for plane in (0, 1):
        diff = np.abs(K[:, plane] - Kref[:, plane])
        assert np.all(diff <= TOL_K * Ktot), f"plane {plane}: max {np.max(diff / Ktot):.3e}"
    assert np.all(K >= 0.0)


def test_kernel_with_vphi_and_scalar_alpha():
    cfg, d = _disc(1)
    po, pc = params_pair(cfg)
    rng = np.random.default_rng(5)
    vphi = rng.normal(scale=30.0, size=d.v_R.shape)
    g = GpuDisc(d, pc, use_alpha_array=False, v_phi=vphi)
    K = g.kernel().cpu().numpy()
    Kref = orc.kernel_cells(*oracle_args(d), po, vphi=vphi)
    Ktot = Kref[:, 0] + Kref[:, 1]
    assert np.all(np.abs(K - Kref) <= TOL_K * Ktot[:, None, :])
    # v_phi really entered
    Kno = orc.kernel_cells(*oracle_args(d), po)
    assert np.max(np.abs(Kno - Kref) / Ktot[:, None, :]) > 1e-3


# ------------------------------------------------------------------------------------------ rates
@pytest.mark.parametrize("index,n_cells", [(1, None), (2, 40), (3, 40), (4, 20), (5, 10)])
def test_rates_from_supplied_kernel_match_oracle(index, n_cells):
    import torch
    cfg, d = _disc(index, n_cells)
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc)
    Kref = orc.kernel_cells(*oracle_args(d), po)                    # the ORACLE's kernel as input
    dref, gain, loss = orc.rates_cells_planes(d.n_bins, d.a_min, d.a_max, d.rho_m, Kref, d.rho_dust,
                                              eta=cfg.eta, chi=cfg.chi_im)
    out = g.rates(torch.from_numpy(Kref).cuda()).cpu().numpy()
    assert_rates_close(out, dref, gain, loss, what=f"cfg{index} rates")
    # mass conservation of the rates: sum_k drho_k = 0 up to rounding of the gain/loss magnitudes
    assert np.all(np.abs(out.sum(axis=1)) <= 1e-12 * (gain + loss).sum(axis=1))


@pytest.mark.parametrize("index,n_cells", [(1, None), (2, 40), (3, 40), (4, 20), (5, 10)])
def test_rates_on_the_fly_match_oracle(index, n_cells):
    cfg, d = _disc(index, n_cells)
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc)
    dref, _, _ = orc.rates_cells(*oracle_args(d), po, d.rho_dust)
    gain, loss = split_free_magnitudes(d, po, cfg)
    out = g.rates_otf().cpu().numpy()
    assert_rates_close(out, dref, gain, loss, what=f"cfg{index} rates_otf")


# ------------------------------------------------------------------------------------------ step
def test_config1_one_rate_evaluation_and_one_step():
    """BASELINE.json config 1 exactly: 1 rate evaluation + 1 step, dt = 1 yr."""
    cfg, d = _disc(1)
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc, n_r=cfg.n_r, n_z=cfg.n_z)
    dt = dt_of(1)
    rho_ref, k4_ref, err_ref = orc.step_cells(*oracle_args(d), po, d.rho_dust, dt)
    rho = g.rho.clone()
    err = g.step(rho, dt).cpu().numpy()
    rho = rho.cpu().numpy()
    assert_rho_close(rho, rho_ref, TOL_RHO_1, "cfg1 step")
    drift = np.abs(rho.sum(axis=1) - d.rho_dust.sum(axis=1)) / d.rho_dust.sum(axis=1)
    assert drift.max() <= TOL_MASS
    np.testing.assert_allclose(err, err_ref, rtol=1e-6)


@pytest.mark.parametrize("index,n_cells,n_steps", [(2, 48, 100), (3, 48, 100), (4, 16, 100), (5, 8, 10)])
def test_many_steps_match_oracle(index, n_cells, n_steps):
    cfg, d = _disc(index, n_cells)
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc)
    dt = dt_of(index)
    rho = g.rho.clone()
    rho_ref = d.rho_dust.copy()
    k_ref = None
    m0 = rho_ref.sum(axis=1)
    worst_drift = 0.0
    for s in range(n_steps):
        rho_ref, k_ref, err_ref = orc.step_cells(*oracle_args(d), po, rho_ref, dt, k1=k_ref)
        before = rho.sum(dim=1)
        err = g.step(rho, dt)
        worst_drift = max(worst_drift, float(((rho.sum(dim=1) - before).abs() / before).max()))
        if s == 0:
            assert_rho_close(rho.cpu().numpy(), rho_ref, TOL_RHO_1, f"cfg{index} step 1")
    assert_rho_close(rho.cpu().numpy(), rho_ref, TOL_RHO_100 if n_steps >= 100 else 10 * TOL_RHO_1,
                     f"cfg{index} after {n_steps} steps")
    np.testing.assert_allclose(err.cpu().numpy(), err_ref, rtol=1e-5, atol=1e-12)
    assert worst_drift <= TOL_MASS
    assert np.abs(rho.cpu().numpy().sum(axis=1) - m0).max() / m0.max() <= n_steps * TOL_MASS


def test_fsal_reuse_and_reset():
    """Second step reuses k4 (3 evaluations); reset_fsal recomputes k1: both give the same state."""
    cfg, d = _disc(2, 16)
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc)
    dt = dt_of(2)
    a = g.rho.clone()
    g.step(a, dt); g.step(a, dt)
    b = g.rho.clone()
    g.grid.reset_fsal()
    g.step(b, dt)
    g.grid.reset_fsal()
    g.step(b, dt)
    assert_rho_close(a.cpu().numpy(), b.cpu().numpy(), 1e-13, "FSAL vs recomputed k1")


def test_bit_reproducible_run_to_run():
    import torch
    cfg, d = _disc(4, 300)
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc)
    outs = []
    for _ in range(2):
        g.grid.reset_fsal()
        rho = g.rho.clone()
        err = g.step(rho, dt_of(4))
        outs.append((rho.clone(), err.clone()))
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
