"""-m gpu: the BASELINE.json configs at their stated sizes and run lengths.

  cfg 2, 3   100 steps on ALL 8000 cells, every cell against the oracle at 1e-9
  cfg 4      cudisc_coag_integrate_steps: 1000 accepted adaptive steps on all 32000 cells; the oracle
             replays the first 100 recorded step sizes on sampled cells at 1e-9; mass drift over the 1000
  cfg 5      one launch at 128000 cells x 200 bins (the general kernel with its per-CTA L2 slabs, every
             CTA's slab exercised), sampled cells including the last wave, then 10 steps
"""
import numpy as np
import pytest

import oracle as orc
import paper_2402_18471_b200 as cd
from paper_2402_18471_b200 import synth_disc

from gpu_common import (TOL_MASS, TOL_RHO_1, TOL_RHO_100, GpuDisc, assert_rho_close, dt_of, oracle_args,
                        params_pair)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("index", [2, 3])
def test_config_100_steps_on_every_cell(index):
    cfg = synth_disc.CONFIGS[index]
    d = synth_disc.make_disc(index)
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc, n_r=cfg.n_r, n_z=cfg.n_z)
    dt = dt_of(index)
    rho = g.rho.clone()
    rho_ref, k_ref = d.rho_dust.copy(), None
    worst = 0.0
    for s in range(cfg.n_steps):
        before = rho.sum(dim=1)
        err = g.step(rho, dt)
        worst = max(worst, float(((rho.sum(dim=1) - before).abs() / before).max()))
        rho_ref, k_ref, err_ref = orc.step_cells(*oracle_args(d), po, rho_ref, dt, k1=k_ref)
    assert cfg.n_steps == 100 and d.n_cells == 8000
    assert_rho_close(rho.cpu().numpy(), rho_ref, TOL_RHO_100, f"cfg{index}, 100 steps, all cells")
    np.testing.assert_allclose(err.cpu().numpy(), err_ref, rtol=1e-5, atol=1e-12)
    assert worst <= TOL_MASS


def test_config4_thousand_adaptive_steps_full_grid():
    import torch
    cfg = synth_disc.CONFIGS[4]
    d = synth_disc.make_disc(4)
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc, n_r=cfg.n_r, n_z=cfg.n_z)
    dt0 = dt_of(4)
    rho = g.rho.clone()
    m0 = d.rho_dust.sum(axis=1)
    info, log = cd.cudisc_coag_integrate_steps(g.grid, g.bins, rho, 100, dt0, max_steps=400)
    torch.cuda.synchronize()
    acc = log[log > 0]
    assert info["n_accepted"] == 100 == acc.size and info["t_done"] == pytest.approx(acc.sum(), rel=1e-12)
    cells = synth_disc.sample_cells(cfg, 24, seed=5)
    ds = d.subset(cells)
    step = lambda r, h, k1: orc.step_cells(*oracle_args(ds), po, r, h, k1=k1)
    rho_ref = orc.replay(step, ds.rho_dust, acc)
    assert_rho_close(rho.cpu().numpy()[cells], rho_ref, TOL_RHO_100, "cfg4, first 100 accepted steps, sampled cells")
    # the remaining 900 accepted steps continue from the returned size and the saved FSAL derivative
    info2, log2 = cd.cudisc_coag_integrate_steps(g.grid, g.bins, rho, 900, info["dt_next"], max_steps=3600)
    torch.cuda.synchronize()
    assert info2["n_accepted"] == 900
    out = rho.cpu().numpy()
    assert np.all(np.isfinite(out))
    assert np.max(np.abs(out.sum(axis=1) - m0) / m0) <= 1000 * TOL_MASS
    # growth happened: mass moved out of the initial MRN range (bins above 1 micron were exactly empty)
    a_e, a_c = synth_disc.size_bins(cfg.n_bins, cfg.a_min, cfg.a_max)
    assert np.all(d.rho_dust[:, a_c > 2e-4] == 0.0) and np.median(out[:, a_c > 2e-4].sum(axis=1) / m0) > 1e-6


def test_config5_full_size_launch_and_ten_steps():
    import torch
    cfg = synth_disc.CONFIGS[5]
    d = synth_disc.make_disc(5)
    assert d.n_cells == 128000 and d.n_bins == 200
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc, n_r=cfg.n_r, n_z=cfg.n_z)
    assert not g.bins.fast_path()[0]               # 200 bins: the general kernel with L2 slabs
    dt = dt_of(5)
    # sampled cells: a spread over the disc plus the last wave of the persistent CTAs
    sm = torch.cuda.get_device_properties(0).multi_processor_count
    C = d.n_cells
    cells = np.unique(np.concatenate([synth_disc.sample_cells(cfg, 48, seed=3), np.arange(C - 16, C),
                                      np.arange(C - sm - 2, C - sm + 2)]))
    assert cells.size >= 64
    ds = d.subset(cells)
    # 10 rate evaluations (BASELINE.json): the first against the oracle, all ten identical in bits
    out0 = g.rates_otf()
    dref, _, _ = orc.rates_cells(*oracle_args(ds), po, ds.rho_dust)
    from gpu_common import assert_rates_close, split_free_magnitudes
    gain, loss = split_free_magnitudes(ds, po, cfg)
    assert_rates_close(out0.cpu().numpy()[cells], dref, gain, loss, what="cfg5 full size, rates")
    for _ in range(9):
        assert torch.equal(g.rates_otf(), out0)
    # 10 steps
    rho = g.rho.clone()
    rho_ref, k_ref = ds.rho_dust.copy(), None
    m0 = d.rho_dust.sum(axis=1)
    for s in range(10):
        err = g.step(rho, dt)
        rho_ref, k_ref, err_ref = orc.step_cells(*oracle_args(ds), po, rho_ref, dt, k1=k_ref)
        if s == 0:
            assert_rho_close(rho.cpu().numpy()[cells], rho_ref, TOL_RHO_1, "cfg5 full size, step 1")
    out = rho.cpu().numpy()
    assert_rho_close(out[cells], rho_ref, 10 * TOL_RHO_1, "cfg5 full size, 10 steps")
    np.testing.assert_allclose(err.cpu().numpy()[cells], err_ref, rtol=1e-5, atol=1e-12)
    assert np.all(np.isfinite(out)) and np.max(np.abs(out.sum(axis=1) - m0) / m0) <= 10 * TOL_MASS
