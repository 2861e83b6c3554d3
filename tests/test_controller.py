"""Adaptive sub-cycling (R10): the oracle's controller against closed
forms, the library's host controller against the same values (no GPU), and -- on the GPU -- the
library's integrator against the oracle replaying its accepted step sizes."""
import numpy as np
import pytest

import oracle as orc
import paper_2402_18471_b200 as cd
from paper_2402_18471_b200 import synth_disc

from test_oracle_closed_forms import MBAR, _grid, _initial, _planes

PINS = [  # (E, factor): 0.9 E^(-1/3) clamped to [0.2, 5]
    (0.729, 1.0), (1.0, 0.9), (0.0, 5.0), (1e-9, 5.0), (1e9, 0.2), (8.0, 0.45), (0.001, 5.0), (0.125, 1.8),
]


@pytest.mark.parametrize("E,f", PINS)
def test_oracle_controller_closed_forms(E, f):
    assert orc.controller_next_dt(E, 3.0) == pytest.approx(3.0 * f, rel=1e-14)


@pytest.mark.parametrize("E,f", PINS)
def test_library_controller_matches(E, f):
    assert cd.cudisc_controller_next_dt(E, 3.0) == pytest.approx(3.0 * f, rel=1e-14)
    assert cd.cudisc_controller_next_dt(E, 3.0) == pytest.approx(orc.controller_next_dt(E, 3.0), rel=1e-15)


def test_oracle_integrate_constant_kernel_closed_form():
    """Adaptive run of the constant kernel: lands exactly on t_span, conserves mass, M0(t) = N0/(1+tau)
    within the grid's numerical diffusion, every accepted step has E <= 1 by construction."""
    g = _grid(120)
    Kp = _planes(g, "const")
    rho0 = _initial(g)
    tau = 20.0
    t_end = 2.0 * tau                                 # K N0 t / 2 = tau with K = N0 = 1
    step = lambda rho, h, k1: orc.step_cells_planes(g.N, g.a_min, g.a_max, g.rho_m, Kp, rho, h, k1=k1)
    rho, log, dt_next = orc.integrate(step, rho0[None, :], t_end, dt_try=1e-3)
    acc = [h for h in log if h > 0]
    assert sum(acc) == pytest.approx(t_end, rel=1e-12)
    assert abs(rho.sum() - rho0.sum()) <= 1e-12 * rho0.sum()
    M0 = (rho[0] / g.m_c).sum()
    assert M0 == pytest.approx(1.0 / (1.0 + tau), rel=0.05)
    assert dt_next > 0 and len(acc) < 400             # the controller opens the step up from 1e-3
    # replaying the accepted schedule reproduces the state bit for bit
    assert np.array_equal(orc.replay(step, rho0[None, :], acc), rho)


@pytest.mark.gpu
@pytest.mark.parametrize("index,n_cells,factor", [(2, 32, 6.0), (3, 32, 6.0), (4, 300, 12.0)])
def test_integrate_matches_oracle_replay(index, n_cells, factor):
    import torch
    from gpu_common import TOL_MASS, TOL_RHO_1, GpuDisc, assert_rho_close, dt_of, oracle_args, params_pair
    cfg = synth_disc.CONFIGS[index]
    d = synth_disc.make_disc(index, cells=synth_disc.sample_cells(cfg, n_cells))
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc)
    dt0 = dt_of(index)
    t_span = factor * dt0
    rho = g.rho.clone()
    info, log = cd.cudisc_coag_integrate(g.grid, g.bins, rho, t_span, 4.0 * dt0, max_steps=400)
    torch.cuda.synchronize()
    acc = log[log > 0]
    assert info["t_done"] == t_span and info["n_accepted"] == acc.size and info["n_rejected"] == (log < 0).sum()
    assert acc.sum() == pytest.approx(t_span, rel=1e-12)
    assert info["n_rejected"] >= 1                   # 4 x the stability-limited step must be rejected
    assert info["err_last"] <= 1.0 and info["dt_next"] > 0
    step = lambda r, h, k1: orc.step_cells(*oracle_args(d), po, r, h, k1=k1)
    rho_ref = orc.replay(step, d.rho_dust, acc)
    assert_rho_close(rho.cpu().numpy(), rho_ref, TOL_RHO_1 * max(acc.size, 1), f"cfg{index} integrate")
    m0 = d.rho_dust.sum(axis=1)
    assert np.max(np.abs(rho.cpu().numpy().sum(axis=1) - m0) / m0) <= acc.size * TOL_MASS
    # a second call continues from the returned step size and the saved FSAL derivative
    info2, log2 = cd.cudisc_coag_integrate(g.grid, g.bins, rho, t_span, info["dt_next"], max_steps=400)
    assert info2["t_done"] == t_span and np.all(np.isfinite(rho.cpu().numpy()))
