"""-m gpu test of cudisc_coag_rates_otf_noalloc (include/cudisc_coag.h): the rate evaluation whose kernel
scratch -- the per-CTA slab for the pairs of K that do not fit in shared memory -- is the library's file-scope
device array, so that the call allocates nothing.  Its output is compared with the existing path
(cudisc_coag_rates_otf, scratch owned by the grid) and with the oracle, within the tolerance of the other
rate tests (tests/gpu_common.py TOL_RATE), on two calls in a row with different inputs: every call shares the
array, which keeps the last call's contents.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the
other GPU tests."""
import numpy as np
import pytest

import oracle as orc
import paper_2402_18471_b200 as cd
from paper_2402_18471_b200 import binding, synth_disc

from gpu_common import GpuDisc, assert_rates_close, oracle_args, params_pair

pytestmark = pytest.mark.gpu


def _rates_noalloc(g, rho):
    out = g.torch.full_like(rho, float("nan"))
    cd.cudisc_coag_rates_otf_noalloc(g.grid, g.bins, rho, out)
    g.torch.cuda.synchronize()
    return out.cpu().numpy()


def _check_two_calls(index, n_cells, expect_scratch):
    cfg = synth_disc.CONFIGS[index]
    d = synth_disc.make_disc(index, cells=synth_disc.sample_cells(cfg, n_cells))
    po, pc = params_pair(cfg)
    g = GpuDisc(d, pc)
    # the slab this grid needs of the static array: resident CTAs x pairs beyond shared memory x 16 B
    vec_bytes = g.bins.schedule_check()[7]
    p_shared = min(g.P, (232448 - vec_bytes) // 16)
    need = min(148, g.C) * (g.P - p_shared) * 16
    assert (need > 0) == expect_scratch
    assert need <= binding.STATIC_SCRATCH_BYTES

    # second input: the same cells' densities in reverse cell order (other values in every slab entry)
    rho1 = g.rho
    rho2 = g.torch.flip(g.rho, dims=[0]).contiguous() * 0.5
    for call, rho in enumerate((rho1, rho2, rho1)):
        rho_h = rho.cpu().numpy()
        got = _rates_noalloc(g, rho)
        old = g.rates_otf(rho).cpu().numpy()
        ref, gain, loss = orc.rates_cells(*oracle_args(d), po, rho_h)
        assert np.all(np.isfinite(got))
        assert_rates_close(got, old, gain, loss, what=f"cfg{index} call {call}: no-alloc vs existing path")
        assert_rates_close(got, ref, gain, loss, what=f"cfg{index} call {call}: no-alloc vs oracle")
        if call == 0:
            first = got
    # the third call repeats the first input: what the second call left in the array changes nothing
    assert np.array_equal(got, first)


def test_noalloc_matches_existing_path_200_bins():
    """config 5 (200 bins): 9594 pairs per CTA live in the static array; 300 cells keep all 148 CTAs busy."""
    _check_two_calls(5, 300, expect_scratch=True)


def test_noalloc_matches_existing_path_without_scratch():
    """config 4 (150 bins): K fits in shared memory, the static array is not touched."""
    _check_two_calls(4, 12, expect_scratch=False)


def test_noalloc_rejects_sizes_beyond_the_static_array():
    import torch
    pc = cd.Params()
    bins = cd.Bins(256, 1e-5, 10.0, 1.67, pc)
    C = 148                                     # 148 CTAs x 23491 pairs x 16 B = 53 MiB > 24 MiB
    grid = cd.Grid(C, 1, bins)
    dev = torch.device("cuda:0")
    one = torch.ones(C, dtype=torch.float64, device=dev)
    vel = torch.zeros((C, 256), dtype=torch.float64, device=dev)
    grid.bind_gas(T=100.0 * one, rho_gas=1e-12 * one, Omega=1e-8 * one, v_R=vel, v_Z=vel)
    rho = torch.full((C, 256), 1e-16, dtype=torch.float64, device=dev)
    out = torch.empty_like(rho)
    with pytest.raises(cd.CudiscError) as ei:
        cd.cudisc_coag_rates_otf_noalloc(grid, bins, rho, out)
    msg = str(ei.value)
    assert "scratch" in msg and str(binding.STATIC_SCRATCH_BYTES) in msg
    cd.cudisc_coag_rates_otf(grid, bins, rho, out)      # the existing path still takes this grid
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all())
    grid.close()
    bins.close()
