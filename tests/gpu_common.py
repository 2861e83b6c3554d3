"""Shared plumbing of the -m gpu parity tests: moves seeded inputs to the device, calls the CUDA
path through the C-ABI binding, calls the oracle on the same inputs.  No method arithmetic."""
import json
import os

import numpy as np

import oracle as orc
import paper_2402_18471_b200 as cd
from paper_2402_18471_b200 import synth_disc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

# Tolerances (BASELINE.json north_star)
TOL_K = 1e-12          # |dKc|, |dKf| <= TOL_K * K_ij
TOL_RATE = 1e-11       # |d drho_k| <= TOL_RATE * (gain_k + loss_k)
TOL_RHO_1 = 1e-11      # one step, relative, bins with rho_k > 1e-30 sum(rho)
TOL_RHO_100 = 1e-9     # after 100 steps
TOL_MASS = 1e-13       # relative drift of sum_k rho_k per step
# Underflow guard of the rate comparison: a sum whose terms lie below DBL_MIN / u ~ 2e-292 is built
# from subnormal products and carries no relative accuracy on either side.
RATE_ABS_FLOOR = 1e-290


def dt_of(index: int) -> float:
    with open(os.path.join(ROOT, "tests", "golden", "dt_manifest.json")) as f:
        return float(json.load(f)[str(index)]["dt_s"])


def params_pair(cfg):
    po = orc.Params(mu=cfg.mu, v_frag=cfg.v_frag, eta=cfg.eta, chi_im=cfg.chi_im, sigma_mol=cfg.sigma_mol)
    pc = cd.Params(mu=cfg.mu, v_frag=cfg.v_frag, alpha=cfg.alpha, eta=cfg.eta, chi_im=cfg.chi_im,
                   sigma_mol=cfg.sigma_mol)
    return po, pc


class GpuDisc:
    """Device copy of a DiscInputs plus the library handles."""

    def __init__(self, d, pc, n_r=None, n_z=None, use_alpha_array=True, v_phi=None):
        import torch
        self.torch = torch
        self.d = d
        self.pc = pc
        dev = torch.device("cuda:0")
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        self.gas = dict(T=t(d.T), rho_gas=t(d.rho_gas), Omega=t(d.Omega), v_R=t(d.v_R), v_Z=t(d.v_Z),
                        alpha=t(d.alpha) if use_alpha_array else None,
                        v_phi=t(v_phi) if v_phi is not None else None)
        self.rho = t(d.rho_dust)
        self.bins = cd.Bins(d.n_bins, d.a_min, d.a_max, d.rho_m, pc)
        C = d.n_cells
        if n_r is None:
            n_r, n_z = C, 1
        self.grid = cd.Grid(n_r, n_z, self.bins)
        self.grid.bind_gas(**self.gas)
        self.C, self.N, self.P = C, d.n_bins, self.bins.n_pairs

    def kernel(self):
        K = self.torch.empty((self.C, 2, self.P), dtype=self.torch.float64, device="cuda:0")
        cd.cudisc_coag_kernel(self.grid, self.bins, self.gas, self.pc, K)
        self.torch.cuda.synchronize()
        return K

    def rates(self, K, rho=None):
        rho = self.rho if rho is None else rho
        out = self.torch.empty_like(rho)
        cd.cudisc_coag_rates(self.grid, self.bins, K, rho, out)
        self.torch.cuda.synchronize()
        return out

    def rates_otf(self, rho=None):
        rho = self.rho if rho is None else rho
        out = self.torch.empty_like(rho)
        cd.cudisc_coag_rates_otf(self.grid, self.bins, rho, out)
        self.torch.cuda.synchronize()
        return out

    def step(self, rho, dt):
        err = self.torch.empty(self.C, dtype=self.torch.float64, device="cuda:0")
        cd.cudisc_coag_step(self.grid, self.bins, rho, dt, err)
        self.torch.cuda.synchronize()
        return err


def oracle_args(d):
    return (d.n_bins, d.a_min, d.a_max, d.rho_m, d.T, d.rho_gas, d.Omega, d.alpha, d.v_R, d.v_Z)


def split_free_magnitudes(d, po, cfg):
    """Gain and loss magnitudes of every bin with p_coag = p_frag = 1 (both planes = the oracle's
    K_ij): the scale of the rate comparison when BOTH sides build the kernel themselves.  Eq. 55's
    p_coag = 1 - p_frag carries an absolute rounding error u on either side, so K p_coag is only
    good to u K_ij, not to u K_ij p_coag."""
    Kref = orc.kernel_cells(*oracle_args(d), po)
    Ktot = Kref[:, 0] + Kref[:, 1]
    planes = np.ascontiguousarray(np.stack([Ktot, Ktot], axis=1))
    _, gain, loss = orc.rates_cells_planes(d.n_bins, d.a_min, d.a_max, d.rho_m, planes, d.rho_dust,
                                           eta=cfg.eta, chi=cfg.chi_im)
    return gain, loss


def assert_rho_close(rho_gpu, rho_ref, tol, what=""):
    """relative per-bin parity on bins with |rho_k| > 1e-30 * cell total (north_star)."""
    tot = rho_ref.sum(axis=1, keepdims=True)
    mask = np.abs(rho_ref) > 1e-30 * tot
    rel = np.abs(rho_gpu - rho_ref) / np.where(mask, np.abs(rho_ref), 1.0)
    rel = np.where(mask, rel, 0.0)
    worst = np.unravel_index(np.argmax(rel), rel.shape)
    assert rel.max() <= tol, f"{what}: max rel diff {rel.max():.3e} at cell/bin {worst} (tol {tol})"
    # bins below the mask: must still be tiny
    small = ~mask
    if small.any():
        assert np.all(np.abs(rho_gpu[small]) <= 1e-29 * np.broadcast_to(tot, rho_ref.shape)[small] + 1e-300), what
    return rel.max()


def assert_rates_close(d_gpu, d_ref, gain, loss, tol=TOL_RATE, what=""):
    scale = gain + loss
    diff = np.abs(d_gpu - d_ref)
    bad = diff > tol * scale + RATE_ABS_FLOOR
    if bad.any():
        w = np.unravel_index(np.argmax(diff / np.where(scale > 0, scale, 1.0)), diff.shape)
        raise AssertionError(f"{what}: {bad.sum()} bins off; worst at {w}: gpu {d_gpu[w]:.17e} ref {d_ref[w]:.17e} "
                             f"gain+loss {scale[w]:.3e}")
    nz = scale > RATE_ABS_FLOOR / tol
    return float((diff[nz] / scale[nz]).max()) if nz.any() else 0.0


def assert_planes_strict(K_gpu, K_ref, what=""):
    """SURVEY 8(c) "rel. 1e-12 per entry", applied to each plane on its own: 1e-12 where p_coag and p_frag
    both exceed 1e-2, 1e-11 where they exceed 1e-3.  Eq. 55's K p_coag = K - K p_frag carries an ABSOLUTE
    error of a few u K_ij on either side, i.e. a relative one of a few u / p: the
    per-entry bar is only meaningful where p is not small, and elsewhere the bar is TOL_K * K_ij.
    K_*: [2, P].  Returns the number of entries checked at 1e-12."""
    Kt = K_ref[0] + K_ref[1]
    n = 0
    for pmin, tol in ((1e-2, TOL_K), (1e-3, 10 * TOL_K)):
        ok = (K_ref[0] > pmin * Kt) & (K_ref[1] > pmin * Kt)
        for plane in (0, 1):
            rel = np.abs(K_gpu[plane] - K_ref[plane])[ok] / K_ref[plane][ok]
            assert rel.size == 0 or rel.max() <= tol, \
                f"{what}: plane {plane} strict rel diff {rel.max():.3e} (p > {pmin})"
        n = n or int(ok.sum())
    return n


def strict_rate_scale(d, po, cfg):
    """The oracle's OWN gain + loss magnitudes (real p_coag, p_frag) and the bins where they are the valid
    scale of the on-the-fly rate comparison: those whose magnitude is at least 1e-3 of the split-free one
    (the pairs feeding them have effective probabilities above 1e-3, so Eq. 55's absolute error u K_ij is
    at most 1e3 u of the true terms)."""
    _, gain, loss = orc.rates_cells(*oracle_args(d), po, d.rho_dust)
    gfree, lfree = split_free_magnitudes(d, po, cfg)
    scale = gain + loss
    ok = (scale >= 1e-3 * (gfree + lfree)) & (scale > 0)
    return scale, ok
