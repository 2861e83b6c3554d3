"""Seeded synthetic protoplanetary-disc inputs for the five BASELINE.json configs.

This module holds the INPUT RECIPE only: a power-law disc
(Sigma_g ~ R^-1, T ~ R^-1/2, Gaussian rho_gas(Z)), terminal-velocity dust drift/settling
velocities and seeded dust size distributions shaped like the paper's runs
(MRN start, dust-to-gas 0.01, alpha = 1e-3, v_frag = 100/1000 cm/s).
It contains none of the coagulation method's arithmetic (no collision kernel, no rates, no
integrator) and is the only module that both the oracle-side tests and the CUDA-side
binding/bench consume.  Neither `oracle/` nor `csrc/` imports it for arithmetic: they
receive plain arrays plus (n_bins, a_min, a_max, rho_m) and build their own mass grids.

All quantities CGS.  Layout of every [C x N] array: row-major, bin fastest,
cell index c = i_R * N_Z + j_Z.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Optional

import numpy as np

# Physical constants (CGS); values fixed in DESIGN.md reading G16.
K_B = 1.380649e-16
M_H = 1.6735575e-24
G_GRAV = 6.67430e-8
M_SUN = 1.98847e33
AU = 1.495978707e13
YEAR = 3.15576e7

SEED_BASE = 18471000


@dataclass(frozen=True)
class DiscConfig:
    """One BASELINE.json config (index 1..5)."""
    index: int
    n_r: int
    n_z: int
    n_bins: int
    a_min: float            # cm
    a_max: float            # cm
    r_in_au: float
    r_out_au: float
    v_frag: float           # cm/s
    alpha: float
    t0: float               # K at 1 AU
    dust: str               # "mrn" | "lognormal" | "bimodal" | "mix3"
    n_steps: int
    dt_years: Optional[float]   # None -> taken from tests/golden/dt_manifest.json
    rho_m: float = 1.67
    mu: float = 2.4
    eta: float = 11.0 / 6.0
    chi_im: float = 1.0
    sigma_mol: float = 2.0e-15
    tan_theta_max: float = 0.15
    dust_to_gas: float = 0.01
    sigma0: float = 1000.0  # g/cm^2 at 1 AU

    @property
    def n_cells(self) -> int:
        return self.n_r * self.n_z

    @property
    def n_pairs(self) -> int:
        return self.n_bins * (self.n_bins + 1) // 2

    @property
    def name(self) -> str:
        return f"cfg{self.index}_{self.n_r}x{self.n_z}x{self.n_bins}"


CONFIGS: Dict[int, DiscConfig] = {
    1: DiscConfig(1, 4, 8, 40, 1e-5, 1.0, 10.0, 20.0, 100.0, 1e-3, 150.0, "mrn", 1, 1.0),
    2: DiscConfig(2, 125, 64, 100, 1e-5, 10.0, 5.0, 100.0, 100.0, 1e-3, 150.0, "lognormal", 100, None),
    3: DiscConfig(3, 125, 64, 100, 1e-5, 10.0, 5.0, 100.0, 1000.0, 1e-4, 150.0, "bimodal", 100, None),
    4: DiscConfig(4, 250, 128, 150, 1e-5, 10.0, 5.0, 100.0, 100.0, 1e-3, 150.0, "mrn", 1000, None),
    5: DiscConfig(5, 500, 256, 200, 1e-6, 100.0, 5.0, 100.0, 500.0, 3e-3, 300.0, "mix3", 10, None),
}


@dataclass
class DiscInputs:
    cfg: DiscConfig
    # grid-of-sizes description handed to both sides (they build their own mass grids)
    n_bins: int
    a_min: float
    a_max: float
    rho_m: float
    # per cell [C]
    T: np.ndarray
    rho_gas: np.ndarray
    Omega: np.ndarray
    alpha: np.ndarray
    R: np.ndarray
    Z: np.ndarray
    # per (cell, bin) [C x N]
    v_R: np.ndarray
    v_Z: np.ndarray
    rho_dust: np.ndarray
    extras: dict = field(default_factory=dict)

    @property
    def n_cells(self) -> int:
        return self.T.shape[0]

    def subset(self, cells: np.ndarray) -> "DiscInputs":
        """Same inputs restricted to the given cell indices (used for sampled parity)."""
        cells = np.asarray(cells, dtype=np.int64)
        return DiscInputs(
            cfg=self.cfg, n_bins=self.n_bins, a_min=self.a_min, a_max=self.a_max, rho_m=self.rho_m,
            T=np.ascontiguousarray(self.T[cells]), rho_gas=np.ascontiguousarray(self.rho_gas[cells]),
            Omega=np.ascontiguousarray(self.Omega[cells]), alpha=np.ascontiguousarray(self.alpha[cells]),
            R=np.ascontiguousarray(self.R[cells]), Z=np.ascontiguousarray(self.Z[cells]),
            v_R=np.ascontiguousarray(self.v_R[cells]), v_Z=np.ascontiguousarray(self.v_Z[cells]),
            rho_dust=np.ascontiguousarray(self.rho_dust[cells]), extras=dict(self.extras),
        )


def size_bins(n_bins: int, a_min: float, a_max: float):
    """Bin edges and geometric-mean centres in grain radius, for placing the initial dust only."""
    k = np.arange(n_bins + 1, dtype=np.float64)
    a_e = a_min * (a_max / a_min) ** (k / n_bins)
    a_c = np.sqrt(a_e[:-1] * a_e[1:])
    return a_e, a_c


def _mrn_weights(a_e: np.ndarray, a_cut: float) -> np.ndarray:
    """MRN n(a) ~ a^-3.5: mass in a bin ~ a_hi^0.5 - a_lo^0.5 for bins entirely below a_cut, else 0."""
    w = np.sqrt(a_e[1:]) - np.sqrt(a_e[:-1])
    w = np.where(a_e[1:] <= a_cut * (1.0 + 1e-12), w, 0.0)
    return w / w.sum()


def _lognormal_weights(a_c: np.ndarray, a_peak, width_dex) -> np.ndarray:
    x = (np.log10(a_c) - np.log10(a_peak)) / width_dex
    w = np.exp(-0.5 * x * x)
    return w / w.sum(axis=-1, keepdims=True)


def make_disc(index: int, *, cells: Optional[np.ndarray] = None, seed: Optional[int] = None) -> DiscInputs:
    """Build config `index` (1..5).  `cells` restricts the OUTPUT to those cell indices, but the
    random stream is always drawn for the full grid in C order so a subset sees the same numbers
    as the full problem would."""
    cfg = CONFIGS[index]
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + index if seed is None else seed))
    n_r, n_z, nb = cfg.n_r, cfg.n_z, cfg.n_bins
    C = n_r * n_z

    # ---- grid (cells bounded by constant R and constant theta; Z = R tan(theta))
    r_e = cfg.r_in_au * (cfg.r_out_au / cfg.r_in_au) ** (np.arange(n_r + 1) / n_r) * AU
    r_c = np.sqrt(r_e[:-1] * r_e[1:])
    tan_e = cfg.tan_theta_max * np.arange(n_z + 1) / n_z
    tan_c = 0.5 * (tan_e[:-1] + tan_e[1:])
    R = np.repeat(r_c, n_z)
    Z = (r_c[:, None] * tan_c[None, :]).reshape(C)

    # ---- gas
    r_au = R / AU
    sigma_g = cfg.sigma0 / r_au
    T = cfg.t0 * r_au ** -0.5
    c_s = np.sqrt(K_B * T / (cfg.mu * M_H))
    omega_k = np.sqrt(G_GRAV * M_SUN / R ** 3)
    H = c_s / omega_k
    rho_mid = sigma_g / (np.sqrt(2.0 * np.pi) * H)
    rho_gas = rho_mid * np.exp(-0.5 * (Z / H) ** 2)
    Omega = np.sqrt(G_GRAV * M_SUN / (R * R + Z * Z) ** 1.5)
    alpha = np.full(C, cfg.alpha)

    # ---- sizes, Stokes numbers (Epstein) for the prescribed velocities only
    a_e, a_c = size_bins(nb, cfg.a_min, cfg.a_max)
    v_th = np.sqrt(8.0 / np.pi) * c_s
    St = cfg.rho_m * a_c[None, :] * Omega[:, None] / (rho_gas[:, None] * v_th[:, None])
    v_k = np.sqrt(G_GRAV * M_SUN / R)
    eta_vk = 0.5 * (c_s ** 2 / v_k) * 2.75
    fac = St / (1.0 + St * St)
    v_Z = -(Omega * Z)[:, None] * fac
    v_R = -2.0 * eta_vk[:, None] * fac

    # ---- dust
    St_mid = 0.5 * np.pi * cfg.rho_m * a_c[None, :] / sigma_g[:, None]

    def settled(weights_2d):
        """Column weights -> local densities with H_d = H sqrt(alpha/(alpha+St_mid))."""
        h_d = H[:, None] * np.sqrt(cfg.alpha / (cfg.alpha + St_mid))
        sig_d = cfg.dust_to_gas * sigma_g[:, None] * weights_2d
        return sig_d / (np.sqrt(2.0 * np.pi) * h_d) * np.exp(-0.5 * (Z[:, None] / h_d) ** 2)

    extras = {}
    if cfg.dust == "mrn":
        w = _mrn_weights(a_e, 1e-4)
        rho = cfg.dust_to_gas * rho_gas[:, None] * w[None, :]
    elif cfg.dust == "lognormal":
        w = _lognormal_weights(a_c, 1e-2, 1.0)
        rho = settled(np.broadcast_to(w, (C, nb)))
    elif cfg.dust == "bimodal":
        w = 0.5 * _mrn_weights(a_e, 1e-4) + 0.5 * _lognormal_weights(a_c, 1e-1, 0.5)
        rho = settled(np.broadcast_to(w, (C, nb)))
    elif cfg.dust == "mix3":
        peaks = 10.0 ** rng.uniform(-4.0, 0.0, size=(C, 3))
        wts = rng.uniform(size=(C, 3))
        wts /= wts.sum(axis=1, keepdims=True)
        w = np.zeros((C, nb))
        for s in range(3):
            w += wts[:, s:s + 1] * _lognormal_weights(a_c[None, :], peaks[:, s:s + 1], 0.3)
        rho = cfg.dust_to_gas * rho_gas[:, None] * w
        extras["peaks"] = peaks
    else:  # pragma: no cover
        raise ValueError(cfg.dust)
    jitter = np.exp(0.1 * rng.standard_normal(size=(C, nb)))
    rho = np.ascontiguousarray(rho * jitter)

    out = DiscInputs(cfg=cfg, n_bins=nb, a_min=cfg.a_min, a_max=cfg.a_max, rho_m=cfg.rho_m,
                     T=T, rho_gas=rho_gas, Omega=Omega, alpha=alpha, R=R, Z=Z,
                     v_R=np.ascontiguousarray(v_R), v_Z=np.ascontiguousarray(v_Z),
                     rho_dust=rho, extras=extras)
    if cells is not None:
        out = out.subset(cells)
    return out


def sample_cells(cfg: DiscConfig, n: int, seed: int = 7) -> np.ndarray:
    """Deterministic spread of cell indices covering mid-plane, surface, inner and outer disc."""
    C = cfg.n_cells
    if n >= C:
        return np.arange(C, dtype=np.int64)
    rng = np.random.Generator(np.random.PCG64(seed + cfg.index))
    fixed = np.array([0, cfg.n_z - 1, C - cfg.n_z, C - 1, C // 2], dtype=np.int64)
    rest = rng.choice(C, size=max(n - fixed.size, 0), replace=False)
    return np.unique(np.concatenate([fixed, rest]))[:n]


# ------------------------------------------------------------------------------------------ Fig. 10 set-up
@dataclass
class Fig10Inputs:
    """Single-radius, vertically integrated coagulation test of PAPER.md:482-491 (Fig. 10): one cell per
    alpha value at R = 20 AU.  rho_dust holds dust SURFACE densities (g/cm^2), h_dust the dust scale
    heights, v_Z the terminal settling velocities at Z = h_i, rho_gas the mid-plane gas density."""
    n_bins: int
    a_min: float
    a_max: float
    rho_m: float
    mu: float
    v_frag: float
    T: np.ndarray
    rho_gas: np.ndarray
    Omega: np.ndarray
    alpha: np.ndarray
    sigma_g: np.ndarray
    c_s: np.ndarray
    v_R: np.ndarray
    v_Z: np.ndarray
    h_dust: np.ndarray
    rho_dust: np.ndarray
    a_frag: np.ndarray      # (2 / 3 pi) Sigma_g / (rho_m alpha) (v_frag / c_s)^2, the fragmentation limit

    @property
    def n_cells(self) -> int:
        return self.T.shape[0]


def make_fig10(alphas=(1e-3, 1e-4), n_bins: int = 200, a_min: float = 1e-5, a_max: float = 10.0,
               r_au: float = 20.0, T0: float = 36.0, mu: float = 2.4, v_frag: float = 100.0,
               sigma0: float = 1000.0, rho_m: float = 1.67, dust_to_gas: float = 0.01) -> Fig10Inputs:
    """PAPER.md:482-491 gives R = 20 AU, T = 36 K, mu = 2.4, alpha = 1e-3, v_frag = 100 cm/s, 200 species;
    it does not give Sigma_g, the size range or the initial condition: Sigma_g = 1000 (R/AU)^-1 g/cm^2 (the
    recipe of the five configs), 0.1 um - 10 cm, MRN up to 1 um with dust-to-gas 0.01 (R19).  A
    second cell with alpha = 1e-4 moves the fragmentation limit by a factor 10 (scaling check)."""
    alphas = np.asarray(alphas, dtype=np.float64)
    C = alphas.size
    R = r_au * AU
    T = np.full(C, T0)
    c_s = np.sqrt(K_B * T / (mu * M_H))
    Om = np.full(C, np.sqrt(G_GRAV * M_SUN / R ** 3))
    H = c_s / Om
    sigma_g = np.full(C, sigma0 / r_au)
    rho_mid = sigma_g / (np.sqrt(2.0 * np.pi) * H)
    a_e, a_c = size_bins(n_bins, a_min, a_max)
    St = 0.5 * np.pi * rho_m * a_c[None, :] / sigma_g[:, None]                 # mid-plane, Epstein
    h = H[:, None] * np.sqrt(alphas[:, None] / (alphas[:, None] + St))
    fac = St / (1.0 + St * St)
    v_Z = -(Om[:, None] * h) * fac                                             # terminal settling at Z = h_i
    v_k = np.sqrt(G_GRAV * M_SUN / R)
    v_R = -2.0 * (0.5 * (c_s ** 2 / v_k) * 2.75)[:, None] * fac
    w = _mrn_weights(a_e, 1e-4)
    sig_d = dust_to_gas * sigma_g[:, None] * w[None, :]
    a_frag = (2.0 / (3.0 * np.pi)) * sigma_g / (rho_m * alphas) * (v_frag / c_s) ** 2
    return Fig10Inputs(n_bins=n_bins, a_min=a_min, a_max=a_max, rho_m=rho_m, mu=mu, v_frag=v_frag, T=T,
                       rho_gas=rho_mid, Omega=Om, alpha=alphas, sigma_g=sigma_g, c_s=c_s,
                       v_R=np.ascontiguousarray(v_R), v_Z=np.ascontiguousarray(v_Z),
                       h_dust=np.ascontiguousarray(h), rho_dust=np.ascontiguousarray(sig_d), a_frag=a_frag)
