"""Writes tests/golden/dt_manifest.json: the fixed step size of configs 2-5 (BASELINE.json gives
none).  Recipe: dt = 0.3 / lambda, lambda = max over
cells and over bins with rho_k > 1e-30 sum(rho) of D-_k / rho_k, where D-_k is the sum of the
negative contributions to bin k in the oracle's first rate evaluation; rounded to 3 digits.
Calls only oracle/ and the input generator.  Run:  python tests/golden/make_dt_manifest.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle as orc  # noqa: E402
from paper_2402_18471_b200 import synth_disc  # noqa: E402


def main():
    out = {"_about": "dt = 0.3/lambda from the oracle's first rate evaluation; see make_dt_manifest.py",
           "1": {"dt_s": 1.0 * synth_disc.YEAR, "source": "BASELINE.json config 1: dt = 1 yr"}}
    for idx in (2, 3, 4, 5):
        cfg = synth_disc.CONFIGS[idx]
        lam = 0.0
        chunk = 8000
        d = synth_disc.make_disc(idx)
        p = orc.Params(mu=cfg.mu, v_frag=cfg.v_frag, eta=cfg.eta, chi_im=cfg.chi_im, sigma_mol=cfg.sigma_mol)
        for c0 in range(0, d.n_cells, chunk):
            s = slice(c0, min(c0 + chunk, d.n_cells))
            _, _, loss = orc.rates_cells(d.n_bins, d.a_min, d.a_max, d.rho_m, d.T[s], d.rho_gas[s], d.Omega[s],
                                         d.alpha[s], d.v_R[s], d.v_Z[s], p, d.rho_dust[s])
            rho = d.rho_dust[s]
            mask = rho > 1e-30 * rho.sum(axis=1, keepdims=True)
            lam = max(lam, float(np.max(np.where(mask, loss / np.where(mask, rho, 1.0), 0.0))))
            print(idx, c0, lam, flush=True)
        dt = float(f"{0.3 / lam:.2e}")
        out[str(idx)] = {"dt_s": dt, "lambda_per_s": lam, "source": "0.3/lambda, 3 significant digits"}
    with open(os.path.join(ROOT, "tests", "golden", "dt_manifest.json"), "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")


if __name__ == "__main__":
    main()
