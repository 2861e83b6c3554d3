#!/usr/bin/env python
"""bench.py -- cudisc_coag_step throughput on a synthetic disc shaped like the paper's runs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

One "step" = one Bogacki-Shampine 3(2) step of EVERY cell of the workload through
the C ABI (cudisc_coag_step): per cell the collision kernel is built on the fly (Eqs. 55-62) and
three rate evaluations (Eqs. 53, 54, 61-68; FSAL) are run -- all of SURVEY.md section 8(a) in one
kernel launch.  Workload: BASELINE.json config 4 (250 x 128 cells, 150 bins), the configuration the
north_star's roofline target is quoted on.  Prints ONE JSON line (rank 0).

  value        cell-updates/s, inputs resident in HBM, CUDA events around each step's launch on the
               launching stream, L2 flushed between timed steps, max over ranks
  e2e          same metric through cudisc_coag_step_host: pinned HOST buffers, H2D + step + D2H
               inside the timed region
  roofline     "alu": algorithmic FP64 instructions / launch duration against
               148 SMs x 64 FP64 lanes x max SM clock; the DFMA rate measured by the library's
               microbenchmark in the same process is reported beside it
  cpu_baseline the oracle (oracle/coag_oracle.c, as it stands) on the host cores, bounded sample

--impl reference times the oracle itself (there is no reference code: PAPER.md is a paper).
--gpus N > 1 (under torchrun): N independent replicas of the workload ("replicas
only"; cells are independent, the path has no exchange step), value = all cells / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

# Algorithmic FP64 instruction counts of the minimal pair formulas (an FMA,
# add, mul or max each count 1; per-bin hoistable terms excluded).
I_BUILD = 41      # per pair, once per step: Eqs. 56-62 on a log grid (FP64-pipe instructions of pair_kernel)
I_EVAL = 6        # per pair per rate evaluation: 4 row-sum + 2 column-sum FMAs
F_BUILD = 58      # the same formulas counted in flops (FMA = 2, add / mul = 1): 17 FMAs + 24 others
F_EVAL = 12
EVALS_PER_STEP = 3
FP64_LANES_PER_SM = 64
METRIC = "coagulation cell-updates/sec (FP64 BS3(2) step, kernel built on the fly)"


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def load_dt(index: int) -> float:
    with open(os.path.join(ROOT, "tests", "golden", "dt_manifest.json")) as f:
        return float(json.load(f)[str(index)]["dt_s"])


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU while the timed region runs (NVML)."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, torch_device_index: int, period_s: float = 0.01):
        self.period = period_s
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self._h = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self._nv = pynvml
            try:
                uuid = str(torch.cuda.get_device_properties(torch_device_index).uuid)
                if not uuid.startswith("GPU-"):
                    uuid = "GPU-" + uuid
                self._h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode())
            except Exception:
                self._h = pynvml.nvmlDeviceGetHandleByIndex(torch_device_index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception as exc:  # pragma: no cover
            self.error = repr(exc)

    def _once(self):
        nv = self._nv
        self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
        try:
            mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
        except Exception:
            mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
        for bit, name in self.REASONS.items():
            if mask & bit:
                self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._once()
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self._h is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr is not None:
            self._stop.set()
            self._thr.join()
            self._thr = None
            self._stop = threading.Event()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(statistics.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "sm_mhz_min": min(self.samples), "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------ oracle legs
def oracle_step_rate(index: int, budget_s: float, warmup: int = 0, steps: int = 1):
    """Times the oracle's BS3(2) step (kernel build + 4 rate evaluations on the first step, as it
    stands) on a bounded sample of config `index`.  Returns (cell-updates/s, info dict)."""
    import oracle as orc
    from paper_2402_18471_b200 import synth_disc
    cfg = synth_disc.CONFIGS[index]
    threads = orc.num_threads()
    po = orc.Params(mu=cfg.mu, v_frag=cfg.v_frag, eta=cfg.eta, chi_im=cfg.chi_im, sigma_mol=cfg.sigma_mol)
    dt = load_dt(index)

    def run(cells, k1=None, rho=None):
        d = run.cache.get(len(cells))
        if d is None:
            d = synth_disc.make_disc(index, cells=cells)
            run.cache[len(cells)] = d
        r = d.rho_dust if rho is None else rho
        t0 = time.perf_counter()
        rho_new, k4, _ = orc.step_cells(d.n_bins, d.a_min, d.a_max, d.rho_m, d.T, d.rho_gas, d.Omega, d.alpha,
                                        d.v_R, d.v_Z, po, r, dt, k1=k1)
        return time.perf_counter() - t0, rho_new, k4
    run.cache = {}

    probe_cells = synth_disc.sample_cells(cfg, min(cfg.n_cells, max(2 * threads, 8)))
    t_probe, _, _ = run(probe_cells)
    per_cell = t_probe / len(probe_cells)
    n = int(min(cfg.n_cells, max(len(probe_cells), budget_s / max(per_cell, 1e-9) / max(steps + warmup, 1))))
    cells = synth_disc.sample_cells(cfg, n)
    rho, k1 = None, None
    for _ in range(warmup):
        _, rho, k1 = run(cells, k1, rho)
    times = []
    for _ in range(steps):
        t, rho, k1 = run(cells, k1, rho)
        times.append(t)
    total = sum(times)
    rate = len(cells) * steps / total
    info = {"cores": threads, "kind": "oracle",
            "sample": f"{len(cells)} of {cfg.n_cells} cells of config {index} ({cfg.n_bins} bins), "
                      f"{steps} step(s) of oracle orc_step_cells (OpenMP over cells) after {warmup} untimed "
                      f"step(s) ({'FSAL: 3' if warmup else 'first step: 4'} rate evaluations per step), {total:.1f} s"}
    return rate, info, total / steps


def run_reference(args):
    rank = env_int("RANK", 0)
    if rank != 0:
        return 0
    from paper_2402_18471_b200 import synth_disc
    cfg = synth_disc.CONFIGS[args.config]
    rate, info, s_per_step = oracle_step_rate(args.config, budget_s=90.0, warmup=args.warmup, steps=args.steps)
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": "cell-updates/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * s_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, args),
        "pair_evals_per_s": rate * EVALS_PER_STEP * cfg.n_pairs,
        "cpu_baseline": {"value": rate, "unit": "cell-updates/s", **info},
        "e2e": {"value": rate, "unit": "cell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_config(cfg, args):
    return {"workload": f"BASELINE.json config {cfg.index}: {cfg.n_r}x{cfg.n_z} cells, {cfg.n_bins} bins "
                        f"({cfg.a_min:g}-{cfg.a_max:g} cm), v_frag={cfg.v_frag:g} cm/s, alpha={cfg.alpha:g}, "
                        f"dust={cfg.dust}, fixed dt from tests/golden/dt_manifest.json",
            "n_cells": cfg.n_cells, "n_bins": cfg.n_bins, "pairs_per_cell": cfg.n_pairs,
            "rate_evals_per_step": EVALS_PER_STEP,
            "l2": "flushed between timed steps (256 MiB memset outside the event pair)",
            "parallelism": f"replicas x{args.gpus}" if args.gpus > 1 else "single GPU"}


# ------------------------------------------------------------------------------------------ ours
def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2402_18471_b200 as cd
    from paper_2402_18471_b200 import synth_disc
    from paper_2402_18471_b200.replicas import max_over_ranks, replica_seed

    rank, world, local = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cd.lib()

    cfg = synth_disc.CONFIGS[args.config]
    d = synth_disc.make_disc(args.config, seed=replica_seed(synth_disc.SEED_BASE + args.config, rank))
    C, N, P = d.n_cells, d.n_bins, cfg.n_pairs
    pc = cd.Params(mu=cfg.mu, v_frag=cfg.v_frag, alpha=cfg.alpha, eta=cfg.eta, chi_im=cfg.chi_im,
                   sigma_mol=cfg.sigma_mol)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    gas = dict(T=t(d.T), rho_gas=t(d.rho_gas), Omega=t(d.Omega), v_R=t(d.v_R), v_Z=t(d.v_Z), alpha=t(d.alpha))
    bins = cd.Bins(N, d.a_min, d.a_max, d.rho_m, pc)
    grid = cd.Grid(cfg.n_r, cfg.n_z, bins)
    grid.bind_gas(**gas)
    dt = load_dt(args.config)
    rho = t(d.rho_dust)
    err = torch.empty(C, dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    # roofline denominators measured in this process (north_star)
    dfma_per_s, _ = cd.cudisc_microbench_dfma(0)
    copy_bps, _ = cd.cudisc_microbench_copy(1 << 30)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing
    for _ in range(args.warmup):
        cd.cudisc_coag_step(grid, bins, rho, dt, err)
    sampler = ClockSampler(local)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    n0 = cd.cudisc_launch_count()
    sampler.start()
    t_wall0 = time.perf_counter()
    for e0, e1 in ev:
        flush.zero_()
        e0.record(stream)
        cd.cudisc_coag_step(grid, bins, rho, dt, err)
        e1.record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    sampler.stop()
    launches = cd.cudisc_launch_count() - n0
    step_ms = [e0.elapsed_time(e1) for e0, e1 in ev]
    total_s = max_over_ranks(sum(step_ms) * 1e-3, world, dev)
    mass0 = float(t(d.rho_dust).sum())
    mass_drift = abs(float(rho.sum()) - mass0) / mass0
    err_max = float(err.max())

    # ---- end to end: pinned host buffers through cudisc_coag_step_host
    rho_h = torch.from_numpy(np.ascontiguousarray(d.rho_dust)).pin_memory()
    err_h = torch.empty(C, dtype=torch.float64).pin_memory()
    grid.reset_fsal()
    for _ in range(max(1, min(args.warmup, 3))):
        cd.cudisc_coag_step_host(grid, bins, rho_h, dt, err_h)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        cd.cudisc_coag_step_host(grid, bins, rho_h, dt, err_h)
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0, world, dev)

    if rank == 0:
        ms = 1e3 * total_s / args.steps
        value = world * C * args.steps / total_s
        alg_instr = float(C) * P * (I_BUILD + EVALS_PER_STEP * I_EVAL)
        kernel_s = statistics.mean(step_ms) * 1e-3
        clocks = sampler.summary()
        sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
        max_mhz = clocks.get("sm_max_mhz") or 1965
        peak_tflops = 2.0 * sm_count * FP64_LANES_PER_SM * max_mhz * 1e6 / 1e12
        achieved_tflops = 2.0 * alg_instr / kernel_s / 1e12
        line = {
            "metric": METRIC, "value": value, "unit": "cell-updates/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args),
            "pair_evals_per_s": value * EVALS_PER_STEP * P,
            "wall_s_timed_region": t_wall,
            "mass_drift_rel": mass_drift, "err_norm_max_last_step": err_max,
            "clocks": clocks,
            "e2e": {"value": world * C * args.steps / e2e_s, "unit": "cell-updates/s",
                    "h2d_bytes_per_step": C * N * 8, "d2h_bytes_per_step": C * N * 8 + C * 8,
                    "ms_per_step": 1e3 * e2e_s / args.steps,
                    "api": "cudisc_coag_step_host (pinned host buffers)"},
            "gpu_launches": int(launches),
            "roofline": {
                "bound": "alu",
                "kernel": "cudisc::coag_v3_kernel<512, MODE_STEP>" if bins.fast_path()[0] else
                          "cudisc::coag_cells_kernel<512, MODE_STEP, SLAB, false>",
                "achieved": achieved_tflops, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved_tflops / peak_tflops,
                # dram__bytes_read.sum + dram__bytes_write.sum of one launch (ncu --set full), profiles/r02_kernels.md
                "traffic": 193767936 if (args.config == 4 and world == 1) else
                           (1226387200 if (args.config == 5 and world == 1) else None),
                "how": f"algorithmic FP64 instructions per launch = C*P*({I_BUILD} + {EVALS_PER_STEP}*{I_EVAL}) "
                       f"= {alg_instr:.4g} (DESIGN.md 'Roofline'), x2 flop per FP64 issue slot, / mean CUDA-event "
                       f"launch duration {1e3 * kernel_s:.3f} ms; peak = {sm_count} SMs x {FP64_LANES_PER_SM} "
                       f"FP64 lanes x {max_mhz} MHz x 2 (derived from unit counts and max clock, not measured)",
                "peak_measured_dfma_tflops": 2.0 * dfma_per_s / 1e12,
                "frac_of_measured_dfma": achieved_tflops / (2.0 * dfma_per_s / 1e12),
                "hbm_copy_measured_gbs": copy_bps / 1e9,
                "hbm_algorithmic_gbs": (6.0 * C * N * 8 + 5.0 * C * 8) / kernel_s / 1e9,
                "note": "the FP64 pipe is the roofline BASELINE.json names; frac is the share of FP64 issue slots the "
                        "algorithmic instructions would need, not a FLOP/s claim.  ncu (profiles/r02_kernels.md): the "
                        "kernel is latency-bound (16 warps per SM, issue slots 53 %, FP64 pipe 31 %, shared-memory pipe "
                        "58 %), see DESIGN.md 'Roofline'",
            },
        }
        if world == 1 and not args.no_cpu_baseline:
            rate, info, _ = oracle_step_rate(args.config, budget_s=20.0, warmup=1, steps=1)   # a FSAL step, like the GPU's
            line["cpu_baseline"] = {"value": rate, "unit": "cell-updates/s", **info}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def measured_peaks():
    """MEASURED_PEAKS.json (driver-written) if present: HBM copy GB/s of this pool's B200s."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


def run_hydro(args, dev):
    """--entry hydro: cudisc_hydrostatic (Eqs. 32-37) on a grid large enough to leave the L2
    (4096 x 1024 cells: 32 MiB read + 32 MiB written per launch); HBM-bound, 16 B per cell."""
    import torch

    import paper_2402_18471_b200 as cd
    from paper_2402_18471_b200 import synth_disc as sd
    n_r, n_z = 4096, 1024
    R_e = 1.0 * sd.AU * 200.0 ** (np.arange(n_r + 1) / n_r)
    R_c = np.sqrt(R_e[:-1] * R_e[1:])
    tan_e = 0.3 * np.arange(n_z + 1) / n_z
    tan_c = 0.5 * (tan_e[:-1] + tan_e[1:])
    T = 150.0 * (R_c[:, None] / sd.AU) ** -0.5 * (1.0 + 3.0 * (tan_c[None, :] / 0.3) ** 2)
    cs2 = torch.from_numpy(np.ascontiguousarray(sd.K_B * T / (2.4 * sd.M_H))).to(dev)
    Sigma = torch.from_numpy(1000.0 * (R_c / sd.AU) ** -1.0).to(dev)
    out = torch.empty_like(cs2)
    h = cd.Hydro(R_e, tan_e, R_c, tan_c)
    GM = sd.G_GRAV * sd.M_SUN
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    copy_bps, _ = cd.cudisc_microbench_copy(1 << 30)
    peaks = measured_peaks()
    hbm_peak = float(peaks.get("hbm_gbs") or copy_bps / 1e9)
    n0 = cd.cudisc_launch_count()
    for _ in range(args.warmup):
        cd.cudisc_hydrostatic(h, cs2, Sigma, GM, out)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    torch.cuda.synchronize()
    for e0, e1 in ev:
        flush.zero_()
        e0.record(stream)
        cd.cudisc_hydrostatic(h, cs2, Sigma, GM, out)
        e1.record(stream)
    torch.cuda.synchronize()
    sec = statistics.mean(e0.elapsed_time(e1) for e0, e1 in ev) * 1e-3
    gbs = 16.0 * n_r * n_z / sec / 1e9
    print(json.dumps({"entry": "hydro", "metric": "hydrostatic-equilibrium cells/s (cudisc_hydrostatic)",
                      "value": n_r * n_z / sec, "unit": "cells/s", "ms_per_launch": 1e3 * sec, "dtype": "f64",
                      "data": "synthetic", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
                      "config": {"workload": f"{n_r} x {n_z} cells, warm-surface temperature structure",
                                 "l2": "flushed between timed launches"},
                      "gpu_launches": int(cd.cudisc_launch_count() - n0),
                      "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                                   "frac": gbs / hbm_peak, "traffic": None,
                                   "how": "16 B per cell (c_s^2 read, rho_g written) / mean CUDA-event launch duration",
                                   "hbm_copy_measured_gbs": copy_bps / 1e9}}), flush=True)
    return 0


def run_entry(args):
    """--entry kernel | rates | step_cached | integrate: the other C-ABI entry points on the same workload
    (config 4 by default), each against its own roof: FP64 issue slots for `kernel`, HBM
    for `rates` / `step_cached` (16 B per pair read); `integrate` = BASELINE.json config 4 as stated
    (1000 accepted adaptive steps: time to solution and mass drift)."""
    import torch

    import paper_2402_18471_b200 as cd
    from paper_2402_18471_b200 import synth_disc

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    dev = torch.device("cuda", env_int("LOCAL_RANK", 0))
    torch.cuda.set_device(dev)
    if args.entry == "hydro":
        return run_hydro(args, dev)
    cfg = synth_disc.CONFIGS[args.config]
    full = args.entry == "integrate"
    n_cells = cfg.n_cells if full else min(cfg.n_cells, args.cells)
    cells = None if n_cells == cfg.n_cells else np.arange(n_cells)        # the first n_cells cells of the grid
    d = synth_disc.make_disc(args.config, cells=cells)
    C, N, P = d.n_cells, d.n_bins, cfg.n_pairs
    pc = cd.Params(mu=cfg.mu, v_frag=cfg.v_frag, alpha=cfg.alpha, eta=cfg.eta, chi_im=cfg.chi_im,
                   sigma_mol=cfg.sigma_mol)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    gas = dict(T=t(d.T), rho_gas=t(d.rho_gas), Omega=t(d.Omega), v_R=t(d.v_R), v_Z=t(d.v_Z), alpha=t(d.alpha))
    bins = cd.Bins(N, d.a_min, d.a_max, d.rho_m, pc)
    grid = cd.Grid(cfg.n_r, cfg.n_z, bins) if full else cd.Grid(C, 1, bins)
    grid.bind_gas(**gas)
    dt = load_dt(args.config)
    rho = t(d.rho_dust)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    dfma_per_s, _ = cd.cudisc_microbench_dfma(0)
    copy_bps, _ = cd.cudisc_microbench_copy(1 << 30)
    peaks = measured_peaks()
    hbm_peak = float(peaks.get("hbm_gbs") or copy_bps / 1e9)
    hbm_src = "MEASURED_PEAKS.json hbm_gbs" if peaks.get("hbm_gbs") else "in-process copy microbenchmark"
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    sampler = ClockSampler(dev.index or 0)
    n0 = cd.cudisc_launch_count()
    base = {"entry": args.entry, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "dtype": "f64",
            "data": "synthetic", "higher_is_better": True, "vs_baseline": None,
            "config": {"workload": f"BASELINE.json config {cfg.index}: {C} of {cfg.n_cells} cells, {N} bins",
                       "n_cells": C, "n_bins": N, "pairs_per_cell": P,
                       "l2": "flushed between timed launches (256 MiB memset outside the event pair)"}}

    if args.entry == "integrate":
        m0 = rho.sum(dim=1)
        torch.cuda.synchronize()
        sampler.start()
        t0 = time.perf_counter()
        info, log = cd.cudisc_coag_integrate_steps(grid, bins, rho, args.accepted, dt, max_steps=4 * args.accepted)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        sampler.stop()
        drift = float(((rho.sum(dim=1) - m0).abs() / m0).max())
        line = dict(base, metric="time to solution of 1000 accepted adaptive BS3(2) steps (cudisc_coag_integrate)",
                    value=wall, unit="s", higher_is_better=False,
                    n_accepted=info["n_accepted"], n_rejected=info["n_rejected"], t_done_s=info["t_done"],
                    dt_last_s=info["dt_last"], mass_drift_rel_max=drift,
                    mass_drift_per_accepted_step=drift / max(info["n_accepted"], 1),
                    cell_updates_per_s=C * (info["n_accepted"] + info["n_rejected"]) / wall,
                    min_rho=float(rho.min()), clocks=sampler.summary(),
                    gpu_launches=int(cd.cudisc_launch_count() - n0))
        print(json.dumps(line), flush=True)
        return 0

    K = torch.empty((C, 2, P), dtype=torch.float64, device=dev)
    cd.cudisc_coag_kernel(grid, bins, gas, pc, K)
    out = torch.empty_like(rho)
    err = torch.empty(C, dtype=torch.float64, device=dev)

    def launch():
        if args.entry == "kernel":
            cd.cudisc_coag_kernel(grid, bins, gas, pc, K)
        elif args.entry == "rates":
            cd.cudisc_coag_rates(grid, bins, K, rho, out)
        else:
            cd.cudisc_coag_step_cached(grid, bins, K, rho, dt, err)

    for _ in range(args.warmup):
        launch()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    torch.cuda.synchronize()
    sampler.start()
    for e0, e1 in ev:
        flush.zero_()
        e0.record(stream)
        launch()
        e1.record(stream)
    torch.cuda.synchronize()
    sampler.stop()
    sec = statistics.mean(e0.elapsed_time(e1) for e0, e1 in ev) * 1e-3
    fast = bool(bins.fast_path()[0])          # the mass grid takes the stencil kernel (coag_v3.cu)
    pairs = float(C) * P
    evals = {"kernel": 0, "rates": 1, "step_cached": EVALS_PER_STEP}[args.entry]
    hbm_bytes = 16.0 * pairs + (2 if args.entry == "rates" else 6 if args.entry == "step_cached" else 0) * 8.0 * C * N
    gbs = hbm_bytes / sec / 1e9
    alu_instr = pairs * (I_BUILD if args.entry == "kernel" else evals * I_EVAL)
    alu_frac = alu_instr / sec / (sm_count * FP64_LANES_PER_SM * (sampler.summary().get("sm_max_mhz") or 1965) * 1e6)
    hbm_frac = gbs / hbm_peak
    bound = "alu" if (args.entry == "kernel" and alu_frac > hbm_frac) else "hbm"
    line = dict(base, metric={"kernel": "kernel pairs/s (cudisc_coag_kernel, K written to HBM)",
                              "rates": "rate-evaluation pairs/s (cudisc_coag_rates, K read from HBM)",
                              "step_cached": "cell-updates/s (cudisc_coag_step_cached, K read from HBM)"}[args.entry],
                value=(C / sec) if args.entry == "step_cached" else pairs * max(evals, 1) / sec,
                unit="cell-updates/s" if args.entry == "step_cached" else "pairs/s", ms_per_launch=1e3 * sec,
                clocks=sampler.summary(), gpu_launches=int(cd.cudisc_launch_count() - n0),
                roofline={"bound": bound,
                          "achieved": gbs if bound == "hbm" else 2.0 * alu_instr / sec / 1e12,
                          "peak": hbm_peak if bound == "hbm" else 2.0 * sm_count * FP64_LANES_PER_SM * 1965e6 / 1e12,
                          "unit": "GB/s" if bound == "hbm" else "TFLOP/s",
                          "frac": hbm_frac if bound == "hbm" else alu_frac,
                          # dram__bytes_read.sum + dram__bytes_write.sum of one launch (ncu --set full, profiles/
                          # r02_kernels.md sections 3 - 5), for the profiled workload (config 4, 16000 cells) only
                          "traffic": ({"kernel": 2897776856, "rates": 2940610528, "step_cached": 2979018016}[args.entry]
                                      if (args.config == 4 and C == 16000 and fast) else None),
                          "kernel": ("cudisc::coag_v3_kernel<512, MODE_%s>"
                                     % {"kernel": "KERNEL", "rates": "RATES", "step_cached": "STEPK"}[args.entry]
                                     if fast else "cudisc::coag_cells_kernel<512, MODE, SLAB, false>"),
                          "hbm_gbs": gbs, "hbm_frac": hbm_frac, "alu_frac": alu_frac,
                          "how": f"algorithmic HBM bytes per launch = 16 B x {pairs:.4g} pairs (+ the [C x N] arrays) "
                                 f"= {hbm_bytes:.4g} / mean CUDA-event launch duration {1e3 * sec:.3f} ms; HBM peak "
                                 f"{hbm_peak:.0f} GB/s from {hbm_src}; alu_frac = FP64 instructions of the minimal "
                                 f"formulas / (SMs x 64 lanes x max clock)",
                          "hbm_copy_measured_gbs": copy_bps / 1e9,
                          "peak_measured_dfma_tflops": 2.0 * dfma_per_s / 1e12})
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--entry", choices=["step", "kernel", "rates", "step_cached", "integrate", "hydro"], default="step",
                    help="C-ABI entry point to time (default: cudisc_coag_step, the contract line)")
    ap.add_argument("--cells", type=int, default=16000, help="cells of the workload for --entry kernel/rates/step_cached")
    ap.add_argument("--accepted", type=int, default=1000, help="accepted steps of --entry integrate")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.entry != "step":
        return run_entry(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
