"""ctypes front end of the CPU oracle (oracle/coag_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2402_18471_b200 (the CUDA path) and the
CUDA path imports nothing from here.

The C file is compiled on first use with plain gcc (-O2, no fast-math, no FP contraction,
OpenMP over cells only) into oracle/_build/liboracle.so.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading
from dataclasses import dataclass
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "coag_oracle.c"
_SRC2 = _HERE / "hydro_oracle.c"
_LIB = _HERE / "_build" / "liboracle.so"
_lock = threading.Lock()
_lib = None

c_dp = C.POINTER(C.c_double)


class OrcParams(C.Structure):
    _fields_ = [("mu", C.c_double), ("v_frag", C.c_double), ("eta", C.c_double),
                ("chi_im", C.c_double), ("sigma_mol", C.c_double), ("rtol", C.c_double),
                ("atol_factor", C.c_double)]


@dataclass
class Params:
    mu: float = 2.4
    v_frag: float = 100.0
    eta: float = 11.0 / 6.0
    chi_im: float = 1.0
    sigma_mol: float = 2.0e-15
    rtol: float = 1e-2
    atol_factor: float = 1e-10

    def c(self) -> OrcParams:
        return OrcParams(self.mu, self.v_frag, self.eta, self.chi_im, self.sigma_mol, self.rtol,
                         self.atol_factor)


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc.  Building the checker is not using it."""
    with _lock:
        if force or not _LIB.exists() or _LIB.stat().st_mtime < max(_SRC.stat().st_mtime, _SRC2.stat().st_mtime):
            _LIB.parent.mkdir(exist_ok=True)
            tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
            cmd = ["gcc", "-O2", "-std=gnu11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                   "-o", str(tmp), str(_SRC), str(_SRC2), "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.orc_pfrag.restype = C.c_double
        L.orc_pfrag.argtypes = [C.c_double, C.c_double]
        L.orc_ystar.restype = C.c_double
        L.orc_ystar.argtypes = [C.c_double]
        L.orc_ststar.restype = C.c_double
        L.orc_ststar.argtypes = [C.c_double, C.c_double]
        L.orc_vrel2_turb.restype = C.c_double
        L.orc_vrel2_turb.argtypes = [C.c_double] * 4
        L.orc_split.restype = C.c_int
        L.orc_lbin.restype = C.c_int
        L.orc_bs32_step.restype = C.c_double
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(c_dp)


def _in(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


# ------------------------------------------------------------------------------------------ grid
@dataclass
class MassGrid:
    N: int
    a_e: np.ndarray
    m_e: np.ndarray
    a_c: np.ndarray
    m_c: np.ndarray
    rho_m: float
    a_min: float
    a_max: float


def mass_grid(N: int, a_min: float, a_max: float, rho_m: float) -> MassGrid:
    a_e = np.empty(N + 1); m_e = np.empty(N + 1); a_c = np.empty(N); m_c = np.empty(N)
    lib().orc_mass_grid(C.c_int(N), C.c_double(a_min), C.c_double(a_max), C.c_double(rho_m),
                        _p(a_e), _p(m_e), _p(a_c), _p(m_c))
    return MassGrid(N, a_e, m_e, a_c, m_c, rho_m, a_min, a_max)


def grid_from_masses(m_c, m_e) -> MassGrid:
    """A MassGrid with arbitrary (monotone) centres/edges for the single-cell functions."""
    m_c = _in(m_c); m_e = _in(m_e)
    N = m_c.size
    return MassGrid(N, np.zeros(N + 1), m_e, np.zeros(N), m_c, 0.0, 0.0, 0.0)


# ------------------------------------------------------------------------------------------ scalars
def pfrag(v_frag: float, dv: float) -> float:
    return float(lib().orc_pfrag(v_frag, dv))


def ystar(St: float) -> float:
    return float(lib().orc_ystar(St))


def ststar(St: float, St_eta: float) -> float:
    return float(lib().orc_ststar(St, St_eta))


def vrel2_turb(St1: float, St2: float, S: float, St_eta: float) -> float:
    return float(lib().orc_vrel2_turb(St1, St2, S, St_eta))


VAR_NUMBER_SPLIT, VAR_TOTAL_LOOKUP = 1, 2


def set_variant(v: int) -> None:
    """Switches the two unpinned readings for the whole oracle (coag_oracle.c, orc_set_variant): bit 0 =
    number-conserving two-bin split (G11), bit 1 = fragment l-bin looked up with the total fragment mass (G2)."""
    lib().orc_set_variant(C.c_int(int(v)))


def split(g: MassGrid, m: float):
    eps = C.c_double()
    l = lib().orc_split(C.c_int(g.N), _p(g.m_c), C.c_double(m), C.byref(eps))
    return int(l), float(eps.value)


def lbin(g: MassGrid, m: float) -> int:
    return int(lib().orc_lbin(C.c_int(g.N), _p(g.m_e), C.c_double(m)))


# ------------------------------------------------------------------------------------------ one cell
def cell_kernel(g: MassGrid, T, rho_g, Omega, alpha, vR, vZ, p: Params, vphi=None):
    """Returns K[N,N], p_frag[N,N], St[N], Ststar[N] of one cell (Eqs. 55-62)."""
    N = g.N
    K = np.empty((N, N)); pf = np.empty((N, N)); St = np.empty(N); Ss = np.empty(N)
    vR = _in(vR); vZ = _in(vZ)
    vp = _p(_in(vphi)) if vphi is not None else None
    cp = p.c()
    lib().orc_cell_kernel(C.c_int(N), _p(g.a_c), _p(g.m_c), C.c_double(g.rho_m), C.c_double(T),
                          C.c_double(rho_g), C.c_double(Omega), C.c_double(alpha), _p(vR), _p(vZ), vp,
                          C.byref(cp), _p(K), _p(pf), _p(St), _p(Ss))
    return K, pf, St, Ss


def rates_literal(g: MassGrid, K, pf, rho, eta=11.0 / 6.0, chi=1.0) -> np.ndarray:
    """Literal Eq. 53/54/61 triple loop in __float128 (O1)."""
    K = _in(K); pf = _in(pf); rho = _in(rho)
    out = np.empty(g.N)
    lib().orc_rates_literal_q(C.c_int(g.N), _p(g.m_c), _p(g.m_e), _p(K), _p(pf), _p(rho),
                              C.c_double(eta), C.c_double(chi), _p(out))
    return out


def rates_flux(g: MassGrid, K, pf, rho, eta=11.0 / 6.0, chi=1.0):
    """Pair-flux form (O2).  Returns drho, gain, loss, S (all [N])."""
    K = _in(K); pf = _in(pf); rho = _in(rho)
    N = g.N
    d = np.empty(N); ga = np.empty(N); lo = np.empty(N); S = np.empty(N)
    lib().orc_rates_flux(C.c_int(N), _p(g.m_c), _p(g.m_e), _p(K), _p(pf), _p(rho), C.c_double(eta),
                         C.c_double(chi), _p(d), _p(ga), _p(lo), _p(S))
    return d, ga, lo, S


def frag_redistribute(g: MassGrid, S, eta=11.0 / 6.0) -> np.ndarray:
    S = _in(S)
    d = np.zeros(g.N)
    lib().orc_frag_redistribute(C.c_int(g.N), _p(g.m_e), C.c_double(eta), _p(S), _p(d), None)
    return d


def bs32_step(g: MassGrid, K, pf, y, h, k1=None, eta=11.0 / 6.0, chi=1.0, rtol=1e-2, atol_factor=1e-10):
    """One BS3(2) step of one cell with (K, p_frag).  Returns y_new, k4, E."""
    K = _in(K); pf = _in(pf)
    Kc = np.ascontiguousarray(K * (1.0 - pf)); Kf = np.ascontiguousarray(K * pf)
    y = _in(y).copy()
    have = k1 is not None
    k = _in(k1).copy() if have else np.zeros(g.N)
    E = lib().orc_bs32_step(C.c_int(g.N), _p(g.m_c), _p(g.m_e), _p(Kc), _p(Kf), C.c_double(eta),
                            C.c_double(chi), C.c_double(rtol), C.c_double(atol_factor), _p(y), _p(k),
                            C.c_int(1 if have else 0), C.c_double(h))
    return y, k, float(E)


# ------------------------------------------------------------------------------------------ batches
_HD_KEEP = []


def _hd(h_dust):
    """Optional [C x N] dust scale heights (vertically integrated kernel) as a C pointer."""
    if h_dust is None:
        return None
    a = _in(h_dust)
    _HD_KEEP[:] = [a]
    return _p(a)


def vint_scale(hd, K):
    """K_ij / sqrt(2 pi (h_i^2 + h_j^2)) of one cell."""
    K = _in(K).copy(); hd = _in(hd)
    lib().orc_vint_scale(C.c_int(hd.size), _p(hd), _p(K))
    return K


def _gas_args(T, rho_g, Omega, alpha, vR, vZ, vphi):
    T = _in(T); rho_g = _in(rho_g); Omega = _in(Omega); alpha = _in(alpha); vR = _in(vR); vZ = _in(vZ)
    keep = [T, rho_g, Omega, alpha, vR, vZ]
    vp = None
    if vphi is not None:
        vphi = _in(vphi); keep.append(vphi); vp = _p(vphi)
    return keep, [_p(T), _p(rho_g), _p(Omega), _p(alpha), _p(vR), _p(vZ), vp]


def kernel_cells(N, a_min, a_max, rho_m, T, rho_g, Omega, alpha, vR, vZ, p: Params, vphi=None,
                 h_dust=None) -> np.ndarray:
    """Packed planes [C, 2, P] (plane 0 = K p_coag, plane 1 = K p_frag)."""
    keep, ga = _gas_args(T, rho_g, Omega, alpha, vR, vZ, vphi)
    Cn = keep[0].size
    P = N * (N + 1) // 2
    out = np.empty((Cn, 2, P))
    cp = p.c()
    lib().orc_kernel_cells(C.c_int(Cn), C.c_int(N), C.c_double(a_min), C.c_double(a_max),
                           C.c_double(rho_m), *ga, C.byref(cp), _p(out), _hd(h_dust))
    return out


def rates_cells(N, a_min, a_max, rho_m, T, rho_g, Omega, alpha, vR, vZ, p: Params, rho, vphi=None, h_dust=None):
    keep, ga = _gas_args(T, rho_g, Omega, alpha, vR, vZ, vphi)
    rho = _in(rho)
    Cn = keep[0].size
    d = np.empty((Cn, N)); g = np.empty((Cn, N)); l = np.empty((Cn, N))
    cp = p.c()
    lib().orc_rates_cells(C.c_int(Cn), C.c_int(N), C.c_double(a_min), C.c_double(a_max),
                          C.c_double(rho_m), *ga, C.byref(cp), _p(rho), _p(d), _p(g), _p(l), _hd(h_dust))
    return d, g, l


def rates_cells_planes(N, a_min, a_max, rho_m, Kp, rho, eta=11.0 / 6.0, chi=1.0):
    """Rates from packed planes Kp: [2, P] shared by all cells, or [C, 2, P]."""
    Kp = _in(Kp); rho = _in(rho)
    Cn = rho.shape[0]
    per_cell = 1 if Kp.ndim == 3 else 0
    d = np.empty((Cn, N)); g = np.empty((Cn, N)); l = np.empty((Cn, N))
    lib().orc_rates_cells_planes(C.c_int(Cn), C.c_int(N), C.c_double(a_min), C.c_double(a_max),
                                 C.c_double(rho_m), C.c_double(eta), C.c_double(chi), _p(Kp),
                                 C.c_int(per_cell), _p(rho), _p(d), _p(g), _p(l))
    return d, g, l


def step_cells(N, a_min, a_max, rho_m, T, rho_g, Omega, alpha, vR, vZ, p: Params, rho, dt, k1=None,
               vphi=None, h_dust=None):
    """One BS3(2) step of every cell.  Returns rho_new [C,N], k4 [C,N], err [C]."""
    keep, ga = _gas_args(T, rho_g, Omega, alpha, vR, vZ, vphi)
    rho = _in(rho).copy()
    Cn = keep[0].size
    have = k1 is not None
    k = _in(k1).copy() if have else np.zeros((Cn, N))
    err = np.empty(Cn)
    cp = p.c()
    lib().orc_step_cells(C.c_int(Cn), C.c_int(N), C.c_double(a_min), C.c_double(a_max),
                         C.c_double(rho_m), *ga, C.byref(cp), _p(rho), _p(k), C.c_int(1 if have else 0),
                         C.c_double(dt), _p(err), _hd(h_dust))
    return rho, k, err


def step_cells_planes(N, a_min, a_max, rho_m, Kp, rho, dt, k1=None, eta=11.0 / 6.0, chi=1.0,
                      rtol=1e-2, atol_factor=1e-10):
    Kp = _in(Kp); rho = _in(rho).copy()
    Cn = rho.shape[0]
    have = k1 is not None
    k = _in(k1).copy() if have else np.zeros((Cn, N))
    err = np.empty(Cn)
    lib().orc_step_cells_planes(C.c_int(Cn), C.c_int(N), C.c_double(a_min), C.c_double(a_max),
                                C.c_double(rho_m), C.c_double(eta), C.c_double(chi), C.c_double(rtol),
                                C.c_double(atol_factor), _p(Kp), _p(rho), _p(k),
                                C.c_int(1 if have else 0), C.c_double(dt), _p(err))
    return rho, k, err


def pack_planes(K: np.ndarray, pf: np.ndarray) -> np.ndarray:
    """Full (K, p_frag) [N,N] -> packed planes [2, P] (layout helper, no method arithmetic beyond Eq. 55)."""
    N = K.shape[0]
    il = np.tril_indices(N)
    return np.ascontiguousarray(np.stack([(K * (1.0 - pf))[il], (K * pf)[il]]))


# ------------------------------------------------------------------------------------------ adaptive sub-cycling
def controller_next_dt(E: float, h: float) -> float:
    """Step-size controller of the embedded pair (R10; PAPER.md:478 names the method and the
    tolerances only): next trial size h * clamp(0.9 E^(-1/3), 0.2, 5), factor 5 for E = 0.  A step is
    accepted iff E <= 1.  Pins: E = 0.729 keeps h (0.9 / 0.9); E = 1 gives 0.9 h; clamps at 0.2 and 5."""
    f = 5.0 if E <= 0.0 else 0.9 * E ** (-1.0 / 3.0)
    return h * min(5.0, max(0.2, f))


def integrate(step, rho, t_span: float, dt_try: float, max_steps: int = 100000):
    """Adaptive sub-cycling over t_span with ONE global step size: `step(rho, dt, k1)` is
    one BS3(2) step of every cell returning (rho_new, k4, err[C]); the global error norm is max_c err_c;
    the last step is cut to land on t_span (a cut step does not shrink the next trial size).
    Returns rho, list of trial step sizes (negative = rejected), dt_next."""
    t, dt, k1, log = 0.0, float(dt_try), None, []
    rho = np.array(rho, dtype=np.float64, copy=True)
    while t < t_span and len(log) < max_steps:
        left = t_span - t
        cut = dt >= left
        h = left if cut else dt
        rho_new, k4, err = step(rho, h, k1)
        E = float(np.max(err))
        if not np.isfinite(E):
            raise FloatingPointError("non-finite error norm")
        if E <= 1.0:
            rho, k1 = rho_new, k4
            t = t_span if cut else t + h
            log.append(h)
            sug = controller_next_dt(E, h)
            dt = max(sug, dt) if cut else sug
        else:
            log.append(-h)
            dt = controller_next_dt(E, h)
    return rho, log, dt


def replay(step, rho, dts):
    """Fixed schedule: the accepted steps of a recorded run (parity under adaptivity)."""
    rho = np.array(rho, dtype=np.float64, copy=True)
    k1 = None
    for h in dts:
        rho, k1, _ = step(rho, float(h), k1)
    return rho


# ------------------------------------------------------------------------------------------ hydrostatic equilibrium
def hydrostatic(R_e, tan_e, R_c, tan_c, cs2, Sigma, GM: float) -> np.ndarray:
    """Gas density [n_r, n_z] of the vertical hydrostatic solve (Eqs. 32-37)."""
    R_e = _in(R_e); tan_e = _in(tan_e); R_c = _in(R_c); tan_c = _in(tan_c); cs2 = _in(cs2); Sigma = _in(Sigma)
    n_r, n_z = cs2.shape
    assert R_e.size == n_r + 1 and tan_e.size == n_z + 1 and R_c.size == n_r and tan_c.size == n_z and Sigma.size == n_r
    out = np.empty((n_r, n_z))
    lib().orc_hydrostatic(C.c_int(n_r), C.c_int(n_z), _p(R_e), _p(tan_e), _p(R_c), _p(tan_c), _p(cs2), _p(Sigma),
                          C.c_double(GM), _p(out))
    return out
