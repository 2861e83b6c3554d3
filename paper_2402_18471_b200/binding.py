"""Thin ctypes binding of libcudisc_coag.so (include/cudisc_coag.h).  Argument marshalling only:
every step of the path runs inside the library's CUDA kernels.  PyTorch supplies device memory
and streams (tensor.data_ptr(), torch.cuda.current_stream()).

There is no fallback of any kind: if the shared library is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from pathlib import Path
from typing import Optional

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libcudisc_coag.so"

STATUS = {0: "OK", 1: "INVALID", 2: "HANDLE", 3: "CUDA", 4: "UNSUPPORTED"}


class CudiscError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"cudisc status {code} ({STATUS.get(code, '?')}): {msg}")
        self.code = code


class cudisc_params(C.Structure):
    _fields_ = [("mu", C.c_double), ("v_frag", C.c_double), ("alpha", C.c_double), ("eta", C.c_double),
                ("chi_im", C.c_double), ("sigma_mol", C.c_double), ("rtol", C.c_double),
                ("atol_factor", C.c_double), ("readings", C.c_int)]


class cudisc_gas_state(C.Structure):
    _fields_ = [("T", C.c_void_p), ("rho_gas", C.c_void_p), ("Omega", C.c_void_p), ("alpha", C.c_void_p),
                ("v_R", C.c_void_p), ("v_Z", C.c_void_p), ("v_phi", C.c_void_p), ("h_dust", C.c_void_p)]


class cudisc_integrate_info(C.Structure):
    _fields_ = [("t_done", C.c_double), ("dt_last", C.c_double), ("dt_next", C.c_double),
                ("err_last", C.c_double), ("n_accepted", C.c_int), ("n_rejected", C.c_int)]


EXPORTS = [
    "cudisc_bins_create", "cudisc_bins_create_general", "cudisc_bins_destroy", "cudisc_bins_query",
    "cudisc_bins_expand_outcomes", "cudisc_bins_schedule_check", "cudisc_bins_fast_path", "cudisc_grid_create", "cudisc_grid_bind_gas", "cudisc_grid_reset_fsal",
    "cudisc_grid_destroy", "cudisc_coag_kernel", "cudisc_coag_rates", "cudisc_coag_rates_otf",
    "cudisc_coag_rates_otf_noalloc",
    "cudisc_coag_step", "cudisc_coag_step_cached", "cudisc_coag_step_host", "cudisc_coag_integrate", "cudisc_coag_integrate_steps", "cudisc_controller_next_dt",
    "cudisc_microbench_dfma",
    "cudisc_microbench_copy", "cudisc_launch_count", "cudisc_last_error", "cudisc_version",
    "cudisc_hydro_create", "cudisc_hydro_destroy", "cudisc_hydrostatic", "cudisc_hydro_last_error",
]

_lib = None


def lib() -> C.CDLL:
    """Load the C-ABI library (built in-tree by paper_2402_18471_b200.build_ext)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2402_18471_b200.build_ext` "
                              "(there is no CPU or PyTorch fallback)")
        L = C.CDLL(str(LIB_PATH))
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.cudisc_bins_create.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, cudisc_params, C.POINTER(vp)]
        L.cudisc_bins_create_general.argtypes = [C.c_int, dp, dp, C.c_double, cudisc_params, C.POINTER(vp)]
        L.cudisc_bins_destroy.argtypes = [vp]
        L.cudisc_bins_query.argtypes = [vp, ip, dp, dp, dp, ip, ip]
        L.cudisc_bins_expand_outcomes.argtypes = [vp, C.POINTER(C.c_longlong), ip, ip, ip, ip, dp, dp, dp]
        L.cudisc_bins_schedule_check.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.cudisc_bins_fast_path.argtypes = [vp, ip, C.POINTER(C.c_longlong), ip]
        L.cudisc_grid_create.argtypes = [C.c_int, C.c_int, vp, C.POINTER(vp)]
        L.cudisc_grid_bind_gas.argtypes = [vp, C.POINTER(cudisc_gas_state)]
        L.cudisc_grid_reset_fsal.argtypes = [vp]
        L.cudisc_grid_destroy.argtypes = [vp]
        L.cudisc_coag_kernel.argtypes = [vp, vp, C.POINTER(cudisc_gas_state), cudisc_params, vp, vp]
        L.cudisc_coag_rates.argtypes = [vp, vp, vp, vp, vp, vp]
        L.cudisc_coag_rates_otf.argtypes = [vp, vp, vp, vp, vp]
        L.cudisc_coag_rates_otf_noalloc.argtypes = [vp, vp, vp, vp, vp]
        L.cudisc_coag_step.argtypes = [vp, vp, vp, C.c_double, vp, vp]
        L.cudisc_coag_step_host.argtypes = [vp, vp, vp, C.c_double, vp, vp]
        L.cudisc_coag_step_cached.argtypes = [vp, vp, vp, vp, C.c_double, vp, vp]
        L.cudisc_coag_integrate.argtypes = [vp, vp, vp, C.c_double, C.c_double, C.c_int, dp,
                                            C.POINTER(cudisc_integrate_info), vp]
        L.cudisc_coag_integrate_steps.argtypes = [vp, vp, vp, C.c_int, C.c_double, C.c_int, dp,
                                                  C.POINTER(cudisc_integrate_info), vp]
        L.cudisc_controller_next_dt.argtypes = [C.c_double, C.c_double]
        L.cudisc_controller_next_dt.restype = C.c_double
        L.cudisc_microbench_dfma.argtypes = [C.c_int, dp, dp]
        L.cudisc_microbench_copy.argtypes = [C.c_longlong, dp, dp]
        L.cudisc_launch_count.restype = C.c_longlong
        L.cudisc_hydro_create.argtypes = [C.c_int, C.c_int, dp, dp, dp, dp, C.POINTER(vp)]
        L.cudisc_hydro_destroy.argtypes = [vp]
        L.cudisc_hydrostatic.argtypes = [vp, vp, vp, C.c_double, vp, vp]
        L.cudisc_hydro_last_error.restype = C.c_char_p
        L.cudisc_last_error.restype = C.c_char_p
        L.cudisc_version.restype = C.c_char_p
        for name in EXPORTS:
            getattr(L, name)       # AttributeError if the library does not export it
        _lib = L
    return _lib


def _check(code: int) -> None:
    if code != 0:
        raise CudiscError(code, lib().cudisc_last_error().decode())


@dataclass
class Params:
    mu: float = 2.4
    v_frag: float = 100.0
    alpha: float = 1e-3
    eta: float = 11.0 / 6.0
    chi_im: float = 1.0
    sigma_mol: float = 2.0e-15
    rtol: float = 1e-2
    atol_factor: float = 1e-10
    readings: int = 0      # bit 0: number-conserving split, bit 1: total-mass fragment lookup (cudisc_coag.h)

    def c(self) -> cudisc_params:
        return cudisc_params(self.mu, self.v_frag, self.alpha, self.eta, self.chi_im, self.sigma_mol,
                             self.rtol, self.atol_factor, int(self.readings))


def _dev_ptr(t, name: str, numel: Optional[int] = None) -> int:
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name}: expected a CUDA tensor")
    if t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous float64 tensor")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name}: expected {numel} elements, got {t.numel()}")
    return t.data_ptr()


def _stream(stream=None) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


class Bins:
    """cudisc_bins handle: mass grid + grid-only tables."""

    def __init__(self, n_bins: int, a_min: float, a_max: float, rho_m: float, params: Params,
                 m_centres=None, m_edges=None):
        self.params = params
        self._h = C.c_void_p()
        if m_centres is None:
            _check(lib().cudisc_bins_create(n_bins, a_min, a_max, rho_m, params.c(), C.byref(self._h)))
        else:
            mc = np.ascontiguousarray(m_centres, dtype=np.float64)
            me = np.ascontiguousarray(m_edges, dtype=np.float64)
            dp = C.POINTER(C.c_double)
            _check(lib().cudisc_bins_create_general(n_bins, mc.ctypes.data_as(dp), me.ctypes.data_as(dp),
                                                    rho_m, params.c(), C.byref(self._h)))
        self.n_bins = n_bins
        self.n_pairs = n_bins * (n_bins + 1) // 2

    @property
    def handle(self):
        return self._h

    def query(self):
        N = self.n_bins
        n = C.c_int(); nband = C.c_int()
        m = np.empty(N); me = np.empty(N + 1); a = np.empty(N); nb = np.empty(N, dtype=np.int32)
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        _check(lib().cudisc_bins_query(self._h, C.byref(n), m.ctypes.data_as(dp), me.ctypes.data_as(dp),
                                       a.ctypes.data_as(dp), nb.ctypes.data_as(ip), C.byref(nband)))
        return {"n_bins": n.value, "m_centres": m, "m_edges": me, "a_centres": a, "n_bulk": nb,
                "n_band": nband.value}

    def expand_outcomes(self):
        """Expanded gather form of every pair outcome (host tables; no GPU needed)."""
        N = self.n_bins
        cnt = C.c_longlong()
        L = lib()
        _check(L.cudisc_bins_expand_outcomes(self._h, C.byref(cnt), None, None, None, None, None, None, None))
        E = cnt.value
        tgt = np.empty(E, dtype=np.int32); i = np.empty(E, dtype=np.int32); j = np.empty(E, dtype=np.int32)
        pl = np.empty(E, dtype=np.int32); coef = np.empty(E); fA = np.empty(N); fiB = np.empty(N)
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        _check(L.cudisc_bins_expand_outcomes(self._h, C.byref(cnt), tgt.ctypes.data_as(ip), i.ctypes.data_as(ip),
                                             j.ctypes.data_as(ip), pl.ctypes.data_as(ip), coef.ctypes.data_as(dp),
                                             fA.ctypes.data_as(dp), fiB.ctypes.data_as(dp)))
        return {"target": tgt, "i": i, "j": j, "plane": pl, "coef": coef, "frag_A": fA, "frag_invB": fiB}

    def schedule_check(self):
        """Host-side self-check of the kernels' work-item schedule (no GPU needed): 8 counters, the
        first six must be zero (include/cudisc_coag.h)."""
        out = (C.c_longlong * 8)()
        _check(lib().cudisc_bins_schedule_check(self._h, out))
        return [int(v) for v in out]

    def fast_path(self):
        """(on, shared-memory bytes, tensor-memory columns) of the tensor-memory kernel for this grid."""
        on = C.c_int(); sm = C.c_longlong(); tm = C.c_int()
        _check(lib().cudisc_bins_fast_path(self._h, C.byref(on), C.byref(sm), C.byref(tm)))
        return bool(on.value), int(sm.value), int(tm.value)

    def close(self):
        if self._h:
            lib().cudisc_bins_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Grid:
    """cudisc_grid handle: n_r x n_z cells on mass grid `bins`."""

    def __init__(self, n_r: int, n_z: int, bins: Bins):
        self.bins = bins
        self.n_r, self.n_z = n_r, n_z
        self.n_cells = n_r * n_z
        self._h = C.c_void_p()
        self._gas_keep = None
        _check(lib().cudisc_grid_create(n_r, n_z, bins.handle, C.byref(self._h)))

    @property
    def handle(self):
        return self._h

    def _gas_struct(self, T, rho_gas, Omega, v_R, v_Z, alpha=None, v_phi=None, h_dust=None):
        Cn, N = self.n_cells, self.bins.n_bins
        gs = cudisc_gas_state(
            _dev_ptr(T, "T", Cn), _dev_ptr(rho_gas, "rho_gas", Cn), _dev_ptr(Omega, "Omega", Cn),
            _dev_ptr(alpha, "alpha", Cn) if alpha is not None else None,
            _dev_ptr(v_R, "v_R", Cn * N), _dev_ptr(v_Z, "v_Z", Cn * N),
            _dev_ptr(v_phi, "v_phi", Cn * N) if v_phi is not None else None,
            _dev_ptr(h_dust, "h_dust", Cn * N) if h_dust is not None else None)
        return gs, (T, rho_gas, Omega, alpha, v_R, v_Z, v_phi, h_dust)

    def bind_gas(self, T, rho_gas, Omega, v_R, v_Z, alpha=None, v_phi=None, h_dust=None):
        gs, keep = self._gas_struct(T, rho_gas, Omega, v_R, v_Z, alpha, v_phi, h_dust)
        _check(lib().cudisc_grid_bind_gas(self._h, C.byref(gs)))
        self._gas_keep = keep      # the library keeps the pointers, not the arrays

    def reset_fsal(self):
        _check(lib().cudisc_grid_reset_fsal(self._h))

    def close(self):
        if self._h:
            lib().cudisc_grid_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ------------------------------------------------------------------------------------------ hot calls
def cudisc_coag_kernel(grid: Grid, bins: Bins, gas: dict, params: Params, K_out, stream=None) -> None:
    """K_out [C, 2, P] <- (K p_coag, K p_frag) of every cell (Eqs. 55-62)."""
    gs, _keep = grid._gas_struct(**gas)
    _check(lib().cudisc_coag_kernel(grid.handle, bins.handle, C.byref(gs), params.c(),
                                    _dev_ptr(K_out, "K_out", grid.n_cells * 2 * bins.n_pairs), _stream(stream)))


def cudisc_coag_rates(grid: Grid, bins: Bins, K, rho_dust, drho_dt, stream=None) -> None:
    """drho_dt [C, N] <- rates from the supplied packed kernel planes K [C, 2, P]."""
    Cn, N = grid.n_cells, bins.n_bins
    _check(lib().cudisc_coag_rates(grid.handle, bins.handle, _dev_ptr(K, "K", Cn * 2 * bins.n_pairs),
                                   _dev_ptr(rho_dust, "rho_dust", Cn * N), _dev_ptr(drho_dt, "drho_dt", Cn * N),
                                   _stream(stream)))


def cudisc_coag_rates_otf(grid: Grid, bins: Bins, rho_dust, drho_dt, stream=None) -> None:
    Cn, N = grid.n_cells, bins.n_bins
    _check(lib().cudisc_coag_rates_otf(grid.handle, bins.handle, _dev_ptr(rho_dust, "rho_dust", Cn * N),
                                       _dev_ptr(drho_dt, "drho_dt", Cn * N), _stream(stream)))


STATIC_SCRATCH_BYTES = 24 << 20     # CUDISC_STATIC_SCRATCH_BYTES of include/cudisc_coag.h


def cudisc_coag_rates_otf_noalloc(grid: Grid, bins: Bins, rho_dust, drho_dt, stream=None) -> None:
    """cudisc_coag_rates_otf without any allocation: the kernel's scratch is the library's static device array."""
    Cn, N = grid.n_cells, bins.n_bins
    _check(lib().cudisc_coag_rates_otf_noalloc(grid.handle, bins.handle, _dev_ptr(rho_dust, "rho_dust", Cn * N),
                                               _dev_ptr(drho_dt, "drho_dt", Cn * N), _stream(stream)))


def cudisc_coag_step(grid: Grid, bins: Bins, rho_dust, dt: float, err_out, stream=None) -> None:
    """One BS3(2) step of every cell, in place on rho_dust [C, N]; err_out [C]."""
    Cn, N = grid.n_cells, bins.n_bins
    _check(lib().cudisc_coag_step(grid.handle, bins.handle, _dev_ptr(rho_dust, "rho_dust", Cn * N),
                                  float(dt), _dev_ptr(err_out, "err_out", Cn), _stream(stream)))


def _host_ptr(t, name: str, numel: int) -> int:
    import torch
    if isinstance(t, np.ndarray):
        if t.dtype != np.float64 or not t.flags.c_contiguous or t.size != numel:
            raise TypeError(f"{name}: expected a C-contiguous float64 array of {numel} elements")
        return t.ctypes.data
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() \
            or t.numel() != numel:
        raise TypeError(f"{name}: expected a contiguous float64 HOST tensor of {numel} elements")
    return t.data_ptr()


def cudisc_coag_step_cached(grid: Grid, bins: Bins, K, rho_dust, dt: float, err_out, stream=None) -> None:
    """cudisc_coag_step with the kernel read from K [C][2][P] instead of being built."""
    Cn, N = grid.n_cells, bins.n_bins
    _check(lib().cudisc_coag_step_cached(grid.handle, bins.handle, _dev_ptr(K, "K", Cn * 2 * bins.n_pairs),
                                         _dev_ptr(rho_dust, "rho_dust", Cn * N), float(dt),
                                         _dev_ptr(err_out, "err_out", Cn), _stream(stream)))


def cudisc_coag_step_host(grid: Grid, bins: Bins, rho_host, dt: float, err_host, stream=None) -> None:
    """cudisc_coag_step with HOST buffers (pinned torch tensors or numpy arrays): H2D copy, step,
    D2H copies, stream wait -- all inside the library call."""
    Cn, N = grid.n_cells, bins.n_bins
    _check(lib().cudisc_coag_step_host(grid.handle, bins.handle, _host_ptr(rho_host, "rho_host", Cn * N),
                                       float(dt), _host_ptr(err_host, "err_host", Cn), _stream(stream)))


def cudisc_controller_next_dt(E: float, h: float) -> float:
    return float(lib().cudisc_controller_next_dt(float(E), float(h)))


def _info_dict(info, log):
    n = info.n_accepted + info.n_rejected
    return ({"t_done": info.t_done, "dt_last": info.dt_last, "dt_next": info.dt_next, "err_last": info.err_last,
             "n_accepted": info.n_accepted, "n_rejected": info.n_rejected}, log[:n].copy())


def cudisc_coag_integrate(grid: Grid, bins: Bins, rho_dust, t_span: float, dt_try: float, max_steps: int = 10000,
                          stream=None):
    """Adaptive BS3(2) sub-cycling over t_span.  Returns (info dict, dt_log): dt_log holds
    the size of every trial step, negated when rejected."""
    Cn, N = grid.n_cells, bins.n_bins
    log = np.zeros(max_steps)
    info = cudisc_integrate_info()
    _check(lib().cudisc_coag_integrate(grid.handle, bins.handle, _dev_ptr(rho_dust, "rho_dust", Cn * N),
                                       float(t_span), float(dt_try), int(max_steps),
                                       log.ctypes.data_as(C.POINTER(C.c_double)), C.byref(info), _stream(stream)))
    return _info_dict(info, log)


def cudisc_coag_integrate_steps(grid: Grid, bins: Bins, rho_dust, n_accepted: int, dt_try: float,
                                max_steps: int = 10000, stream=None):
    """Adaptive sub-cycling until n_accepted steps were accepted (BASELINE.json config 4)."""
    Cn, N = grid.n_cells, bins.n_bins
    log = np.zeros(max_steps)
    info = cudisc_integrate_info()
    _check(lib().cudisc_coag_integrate_steps(grid.handle, bins.handle, _dev_ptr(rho_dust, "rho_dust", Cn * N),
                                             int(n_accepted), float(dt_try), int(max_steps),
                                             log.ctypes.data_as(C.POINTER(C.c_double)), C.byref(info),
                                             _stream(stream)))
    return _info_dict(info, log)


class Hydro:
    """cudisc_hydro handle: geometry of the (R, theta) grid for cudisc_hydrostatic."""

    def __init__(self, R_edges, tan_edges, R_centres, tan_centres):
        dp = C.POINTER(C.c_double)
        a = [np.ascontiguousarray(x, dtype=np.float64) for x in (R_edges, tan_edges, R_centres, tan_centres)]
        self.n_r, self.n_z = a[2].size, a[3].size
        if a[0].size != self.n_r + 1 or a[1].size != self.n_z + 1:
            raise ValueError("edge arrays must have one more entry than the centre arrays")
        self._h = C.c_void_p()
        code = lib().cudisc_hydro_create(self.n_r, self.n_z, *[x.ctypes.data_as(dp) for x in a], C.byref(self._h))
        if code:
            raise CudiscError(code, lib().cudisc_hydro_last_error().decode())

    @property
    def handle(self):
        return self._h

    def close(self):
        if self._h:
            lib().cudisc_hydro_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def cudisc_hydrostatic(hydro: Hydro, cs2, Sigma_g, GM: float, rho_gas_out, stream=None) -> None:
    """rho_gas_out [n_r, n_z] <- vertical hydrostatic equilibrium of every column (Eqs. 32-37)."""
    n = hydro.n_r * hydro.n_z
    code = lib().cudisc_hydrostatic(hydro.handle, _dev_ptr(cs2, "cs2", n), _dev_ptr(Sigma_g, "Sigma_g", hydro.n_r),
                                    float(GM), _dev_ptr(rho_gas_out, "rho_gas_out", n), _stream(stream))
    if code:
        raise CudiscError(code, lib().cudisc_hydro_last_error().decode())


def cudisc_microbench_dfma(n_iter: int = 0):
    v = C.c_double(); ms = C.c_double()
    _check(lib().cudisc_microbench_dfma(n_iter, C.byref(v), C.byref(ms)))
    return v.value, ms.value


def cudisc_microbench_copy(n_bytes: int = 0):
    v = C.c_double(); ms = C.c_double()
    _check(lib().cudisc_microbench_copy(n_bytes, C.byref(v), C.byref(ms)))
    return v.value, ms.value


def cudisc_launch_count() -> int:
    return int(lib().cudisc_launch_count())


def cudisc_version() -> str:
    return lib().cudisc_version().decode()
