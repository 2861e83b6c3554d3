"""cudisc-coag-b200: the per-cell Smoluchowski coagulation/fragmentation update of cuDisc
(arXiv 2402.18471, section 5) as hand-written FP64 CUDA kernels for sm_100a behind a C ABI
(include/cudisc_coag.h).  This package is the thin Python binding plus the seeded input recipe.
"""
from .binding import (Bins, CudiscError, Grid, Hydro, Params, cudisc_hydrostatic, cudisc_coag_kernel, cudisc_coag_rates,  # noqa: F401
                      cudisc_coag_rates_otf, cudisc_coag_rates_otf_noalloc, cudisc_coag_step, cudisc_coag_step_cached, cudisc_coag_step_host, cudisc_coag_integrate,
                      cudisc_coag_integrate_steps, cudisc_controller_next_dt,
                      cudisc_launch_count,
                      cudisc_microbench_copy, cudisc_microbench_dfma, cudisc_version, lib)
