/*
 * cudisc_coag.h -- C ABI of libcudisc_coag.so: the per-cell Smoluchowski coagulation /
 * fragmentation update of cuDisc (arXiv 2402.18471, section 5) as
 * hand-written FP64 CUDA kernels for sm_100a (NVIDIA B200).
 *
 * Conventions
 *   - All floating point is FP64, all quantities CGS.
 *   - C = n_r * n_z cells, N = n_bins mass bins, P = N (N + 1) / 2 unordered pairs (i >= j).
 *   - Every [C x N] array is row-major, bin fastest; cell index c = i_R * n_z + j_Z.
 *   - "DEVICE" pointers are caller-owned CUDA device buffers (e.g. a torch tensor's data_ptr());
 *     the library never frees or reallocates them.  "HOST" pointers are plain host memory.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  The three
 *     hot calls only enqueue work on `stream` and return; they do not allocate and do not
 *     synchronise with the host.
 *   - Every function returns a cudisc_status.  No C++ exception crosses the ABI.
 *     cudisc_last_error() returns a thread-local, NUL-terminated description of the last
 *     non-zero status returned on the calling thread.
 *   - Non-finite inputs are not checked on the hot path; NaN propagates into the outputs
 *     (err_out in particular).
 *   - There is no CPU fallback: without a CUDA device every call that needs one returns
 *     CUDISC_ERR_CUDA.
 *
 * Readings of the paper where it is silent or garbled are listed in DESIGN.md ("Readings",
 * R1..R16) and referenced below.
 */
#ifndef CUDISC_COAG_H
#define CUDISC_COAG_H

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    CUDISC_OK = 0,
    CUDISC_ERR_INVALID = 1,     /* NULL pointer, n_bins < 2, a_min >= a_max, non-monotone masses ... */
    CUDISC_ERR_HANDLE = 2,      /* bad handle, or grid was created for different bins             */
    CUDISC_ERR_CUDA = 3,        /* CUDA runtime error (launch failure, no device, sticky error)   */
    CUDISC_ERR_UNSUPPORTED = 4  /* size outside what the kernels support (n_bins > 256)           */
} cudisc_status;

typedef struct cudisc_bins_s *cudisc_bins;   /* mass grid + grid-only tables; owned by the library */
typedef struct cudisc_grid_s *cudisc_grid;   /* cell grid: bound gas state, FSAL buffer, scratch   */
typedef void *cudisc_stream;                 /* cudaStream_t */

/* Physical / numerical parameters, passed by value. */
typedef struct {
    double mu;           /* mean molecular weight of the gas (default 2.4)          */
    double v_frag;       /* fragmentation threshold velocity, cm/s (Eq. 62)         */
    double alpha;        /* turbulent alpha used when gas_state.alpha == NULL      */
    double eta;          /* fragment power-law slope (Eq. 66; default 11/6)         */
    double chi_im;       /* fragment mass in units of the impactor mass (default 1) */
    double sigma_mol;    /* H2 collision cross-section for nu_mol, cm^2 (reading R6; 2e-15)       */
    double rtol;         /* BS3(2) relative tolerance (default 1e-2)                */
    double atol_factor;  /* absolute tolerance = atol_factor * sum_k rho_k (1e-10)  */
    int readings;        /* variants of two readings the paper leaves open (R2, R11); 0 = the
                            readings taken.  Bit 0: number-conserving two-bin split (the bins
                            receive the number fractions eps, 1 - eps of the product instead of its mass
                            fractions).  Bit 1: the fragment l-bin is looked up with the total fragment mass
                            m_j + min(chi m_j, m_i) instead of min(chi m_j, m_i).
                            Other bits: CUDISC_ERR_INVALID.  Grid-only: fixed per cudisc_bins handle.     */
} cudisc_params;

/* Frozen per-cell inputs from the other solvers.  DEVICE pointers. */
typedef struct {
    const double *T;        /* [C]  gas temperature, K                                            */
    const double *rho_gas;  /* [C]  gas density, g/cm^3                                           */
    const double *Omega;    /* [C]  Keplerian angular frequency, 1/s                              */
    const double *alpha;    /* [C]  or NULL -> params.alpha in every cell                         */
    const double *v_R;      /* [C x N] dust radial velocity per size, cm/s                        */
    const double *v_Z;      /* [C x N] dust vertical velocity per size, cm/s                      */
    const double *v_phi;    /* [C x N] or NULL (term left out of Delta v_lam)                     */
    const double *h_dust;   /* [C x N] dust scale heights, cm, or NULL.  Non-NULL selects the
                               vertically integrated kernel of PAPER.md:486: K_ij / sqrt(2 pi (h_i^2 +
                               h_j^2)), rho_dust then holds surface densities and v_Z the settling
                               velocities at Z = h.  Not together with v_phi (UNSUPPORTED).         */
} cudisc_gas_state;

/* ---------------------------------------------------------------------------------------------
 * Handles
 * ------------------------------------------------------------------------------------------- */

/* Mass grid of PAPER.md:442, 467, 503: n_bins bins <-> n_bins + 1 log-spaced edges in grain
 * radius over [a_min, a_max] (cm); m^e_k = (4 pi / 3) rho_m (a^e_k)^3; centres are geometric
 * means of the edges.  Also builds every grid-only table of the rate evaluation (two-bin split
 * of Eqs. 63-65, remnant / fragment masses of Eq. 68, l-bins and N_k of Eq. 67) from p.eta and
 * p.chi_im, on the host; they are uploaded to the current CUDA device on first use.
 * p is stored: cudisc_coag_step uses it.  Works without a CUDA device (tables stay on the host).
 * One device per handle: the device copy of the tables follows the CURRENT device of the call that needs it,
 * so a bins handle (and the grids made from it) must be used from one device only; use one handle per device.
 * Errors: INVALID (n_bins < 2, a_min <= 0, a_min >= a_max, rho_m <= 0, eta >= 2, chi_im <= 0,
 * out == NULL), UNSUPPORTED (n_bins > 256). */
int cudisc_bins_create(int n_bins, double a_min, double a_max, double rho_m,
                       cudisc_params p, cudisc_bins *out);

/* Same for an arbitrary monotone mass grid: m_centres [n_bins], m_edges [n_bins + 1] (HOST,
 * copied), strictly increasing with m_edges[k] < m_centres[k] < m_edges[k+1].  Grain radii are
 * a_k = (3 m_k / (4 pi rho_m))^(1/3). */
int cudisc_bins_create_general(int n_bins, const double *m_centres, const double *m_edges,
                               double rho_m, cudisc_params p, cudisc_bins *out);

int cudisc_bins_destroy(cudisc_bins b);

/* Introspection of the host tables (HOST output pointers, any may be NULL):
 *   m_centres [N], m_edges [N+1], a_centres [N]; n_bulk [N] = number of leading impactor bins j
 *   of target row i whose collision outcomes are handled by the structured ("bulk") row sums;
 *   *n_band = number of entries of the band gather lists (all remaining pair outcomes). */
int cudisc_bins_query(cudisc_bins b, int *n_bins, double *m_centres, double *m_edges,
                      double *a_centres, int *n_bulk, int *n_band);

/* The full outcome table in gather form, for checking the host logic without a GPU.
 * For every output bin k the rate is
 *   drho_k = sum_e  coef[e] * n_{i[e]} * n_{j[e]} * Kplane[e]_{i[e] j[e]}     (entries with target k)
 *          + A_k * sum_{l >= k} S_l / B_l,      S_l = same form over the S-entries with target l,
 * where the lists returned here are the EXPANDED ones (bulk row/column sums written out pair by
 * pair), so that a test can evaluate them with plain loops.  Call with all pointers NULL to get
 * the counts.  target < N: density bin; target >= N: S bin (target - N).  plane 0 = K p_coag,
 * 1 = K p_frag; the diagonal factor 1/2 is already folded into coef.
 * frag_A [N], frag_invB [N]: A_k and 1 / B_l of PAPER.md:465-469. */
int cudisc_bins_expand_outcomes(cudisc_bins b, long long *n_entries, int *target, int *i, int *j,
                                int *plane, double *coef, double *frag_A, double *frag_invB);

/* Host-side self-check of the work-item schedule the kernels run for this mass grid (no device
 * needed): decodes the packed items exactly as the device code does and counts what is wrong.
 *   out[0] pairs (i >= j) not built exactly once by the build items
 *   out[1] (row i, column j < n_bulk[i]) not summed exactly once by the row-pass items
 *   out[2] (i >= j) not summed exactly once by the column-pass items
 *   out[3] partial-sum slots out of range, written twice, or read by the combine step but never written
 *   out[4] band indices out of range of what they address, or band entries lost
 *   out[5] band gather tasks: target groups without exactly one covering set of tasks
 *   out[6] number of items (build + eval);  out[7] shared-memory bytes needed besides the K store
 * out[0..5] are 0 for a correct schedule.  out: HOST [8].  When the grid takes the tensor-memory kernel
 * (cudisc_bins_fast_path) its static per-warp task lists are checked as well and counted in the same
 * slots: pairs built once, bulk (row, column) and (i >= j) summed once, partial-sum parts written once,
 * tensor-memory columns written by the build exactly where the column tasks of the same quarter read them
 * and disjoint from the tables, band entries complete, at most two band halves per warp. */
int cudisc_bins_schedule_check(cudisc_bins b, long long *out);

/* Whether this mass grid takes the tensor-memory kernel for cudisc_coag_step / cudisc_coag_rates_otf
 * (second copy of the cell's kernel in the SM's tensor memory, static per-warp
 * schedule; needs 64 <= n_bins, the band tables and the row copy to fit: up to ~155 bins at 227 KB of
 * shared memory), the dynamic shared memory it needs and the 32-bit tensor-memory columns (of 4 x 512)
 * its tables and column copy occupy.  Otherwise the general kernel runs (any n_bins <= 256).  Host only. */
int cudisc_bins_fast_path(cudisc_bins b, int *on, long long *smem_bytes, int *tmem_cols_used);

/* Cell grid of n_r x n_z cells using mass grid b.  Allocates on the current CUDA device: the
 * FSAL buffer [C x N], and the kernel scratch.  The handle remembers b. */
int cudisc_grid_create(int n_r, int n_z, cudisc_bins b, cudisc_grid *out);

/* Bind the frozen gas state used by cudisc_coag_step.  The struct is copied, the arrays are NOT:
 * they must stay valid and unchanged while steps are enqueued.  Invalidates the FSAL buffer. */
int cudisc_grid_bind_gas(cudisc_grid g, const cudisc_gas_state *gs);

/* Invalidate the saved last-stage derivative k4 (call after changing rho_dust outside the
 * library, or the gas arrays in place): the next step recomputes k1 = f(rho). */
int cudisc_grid_reset_fsal(cudisc_grid g);

int cudisc_grid_destroy(cudisc_grid g);

/* ---------------------------------------------------------------------------------------------
 * Hot path
 * ------------------------------------------------------------------------------------------- */

/* Collision kernel of every cell, PAPER.md:410-440 (Eqs. 55-62): K_ij = sigma_ij dv_ij with
 * sigma_ij = pi (a_i + a_j)^2 (R3), dv_ij^2 = Brownian (Eq. 58) + turbulent (Eqs. 59-60, Ormel &
 * Cuzzi 2007 closed forms, R4) + laminar (v_R, v_Z [, v_phi] differences), and the
 * fragmentation probability p_frag of Eq. 62.
 * K_out: DEVICE [C][2][P], packed lower-triangular (i >= j at index i (i + 1) / 2 + j):
 *        plane 0 = K_ij (1 - p_frag,ij), plane 1 = K_ij p_frag,ij; the diagonal is NOT halved.
 * Uses p.mu, p.v_frag, p.alpha (if gs->alpha == NULL) and p.sigma_mol; gs must be non-NULL. */
int cudisc_coag_kernel(cudisc_grid g, cudisc_bins b, const cudisc_gas_state *gs,
                       cudisc_params p, double *K_out, cudisc_stream stream);

/* Rate evaluation from a supplied kernel, PAPER.md:396-404, 432-476 (Eqs. 53, 54, 61-68) in the
 * cancellation-free pair-flux form (R9): drho_dt_k for every cell.
 * K: DEVICE [C][2][P] as written by cudisc_coag_kernel -- ANY symmetric kernel is accepted
 *    (closed-form tests pass plane 0 = K, plane 1 = 0).
 * rho_dust: DEVICE [C x N] in; drho_dt: DEVICE [C x N] out.  May not alias. */
int cudisc_coag_rates(cudisc_grid g, cudisc_bins b, const double *K,
                      const double *rho_dust, double *drho_dt, cudisc_stream stream);

/* Extension: the same rate evaluation with K built on the fly from the gas state bound to g
 * (never written to HBM). */
int cudisc_coag_rates_otf(cudisc_grid g, cudisc_bins b, const double *rho_dust, double *drho_dt,
                          cudisc_stream stream);

/* cudisc_coag_rates_otf for callers that may not allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same operation, same arguments, same results, on the general cell
 * kernel (coag_kernels.cu), whose scratch -- the per-CTA slab for the pairs of K that do not fit in shared
 * memory, (P - P_shared) x 16 B per resident CTA -- lives in a file-scope device array of the library instead
 * of the grid's own buffer.  The call performs no cudaMalloc / cudaFree and calls no allocating library
 * routine; g and b must exist already (cudisc_grid_create uploads the tables), and the first call on a device
 * looks the array's address up (cudaGetSymbolAddress: no allocation), so make one call at set-up.
 * Limit: the array holds CUDISC_STATIC_SCRATCH_BYTES = 24 MiB on every GPU that loads the library, until
 * the process exits: enough for every grid of up to 200 bins on a 148-SM GPU (21.7 MiB); a grid that needs more
 * is rejected with CUDISC_ERR_UNSUPPORTED and a message that states both sizes (use cudisc_coag_rates_otf).
 * Grids whose K fits in shared memory use no scratch at all.
 * All calls share the array and it keeps the last call's contents; the kernel writes every slab entry of a
 * cell before reading it, so nothing needs clearing -- but two calls of this entry point that OVERLAP on
 * the GPU (different streams, or graph branches) race on it: serialise them.
 * rho_dust: DEVICE [C x N] in; drho_dt: DEVICE [C x N] out.  May not alias. */
#define CUDISC_STATIC_SCRATCH_BYTES (24u << 20)
int cudisc_coag_rates_otf_noalloc(cudisc_grid g, cudisc_bins b, const double *rho_dust, double *drho_dt,
                                  cudisc_stream stream);

/* One Bogacki-Shampine 3(2) step of size dt (s) of every cell, with the kernel
 * built on the fly, once per cell per step, from the gas state bound to g and frozen over the
 * stages; parameters are those given to cudisc_bins_create.
 * rho_dust: DEVICE [C x N] in/out.  err_out: DEVICE [C], the scaled error norm of each cell
 *   E_c = max_k |e_k| / (atol_factor * sum_k rho_k + rtol * max(|rho_k|, |rho_k^new|))   (R10);
 * the step is accepted by the caller iff max_c E_c <= 1 (this call always advances rho_dust).
 * The first call after create / bind_gas / reset_fsal evaluates k1 = f(rho) (4 rate evaluations);
 * later calls reuse the saved k4 (FSAL, 3 evaluations) -- only for the same rho_dust array (a different
 * pointer, or a switch between this call and cudisc_coag_step_cached, recomputes k1); call
 * cudisc_grid_reset_fsal after modifying rho_dust in place.  One device per process is assumed for a
 * given handle: tables and scratch live on the device that was current at cudisc_grid_create. */
int cudisc_coag_step(cudisc_grid g, cudisc_bins b, double *rho_dust, double dt,
                     double *err_out, cudisc_stream stream);

/* Cached-kernel form of cudisc_coag_step: the same Bogacki-Shampine 3(2) step with the
 * kernel read from K (DEVICE [C][2][P], as written by cudisc_coag_kernel; ANY symmetric kernel is
 * accepted, e.g. the closed-form test kernels with plane 1 = 0) instead of being built from the gas
 * state.  16 B of HBM traffic per pair and step.  Shares the FSAL buffer with cudisc_coag_step:
 * call cudisc_grid_reset_fsal when switching between the two or changing K. */
int cudisc_coag_step_cached(cudisc_grid g, cudisc_bins b, const double *K, double *rho_dust, double dt,
                            double *err_out, cudisc_stream stream);

/* End-to-end form of cudisc_coag_step for callers whose dust array lives in HOST memory (the
 * other solvers of the paper's global loop, when they run elsewhere):
 * rho_host: HOST [C x N] in/out, err_host: HOST [C] out (page-locked memory makes the copies
 * asynchronous and full-speed; pageable memory works).  Enqueues on `stream`: host->device copy
 * of rho_host into a staging buffer owned by g (allocated on the first call, the only allocation
 * this call ever makes), the same kernel as cudisc_coag_step, device->host copies of the new
 * densities and of the error norms; then WAITS for the stream, so the host buffers are valid on
 * return.  The FSAL derivative is kept on the device exactly as for cudisc_coag_step: call
 * cudisc_grid_reset_fsal if rho_host was modified between steps. */
int cudisc_coag_step_host(cudisc_grid g, cudisc_bins b, double *rho_host, double dt,
                          double *err_host, cudisc_stream stream);

/* ---------------------------------------------------------------------------------------------
 * Adaptive sub-cycling (reading R10)
 * ------------------------------------------------------------------------------------------- */

typedef struct {
    double t_done;        /* time covered, s (== t_span unless max_steps ran out)                  */
    double dt_last;       /* size of the last accepted step (possibly truncated to land on t_span) */
    double dt_next;       /* the controller's suggestion for the next step: hand it back as dt_try
                             of the next call ("the final sub-timestep")             */
    double err_last;      /* max_c E_c of the last accepted step                                   */
    int n_accepted, n_rejected;
} cudisc_integrate_info;

/* Step-size controller of the embedded pair (R10, textbook): a step of size h with error norm
 * E = max_c E_c is accepted iff E <= 1; the next trial size is h * clamp(0.9 E^(-1/3), 0.2, 5)
 * (factor 5 for E == 0).  Pure host function, no device needed. */
double cudisc_controller_next_dt(double E, double h);

/* Integrates every cell over t_span seconds with adaptive BS3(2) sub-steps of ONE global size
 * (coagulation sub-cycles inside the global step with the gas state frozen).
 * The controller runs on the DEVICE: every trial is one step launch that reads its size and
 * its buffer roles from a controller state in device memory, followed by a one-block kernel that reduces
 * the per-cell error norms, accepts or rejects, and writes the next size; trials are enqueued in batches
 * of 32 without a host round trip (launches after the end return at once) and the host reads the state
 * once per batch.  Rejected steps leave the state untouched.  The last step is cut to land on t_span.
 * rho_dust: DEVICE [C x N] in/out.  dt_try: first trial size, s (> 0).  max_steps: bound on accepted
 * + rejected steps.  dt_log: HOST [max_steps] or NULL; receives the size of every trial step in
 * order, negated when the step was rejected.  info: HOST, may be NULL.
 * SYNCHRONISES with `stream` (once per batch).  Buffers owned by g are allocated on the first call, all or
 * nothing.  A non-finite error norm stops the integration with CUDISC_ERR_INVALID (rho_dust then holds
 * the last accepted state).
 * FSAL: the saved derivative is reused only if it was produced from this same rho_dust array with the
 * kernel built on the fly (the library remembers both); after rho_dust was modified IN PLACE by the caller
 * (dust transport between coagulation calls) cudisc_grid_reset_fsal must be called. */
int cudisc_coag_integrate(cudisc_grid g, cudisc_bins b, double *rho_dust, double t_span, double dt_try,
                          int max_steps, double *dt_log, cudisc_integrate_info *info,
                          cudisc_stream stream);

/* Same, but stops after n_accepted accepted steps instead of at a time (BASELINE.json config 4:
 * "integrate 1000 coagulation steps"); info->t_done is the time reached. */
int cudisc_coag_integrate_steps(cudisc_grid g, cudisc_bins b, double *rho_dust, int n_accepted, double dt_try,
                                int max_steps, double *dt_log, cudisc_integrate_info *info,
                                cudisc_stream stream);

/* ---------------------------------------------------------------------------------------------
 * Vertical hydrostatic equilibrium of the gas (Eqs. 32-37): the step
 * that produces the rho_gas the coagulation path consumes.
 * ------------------------------------------------------------------------------------------- */

typedef struct cudisc_hydro_s *cudisc_hydro;   /* grid geometry on the device; owned by the library */

/* Geometry of the (R, theta) grid of PAPER.md:29-38: R_edges [n_r + 1], tan_edges [n_z + 1] (tan theta at
 * the cell interfaces, j = 0 nearest the mid-plane), R_centres [n_r], tan_centres [n_z] (HOST, copied;
 * strictly increasing, centres inside their cells).  Uploads d(R^3)_i (Eq. 1), (R dR)_i = d(R^2)_i / 2
 * (PAPER.md:264), d(tan theta)_j and the centres to the current device.  n_z <= 4096. */
int cudisc_hydro_create(int n_r, int n_z, const double *R_edges, const double *tan_edges,
                        const double *R_centres, const double *tan_centres, cudisc_hydro *out);
int cudisc_hydro_destroy(cudisc_hydro h);

/* rho_gas_out [n_r x n_z] (DEVICE, j fastest) <- hydrostatic gas density of every radial column:
 *   P_{i,j} / P_{i,j-1} = exp[ GM <1/c_s^2>_{i,j} (1/r_{i,j} - 1/r_{i,j-1}) ]   (Eqs. 34, 35),
 *   r_{i,j} = R^c_i sqrt(1 + tan^2 theta^c_j); multiplicative scan over j from the cell nearest the
 *   mid-plane (Eq. 36; reading R17); omega = P / c_s^2; rho = Sigma_g (R dR) omega / sum_k omega V (Eq. 37,
 *   taken literally: the cells on the grid carry Sigma_g, reading R18).
 * cs2: DEVICE [n_r x n_z] isothermal sound speed squared, cm^2/s^2 (k_B T / mu m_H); Sigma_g: DEVICE [n_r],
 * g/cm^2; GM: G M_*, cm^3/s^2.  May not alias.  Only enqueues on `stream`; allocates nothing. */
int cudisc_hydrostatic(cudisc_hydro h, const double *cs2, const double *Sigma_g, double GM,
                       double *rho_gas_out, cudisc_stream stream);

const char *cudisc_hydro_last_error(void);

/* ---------------------------------------------------------------------------------------------
 * Roofline denominators measured in the same process (north_star: "peaks measured by a
 * microbenchmark in the same run").  Both synchronise the device.
 * ------------------------------------------------------------------------------------------- */

/* Dependent-chain-free DFMA loop on every SM: *dfma_per_s = FP64 fused multiply-adds per second
 * (thread-level operations).  n_iter <= 0 picks a default that runs for ~50 ms. */
int cudisc_microbench_dfma(int n_iter, double *dfma_per_s, double *elapsed_ms);

/* STREAM-style device copy of n_bytes (read + write counted): *bytes_per_s. */
int cudisc_microbench_copy(long long n_bytes, double *bytes_per_s, double *elapsed_ms);

/* Number of kernels this library has launched in this process (bench.py's gpu_launches). */
long long cudisc_launch_count(void);

const char *cudisc_last_error(void);
const char *cudisc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CUDISC_COAG_H */
