/*
 * coag_oracle.c -- TEST INFRASTRUCTURE.  Plain, slow, obviously-correct CPU restatement of the
 * per-cell Smoluchowski coagulation/fragmentation update of cuDisc, written from
 * /root/reference/PAPER.md section 5.  Every function cites the passage it
 * follows.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_2402_18471_b200/csrc/ and is only ever called from tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs.
 *
 * All FP64 (the paper fixes no precision; BASELINE.json asks for FP64), CGS units.
 * [C x N] arrays are row-major, bin fastest.
 *
 * Readings of the paper where it is silent/garbled are DESIGN.md "Readings" R1..R16 (named
 * G1..G16 in SURVEY.md section 8(c)); each is flagged at its use below.
 *
 * Pin status (tests/test_oracle_*.py, -m "not gpu"):
 *   orc_mass_grid ............ pinned (PAPER.md:503 mass ratio 1.38 for both published grids)
 *   orc_pfrag ................ pinned (closed form 2.5 e^-1.5 at dv = v_frag; limits 0 and 1)
 *   orc_split ................ pinned (weights sum to 1, mass m reproduced, brute force)
 *   orc_rates_literal_q ...... pinned (exact-rational brute force on 8-bin grids in the test)
 *   orc_rates_flux ........... pinned (== literal form in exact arithmetic; sum_k = 0; closed-form
 *                              constant and additive kernel solutions; pure-sticking invariant)
 *   orc_frag_redistribute .... pinned (telescoping sum = 1; brute force against Eq. 67 directly)
 *   orc_bs32_step ............ pinned (order of convergence 3, exact on cubic-in-t test ODE via
 *                              the generic-rhs twin in the tests; conservation 1e-13)
 *   orc_vint_scale ........... pinned (quadrature of the product of two Gaussian vertical profiles)
 *   orc_cell_kernel .......... Brownian/laminar parts + regime limits of the turbulent part pinned;
 *                              PARITY UNPINNED for: sigma_ij = pi (a_i+a_j)^2 (R3), the Ormel &
 *                              Cuzzi formulas as recalled (R4, limits pinned only), nu_mol (R6),
 *                              fragment l-bin lookup mass (R2), linear mass-fraction split (R11),
 *                              error norm (R10).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_KB 1.380649e-16   /* erg/K   (R16) */
#define ORC_MH 1.6735575e-24  /* g       (R16) */
#define ORC_PI 3.14159265358979323846

typedef struct {
    double mu;        /* mean molecular weight */
    double v_frag;    /* cm/s */
    double eta;       /* fragment slope */
    double chi_im;
    double sigma_mol; /* cm^2, R6 */
    double rtol;
    double atol_factor;
} orc_params;

/* ------------------------------------------------------------------------------------------
 * S0  Mass grid.  PAPER.md:442 (log mass grid), :467 (bin edges m^e_k, m^e_{k+1}), :503
 * ("100 dust species with grain sizes logarithmically spaced between 0.1 um and 0.5 cm ...
 * m_{n+1}/m_n = 1.38"): N bins <-> N+1 log-spaced edges spanning [a_min, a_max]; centres are the
 * geometric means of the edges.
 * ------------------------------------------------------------------------------------------ */
void orc_mass_grid(int N, double a_min, double a_max, double rho_m,
                   double *a_e, double *m_e, double *a_c, double *m_c)
{
    for (int k = 0; k <= N; ++k) {
        a_e[k] = a_min * pow(a_max / a_min, (double)k / (double)N);
        m_e[k] = (4.0 * ORC_PI / 3.0) * rho_m * a_e[k] * a_e[k] * a_e[k];
    }
    for (int k = 0; k < N; ++k) {
        a_c[k] = sqrt(a_e[k] * a_e[k + 1]);
        m_c[k] = sqrt(m_e[k] * m_e[k + 1]);
    }
}

/* PAPER.md:440, Eq. 62.  dv = 0 -> 0 (limit; R15). */
double orc_pfrag(double v_frag, double dv)
{
    if (!(dv > 0.0)) return 0.0;
    double x = 1.5 * (v_frag / dv) * (v_frag / dv);
    return (x + 1.0) * exp(-x);
}

/* Ormel & Cuzzi (2007) Eq. 21d as recalled in R4: root y* of
 *   (2/3) y (y-1)^2 - 1/(1+y) = -St/(1+St),   St < 1,
 * by exactly 6 Newton iterations from y0 = 1.6 - 0.6 St (no convergence test, so that any other
 * implementation can run the identical fixed procedure).  PAPER.md:430 uses an unpublished
 * quadratic fit "accurate to within 2%" to this root. */
double orc_ystar(double St)
{
    double y = 1.6 - 0.6 * St;
    double rhs = -St / (1.0 + St);
    for (int it = 0; it < 6; ++it) {
        double f = (2.0 / 3.0) * y * (y - 1.0) * (y - 1.0) - 1.0 / (1.0 + y) - rhs;
        double fp = (2.0 / 3.0) * (y - 1.0) * (3.0 * y - 1.0) + 1.0 / ((1.0 + y) * (1.0 + y));
        y -= f / fp;
    }
    return y;
}

/* St* of one grain: PAPER.md:587 (minimum Re^-1/2, maximum 1), R4. */
double orc_ststar(double St, double St_eta)
{
    double s;
    if (St >= 1.0) s = 1.0;
    else s = orc_ystar(St) * St;
    if (s < St_eta) s = St_eta;
    if (s > 1.0) s = 1.0;
    return s;
}

static double t_oc(double x, double a) { return x * x / (x + a); }

/* Ormel & Cuzzi (2007) Eqs. 17 and 18 as recalled in R4 (PAPER.md:430 cites them, does not print
 * them).  St1 >= St2, S = St*_12 = St* of the larger grain.  Returns dV_I^2 + dV_II^2 in units of
 * V_g^2 (Eq. 60 squared). */
double orc_vrel2_turb(double St1, double St2, double S, double St_eta)
{
    double dVI = (St1 - St2) / (St1 + St2) *
                 (t_oc(St1, S) - t_oc(St1, 1.0) - t_oc(St2, S) + t_oc(St2, 1.0));
    double dVII = 2.0 * (S - St_eta) + t_oc(St1, S) - t_oc(St1, St_eta)
                                     + t_oc(St2, S) - t_oc(St2, St_eta);
    if (dVI < 0.0) dVI = 0.0;
    if (dVII < 0.0) dVII = 0.0;
    return dVI + dVII;
}

/* ------------------------------------------------------------------------------------------
 * S1-S3  Collision kernel of one cell.  PAPER.md:410-440 (Eqs. 55-62).
 * Outputs K[i*N+j] = sigma_ij dv_ij (Eq. 56, full symmetric, NOT halved on the diagonal) and
 * pf[i*N+j] = p_frag,ij (Eq. 62).  vphi may be NULL.  St_out/Sstar_out (length N) optional.
 * ------------------------------------------------------------------------------------------ */
void orc_cell_kernel(int N, const double *a_c, const double *m_c, double rho_m,
                     double T, double rho_g, double Omega, double alpha,
                     const double *vR, const double *vZ, const double *vphi,
                     const orc_params *p, double *K, double *pf,
                     double *St_out, double *Sstar_out)
{
    /* S1: per-cell scalars */
    double cs = sqrt(ORC_KB * T / (p->mu * ORC_MH));
    double vth = sqrt(8.0 / ORC_PI) * cs;
    double Vg2 = alpha * cs * cs;                         /* PAPER.md:424, Eq. 59 squared */
    double H = cs / Omega;
    double nu_t = alpha * cs * H;
    double lambda = p->mu * ORC_MH / (rho_g * p->sigma_mol);
    double nu_mol = 0.5 * vth * lambda;                   /* R6 */
    double Re = nu_t / nu_mol;
    double St_eta = 1.0 / sqrt(Re);

    double *St = (double *)malloc(sizeof(double) * (size_t)N);
    double *Ss = (double *)malloc(sizeof(double) * (size_t)N);
    for (int i = 0; i < N; ++i) {
        St[i] = rho_m * a_c[i] / (rho_g * vth) * Omega;   /* PAPER.md:117, Eq. 14 (R14) times Omega */
        Ss[i] = orc_ststar(St[i], St_eta);
        if (St_out) St_out[i] = St[i];
        if (Sstar_out) Sstar_out[i] = Ss[i];
    }
    for (int i = 0; i < N; ++i) {
        for (int j = 0; j <= i; ++j) {
            double sigma = ORC_PI * (a_c[i] + a_c[j]) * (a_c[i] + a_c[j]);          /* R3 */
            double vbm2 = 8.0 * ORC_KB * T * (m_c[i] + m_c[j]) / (ORC_PI * m_c[i] * m_c[j]); /* Eq. 58 */
            double vt2 = Vg2 * orc_vrel2_turb(St[i], St[j], Ss[i], St_eta);         /* Eqs. 59-60 */
            double dR = vR[i] - vR[j], dZ = vZ[i] - vZ[j];
            double vl2 = dR * dR + dZ * dZ;
            if (vphi) { double dP = vphi[i] - vphi[j]; vl2 += dP * dP; }
            double dv = sqrt(vbm2 + vt2 + vl2);                                      /* Eq. 57 */
            double k = sigma * dv;                                                   /* Eq. 56 */
            double f = orc_pfrag(p->v_frag, dv);                                     /* Eq. 62 */
            K[i * N + j] = K[j * N + i] = k;
            pf[i * N + j] = pf[j * N + i] = f;
        }
    }
    free(St); free(Ss);
}

/* Vertically integrated kernel: "constructed by dividing the coagulation kernel (Eqn. 56)
 * by sqrt(2 pi (h_i^2 + h_j^2)), where h_i & h_j are the scale heights of the dust grains, assuming a
 * Gaussian vertical density profile".  hd[N]: dust scale heights (an input, like the velocities).
 * K: full N x N, scaled in place; p_frag is a function of dv only and stays.
 * Pinned (tests/test_oracle_pins.py) by numerical quadrature of the product of two Gaussians. */
void orc_vint_scale(int N, const double *hd, double *K)
{
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j)
            K[i * N + j] /= sqrt(2.0 * ORC_PI * (hd[i] * hd[i] + hd[j] * hd[j]));
}

/* ------------------------------------------------------------------------------------------
 * S5  Two-bin split.  PAPER.md:442-457 (Eqs. 63-65) with reading R7 (non-strict lower bound:
 * l = largest index with m_l <= m) and R8 (off-grid products: everything into bin N-1, resp. 0).
 * Returns l in [-1, N-1]; *eps = mass fraction to bin l, 1-*eps to bin l+1.
 *   m <  m_0      -> l = -1, eps = 0   (all of it to bin 0)
 *   m >= m_{N-1}  -> l = N-1, eps = 1  (all of it to bin N-1)
 * ------------------------------------------------------------------------------------------ */
/* Variants of two readings the paper cannot pin (R2, R11), switched for the
 * whole oracle by orc_set_variant (default 0 = the readings taken):
 *   bit 0 (ORC_VAR_NUMBER_SPLIT)  PAPER.md:446 "fractions of the mass": instead of the literal mass
 *         fractions (eps m, (1 - eps) m) the two bins receive the NUMBER fractions eps, 1 - eps of the
 *         product (Kovetz & Olund 1969): masses eps m_l and (1 - eps) m_u, which also sum to m.
 *   bit 1 (ORC_VAR_TOTAL_LOOKUP)  PAPER.md:469-476: the l-bin of the largest fragment is looked up with
 *         the total fragment mass m_j + min(chi m_j, m_i) instead of min(chi m_j, m_i). */
enum { ORC_VAR_NUMBER_SPLIT = 1, ORC_VAR_TOTAL_LOOKUP = 2 };
static int orc_variant = 0;
void orc_set_variant(int v) { orc_variant = v; }
int orc_get_variant(void) { return orc_variant; }

int orc_split(int N, const double *m_c, double m, double *eps)
{
    if (m < m_c[0]) { *eps = 0.0; return -1; }
    if (m >= m_c[N - 1]) { *eps = 1.0; return N - 1; }
    int l = 0;
    while (l + 1 < N && m_c[l + 1] <= m) ++l;
    *eps = (m_c[l + 1] - m) / (m_c[l + 1] - m_c[l]);     /* Eq. 65 */
    if (orc_variant & ORC_VAR_NUMBER_SPLIT) *eps = *eps * m_c[l] / m;   /* number eps -> mass eps m_l / m */
    return l;
}

/* "the smallest l such that m^e_{l+1} > m_frag". */
int orc_lbin(int N, const double *m_e, double m)
{
    int l = 0;
    while (l < N - 1 && !(m_e[l + 1] > m)) ++l;
    return l;
}

/* Eq. 68 and the sentence after it; R2.
 * tar = heavier (i), im = lighter (j).  m_ft evaluated as m_j + min(chi m_j, m_i), never by
 * subtraction.  m_lf = mass used to look up the largest fragment's bin. */
static void outcome_masses(double mi, double mj, double chi, double *m_rem, double *m_ft, double *m_lf)
{
    double x = chi * mj;
    *m_rem = (x < mi) ? (mi - x) : 0.0;
    *m_lf = (x < mi) ? x : mi;
    *m_ft = mj + *m_lf;
    if (orc_variant & ORC_VAR_TOTAL_LOOKUP) *m_lf = *m_ft;
}

/* ------------------------------------------------------------------------------------------
 * S6-O1  Literal rate equation.  PAPER.md:396-404 (Eqs. 53, 54), :432-436 (Eq. 61 and the
 * diagonal 1/2 rule, reading R1: gain only), with C_ijk, R_ijk (Eqs. 63-64) and
 * F_ijk = N_k(m^e_{l+1}) (Eq. 67, used DIRECTLY here, not via the l-bin shortcut), a full
 * triple loop over (i, j<=i, k), accumulated in __float128.  This is the definition; it is
 * numerically unusable in double on wide grids (R9) and exists to pin orc_rates_flux.
 * K, pf: full N x N.  Output rounded to double.
 * ------------------------------------------------------------------------------------------ */
void orc_rates_literal_q(int N, const double *m_c, const double *m_e, const double *K,
                         const double *pf, const double *rho, double eta, double chi,
                         double *drho)
{
    __float128 *acc = (__float128 *)calloc((size_t)N, sizeof(__float128));
    double ex = 2.0 - eta;
    for (int i = 0; i < N; ++i) {
        for (int j = 0; j <= i; ++j) {
            __float128 ni = (__float128)rho[i] / m_c[i], nj = (__float128)rho[j] / m_c[j];
            __float128 Kij = K[i * N + j];
            if (i == j) Kij *= 0.5;
            __float128 pfr = pf[i * N + j], pco = 1.0 - pfr;            /* Eq. 55 */
            double m_rem, m_ft, m_lf;
            outcome_masses(m_c[i], m_c[j], chi, &m_rem, &m_ft, &m_lf);
            double M = m_c[i] + m_c[j];
            double epsC, epsR = 0.0;
            int lC = orc_split(N, m_c, M, &epsC);
            int lR = -2;
            if (m_rem > 0.0) lR = orc_split(N, m_c, m_rem, &epsR);
            int lF = orc_lbin(N, m_e, m_lf);
            __float128 mmax = powl((long double)m_e[lF + 1], (long double)ex)
                            - powl((long double)m_e[0], (long double)ex);
            for (int k = 0; k < N; ++k) {
                __float128 Cijk = 0, Rijk = 0, Fijk = 0;
                if (lC == N - 1) { if (k == N - 1) Cijk = 1; }
                else { if (k == lC) Cijk = epsC; if (k == lC + 1) Cijk = 1.0 - (__float128)epsC; }
                if (lR != -2) {
                    if (lR == -1) { if (k == 0) Rijk = 1; }
                    else if (lR == N - 1) { if (k == N - 1) Rijk = 1; }
                    else { if (k == lR) Rijk = epsR; if (k == lR + 1) Rijk = 1.0 - (__float128)epsR; }
                }
                if (k <= lF)
                    Fijk = ((__float128)powl((long double)m_e[k + 1], (long double)ex)
                          - (__float128)powl((long double)m_e[k], (long double)ex)) / mmax; /* Eq. 67 */
                acc[k] += ni * nj * Kij * (pco * (__float128)M * Cijk
                          + pfr * ((__float128)m_rem * Rijk + (__float128)m_ft * Fijk)); /* Eq. 61 */
            }
        }
    }
    for (int k = 0; k < N; ++k) {                                        /* Eq. 54, full K_kk (R1) */
        __float128 nk = (__float128)rho[k] / m_c[k];
        for (int i = 0; i < N; ++i) {
            __float128 ni = (__float128)rho[i] / m_c[i];
            acc[k] -= (__float128)m_c[k] * ni * nk * (__float128)K[i * N + k];
        }
    }
    for (int k = 0; k < N; ++k) drho[k] = (double)acc[k];
    free(acc);
}

/* ------------------------------------------------------------------------------------------
 * S7  Fragment redistribution.  PAPER.md:465-469 (Eq. 67 and the l-bin two-stage algorithm):
 * S[l] = total fragment mass rate whose largest fragment falls in bin l; every S[l] is spread
 * over k <= l with N_k(m^e_{l+1}) = A_k / B_l.
 * ------------------------------------------------------------------------------------------ */
void orc_frag_redistribute(int N, const double *m_e, double eta, const double *S,
                           double *drho, double *gain)
{
    double ex = 2.0 - eta;
    double acc = 0.0;
    double p0 = pow(m_e[0], ex);
    for (int l = N - 1; l >= 0; --l) {
        double Bl = pow(m_e[l + 1], ex) - p0;
        double Al = pow(m_e[l + 1], ex) - pow(m_e[l], ex);
        acc += S[l] / Bl;
        drho[l] += Al * acc;
        if (gain) gain[l] += Al * acc;
    }
}

static void addpm(double *drho, double *gain, double *loss, int k, double v)
{
    drho[k] += v;
    if (v >= 0.0) gain[k] += v; else loss[k] -= v;
}

/* ------------------------------------------------------------------------------------------
 * S6-O2  Pair-flux form of Eqs. 53/54/61 (reading R9): algebraically identical to the literal
 * form (pinned in exact arithmetic by tests/test_oracle_rates.py), every term proportional to
 * the swept mass so that no catastrophic cancellation occurs on wide mass grids.
 * Kc = K p_coag and Kf = K p_frag, full N x N (not halved: the diagonal 1/2 is applied here,
 * PAPER.md:436); the rate form only ever uses these two products (R_c = n_i n_j K p_c,
 * R_f = n_i n_j K p_f).  orc_rates_flux() below is the (K, p_frag) front end.
 * Outputs: drho[N] (includes fragment redistribution S7), gain[N], loss[N] = sums of the
 * positive / |negative| contributions to each bin (for parity tolerances), S_out[N] optional.
 * ------------------------------------------------------------------------------------------ */
void orc_rates_flux_cf(int N, const double *m_c, const double *m_e, const double *Kc,
                       const double *Kf, const double *rho, double eta, double chi,
                       double *drho, double *gain, double *loss, double *S_out)
{
    double *S = (double *)calloc((size_t)N, sizeof(double));
    double *g = gain, *l = loss;
    int own = 0;
    if (!g) { g = (double *)calloc((size_t)N, sizeof(double)); l = (double *)calloc((size_t)N, sizeof(double)); own = 1; }
    else { memset(g, 0, sizeof(double) * (size_t)N); memset(l, 0, sizeof(double) * (size_t)N); }
    memset(drho, 0, sizeof(double) * (size_t)N);

    for (int i = 0; i < N; ++i) {
        double ni = rho[i] / m_c[i];
        for (int j = 0; j <= i; ++j) {
            double nj = rho[j] / m_c[j];
            double half = (i == j) ? 0.5 : 1.0;
            double Rf = half * ni * nj * Kf[i * N + j];
            double Rc = half * ni * nj * Kc[i * N + j];
            double mi = m_c[i], mj = m_c[j];

            /* --- coagulation product m_i + m_j (Eq. 63) */
            if (i < N - 1 && mj < m_c[i + 1] - mi) {
                double D = m_c[i + 1] - mi;                              /* product inside [m_i, m_{i+1}) */
                if (orc_variant & ORC_VAR_NUMBER_SPLIT) {
                    /* number eps = (D - m_j)/D stays in bin i (mass eps m_i, minus the m_i removed), number
                       m_j / D arrives in bin i+1 with mass m_{i+1} each: -m_i m_j / D and + m_{i+1} m_j / D */
                    addpm(drho, g, l, i, -Rc * mj * mi / D);
                    addpm(drho, g, l, i + 1, Rc * mj * m_c[i + 1] / D);
                } else {
                    addpm(drho, g, l, i, Rc * mj * (m_c[i + 1] - 2.0 * mi - mj) / D);
                    addpm(drho, g, l, i + 1, Rc * mj * (mi + mj) / D);
                }
                addpm(drho, g, l, j, -Rc * mj);
            } else if (i == N - 1) {                                     /* R8: stays in the top bin */
                addpm(drho, g, l, N - 1, Rc * mj);
                addpm(drho, g, l, j, -Rc * mj);
            } else {
                double eps; double M = mi + mj;
                int lo = orc_split(N, m_c, M, &eps);
                addpm(drho, g, l, i, -Rc * mi);
                addpm(drho, g, l, j, -Rc * mj);
                if (lo == N - 1) addpm(drho, g, l, N - 1, Rc * M);
                else { addpm(drho, g, l, lo, Rc * M * eps); addpm(drho, g, l, lo + 1, Rc * M * (1.0 - eps)); }
            }

            /* --- fragmentation: remnant (Eqs. 64, 68) and fragments (Eq. 67 via l-bins) */
            double m_rem, m_ft, m_lf;
            outcome_masses(mi, mj, chi, &m_rem, &m_ft, &m_lf);
            if (i >= 1 && chi * mj <= mi - m_c[i - 1]) {                 /* remnant inside (m_{i-1}, m_i] */
                double Dp = mi - m_c[i - 1];
                if (orc_variant & ORC_VAR_NUMBER_SPLIT) {
                    /* number chi m_j / D' of the remnant drops to bin i-1 (mass m_{i-1} each) */
                    addpm(drho, g, l, i, -Rf * chi * mj * mi / Dp);
                    addpm(drho, g, l, i - 1, Rf * chi * mj * m_c[i - 1] / Dp);
                } else {
                    addpm(drho, g, l, i, -Rf * chi * mj * (1.0 + m_rem / Dp));
                    addpm(drho, g, l, i - 1, Rf * m_rem * chi * mj / Dp);
                }
                addpm(drho, g, l, j, -Rf * mj);
            } else {
                addpm(drho, g, l, i, -Rf * mi);
                addpm(drho, g, l, j, -Rf * mj);
                if (m_rem > 0.0) {
                    double eps;
                    int lo = orc_split(N, m_c, m_rem, &eps);
                    if (lo == -1) addpm(drho, g, l, 0, Rf * m_rem);      /* R8 */
                    else if (lo == N - 1) addpm(drho, g, l, N - 1, Rf * m_rem);
                    else { addpm(drho, g, l, lo, Rf * m_rem * eps); addpm(drho, g, l, lo + 1, Rf * m_rem * (1.0 - eps)); }
                }
            }
            S[orc_lbin(N, m_e, m_lf)] += Rf * m_ft;
        }
    }
    orc_frag_redistribute(N, m_e, eta, S, drho, g);
    if (S_out) memcpy(S_out, S, sizeof(double) * (size_t)N);
    free(S);
    if (own) { free(g); free(l); }
}

/* (K, p_frag) front end: Kc = K (1 - p_frag) (Eq. 55), Kf = K p_frag. */
void orc_rates_flux(int N, const double *m_c, const double *m_e, const double *K,
                    const double *pf, const double *rho, double eta, double chi,
                    double *drho, double *gain, double *loss, double *S_out)
{
    double *Kc = (double *)malloc(sizeof(double) * (size_t)N * N * 2);
    double *Kf = Kc + (size_t)N * N;
    for (int q = 0; q < N * N; ++q) { Kf[q] = K[q] * pf[q]; Kc[q] = K[q] * (1.0 - pf[q]); }
    orc_rates_flux_cf(N, m_c, m_e, Kc, Kf, rho, eta, chi, drho, gain, loss, S_out);
    free(Kc);
}

/* ------------------------------------------------------------------------------------------
 * S8  One Bogacki-Shampine 3(2) step of one cell.  PAPER.md:478 names the method and the default
 * tolerances (rtol 1 %, atol 1e-10 * sum_k rho_k); the tableau is the textbook one
 * (Bogacki & Shampine 1989).  Kc = K p_coag, Kf = K p_frag (full N x N) are frozen over the
 * stages.
 * y[N] in/out; k1[N] in (if have_k1) and out (= k4, FSAL).  Returns the scaled error norm
 * E = max_k |e_k| / (atol + rtol max(|y_k|, |y'_k|))  (R10).
 * ------------------------------------------------------------------------------------------ */
double orc_bs32_step(int N, const double *m_c, const double *m_e, const double *Kc, const double *Kf,
                     double eta, double chi, double rtol, double atol_factor,
                     double *y, double *k1, int have_k1, double h)
{
    double *k2 = (double *)malloc(sizeof(double) * (size_t)N * 5);
    double *k3 = k2 + N, *k4 = k3 + N, *ys = k4 + N, *yn = ys + N;
    if (!have_k1) orc_rates_flux_cf(N, m_c, m_e, Kc, Kf, y, eta, chi, k1, NULL, NULL, NULL);
    for (int k = 0; k < N; ++k) ys[k] = y[k] + 0.5 * h * k1[k];
    orc_rates_flux_cf(N, m_c, m_e, Kc, Kf, ys, eta, chi, k2, NULL, NULL, NULL);
    for (int k = 0; k < N; ++k) ys[k] = y[k] + 0.75 * h * k2[k];
    orc_rates_flux_cf(N, m_c, m_e, Kc, Kf, ys, eta, chi, k3, NULL, NULL, NULL);
    for (int k = 0; k < N; ++k)
        yn[k] = y[k] + h * ((2.0 / 9.0) * k1[k] + (1.0 / 3.0) * k2[k] + (4.0 / 9.0) * k3[k]);
    orc_rates_flux_cf(N, m_c, m_e, Kc, Kf, yn, eta, chi, k4, NULL, NULL, NULL);
    double sum = 0.0;
    for (int k = 0; k < N; ++k) sum += y[k];
    double atol = atol_factor * sum;
    double E = 0.0;
    for (int k = 0; k < N; ++k) {
        double e = h * ((-5.0 / 72.0) * k1[k] + (1.0 / 12.0) * k2[k] + (1.0 / 9.0) * k3[k] - (1.0 / 8.0) * k4[k]);
        double sc = atol + rtol * fmax(fabs(y[k]), fabs(yn[k]));
        double r = (e == 0.0) ? 0.0 : fabs(e) / sc;   /* R10: e_k = 0 counts 0 (an empty cell has sc = 0: no 0/0) */
        if (r > E || r != r) E = r;
    }
    for (int k = 0; k < N; ++k) { y[k] = yn[k]; k1[k] = k4[k]; }
    free(k2);
    return E;
}

/* ------------------------------------------------------------------------------------------
 * Batch drivers over cells (cells are independent; OpenMP over cells only).
 * Packed planes layout (that of the C-ABI calls cudisc_coag_kernel / cudisc_coag_rates):
 * Kp[C][2][P], P = N(N+1)/2, lower-triangular i >= j at index i(i+1)/2 + j;
 * plane 0 = K_ij p_coag,ij, plane 1 = K_ij p_frag,ij, diagonal NOT halved.
 * ------------------------------------------------------------------------------------------ */

static double *grid_alloc(int N, double a_min, double a_max, double rho_m,
                          double **m_e, double **a_c, double **m_c)
{
    double *a_e = (double *)malloc(sizeof(double) * (size_t)(4 * N + 2));
    *m_e = a_e + N + 1; *a_c = *m_e + N + 1; *m_c = *a_c + N;
    orc_mass_grid(N, a_min, a_max, rho_m, a_e, *m_e, *a_c, *m_c);
    return a_e;
}

/* in place: (K, pf) -> (Kc, Kf) = (K (1 - pf), K pf)   (Eq. 55) */
static void to_products(int N, double *K, double *pf)
{
    for (int q = 0; q < N * N; ++q) { double k = K[q], f = pf[q]; pf[q] = k * f; K[q] = k * (1.0 - f); }
}

static void unpack_planes(int N, const double *Kp, double *Kc, double *Kf)
{
    size_t P = (size_t)N * (N + 1) / 2;
    for (int i = 0; i < N; ++i)
        for (int j = 0; j <= i; ++j) {
            size_t q = (size_t)i * (i + 1) / 2 + j;
            Kc[i * N + j] = Kc[j * N + i] = Kp[q];
            Kf[i * N + j] = Kf[j * N + i] = Kp[P + q];
        }
}

void orc_kernel_cells(int C, int N, double a_min, double a_max, double rho_m,
                      const double *T, const double *rho_g, const double *Omega, const double *alpha,
                      const double *vR, const double *vZ, const double *vphi,
                      const orc_params *p, double *K_out, const double *hd)
{
    size_t P = (size_t)N * (N + 1) / 2;
    double *m_e, *a_c, *m_c;
    double *a_e = grid_alloc(N, a_min, a_max, rho_m, &m_e, &a_c, &m_c);
#pragma omp parallel
    {
        double *K = (double *)malloc(sizeof(double) * (size_t)N * N * 2);
        double *pf = K + (size_t)N * N;
#pragma omp for schedule(dynamic, 4)
        for (int c = 0; c < C; ++c) {
            orc_cell_kernel(N, a_c, m_c, rho_m, T[c], rho_g[c], Omega[c], alpha[c],
                            vR + (size_t)c * N, vZ + (size_t)c * N, vphi ? vphi + (size_t)c * N : NULL,
                            p, K, pf, NULL, NULL);
            if (hd) orc_vint_scale(N, hd + (size_t)c * N, K);
            to_products(N, K, pf);
            double *o0 = K_out + (size_t)c * 2 * P, *o1 = o0 + P;
            for (int i = 0; i < N; ++i)
                for (int j = 0; j <= i; ++j) {
                    size_t q = (size_t)i * (i + 1) / 2 + j;
                    o0[q] = K[i * N + j];
                    o1[q] = pf[i * N + j];
                }
        }
        free(K);
    }
    free(a_e);
}

/* Rates from supplied packed planes; planes shared by all cells if per_cell == 0. */
void orc_rates_cells_planes(int C, int N, double a_min, double a_max, double rho_m,
                            double eta, double chi, const double *Kp, int per_cell,
                            const double *rho, double *drho, double *gain, double *loss)
{
    size_t P = (size_t)N * (N + 1) / 2;
    double *m_e, *a_c, *m_c;
    double *a_e = grid_alloc(N, a_min, a_max, rho_m, &m_e, &a_c, &m_c);
#pragma omp parallel
    {
        double *Kc = (double *)malloc(sizeof(double) * (size_t)N * N * 2);
        double *Kf = Kc + (size_t)N * N;
        if (!per_cell) unpack_planes(N, Kp, Kc, Kf);
#pragma omp for schedule(dynamic, 4)
        for (int c = 0; c < C; ++c) {
            if (per_cell) unpack_planes(N, Kp + (size_t)c * 2 * P, Kc, Kf);
            orc_rates_flux_cf(N, m_c, m_e, Kc, Kf, rho + (size_t)c * N, eta, chi, drho + (size_t)c * N,
                              gain ? gain + (size_t)c * N : NULL, loss ? loss + (size_t)c * N : NULL, NULL);
        }
        free(Kc);
    }
    free(a_e);
}

/* Rates with the kernel built from the gas state. */
void orc_rates_cells(int C, int N, double a_min, double a_max, double rho_m,
                     const double *T, const double *rho_g, const double *Omega, const double *alpha,
                     const double *vR, const double *vZ, const double *vphi,
                     const orc_params *p, const double *rho, double *drho, double *gain, double *loss,
                     const double *hd)
{
    double *m_e, *a_c, *m_c;
    double *a_e = grid_alloc(N, a_min, a_max, rho_m, &m_e, &a_c, &m_c);
#pragma omp parallel
    {
        double *K = (double *)malloc(sizeof(double) * (size_t)N * N * 2);
        double *pf = K + (size_t)N * N;
#pragma omp for schedule(dynamic, 4)
        for (int c = 0; c < C; ++c) {
            orc_cell_kernel(N, a_c, m_c, rho_m, T[c], rho_g[c], Omega[c], alpha[c],
                            vR + (size_t)c * N, vZ + (size_t)c * N, vphi ? vphi + (size_t)c * N : NULL,
                            p, K, pf, NULL, NULL);
            if (hd) orc_vint_scale(N, hd + (size_t)c * N, K);
            to_products(N, K, pf);
            orc_rates_flux_cf(N, m_c, m_e, K, pf, rho + (size_t)c * N, p->eta, p->chi_im,
                              drho + (size_t)c * N, gain ? gain + (size_t)c * N : NULL,
                              loss ? loss + (size_t)c * N : NULL, NULL);
        }
        free(K);
    }
    free(a_e);
}

/* One BS3(2) step of every cell with the kernel built from the gas state (once per cell per step,
 * frozen over the stages).  rho [C x N] in/out, k1 [C x N] in/out (FSAL), err [C]. */
void orc_step_cells(int C, int N, double a_min, double a_max, double rho_m,
                    const double *T, const double *rho_g, const double *Omega, const double *alpha,
                    const double *vR, const double *vZ, const double *vphi,
                    const orc_params *p, double *rho, double *k1, int have_k1, double dt, double *err,
                    const double *hd)
{
    double *m_e, *a_c, *m_c;
    double *a_e = grid_alloc(N, a_min, a_max, rho_m, &m_e, &a_c, &m_c);
#pragma omp parallel
    {
        double *K = (double *)malloc(sizeof(double) * (size_t)N * N * 2);
        double *pf = K + (size_t)N * N;
#pragma omp for schedule(dynamic, 4)
        for (int c = 0; c < C; ++c) {
            orc_cell_kernel(N, a_c, m_c, rho_m, T[c], rho_g[c], Omega[c], alpha[c],
                            vR + (size_t)c * N, vZ + (size_t)c * N, vphi ? vphi + (size_t)c * N : NULL,
                            p, K, pf, NULL, NULL);
            if (hd) orc_vint_scale(N, hd + (size_t)c * N, K);
            to_products(N, K, pf);
            err[c] = orc_bs32_step(N, m_c, m_e, K, pf, p->eta, p->chi_im, p->rtol, p->atol_factor,
                                   rho + (size_t)c * N, k1 + (size_t)c * N, have_k1, dt);
        }
        free(K);
    }
    free(a_e);
}

/* Step with supplied packed planes (shared by all cells): closed-form kernel runs. */
void orc_step_cells_planes(int C, int N, double a_min, double a_max, double rho_m,
                           double eta, double chi, double rtol, double atol_factor,
                           const double *Kp, double *rho, double *k1, int have_k1, double dt, double *err)
{
    double *m_e, *a_c, *m_c;
    double *a_e = grid_alloc(N, a_min, a_max, rho_m, &m_e, &a_c, &m_c);
    double *Kc = (double *)malloc(sizeof(double) * (size_t)N * N * 2);
    double *Kf = Kc + (size_t)N * N;
    unpack_planes(N, Kp, Kc, Kf);
#pragma omp parallel for schedule(dynamic, 4)
    for (int c = 0; c < C; ++c)
        err[c] = orc_bs32_step(N, m_c, m_e, Kc, Kf, eta, chi, rtol, atol_factor,
                               rho + (size_t)c * N, k1 + (size_t)c * N, have_k1, dt);
    free(Kc);
    free(a_e);
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
