/* hydro_oracle.c -- CPU oracle of the vertical hydrostatic-equilibrium solve of cuDisc
 * (arXiv 2402.18471 section 3.5; Eqs. 32-37).  TEST INFRASTRUCTURE: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline legs may use it; it shares no code with
 * paper_2402_18471_b200/csrc/.  Plain C, FP64, the paper's order of operations, no blocking.
 *
 * Per radial column i (cells j = 0 .. n_z-1, j = 0 nearest the mid-plane):
 *   Eq. 35   <1/c_s^2>_{i,j} = (1/c_s^2_{i,j} + 1/c_s^2_{i,j-1}) / 2
 *   Eq. 34   P_{i,j} / P_{i,j-1} = exp[ G M_* <1/c_s^2>_{i,j} (1/r_{i,j} - 1/r_{i,j-1}) ],   j >= 1
 *   Eq. 36   P_{i,j} / P_{i,0} = prod_{k=1..j} P_{i,k} / P_{i,k-1}        (sequential product)
 *   omega_{i,j} = (P_{i,j} / P_{i,0}) / c_s^2_{i,j}                        (ideal gas, unnormalised density)
 *   Eq. 37   rho_{g,i,j} = Sigma_{g,i} (R dR)_i / (sum_k omega_{i,k} V_{i,k}) * omega_{i,j}
 * with r_{i,j} = R^c_i sqrt(1 + tan^2 theta^c_j) (Z^c = R^c tan theta^c), V_{i,j} =
 * d(R^3)_i d(tan theta)_j / 3 (Eq. 1) and (R dR)_i = d(R^2)_i / 2.
 *
 * Readings (R17, R18):
 *   R17  PAPER.md:258 says "relative to the cell at i = 0": the scan of Eq. 36 runs over Z, so the
 *        reference cell is j = 0.
 *   R18  Eq. 37 is taken literally: the cells of the column that are ON THE GRID carry Sigma_g (R dR);
 *        on the default one-sided grid (mirror symmetry) the caller passes the surface
 *        density of that side.
 * Pins (tests/test_oracle_hydro.py): the isothermal column against the closed form
 * exp[G M / c_s^2 (1/r - 1/r_0)] and its thin-disc Gaussian limit, sum_k rho V = Sigma (R dR),
 * a stratified column against adaptive quadrature of Eq. 33 with second-order convergence.
 */
#include <math.h>
#include <stddef.h>

/* R_e [n_r+1], tan_e [n_z+1]: edges; R_c [n_r], tan_c [n_z]: centres; cs2 [n_r x n_z] (j fastest);
 * Sigma [n_r]; rho_out [n_r x n_z]. */
void orc_hydrostatic(int n_r, int n_z, const double *R_e, const double *tan_e, const double *R_c,
                     const double *tan_c, const double *cs2, const double *Sigma, double GM,
                     double *rho_out)
{
    for (int i = 0; i < n_r; ++i) {
        const double *c = cs2 + (size_t)i * n_z;
        double *o = rho_out + (size_t)i * n_z;
        double dR3 = R_e[i + 1] * R_e[i + 1] * R_e[i + 1] - R_e[i] * R_e[i] * R_e[i];
        double RdR = 0.5 * (R_e[i + 1] * R_e[i + 1] - R_e[i] * R_e[i]);
        double P = 1.0, sum = 0.0;
        double r_prev = 0.0;
        for (int j = 0; j < n_z; ++j) {
            double r = R_c[i] * sqrt(1.0 + tan_c[j] * tan_c[j]);
            if (j > 0) {
                double avg = 0.5 * (1.0 / c[j] + 1.0 / c[j - 1]);               /* Eq. 35 */
                P *= exp(GM * avg * (1.0 / r - 1.0 / r_prev));                   /* Eqs. 34, 36 */
            }
            r_prev = r;
            double omega = P / c[j];
            double V = dR3 * (tan_e[j + 1] - tan_e[j]) / 3.0;                    /* Eq. 1 */
            o[j] = omega;
            sum += omega * V;
        }
        double norm = Sigma[i] * RdR / sum;                                       /* Eq. 37 */
        for (int j = 0; j < n_z; ++j) o[j] *= norm;
    }
}
