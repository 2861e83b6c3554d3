// coag_tables.h -- host-side, grid-only tables of the rate evaluation (internal header).
//
// Everything here depends only on the mass grid, eta and chi_im: it is
// computed once per cudisc_bins handle on the host and uploaded.  The decomposition of the
// pair-flux form of Eqs. 53/54/61-68 is:
//
//   bulk rows   : for target row i and impactors j < n_bulk[i] both the coagulation product
//                 (inside [m_i, m_{i+1}), or i = N-1) and the remnant (inside (m_{i-1}, m_i])
//                 stay next to bin i, so the deposits into bins i-1, i, i+1 are LINEAR in four
//                 row sums  A1 = sum_j Kc_ij y_j, A2 = sum_j Kc_ij y_j m_j, F1, F2 (same with Kf),
//                 y_j = rho_j.  Coefficients cA*, cB*, cF*, cG* below.
//   columns     : bin j always loses (Rc + Rf) m_j (Eq. 54 restricted to the smaller collider):
//                 G_j = sum_{i >= j} Kc_ij n_i + sum_{i >= iS[j]} Kf_ij n_i, and its fragments land in
//                 l-bin lj[j] with mass (1 + chi) m_j:  H_j = sum_{i >= iS[j]} Kf_ij n_i.
//   band        : every other pair outcome (products that leave the neighbourhood of bin i, rows
//                 near the diagonal, grid boundaries) as explicit gather entries per target bin.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace cudisc {

struct BandEntry {
    int target;   // [0, N): density bin; [N, 2N): S (l-bin) target - N
    int i, j;     // pair, i >= j
    int plane;    // 0: K p_coag, 1: K p_frag
    double coef;  // contribution = coef * n_i * n_j * Kplane_ij  (diagonal K already halved)
};

// Variants of two readings the paper cannot pin (R2, R11; cudisc_params.readings)
enum { kVarNumberSplit = 1,    // the two bins receive NUMBER fractions (masses eps m_l, (1 - eps) m_u)
       kVarTotalLookup = 2 };  // fragment l-bin looked up with the total fragment mass

struct HostTables {
    int N = 0;
    int variant = 0;
    double rho_m = 0, eta = 0, chi = 0;
    std::vector<double> m, me, a, rm;
    // bulk row coefficients: bin i   += n_i (cA1 A1 + cA2 A2 + cF1 F1 + cF2 F2)
    //                        bin i+1 += n_i (cB1 A1 + cB2 A2)
    //                        bin i-1 += n_i (cG1 F1 + cG2 F2)
    std::vector<double> cA1, cA2, cB1, cB2, cF1, cF2, cG1, cG2;
    std::vector<int> n_bulk;   // per row i
    std::vector<int> iS;       // per column j: first row i >= j with m_i > chi m_j (N if none)
    std::vector<int> lj;       // per column j: l-bin of chi m_j
    std::vector<int> jS_lo, jS_hi;   // per l: columns j in [jS_lo, jS_hi) have lj[j] == l
    double sS = 0;             // (1 + chi)
    std::vector<double> fA, finvB;   // Eq. 67: A_k and 1 / B_l
    std::vector<BandEntry> band;     // sorted by (target, i, j, plane)
};

// Returns an empty string on success, else the reason the grid is rejected.
std::string build_log_grid(int N, double a_min, double a_max, double rho_m,
                           std::vector<double> &m, std::vector<double> &me, std::vector<double> &a);
std::string build_tables(const std::vector<double> &m, const std::vector<double> &me,
                         const std::vector<double> &a, double rho_m, double eta, double chi, int variant,
                         HostTables &out);

// Expanded gather form of ALL outcomes (bulk written out pair by pair) for host-side checking;
// here the diagonal 1/2 is folded into coef (K is the plain, un-halved kernel).
void expand_outcomes(const HostTables &t, std::vector<BandEntry> &out);

}  // namespace cudisc
