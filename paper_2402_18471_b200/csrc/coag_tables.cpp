// coag_tables.cpp -- host construction of the grid-only tables (see coag_tables.h).
// Written from PAPER.md:442-476 (Eqs. 63-68) and DESIGN.md readings R1, R2, R7, R8, R9.
// Shares nothing with oracle/.
#include "coag_tables.h"

#include <algorithm>
#include <cmath>
#include <string>

namespace cudisc {

namespace {

constexpr double kPi = 3.14159265358979323846;

// Two-bin split of a product mass (Eqs. 63-65; R7: lower bin = last centre <= mass; R8: masses
// off the grid go entirely to the first / last bin).
struct Split {
    int lo;        // -1: below the grid (all to bin 0); N-1: at/above the top (all to N-1)
    double eps;    // mass fraction to lo; 1 - eps to lo + 1
};

// number_split (reading R11, variant): the bins receive the NUMBER fractions eps, 1 - eps of the product,
// i.e. the masses eps m_lo and (1 - eps) m_lo+1 (they also sum to `mass`): mass fraction eps m_lo / mass.
Split split_mass(const std::vector<double> &m, double mass, bool number_split)
{
    const int N = (int)m.size();
    if (mass < m[0]) return {-1, 0.0};
    if (mass >= m[N - 1]) return {N - 1, 1.0};
    int lo = (int)(std::upper_bound(m.begin(), m.end(), mass) - m.begin()) - 1;
    double eps = (m[lo + 1] - mass) / (m[lo + 1] - m[lo]);
    if (number_split) eps = eps * m[lo] / mass;
    return {lo, eps};
}

// smallest l with upper edge above the mass (clamped to the last bin).
int l_bin(const std::vector<double> &me, double mass)
{
    const int N = (int)me.size() - 1;
    int l = (int)(std::upper_bound(me.begin() + 1, me.end(), mass) - (me.begin() + 1));
    return std::min(l, N - 1);
}

enum CoagCase { COAG_NEXT, COAG_TOP, COAG_FAR };

CoagCase coag_case(const std::vector<double> &m, int i, int j)
{
    const int N = (int)m.size();
    if (i < N - 1 && m[j] < m[i + 1] - m[i]) return COAG_NEXT;   // product inside [m_i, m_{i+1})
    if (i == N - 1) return COAG_TOP;                              // R8
    return COAG_FAR;
}

bool frag_near(const std::vector<double> &m, double chi, int i, int j)
{
    return i >= 1 && chi * m[j] <= m[i] - m[i - 1];               // remnant inside (m_{i-1}, m_i]
}

// All outcomes of pair (i, j) that are NOT covered by the column sums, as (target, plane, coef)
// for unit n_i n_j K; `with_columns` additionally emits the column part (loss of bin j and the
// fragment source), which the expanded form needs.
void pair_outcomes(const HostTables &t, int i, int j, bool with_columns, bool skip_row_part,
                   std::vector<BandEntry> &out)
{
    const std::vector<double> &m = t.m;
    const int N = t.N;
    const double chi = t.chi;
    const double mi = m[i], mj = m[j];
    auto emit = [&](int target, int plane, double coef) {
        out.push_back({target, i, j, plane, coef});
    };
    if (!skip_row_part) {
        // ---- coagulation product m_i + m_j
        switch (coag_case(m, i, j)) {
        case COAG_NEXT: {
            double D = m[i + 1] - mi;
            if (t.variant & kVarNumberSplit) {
                // number m_j / D of the product arrives in bin i + 1 (mass m_{i+1} each), the rest stays in bin i
                emit(i, 0, -mj * mi / D);
                emit(i + 1, 0, mj * m[i + 1] / D);
            } else {
                emit(i, 0, mj * (m[i + 1] - 2.0 * mi - mj) / D);
                emit(i + 1, 0, mj * (mi + mj) / D);
            }
            break;
        }
        case COAG_TOP:
            emit(N - 1, 0, mj);
            break;
        case COAG_FAR: {
            double M = mi + mj;
            Split s = split_mass(m, M, t.variant & kVarNumberSplit);
            emit(i, 0, -mi);
            if (s.lo == N - 1) emit(N - 1, 0, M);
            else { emit(s.lo, 0, M * s.eps); emit(s.lo + 1, 0, M * (1.0 - s.eps)); }
            break;
        }
        }
        // ---- fragmentation: remnant of the target (Eq. 68)
        double x = chi * mj;
        double m_rem = (x < mi) ? mi - x : 0.0;
        if (frag_near(m, chi, i, j)) {
            double Dp = mi - m[i - 1];
            if (t.variant & kVarNumberSplit) {
                // number chi m_j / D' of the remnant drops to bin i - 1 (mass m_{i-1} each)
                emit(i, 1, -x * mi / Dp);
                emit(i - 1, 1, x * m[i - 1] / Dp);
            } else {
                emit(i, 1, -x * (1.0 + m_rem / Dp));
                emit(i - 1, 1, m_rem * x / Dp);
            }
        } else {
            emit(i, 1, -mi);
            if (m_rem > 0.0) {
                Split s = split_mass(m, m_rem, t.variant & kVarNumberSplit);
                if (s.lo == -1) emit(0, 1, m_rem);
                else if (s.lo == N - 1) emit(N - 1, 1, m_rem);
                else { emit(s.lo, 1, m_rem * s.eps); emit(s.lo + 1, 1, m_rem * (1.0 - s.eps)); }
            }
        }
    }
    // ---- column part: the impactor bin j always loses its own mass; fragments (R2)
    const bool col_frag = (i >= t.iS[j]);          // m_i > chi m_j: handled by the column sums
    if (with_columns) {
        emit(j, 0, -mj);
        emit(j, 1, -mj);
        if (col_frag) emit(N + t.lj[j], 1, mj + chi * mj);
    }
    if (!col_frag) {
        // largest fragment limited by the target mass: m_lf = m_i, m_ft = m_j + m_i
        if (!with_columns) emit(j, 1, -mj);        // Kf loss of bin j not in the column sum either
        emit(N + l_bin(t.me, (t.variant & kVarTotalLookup) ? mj + mi : mi), 1, mj + mi);
    }
}

}  // namespace

std::string build_log_grid(int N, double a_min, double a_max, double rho_m,
                           std::vector<double> &m, std::vector<double> &me, std::vector<double> &a)
{
    if (N < 2) return "n_bins < 2";
    if (!(a_min > 0.0) || !(a_max > a_min)) return "need 0 < a_min < a_max";
    if (!(rho_m > 0.0)) return "rho_m <= 0";
    std::vector<double> ae(N + 1);
    me.resize(N + 1); m.resize(N); a.resize(N);
    for (int k = 0; k <= N; ++k) {
        ae[k] = a_min * std::pow(a_max / a_min, (double)k / (double)N);
        me[k] = (4.0 * kPi / 3.0) * rho_m * ae[k] * ae[k] * ae[k];
    }
    for (int k = 0; k < N; ++k) {
        a[k] = std::sqrt(ae[k] * ae[k + 1]);
        m[k] = std::sqrt(me[k] * me[k + 1]);
    }
    return "";
}

std::string build_tables(const std::vector<double> &m, const std::vector<double> &me,
                         const std::vector<double> &a, double rho_m, double eta, double chi, int variant,
                         HostTables &t)
{
    if (variant & ~(kVarNumberSplit | kVarTotalLookup)) return "unknown bits in params.readings";
    const int N = (int)m.size();
    if (N < 2) return "n_bins < 2";
    if ((int)me.size() != N + 1 || (int)a.size() != N) return "inconsistent grid arrays";
    if (!(eta < 2.0)) return "eta must be < 2";
    if (!(chi > 0.0)) return "chi_im must be > 0";
    for (int k = 0; k < N; ++k) {
        if (!(me[k] > 0.0) || !(me[k] < m[k]) || !(m[k] < me[k + 1])) return "mass grid not monotone";
        if (!(a[k] > 0.0)) return "non-positive grain radius";
    }
    t = HostTables();
    t.N = N; t.rho_m = rho_m; t.eta = eta; t.chi = chi; t.variant = variant;
    t.m = m; t.me = me; t.a = a;
    t.rm.resize(N);
    for (int k = 0; k < N; ++k) t.rm[k] = 1.0 / m[k];
    t.sS = 1.0 + chi;

    // ---- columns: iS, lj
    t.iS.assign(N, N); t.lj.assign(N, 0);
    for (int j = 0; j < N; ++j) {
        for (int i = j; i < N; ++i)
            if (chi * m[j] < m[i]) { t.iS[j] = i; break; }
        t.lj[j] = l_bin(me, (variant & kVarTotalLookup) ? m[j] + chi * m[j] : chi * m[j]);
    }
    t.jS_lo.assign(N, 0); t.jS_hi.assign(N, 0);
    for (int l = 0; l < N; ++l) {
        int lo = (int)(std::lower_bound(t.lj.begin(), t.lj.end(), l) - t.lj.begin());
        int hi = (int)(std::upper_bound(t.lj.begin(), t.lj.end(), l) - t.lj.begin());
        t.jS_lo[l] = lo; t.jS_hi[l] = hi;
    }

    // ---- bulk rows: prefix of j where the product stays next to bin i for BOTH outcomes
    t.n_bulk.assign(N, 0);
    t.cA1.assign(N, 0); t.cA2.assign(N, 0); t.cB1.assign(N, 0); t.cB2.assign(N, 0);
    t.cF1.assign(N, 0); t.cF2.assign(N, 0); t.cG1.assign(N, 0); t.cG2.assign(N, 0);
    for (int i = 0; i < N; ++i) {
        int nb = 0;
        for (int j = 0; j <= i; ++j) {
            CoagCase cc = coag_case(m, i, j);
            if (cc == COAG_FAR || !frag_near(m, chi, i, j)) break;
            nb = j + 1;
        }
        t.n_bulk[i] = nb;
        if (nb == 0) continue;
        // coagulation:  Rc m_j (m_{i+1} - 2 m_i - m_j) / D -> bin i ;  Rc m_j (m_i + m_j) / D -> bin i+1
        if (i < N - 1 && (variant & kVarNumberSplit)) {
            double D = m[i + 1] - m[i];             // -Rc m_j m_i / D -> bin i ;  Rc m_j m_{i+1} / D -> bin i+1
            t.cA1[i] = -m[i] / D;
            t.cB1[i] = m[i + 1] / D;
        } else if (i < N - 1) {
            double D = m[i + 1] - m[i];
            t.cA1[i] = (m[i + 1] - 2.0 * m[i]) / D; t.cA2[i] = -1.0 / D;
            t.cB1[i] = m[i] / D;                    t.cB2[i] = 1.0 / D;
        } else {
            t.cA1[i] = 1.0;                         // R8: product stays in the top bin
        }
        // fragmentation: -Rf chi m_j (1 + (m_i - chi m_j)/D') -> bin i ; Rf (m_i - chi m_j) chi m_j / D' -> i-1
        double Dp = m[i] - m[i - 1];               // nb > 0 implies i >= 1
        if (variant & kVarNumberSplit) {           // -Rf chi m_j m_i / D' -> bin i ;  Rf chi m_j m_{i-1} / D' -> i-1
            t.cF1[i] = -chi * m[i] / Dp;
            t.cG1[i] = chi * m[i - 1] / Dp;
        } else {
            t.cF1[i] = -chi * (1.0 + m[i] / Dp);  t.cF2[i] = chi * chi / Dp;
            t.cG1[i] = chi * m[i] / Dp;           t.cG2[i] = -chi * chi / Dp;
        }
    }

    // ---- band: everything outside the bulk prefixes, plus what the column sums do not cover
    for (int i = 0; i < N; ++i)
        for (int j = 0; j <= i; ++j)
            pair_outcomes(t, i, j, /*with_columns=*/false, /*skip_row_part=*/j < t.n_bulk[i], t.band);
    std::stable_sort(t.band.begin(), t.band.end(), [](const BandEntry &x, const BandEntry &y) {
        if (x.target != y.target) return x.target < y.target;
        if (x.i != y.i) return x.i < y.i;
        if (x.j != y.j) return x.j < y.j;
        return x.plane < y.plane;
    });

    // ---- fragment power law (Eq. 67): N_k(m^e_{l+1}) = A_k / B_l for k <= l
    t.fA.resize(N); t.finvB.resize(N);
    const double ex = 2.0 - eta;
    const double p0 = std::pow(me[0], ex);
    for (int k = 0; k < N; ++k) {
        t.fA[k] = std::pow(me[k + 1], ex) - std::pow(me[k], ex);
        t.finvB[k] = 1.0 / (std::pow(me[k + 1], ex) - p0);
    }
    return "";
}

void expand_outcomes(const HostTables &t, std::vector<BandEntry> &out)
{
    out.clear();
    for (int i = 0; i < t.N; ++i)
        for (int j = 0; j <= i; ++j) {
            size_t first = out.size();
            const bool bulk = j < t.n_bulk[i];
            if (bulk) {
                // the row-sum coefficients written out for this pair: y_j = n_j m_j
                const double mj = t.m[j], mj2 = t.m[j] * t.m[j];
                out.push_back({i, i, j, 0, t.cA1[i] * mj + t.cA2[i] * mj2});
                if (i + 1 < t.N) out.push_back({i + 1, i, j, 0, t.cB1[i] * mj + t.cB2[i] * mj2});
                out.push_back({i, i, j, 1, t.cF1[i] * mj + t.cF2[i] * mj2});
                out.push_back({i - 1, i, j, 1, t.cG1[i] * mj + t.cG2[i] * mj2});
            }
            pair_outcomes(t, i, j, /*with_columns=*/true, /*skip_row_part=*/bulk, out);
            if (i == j)
                for (size_t e = first; e < out.size(); ++e) out[e].coef *= 0.5;
        }
}

}  // namespace cudisc
