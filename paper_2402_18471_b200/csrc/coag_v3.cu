// coag_v3.cu -- the stencil cell kernel (sm_100a, FP64): cudisc_coag_step and cudisc_coag_rates_otf on
// mass grids that coag_v3_host.cpp accepts (every exact log grid whose cell fits an SM).
//
// Same mathematics and the same device routines (prologue, pair kernel, BS3(2) algebra) as the general
// kernel of coag_kernels.cu; what differs is where the collision kernel of the cell lives and how the
// work is dealt out (coag_v3.h):
//   * the build writes every K_ij twice: to the packed shared-memory row copy and to the column copy in
//     tensor memory (tcgen05.st, lane <-> column j, 8-row chunks); a 32 x 32 diagonal block is built with
//     its short and long rows folded into full warps, then copied to tensor memory with zeros above the
//     diagonal;
//   * a rate evaluation reads the row copy once (row pass) and the column copy once (column pass, one
//     tcgen05.ld of 8 rows per chunk);
//   * the near-diagonal outcomes are a stencil over the staged products y_i n_{i-d} K[i][i-d] with
//     warp-uniform coefficients from a small table in shared memory (+ a few exception entries at the grid
//     ends);
//   * every warp owns a static list of runs (kernel parameter V3Tables, copied to shared memory once per
//     launch): no queues, no atomics, fixed summation order -> results are bit-reproducible;
//   * nothing that is the same for every bin runs between two block barriers: the per-cell scalars of the
//     prologue are derived two cells ahead by the warp that has no part in the combine phase.
// One persistent CTA of 512 threads per SM; thread k < N owns bin k (state and derivatives in registers).
#include "coag_v3.h"
#include "coag_launch.h"

namespace cudisc {

namespace {

// ------------------------------------------------------------------------------------------ tensor memory
__device__ __forceinline__ uint32_t tq_addr(uint32_t tbase, int quarter, int col)
{
    return tbase + ((uint32_t)(32 * quarter) << 16) + (uint32_t)col;
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&v)[32])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
                 "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
                 "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};\n"
                 :: "r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
                    "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]),
                    "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]), "r"(v[20]), "r"(v[21]), "r"(v[22]), "r"(v[23]),
                    "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]), "r"(v[31])
                 : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                 "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
                   "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
                   "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                 : "r"(taddr) : "memory");
}
// 8-byte asynchronous global -> shared copy (LDGSTS): inputs of a cell are staged in shared memory
// while the build runs, without holding registers across it
__device__ __forceinline__ void cp_async8(void *dst_smem, const void *src_gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n"
                 :: "r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }
__device__ __forceinline__ double u2d(uint32_t lo, uint32_t hi) { return __hiloint2double((int)hi, (int)lo); }
__device__ __forceinline__ uint32_t dlo(double x) { return (uint32_t)__double2loint(x); }
__device__ __forceinline__ uint32_t dhi(double x) { return (uint32_t)__double2hiint(x); }


// ------------------------------------------------------------------------------------------ shared memory
// Fixed arrays at compile-time offsets (coag_v3.h kV3o*): their addresses fold into the instructions.
struct VSm {
    char *base;
    double2 *KR;        // row copy of the kernel, packed lower-triangular, diagonal halved (runtime offset)
    Smem s;             // the arrays the shared device routines address (coag_device.cuh)
    __device__ __forceinline__ double *RED() const { return reinterpret_cast<double *>(base + kV3oRED); }
    __device__ __forceinline__ int2 *BINI() const { return reinterpret_cast<int2 *>(base + kV3oBINI); }
    __device__ __forceinline__ double2 *YY() const { return reinterpret_cast<double2 *>(base + kV3oYY); }
    __device__ __forceinline__ double *NN() const { return reinterpret_cast<double *>(base + kV3oNN); }
    __device__ __forceinline__ double *BANDV() const { return reinterpret_cast<double *>(base + kV3oBANDV); }
    __device__ __forceinline__ double *WST() const { return reinterpret_cast<double *>(base + kV3oUNION); }
    __device__ __forceinline__ const V3Hot *HOT() const { return reinterpret_cast<const V3Hot *>(base + kV3oHOT); }
};

// a pair of the row copy: (Kc, Kf) pairs at KR[p], or -- PLANAR, cudisc_coag_rates: the store is the image of a cell's
// planes in HBM, filled by bulk copies -- two doubles P apart
template <bool PLANAR>
__device__ __forceinline__ double2 v3_kld(const double2 *KR, int P, int p)
{
    if (PLANAR) {
        const double *d = reinterpret_cast<const double *>(KR);
        return make_double2(d[p], d[P + p]);
    }
    return KR[p];
}

__device__ __forceinline__ VSm v3_carve(char *base, const DevTables &tb, const V3Tables &vt)
{
    VSm f;
    f.base = base;
    f.KR = (double2 *)(base + vt.oK);
    Smem &s = f.s;
    double *u = (double *)(base + kV3oUNION);
    s.YY = f.YY(); s.NN = f.NN();
    // grid-only tables of the pair kernel: shared memory if the cell leaves room, else read through L1
    s.DTAB = vt.oDTAB ? (double2 *)(base + vt.oDTAB) : const_cast<double2 *>(tb.dtab);
    s.EXPT = vt.oDTAB ? (double *)(base + vt.oDTAB + 16 * vt.N) : const_cast<double *>(tb.exptab);
    s.RED = f.RED();
    s.BANDV = s.BANDV2 = nullptr; s.WST = nullptr; s.BINC = nullptr; s.BINI = f.BINI();
    s.CTR = nullptr; s.SCHED = nullptr; s.ITB = s.ITE = nullptr; s.PARTR = s.PARTC = nullptr;
    s.RI = (double2 *)u;
    s.B0 = (double2 *)(u + 10 * kV3NpMax); s.B1 = (double2 *)(u + 12 * kV3NpMax);
    s.J2 = (double2 *)(u + 14 * kV3NpMax); s.J3 = (double2 *)(u + 16 * kV3NpMax);
    s.V5 = u + 18 * kV3NpMax;
    return f;
}

// ------------------------------------------------------------------------------------------ build
// rows [32 c + 8 k0, ...) of column block c in chunks of 8 rows (all rows >= 32 c + 32: no diagonal pair);
// lanes <-> columns j = 32 c + lane.  Two rows per iteration.
// KOUT (cudisc_coag_kernel): the pairs go to the planes kout[2][P] in HBM (a warp stores 256 contiguous bytes per
// row and plane) and nowhere else.
template <bool KOUT>
__device__ __forceinline__ void v3_build_rows(const V3Tables &vt, const VSm &f, const PairConst &pc,
                                              const V3ColRun &run, uint32_t tq, int lane, double *kout = nullptr)
{
    const Smem &s = f.s;
    const int N = vt.N;
    const int j = 32 * run.c + lane;                 // < N: the block has rows below it
    const RoleJ B = load_role_j<false>(s, j);
    const int iSj = (f.BINI()[j].x >> 9) & 0x1ff;
    int i = 32 * run.c + 8 * run.k0;
    const int iend = min(N, i + 8 * run.n);
    uint32_t ta = tq + (uint32_t)run.tcol;
    double2 *kr = f.KR + tri(i) + j;
#pragma unroll 1
    for (; i < iend; i += 2, ta += 8) {
        const bool two = i + 1 < iend;
        const int i2 = two ? i + 1 : i;
        const RoleI A1 = load_role_i<false, false>(s, i);
        const RoleI A2 = load_role_i<false, false>(s, i2);
        const double2 k1 = pair_kernel<false, true, false>(A1, B, i - j, pc, s);
        double2 k2 = pair_kernel<false, true, false>(A2, B, i2 - j, pc, s);
        if (KOUT) {
            double *ko = kout + tri(i) + j;
            __stcs(ko, k1.x); __stcs(ko + vt.P, k1.y);
            if (two) { __stcs(ko + i + 1, k2.x); __stcs(ko + vt.P + i + 1, k2.y); }
            continue;
        }
        kr[0] = k1;
        if (two) kr[i + 1] = k2;
        else k2 = make_double2(0.0, 0.0);            // the row past the grid stays 0 in the column copy
        kr += 2 * i + 3;                             // tri(i + 2) - tri(i)
        // column copy: Kf of rows below iS[j] is not part of the column sums (coag_tables.h)
        const double f1 = (i < iSj) ? 0.0 : k1.y, f2 = (i2 < iSj) ? 0.0 : k2.y;
        const uint32_t v[8] = {dlo(k1.x), dhi(k1.x), dlo(f1), dhi(f1), dlo(k2.x), dhi(k2.x), dlo(f2), dhi(f2)};
        tmem_st8(ta, v);
    }
}

// diagonal block c: rows folded two to a warp (V3Tables::foldA / foldB), two folded rows per iteration;
// then the block goes to tensor memory with zeros above the diagonal.  KOUT: straight to the planes in HBM, diagonal
// not halved (the planes hold K itself; the calls that read them halve it).
template <bool KOUT>
__device__ __forceinline__ void v3_build_diag(const V3Tables &vt, const VSm &f, const PairConst &pc,
                                              const V3ColRun &run, uint32_t tq, int lane, double *kout = nullptr)
{
    const Smem &s = f.s;
    const int N = vt.N, c = run.c, nf = f.HOT()->nFold[c];
    auto where = [&](int fi, int &i, int &j) -> bool {
        const int rA = f.HOT()->foldA[c][fi], rB = f.HOT()->foldB[c][fi];
        bool ok = true;
        int r = rA, q = lane;
        if (lane > rA) { r = rB; q = lane - rA - 1; ok = rB != 0xff && q <= rB; }
        if (!ok) { r = rA; q = 0; }
        i = 32 * c + r; j = 32 * c + q;
        return ok;
    };
#pragma unroll 1
    for (int fi = 0; fi < nf; fi += 2) {
        int i1, j1, i2, j2;
        const bool ok1 = where(fi, i1, j1);
        const bool ok2 = (fi + 1 < nf) ? where(fi + 1, i2, j2) : (where(fi, i2, j2), false);
        const RoleI A1 = load_role_i<false, true>(s, i1);
        const RoleJ B1 = load_role_j<false>(s, j1);
        const RoleI A2 = load_role_i<false, true>(s, i2);
        const RoleJ B2 = load_role_j<false>(s, j2);
        double2 k1 = pair_kernel<false, true, true>(A1, B1, i1 - j1, pc, s);
        double2 k2 = pair_kernel<false, true, true>(A2, B2, i2 - j2, pc, s);
        if (KOUT) {
            if (ok1) { double *ko = kout + tri(i1) + j1; __stcs(ko, k1.x); __stcs(ko + vt.P, k1.y); }
            if (ok2) { double *ko = kout + tri(i2) + j2; __stcs(ko, k2.x); __stcs(ko + vt.P, k2.y); }
            continue;
        }
        if (i1 == j1) { k1.x *= 0.5; k1.y *= 0.5; }
        if (i2 == j2) { k2.x *= 0.5; k2.y *= 0.5; }
        if (ok1) f.KR[tri(i1) + j1] = k1;
        if (ok2) f.KR[tri(i2) + j2] = k2;
    }
    if (KOUT) return;
    __syncwarp();
    const int j = 32 * c + lane;
    const int iSj = (j < N) ? ((f.BINI()[j].x >> 9) & 0x1ff) : 0;
#pragma unroll 1
    for (int kk = 0; kk < run.n; ++kk) {
        uint32_t v[32];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int i = 32 * c + 8 * kk + r;
            double2 k2 = make_double2(0.0, 0.0);
            if (i < N && j <= i) k2 = f.KR[tri(i) + j];
            if (i < iSj) k2.y = 0.0;
            v[4 * r] = dlo(k2.x); v[4 * r + 1] = dhi(k2.x); v[4 * r + 2] = dlo(k2.y); v[4 * r + 3] = dhi(k2.y);
        }
        tmem_st32(tq + (uint32_t)(run.tcol + 32 * kk), v);
    }
}

// ------------------------------------------------------------------------------------------ K from HBM
// cudisc_coag_rates / cudisc_coag_step_cached: the row copy is the image of a cell's planes in HBM ([2][P] doubles,
// PLANAR), refilled by 1-D bulk copies (TMA, refill_bulk of coag_device.cuh) that complete on an mbarrier in RED; the
// column copy is then made from the row copy.
constexpr int kV3RedMbar = 90;
// chunks [k0, k0 + n) of column block c: row copy -> tensor memory (lane <-> column j; zeros above the diagonal and
// for Kf of rows below iS[j], as the build writes them)
template <bool PLANAR, bool ONFLY>
__device__ __forceinline__ void v3_fill_tmem(const V3Tables &vt, const VSm &f, const V3ColRun &run, uint32_t tq, int lane)
{
    const int N = vt.N, c = run.c;
    const int j = 32 * c + lane;
    const int iSj = (j < N) ? ((f.BINI()[j].x >> 9) & 0x1ff) : 0;
    const bool halve = ONFLY && run.diag && !vt.diagBulk;     // (only a diagonal block holds diagonal pairs)
#pragma unroll 1
    for (int kk = 0; kk < run.n; ++kk) {
        uint32_t v[32];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int i = 32 * c + 8 * (run.k0 + kk) + r;
            double2 k2 = make_double2(0.0, 0.0);
            if (i < N && j <= i) k2 = v3_kld<PLANAR>(f.KR, vt.P, tri(i) + j);
            if (halve && i == j) { k2.x *= 0.5; k2.y *= 0.5; }           // PAPER.md:436 (the planes hold K itself)
            if (i < iSj) k2.y = 0.0;
            v[4 * r] = dlo(k2.x); v[4 * r + 1] = dhi(k2.x); v[4 * r + 2] = dlo(k2.y); v[4 * r + 3] = dhi(k2.y);
        }
        tmem_st32(tq + (uint32_t)(run.tcol + 32 * kk), v);
    }
}

// ------------------------------------------------------------------------------------------ eval pieces
// column pass of one run: lane <-> impactor column j = 32 c + lane, rows of chunks [k0, k0 + n) from tensor
// memory; G_j += Kc_ij n_i, H_j += Kf_ij n_i (Kf already 0 where the pair does not count).
__device__ __forceinline__ void v3_col_run(const V3Tables &vt, const VSm &f, const V3ColRun &run, uint32_t tq, int lane)
{
    uint32_t ta = tq + (uint32_t)run.tcol;
    const double *nn = f.NN() + 32 * run.c + 8 * run.k0;
    double gc = 0.0, h = 0.0, gc2 = 0.0, h2 = 0.0;
    // one chunk (8 rows) per tcgen05.ld.x32 (tcgen05.wait::ld drains every load in flight, so a deeper
    // pipeline of smaller loads only adds round trips)
#pragma unroll 1
    for (int kk = 0; kk < run.n; ++kk) {
        uint32_t v[32];
        tmem_ld32(ta, v);
        const double2 n01 = *reinterpret_cast<const double2 *>(nn);
        const double2 n23 = *reinterpret_cast<const double2 *>(nn + 2);
        const double2 n45 = *reinterpret_cast<const double2 *>(nn + 4);
        const double2 n67 = *reinterpret_cast<const double2 *>(nn + 6);
        tmem_wait_ld();
        gc = fma(u2d(v[0], v[1]), n01.x, gc);      h = fma(u2d(v[2], v[3]), n01.x, h);
        gc2 = fma(u2d(v[4], v[5]), n01.y, gc2);    h2 = fma(u2d(v[6], v[7]), n01.y, h2);
        gc = fma(u2d(v[8], v[9]), n23.x, gc);      h = fma(u2d(v[10], v[11]), n23.x, h);
        gc2 = fma(u2d(v[12], v[13]), n23.y, gc2);  h2 = fma(u2d(v[14], v[15]), n23.y, h2);
        gc = fma(u2d(v[16], v[17]), n45.x, gc);    h = fma(u2d(v[18], v[19]), n45.x, h);
        gc2 = fma(u2d(v[20], v[21]), n45.y, gc2);  h2 = fma(u2d(v[22], v[23]), n45.y, h2);
        gc = fma(u2d(v[24], v[25]), n67.x, gc);    h = fma(u2d(v[26], v[27]), n67.x, h);
        gc2 = fma(u2d(v[28], v[29]), n67.y, gc2);  h2 = fma(u2d(v[30], v[31]), n67.y, h2);
        ta += 32; nn += 8;
    }
    reinterpret_cast<double2 *>(f.base + vt.oCOLP)[32 * run.slot + lane] = make_double2(gc + gc2, h + h2);
}

// row pass of one run: lane <-> target row i = 32 b + lane, impactor columns [ja, jb) clipped to the bulk
// prefix j < n_bulk[i]:  A1, A2 += Kc_ij (y_j, y_j m_j);  F1, F2 += Kf_ij (y_j, y_j m_j).  The slot takes
// the deposits per unit n_i into bins i - 1, i, i + 1 (coefficients of coag_tables.h, read through L1).
template <bool PLANAR>
__device__ __forceinline__ void v3_row_run(const DevTables &tb, const V3Tables &vt, const VSm &f, const V3RowRun &run,
                                           int lane)
{
    const int N = vt.N;
    const int i = 32 * run.b + lane, iv = min(i, N - 1);
    const int nbi = (i < N) ? (f.BINI()[iv].x & 0x1ff) : 0;
    const double *bc = tb.binc + iv;
    const int Nq = tb.Np;
    const double cA1 = __ldg(bc + BC_A1 * Nq), cA2 = __ldg(bc + BC_A2 * Nq), cB1 = __ldg(bc + BC_B1 * Nq);
    const double cF1 = __ldg(bc + BC_F1 * Nq), cF2 = __ldg(bc + BC_F2 * Nq), cG1 = __ldg(bc + BC_G1 * Nq);
    const double2 *kr = f.KR + tri(iv);                              // (pairs)
    const double *kc = reinterpret_cast<const double *>(f.KR) + tri(iv), *kf = kc + vt.P;     // (PLANAR)
    const double2 *yy = f.YY();
    double a1 = 0.0, a2 = 0.0, f1 = 0.0, f2 = 0.0, b1 = 0.0, b2 = 0.0, g1 = 0.0, g2 = 0.0;
    int j = run.ja;
    const int jr = min(run.jb, f.HOT()->cmin[run.b]);
    // the rectangle: every row of the block has these columns
#pragma unroll 4
    for (; j + 2 <= jr; j += 2) {
        const double2 k2 = PLANAR ? make_double2(kc[j], kf[j]) : kr[j];
        const double2 k3 = PLANAR ? make_double2(kc[j + 1], kf[j + 1]) : kr[j + 1];
        const double2 y2 = yy[j], y3 = yy[j + 1];
        a1 = fma(k2.x, y2.x, a1); a2 = fma(k2.x, y2.y, a2);
        f1 = fma(k2.y, y2.x, f1); f2 = fma(k2.y, y2.y, f2);
        b1 = fma(k3.x, y3.x, b1); b2 = fma(k3.x, y3.y, b2);
        g1 = fma(k3.y, y3.x, g1); g2 = fma(k3.y, y3.y, g2);
    }
    // the ragged rest (and an odd last rectangle column): row i takes j < n_bulk[i]; the loads are
    // unconditional -- past the end of a row they hit the next rows of the packed array
#pragma unroll 4
    for (; j < run.jb; ++j) {
        const double2 k2 = PLANAR ? make_double2(kc[j], kf[j]) : kr[j];
        double2 y2 = yy[j];
        const bool on = j < nbi;                     // (selects, not branches: the warp stays converged)
        y2.x = on ? y2.x : 0.0; y2.y = on ? y2.y : 0.0;
        a1 = fma(k2.x, y2.x, a1); a2 = fma(k2.x, y2.y, a2);
        f1 = fma(k2.y, y2.x, f1); f2 = fma(k2.y, y2.y, f2);
    }
    a1 += b1; a2 += b2; f1 += g1; f2 += g2;
    double *pp = reinterpret_cast<double *>(f.base + vt.oROWP) + 96 * run.slot + lane;
    pp[0] = cG1 * f1 - cF2 * f2;                                     // -> bin i - 1
    pp[32] = (cA1 * a1 + cA2 * a2) + (cF1 * f1 + cF2 * f2);          // -> bin i
    pp[64] = cB1 * a1 - cA2 * a2;                                    // -> bin i + 1
}

// band stage of the bins 32 g + lane (coag_v3.h): W[plane][d][i] = y_i n_{i-d} Kplane[i][i-d], 0 where the
// pair does not exist; yi: the thread's own y (0 for i >= N)
template <bool PLANAR, bool ONFLY>
__device__ __forceinline__ void v3_stage(const V3Tables &vt, const VSm &f, int i, double yi)
{
    const int N = vt.N, D = vt.bandD;
    const int iv = min(i, N - 1);
    const int pd = tri(iv) + iv;                     // the diagonal pair of row iv
    const double *nn = f.NN() + iv;
    double *w = f.WST() + vt.wPad + i;
    const int plane = D * vt.wRow;
#pragma unroll 2
    for (int d = 0; d < D; ++d) {
        double wc = 0.0, wf = 0.0;
        if (d <= iv) {
            const double2 k2 = v3_kld<PLANAR>(f.KR, vt.P, pd - d);
            // (PLANAR: the store holds K itself; the half of the diagonal pair, is taken here and in
            //  v3_fill_tmem -- unless the row pass reads diagonal pairs too, vt.diagBulk: then the store was halved)
            const double yn = (ONFLY && !vt.diagBulk && d == 0 ? 0.5 * yi : yi) * nn[-d];
            wc = yn * k2.x; wf = yn * k2.y;
        }
        if (i < N) {                                 // (rows of the stage hold the N bins + padding)
            w[d * vt.wRow] = wc;
            w[plane + d * vt.wRow] = wf;
        }
    }
}

// exception entries of target block g, kind `kind` (grid ends; coag_v3.h): lanes <-> entries of one target, fixed
// xor tree, the lane that owns the target adds the sum
__device__ __forceinline__ double v3_exceptions(const VSm &f, const double *wst, int g, int kind, int lane, double acc)
{
    const V3Hot *hot = f.HOT();
#pragma unroll 1
    for (int x = 0; x < kV3MaxExcT; ++x) {
        const V3ExcTarget et = hot->excT[x];
        if (et.t < 0) break;
        if (et.kind != kind || (et.t >> 5) != g) continue;
        double v = 0.0;
        if (et.e0 + lane < et.e1) v = hot->exc[et.e0 + lane].c * wst[hot->exc[et.e0 + lane].off];
#pragma unroll
        for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
        if (lane == (et.t & 31)) acc += v;
    }
    return acc;
}

// band stencil of target t over density taps [q0, q1) (multiples of 8) / over the S taps.  A tap is one 16-byte
// load from the table in shared memory; the eight stage loads of a batch are in flight together.
__device__ __forceinline__ double v3_taps(const VSm &f, const double *wst, int t, int q0, int q1)
{
    const double *w = wst + t;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
#pragma unroll 1
    for (int q = q0; q < q1; q += 8) {
        const uint4 *tp = reinterpret_cast<const uint4 *>(f.HOT()->taps + q);
        uint4 e[8];
        double v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) e[u] = tp[u];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = w[(int)e[u].z];
        a0 = fma(u2d(e[0].x, e[0].y), v[0], a0); a1 = fma(u2d(e[1].x, e[1].y), v[1], a1);
        a2 = fma(u2d(e[2].x, e[2].y), v[2], a2); a3 = fma(u2d(e[3].x, e[3].y), v[3], a3);
        a0 = fma(u2d(e[4].x, e[4].y), v[4], a0); a1 = fma(u2d(e[5].x, e[5].y), v[5], a1);
        a2 = fma(u2d(e[6].x, e[6].y), v[6], a2); a3 = fma(u2d(e[7].x, e[7].y), v[7], a3);
    }
    return (a0 + a1) + (a2 + a3);
}
__device__ __forceinline__ double v3_staps(const V3Tables &vt, const VSm &f, const double *wst, int t)
{
    const double *w = wst + t;
    double a0 = 0.0;
#pragma unroll 1
    for (int q = 0; q < vt.nSTaps; ++q) {
        const uint4 e = reinterpret_cast<const uint4 *>(f.HOT()->staps)[q];
        a0 = fma(u2d(e.x, e.y), w[(int)e.z], a0);
    }
    return a0;
}

// ------------------------------------------------------------------------------------------ eval
// One rate evaluation: thread k < N passes y_k and gets drho_k/dt.  c1, c2, c3: per-thread constants of the
// thread's role -- bin owners (warp < nb): m_k, 1 / m_k, A_k; column-combine group (warp nb + g): -, -, 1 / B_k.
template <int NT, bool PLANAR = false, bool ONFLY = false>
__device__ __forceinline__ double v3_eval(const DevTables &tb, const V3Tables &vt, const VSm &f, double y,
                                          double c1, double c2, double c3, int tid, uint32_t tq, int ppart,
                                          const CellDerived &nd, const GasArgs &gs, bool deriveNext, ProlState &ps,
                                          RoleVals &rv, bool storeNext, double nvR, double nvZ,
                                          const double *kin_next = nullptr)
{
    const int N = vt.N, nb = vt.nb;
    const int lane = tid & 31, warp = tid >> 5;
    const int k = tid;
    const bool live = k < N;

    // ---- phase 0
    double nk = 0.0;
    if (live) {
        nk = y * c2;
        f.NN()[k] = nk;
        f.YY()[k] = make_double2(y, y * c1);
    }
    __syncthreads();

    // ---- phase A: the bin-owning warps stage the band products of their bins (and sum the stencil exceptions of
    //      their bins when those only read the warp's own stage entries), run a third of the NEXT cell's prologue
    //      (ppart 1, 2, 3; 4: all of it); then every warp its own runs
    double excA = 0.0;          // density exceptions of the thread's own bin, summed in phase A when they are local
    if (warp < nb) {
        v3_stage<PLANAR, ONFLY>(vt, f, k, live ? y : 0.0);
        if (vt.excLocal) {
            __syncwarp();
            excA = v3_exceptions(f, f.WST(), warp, 0, lane, 0.0);
        }
        if (ppart) {
            if (ppart == 1 || ppart == 4) ps = prologue_begin(tb, nd, k);
            prologue_newton(ps, ppart == 4 ? 6 : 2);
            if (ppart >= 3) rv = prologue_finish(tb, nd, ps, c2, k);
        }
    }
    // (one copy of each run body: the instruction cache matters more than the select chain.  Column runs
    //  first on every warp: starting odd warps on their row runs instead was measured slower.  The packed runs
    //  are read here, not held in registers across the build.)
    const uint4 colw = reinterpret_cast<const uint4 *>(f.base + kV3oRUNS)[2 * warp];
    const uint4 roww = reinterpret_cast<const uint4 *>(f.base + kV3oRUNS)[2 * warp + 1];
#pragma unroll 1
    for (int r = 0; r < kV3ColRuns; ++r) {
        const uint32_t w = r == 0 ? colw.x : (r == 1 ? colw.y : (r == 2 ? colw.z : colw.w));
        if (!w) break;
        v3_col_run(vt, f, v3_unpack_col(w), tq, lane);
    }
#pragma unroll 1
    for (int r = 0; r < kV3RowRuns; ++r) {
        const uint32_t w = r == 0 ? roww.x : (r == 1 ? roww.y : roww.z);
        if (!w) break;
        v3_row_run<PLANAR>(tb, vt, f, v3_unpack_row(w), lane);
    }
    __syncthreads();
    // (kernel read from HBM, last evaluation of a cell: the row copy is dead from here on, the next cell's planes
    //  start to arrive under the combine phase)
    if (PLANAR && kin_next && tid == 0)
        refill_bulk(f.KR, kin_next, vt.P, reinterpret_cast<uint64_t *>(f.RED() + kV3RedMbar));

    // ---- phase B (combine), three groups of warps side by side:
    //   R (warp w < nb, bin 32 w + lane)      row partials -> deposits into bins k-1, k, k+1; first half of the
    //                                         band stencil of its bins (stays in a register)
    //   C (warp nb + w, bin 32 w + lane)      column partials -> loss frequency G_k, fragment source of l-bin k,
    //                                         suffix scan of S_l / B_l (Eq. 67 via l-bins)
    //   D (warp 2 nb + w, bin 32 w + lane)    second half of the band stencil, exception entries -> BANDV
    // G_k and the scanned value travel through NN[k] and YY[k].y, dead by now.
    double d0 = 0.0, dm1 = 0.0, dp1 = 0.0, up = 0.0, dn = 0.0, bandR = 0.0;
    double *wtot = f.RED(), *eUp = f.RED() + 16, *eDn = f.RED() + 32;
    const double *wst = f.WST();
    if (warp < nb) {
        const double *pp = reinterpret_cast<const double *>(f.base + vt.oROWP) + 96 * f.HOT()->rpBase[warp] + lane;
        const int np = f.HOT()->rpCnt[warp];
#pragma unroll 2
        for (int p = 0; p < np; ++p) {
            dm1 += pp[96 * p]; d0 += pp[96 * p + 32]; dp1 += pp[96 * p + 64];
        }
        dm1 *= nk; d0 *= nk; dp1 *= nk;
        if (lane == 0) eDn[warp] = dm1;
        if (lane == 31) eUp[warp] = dp1;
        up = __shfl_up_sync(0xffffffffu, dp1, 1);
        dn = __shfl_down_sync(0xffffffffu, dm1, 1);
        bandR = v3_taps(f, wst, min(k, N - 1), 0, vt.nTapsR);
    } else if (warp < 2 * nb) {
        const int g = warp - nb, kc = 32 * g + lane;
        const double2 *colp = reinterpret_cast<const double2 *>(f.base + vt.oCOLP);
        auto colsum = [&](int j, double &gj, double &hj) {
            const int c = j >> 5, np = f.HOT()->cpCnt[c];
            const double2 *pc2 = colp + 32 * f.HOT()->cpBase[c] + (j & 31);
            gj = 0.0; hj = 0.0;
#pragma unroll 2
            for (int r = 0; r < np; ++r) {
                const double2 u = pc2[32 * r];
                gj += u.x; hj += u.y;
            }
        };
        // S stencil of l-bin kc (stage entries past the bins are 0) and its exceptions
        double sl = v3_staps(vt, f, wst, min(kc, N - 1));
        if (vt.nExcS) sl = v3_exceptions(f, wst, g, 1, lane, sl);
        if (kc < N) {
            const int2 bi = f.BINI()[kc];
            double gc, h;
            colsum(kc, gc, h);
            f.NN()[kc] = gc + h;                           // G_k
            for (int j = bi.y & 0xffff; j < (bi.y >> 16); ++j) {
                double gj, hj = h;
                if (j != kc) colsum(j, gj, hj);
                sl = fma(tb.sS * f.YY()[j].x, hj, sl);
            }
        }
        const double sv = (kc < N) ? sl * c3 : 0.0;
        double suf = sv;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double v = __shfl_down_sync(0xffffffffu, suf, o);
            if (lane + o < 32) suf += v;
        }
        if (lane == 0) wtot[g] = suf;
        if (kc < N) f.YY()[kc].y = suf;
    } else if (warp < 3 * nb) {
        const int g = warp - 2 * nb, t = 32 * g + lane;
        double da = v3_taps(f, wst, min(t, N - 1), vt.nTapsR, vt.nTaps);       // (the list is padded to a multiple of 8)
        if (!vt.excLocal) da = v3_exceptions(f, wst, g, 0, lane, da);
        f.BANDV()[t] = da;
    } else if (deriveNext && warp == kV3Warps - 1) {
        // the warp with no part in the combine: the per-cell scalars of the cell after the next one (its gas
        // values landed in RED[80 .. 83] with this cell's build), for the bin owners to pick up after the next build
        const CellGas g = {f.RED()[80], f.RED()[81], f.RED()[82], gs.alpha ? f.RED()[83] : gs.alpha_const};
        const CellDerived d = derive_cell(g, gs.mu, gs.sigma_mol);
        if (lane == 0) {
            f.RED()[84] = d.Ste; f.RED()[85] = d.den; f.RED()[86] = d.Om; f.RED()[87] = d.Vg2; f.RED()[88] = d.bmc;
        }
    }
    __syncthreads();
    // last evaluation of a cell: the partial sums are consumed, so the role vectors of the NEXT cell go into the
    // union now and the other warps start its build while the bin owners assemble and finish this cell
    if (storeNext) {
        if (warp < nb) {
            prologue_store(tb, rv, nvR, nvZ, 0.0, false, false, f.s, k);
            if (tid == 0) f.RED()[95] = rv.Vg2;
        }
        __syncthreads();
    }
    if (warp >= nb) return 0.0;

    double d = 0.0;
    if (live) {
        double suf = f.YY()[k].y;
#pragma unroll 1
        for (int w = warp + 1; w < nb; ++w) suf += wtot[w];
        const double prev = (lane > 0) ? up : (warp > 0 ? eUp[warp - 1] : 0.0);
        const double next = (lane < 31) ? dn : (warp + 1 < nb ? eDn[warp + 1] : 0.0);
        d = d0;
        if (k > 0) d += prev;
        if (k < N - 1) d += next;
        d += (bandR + excA) + f.BANDV()[k];
        d = fma(-y, f.NN()[k], d);
        d = fma(c3, suf, d);
    }
    return d;
}

template <int NT, int MODE>
__global__ void __launch_bounds__(NT, 1)
coag_v3_kernel(const DevTables tb, const V3Tables vt, const GasArgs gs, const StepArgs sa_in)
{
    StepArgs sa = sa_in;
    constexpr bool KIN = MODE == MODE_RATES || MODE == MODE_STEPK;       // the kernel of a cell is read from HBM
    constexpr bool STEPPING = MODE == MODE_STEP || MODE == MODE_STEPK;   // BS3(2) step (else: one rate evaluation)
    constexpr bool PLANAR = KIN;         // row copy = image of the planes in HBM, refilled by bulk copies
    // The half of the diagonal pairs (the planes hold K itself): taken on the fly by the two readers of
    // diagonal pairs (band stage, tensor-memory fill) in the step, which saves two block barriers per cell; in place
    // for the single evaluation of cudisc_coag_rates, where that measured 4 % faster (0.75 against 0.78 ms).
    constexpr bool ONFLY = MODE == MODE_STEPK;
    if (STEPPING && !apply_ctrl(sa)) return;
    extern __shared__ __align__(16) char smem_v3[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, quarter = warp & 3;
    const int N = vt.N, nb = vt.nb;
    const VSm f = v3_carve(smem_v3, tb, vt);
    const Smem &s = f.s;
    PairConst pc;
    pc.c15vf2 = 1.5 * gs.v_frag * gs.v_frag;
    pc.Vg2 = 0.0;
    const int k = tid;
    const bool live = k < N;

    // ---- per-CTA constants
    for (int q = tid; q < kV3NpMax; q += NT) f.BINI()[q] = q < N ? tb.bini[q] : make_int2(0, 0);
    for (int q = tid; q < kV3NpMax; q += NT) f.YY()[q] = make_double2(0.0, 0.0);
    for (int q = tid; q < kV3NpMax + 16; q += NT) f.NN()[q] = 0.0;
    for (int q = tid; q < kV3NpMax; q += NT) f.BANDV()[q] = 0.0;
    if (vt.oDTAB) {
        for (int q = tid; q < N; q += NT) s.DTAB[q] = tb.dtab[q];
        for (int q = tid; q < 64; q += NT) s.EXPT[q] = tb.exptab[q];
    }
    for (int q = tid; q < (int)(sizeof(V3Hot) / 4); q += NT)
        reinterpret_cast<uint32_t *>(smem_v3 + kV3oHOT)[q] = reinterpret_cast<const uint32_t *>(&vt.hot)[q];
    // the packed runs of every warp (kernel parameters -> shared memory) and the constants of the thread's role
    // (v3_eval)
    static_assert(kV3ColRuns == 4 && kV3RowRuns == 3, "run words: one uint4 of column runs, one of row runs per warp");
    if (tid < 8 * kV3Warps) {
        const int w = tid >> 3, r = tid & 7;
        reinterpret_cast<uint32_t *>(smem_v3 + kV3oRUNS)[tid] = r < 4 ? vt.col[w][r] : (r < 7 ? vt.row[w][r - 4] : 0u);
    }
    double c1 = 0.0, c2 = 0.0, c3 = 0.0;
    if (live) {
        c1 = tb.binc[BC_M * tb.Np + k]; c2 = tb.binc[BC_RM * tb.Np + k]; c3 = tb.binc[BC_FA * tb.Np + k];
    } else if (warp >= nb && warp < 2 * nb && tid - 32 * nb < N) {
        c3 = tb.binc[BC_FIB * tb.Np + tid - 32 * nb];
    }

    uint64_t *kbar = reinterpret_cast<uint64_t *>(f.RED() + kV3RedMbar);
    uint32_t kph = 0u;
    const bool kin_tma = PLANAR && (reinterpret_cast<uintptr_t>(sa.Kin) & 15) == 0;
    if (PLANAR && tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" :: "r"(smem_addr(kbar)), "r"(1) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    uint32_t *slot = reinterpret_cast<uint32_t *>(f.RED());
    if (tid < 32) tmem_alloc_all(slot);
    tmem_fence_before();
    __syncthreads();
    tmem_fence_after();
    const uint32_t tbase = *slot;
    const uint32_t tq = tq_addr(tbase, quarter, 0);
    {   // zero the whole quarter once (rows past the grid of the last chunk of a block are never written)
        uint32_t z[32];
#pragma unroll
        for (int u = 0; u < 32; ++u) z[u] = 0u;
#pragma unroll 1
        for (int q = 0; q < 4; ++q) tmem_st32(tq + (uint32_t)(128 * (warp >> 2) + 32 * q), z);
        tmem_wait_st();
    }
    tmem_fence_before();
    __syncthreads();
    tmem_fence_after();

    // frozen inputs of a cell, fetched ahead: the per-cell scalars two cells ahead (the warp
    // that idles in the combine phase turns them into what the prologue needs, RED[84 .. 88], and the evaluations
    // of the cell before run that prologue piece by piece), the per-bin velocities two evaluations before the
    // end of the cell before
    CellDerived nd = {1.0, 1.0, 1.0, 1.0, 1.0};
    double nvR = 0.0, nvZ = 0.0;
    auto stage_gas = [&](int cell) {        // cp.async of the per-cell scalars into RED[80 .. 83]
        if (cell >= sa.C || tid >= 4) return;
        const double *src = tid == 0 ? gs.T : (tid == 1 ? gs.rho_g : (tid == 2 ? gs.Omega : gs.alpha));
        if (src) cp_async8(s.RED + 80 + tid, src + cell);
    };
    auto raw_gas = [&]() {
        const CellGas g = {s.RED[80], s.RED[81], s.RED[82], gs.alpha ? s.RED[83] : gs.alpha_const};
        return g;
    };
    auto take_derived = [&]() {
        nd.Ste = s.RED[84]; nd.den = s.RED[85]; nd.Om = s.RED[86]; nd.Vg2 = s.RED[87]; nd.bmc = s.RED[88];
    };
    auto fetch_vel = [&](int cell) {
        if (cell >= sa.C || !live) return;
        const size_t g = (size_t)cell * N + k;
        nvR = __ldg(gs.vR + g); nvZ = __ldg(gs.vZ + g);
    };
    // first cell of the CTA: nothing ran ahead, every thread takes the raw values; second cell: its scalars are
    // derived here (once per launch)
    CellGas g0 = {1.0, 1.0, 1.0, 1.0};
    if (!KIN) {
        stage_gas(blockIdx.x);
        cp_async_wait_all();
        __syncthreads();
        g0 = raw_gas();
        fetch_vel(blockIdx.x);
        __syncthreads();
        stage_gas(blockIdx.x + gridDim.x);
        cp_async_wait_all();
        __syncthreads();
    }
    if (!KIN && warp == kV3Warps - 1 && (int)(blockIdx.x + gridDim.x) < sa.C) {
        const CellDerived d = derive_cell(raw_gas(), gs.mu, gs.sigma_mol);
        if (lane == 0) {
            s.RED[84] = d.Ste; s.RED[85] = d.den; s.RED[86] = d.Om; s.RED[87] = d.Vg2; s.RED[88] = d.bmc;
        }
    }
    RoleVals rv;
    rv.Vg2 = 0.0;
    ProlState ps = {2.0, 0.0, 0.0, 0.0};
    bool rv_valid = false;

    if (MODE == MODE_KERNEL) {
        // cudisc_coag_kernel: the build alone, every pair straight to the planes in HBM.  The bin-owning warps also
        // run the whole prologue of the CTA's next cell (in registers) after their share of the rows -- the host
        // deals them fewer rows (V3Tables built with buildOnly) --, and store its role vectors between two barriers.
        rv = prologue_compute(tb, g0, gs.mu, gs.sigma_mol, c2, k);
        if (warp < nb) prologue_store(tb, rv, nvR, nvZ, 0.0, false, false, s, k);
        if (tid == 0) s.RED[95] = rv.Vg2;
        __syncthreads();
        for (int cell = blockIdx.x; cell < sa.C; cell += gridDim.x) {
            pc.Vg2 = s.RED[95];
            const int nxt = cell + (int)gridDim.x;
            const bool pre = nxt < sa.C && warp < nb;
            CellGas gn = {1.0, 1.0, 1.0, 1.0};
            if (pre) {
                gn.T = __ldg(gs.T + nxt); gn.rho_g = __ldg(gs.rho_g + nxt); gn.Om = __ldg(gs.Omega + nxt);
                gn.alpha = gs.alpha ? __ldg(gs.alpha + nxt) : gs.alpha_const;
                fetch_vel(nxt);
            }
            double *kout = sa.out + (size_t)cell * 2 * vt.P;
#pragma unroll 1
            for (int r = 0; r < kV3ColRuns; ++r) {
                const uint32_t w = reinterpret_cast<const uint32_t *>(smem_v3 + kV3oRUNS)[8 * warp + r];
                if (!w) break;
                const V3ColRun run = v3_unpack_col(w);
                if (run.diag) v3_build_diag<true>(vt, f, pc, run, tq, lane, kout);
                else v3_build_rows<true>(vt, f, pc, run, tq, lane, kout);
            }
            if (pre) rv = prologue_compute(tb, gn, gs.mu, gs.sigma_mol, c2, k);
            __syncthreads();                              // the role vectors of this cell are dead
            if (pre) {
                prologue_store(tb, rv, nvR, nvZ, 0.0, false, false, s, k);
                if (tid == 0) s.RED[95] = rv.Vg2;
            }
            __syncthreads();
        }
        tmem_fence_before();
        __syncthreads();
        if (tid < 32) tmem_dealloc_all(tbase);
        return;
    }

    int err_cell = -1;          // cell whose warp error maxima wait in RED[64 ..) for the next barrier
    auto flush_err = [&]() {
        if (STEPPING && tid == NT - 32 && err_cell >= 0) {     // (a thread of the warp that owns no bins)
            unsigned long long m = 0ull;
#pragma unroll 1
            for (int w = 0; w < nb; ++w) {
                const unsigned long long v = reinterpret_cast<const unsigned long long *>(s.RED)[64 + w];
                m = v > m ? v : m;
            }
            sa.err[err_cell] = __longlong_as_double((long long)m);
        }
    };
    for (int cell = blockIdx.x; cell < sa.C; cell += gridDim.x) {
        const size_t row = (size_t)cell * N;
        if (!KIN && !rv_valid) {                      // first cell of the CTA: nothing ran ahead
            rv = prologue_compute(tb, g0, gs.mu, gs.sigma_mol, c2, k);
            prologue_store(tb, rv, nvR, nvZ, 0.0, false, false, s, k);
            if (tid == 0) s.RED[95] = rv.Vg2;
            __syncthreads();
        }
        pc.Vg2 = s.RED[95];
        // state and FSAL derivative of the cell (thread <-> bin) and the next cell's gas scalars: asynchronous
        // copies into (y, y m) -- free during the build -- and RED, landed by the post-build barrier
        if (live) {
            cp_async8(&f.YY()[k].x, sa.rho + row + k);
            if (STEPPING && sa.have_k1) cp_async8(&f.YY()[k].y, sa.k_fsal + row + k);
        }
        if (!KIN) stage_gas(cell + 2 * gridDim.x);
        if (KIN) {
            // the planes of this cell: bulk copies on their way since the last evaluation of the CTA's previous cell
            // (v3_eval: behind the last read of the row copy, under the combine phase); every thread waits for them
            // itself, then every warp copies its chunks to tensor memory
            const double *planes = sa.Kin + (size_t)cell * 2 * vt.P;
            if (kin_tma) {
                if (cell == (int)blockIdx.x && tid == 0) refill_bulk(f.KR, planes, vt.P, kbar);
                mbar_wait_parity(kbar, kph);
                kph ^= 1u;
            } else {                                      // planes not 16-byte aligned: plain copy
                double *img = reinterpret_cast<double *>(f.KR);
                for (int p = tid; p < 2 * vt.P; p += NT) img[p] = __ldcs(planes + p);
                __syncthreads();
            }
            if (!ONFLY || vt.diagBulk) {                  // (always on grids whose bulk row sums reach the diagonal pair)
                __syncthreads();
                if (live) {
                    double *img = reinterpret_cast<double *>(f.KR) + tri(k) + k;
                    img[0] *= 0.5; img[vt.P] *= 0.5;
                }
                __syncthreads();
            }
            // while this cell is evaluated its successor's planes are pulled into L2 (asynchronous bulk prefetch)
            if (cell + (int)gridDim.x < sa.C && (reinterpret_cast<uintptr_t>(sa.Kin) & 15) == 0) {
                const char *nxt = reinterpret_cast<const char *>(sa.Kin + (size_t)(cell + gridDim.x) * 2 * vt.P);
                const size_t bytes = 16 * (size_t)vt.P;
                constexpr size_t kChunk = 8192;
                for (size_t off = (size_t)tid * kChunk; off < bytes; off += (size_t)NT * kChunk) {
                    const uint32_t n = (uint32_t)(bytes - off < kChunk ? bytes - off : kChunk);
                    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(nxt + off), "r"(n) : "memory");
                }
            }
        }
#pragma unroll 1
        for (int r = 0; r < kV3ColRuns; ++r) {
            const uint32_t w = reinterpret_cast<const uint32_t *>(smem_v3 + kV3oRUNS)[8 * warp + r];
            if (!w) break;
            const V3ColRun run = v3_unpack_col(w);
            if (KIN) v3_fill_tmem<PLANAR, ONFLY>(vt, f, run, tq, lane);
            else if (run.diag) v3_build_diag<false>(vt, f, pc, run, tq, lane);
            else v3_build_rows<false>(vt, f, pc, run, tq, lane);
        }
        tmem_wait_st();
        cp_async_wait_all();
        double y0 = 0.0, k1 = 0.0;
        if (live) {                                   // the thread's own copies are complete
            y0 = f.YY()[k].x;
            if (STEPPING && sa.have_k1) k1 = f.YY()[k].y;
        }
        if (STEPPING && warp < nb) {
            double ws = y0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) ws += __shfl_xor_sync(0xffffffffu, ws, o);
            if (lane == 0) s.RED[48 + warp] = ws;
        }
        tmem_fence_before();
        __syncthreads();
        tmem_fence_after();
        if (!KIN) take_derived();
        flush_err();
        // the role vectors are dead: zero the padding of the band stage (its bins are written per evaluation)
        {   // (16 threads per stage row; the host checks that this covers them)
            const int r = tid >> 4, e = tid & 15;
            if (r < 2 * vt.bandD && e < vt.wRow - N) f.WST()[r * vt.wRow + (e < vt.wPad ? e : N + e)] = 0.0;
        }

        const bool more = cell + (int)gridDim.x < sa.C, more2 = cell + 2 * (int)gridDim.x < sa.C;
        const double *kin_next = (KIN && more && kin_tma) ? sa.Kin + (size_t)(cell + gridDim.x) * 2 * vt.P : nullptr;
        if (MODE == MODE_RATES) {
            const double d = v3_eval<NT, PLANAR, ONFLY>(tb, vt, f, y0, c1, c2, c3, tid, tq, 0, nd, gs, false, ps, rv,
                                                        false, nvR, nvZ, kin_next);
            if (live) sa.out[row + k] = d;
            continue;
        }
        if (MODE == MODE_OTF) {
            fetch_vel(cell + gridDim.x);
            const double d = v3_eval<NT>(tb, vt, f, y0, c1, c2, c3, tid, tq, more ? 4 : 0, nd, gs, more2, ps, rv,
                                         more, nvR, nvZ);
            rv_valid = more;
            if (live) sa.out[row + k] = d;
            continue;
        }

        // ---------------- Bogacki-Shampine 3(2)
        const double h = sa.dt;
        double k2 = 0.0, k3 = 0.0, k4 = 0.0, yn = y0;
#pragma unroll 1
        for (int st = sa.have_k1 ? 1 : 0; st < 4; ++st) {
            double ys = y0;
            if (st == 1) ys = y0 + 0.5 * h * k1;
            if (st == 2) ys = y0 + 0.75 * h * k2;
            if (!KIN && st == 2) fetch_vel(cell + gridDim.x);
            if (st == 3) {
                yn = y0 + h * ((2.0 / 9.0) * k1 + (1.0 / 3.0) * k2 + (4.0 / 9.0) * k3);
                ys = yn;
            }
            const double d = KIN ? v3_eval<NT, PLANAR, ONFLY>(tb, vt, f, ys, c1, c2, c3, tid, tq, 0, nd, gs, false, ps,
                                                              rv, false, nvR, nvZ, st == 3 ? kin_next : nullptr)
                                 : v3_eval<NT>(tb, vt, f, ys, c1, c2, c3, tid, tq, more ? st : 0, nd, gs,
                                               more2 && st == 1, ps, rv, more && st == 3, nvR, nvZ);
            if (st == 3) rv_valid = more;
            if (st == 0) k1 = d;
            if (st == 1) k2 = d;
            if (st == 2) k3 = d;
            if (st == 3) k4 = d;
        }
        // error norm (R10) and write-back.  sum_k y0_k: warp sums taken before the post-build
        // barrier; max_k: warp maxima here, combined by thread 0 after the next block barrier (the scaled
        // errors are >= 0 or NaN, so the unsigned order of their bit patterns is the NaN-propagating max)
        if (warp < nb) {
            double ysum = 0.0;
#pragma unroll 1
            for (int w = 0; w < nb; ++w) ysum += s.RED[48 + w];
            const double atol = sa.atol_factor * ysum;
            unsigned long long eb = 0ull;
            if (live) {
                const double e = h * ((-5.0 / 72.0) * k1 + (1.0 / 12.0) * k2 + (1.0 / 9.0) * k3 - (1.0 / 8.0) * k4);
                const double sc = atol + sa.rtol * fmax(fabs(y0), fabs(yn));
                const double emax = (e == 0.0) ? 0.0 : fabs(e) / sc;
                eb = (unsigned long long)__double_as_longlong(emax);
                sa.rho_out[row + k] = yn;
                sa.k_out[row + k] = k4;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const unsigned long long v = __shfl_xor_sync(0xffffffffu, eb, o);
                eb = v > eb ? v : eb;
            }
            if (lane == 0) reinterpret_cast<unsigned long long *>(s.RED)[64 + warp] = eb;
        }
        err_cell = cell;
    }
    tmem_fence_before();
    __syncthreads();
    flush_err();
    if (tid < 32) tmem_dealloc_all(tbase);
}

template <int MODE>
cudaError_t launch_v3_mode(const LaunchCfg &lc, const DevTables &tb, const V3Tables &vt, const GasArgs &gs,
                           const StepArgs &sa, cudaStream_t st)
{
    auto fn = coag_v3_kernel<kThreads, MODE>;
    static bool attr_done[64] = {false};    // the attribute is per device (and per instantiation)
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !attr_done[dev]) {
        e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, lc.smem_optin);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) attr_done[dev] = true;
    }
    fn<<<lc.grid, kThreads, lc.smem_bytes, st>>>(tb, vt, gs, sa);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_v3(int mode, const LaunchCfg &lc, const DevTables &tb, const V3Tables &vt,
                      const GasArgs &gs, const StepArgs &sa, cudaStream_t st)
{
    if (mode == MODE_OTF) return launch_v3_mode<MODE_OTF>(lc, tb, vt, gs, sa, st);
    if (mode == MODE_KERNEL) return launch_v3_mode<MODE_KERNEL>(lc, tb, vt, gs, sa, st);
    if (mode == MODE_RATES) return launch_v3_mode<MODE_RATES>(lc, tb, vt, gs, sa, st);
    if (mode == MODE_STEPK) return launch_v3_mode<MODE_STEPK>(lc, tb, vt, gs, sa, st);
    return launch_v3_mode<MODE_STEP>(lc, tb, vt, gs, sa, st);
}

}  // namespace cudisc
