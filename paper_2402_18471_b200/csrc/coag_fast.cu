// coag_fast.cu -- the tensor-memory cell kernel (sm_100a, FP64): cudisc_coag_step and
// cudisc_coag_rates_otf for mass grids whose tables fit (coag_fast.h).
//
// Same mathematics and the same device routines (prologue, pair kernel, BS3(2) algebra) as the general
// kernel of coag_kernels.cu; what differs is where the collision kernel of the cell lives and how the
// work is dealt out:
//   * the build writes every K_ij twice: to the packed shared-memory row copy and, for the rows below
//     the diagonal blocks, to a column copy in tensor memory (tcgen05.st, lane <-> column j);
//   * a rate evaluation reads the shared-memory copy once (row pass, band products, diagonal blocks)
//     and the tensor-memory copy once (column pass, tcgen05.ld), instead of shared memory twice;
//   * per-bin constants of the combine step and the band tables sit in tensor memory as well;
//   * tasks that touch tensor memory wait in one queue per tensor-memory quarter (a warp reaches only
//     the lanes of quarter warp % 4), everything else in a free queue drained afterwards.
// One persistent CTA of 512 threads per SM; thread k < N owns bin k.
#include "coag_fast.h"
#include "coag_launch.h"

namespace cudisc {

namespace {

// ------------------------------------------------------------------------------------------ tensor memory
__device__ __forceinline__ uint32_t tq_addr(uint32_t tbase, int quarter, int col)
{
    return tbase + ((uint32_t)(32 * quarter) << 16) + (uint32_t)col;
}
__device__ __forceinline__ void tmem_st2(uint32_t taddr, uint32_t a, uint32_t b)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};\n" :: "r"(taddr), "r"(a), "r"(b) : "memory");
}
__device__ __forceinline__ void tmem_st4(uint32_t taddr, const uint32_t (&v)[4])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};\n"
                 :: "r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory");
}
__device__ __forceinline__ void tmem_ld2(uint32_t taddr, uint32_t (&v)[2])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];\n"
                 : "=r"(v[0]), "=r"(v[1]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t (&v)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];\n"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(taddr) : "memory");
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
struct FSm {
    double2 *KR;        // row copy of the kernel, packed lower-triangular, diagonal halved
    Smem s;             // the arrays the shared device routines address (coag_device.cuh)
    uint2 *TB, *TE;     // build / evaluation tasks (per-warp lists, FastTables::bw / ew)
};

// offsets (in doubles) of the arrays, computed on the host (FastTables::off): a pointer the compiler
// has to re-materialise under register pressure costs one add of a kernel parameter
__device__ __forceinline__ FSm fast_carve(double *base, const FastTables &ft)
{
    FSm f;
    f.KR = (double2 *)base;
    Smem &s = f.s;
    s.YY = (double2 *)(base + ft.off[FO_YY]);
    s.DTAB = (double2 *)(base + ft.off[FO_DTAB]);
    s.NN = base + ft.off[FO_NN];
    s.BANDV = base + ft.off[FO_BANDV];
    s.BANDV2 = base + ft.off[FO_BANDV2];
    s.BINC = nullptr;
    s.BINI = (int2 *)(base + ft.off[FO_BINI]);
    s.EXPT = base + ft.off[FO_EXPT];
    s.RED = base + ft.off[FO_RED];
    s.CTR = nullptr; s.SCHED = nullptr; s.ITB = s.ITE = nullptr;
    f.TB = (uint2 *)(base + ft.off[FO_TB]);
    f.TE = (uint2 *)(base + ft.off[FO_TE]);
    s.PARTR = base + ft.off[FO_UNION];
    s.PARTC = base + ft.off[FO_PARTC];
    s.WST = base + ft.off[FO_WST];
    s.RI = (double2 *)(base + ft.off[FO_UNION]);
    s.B0 = (double2 *)(base + ft.off[FO_B0]);
    s.B1 = (double2 *)(base + ft.off[FO_B1]);
    s.J2 = (double2 *)(base + ft.off[FO_J2]);
    s.J3 = (double2 *)(base + ft.off[FO_J3]);
    s.V5 = base + ft.off[FO_V5];
    return f;
}

// ------------------------------------------------------------------------------------------ build
template <bool VPHI, bool LOG>
__device__ __forceinline__ void fast_build(const DevTables &tb, const FastTables &ft, const FSm &f,
                                           const PairConst &pc, uint32_t tbase, int warp, int lane)
{
    const Smem &s = f.s;
    const int N = tb.N, quarter = warp & 3;
    const int it1 = ft.bw[warp + 1];
    for (int it = ft.bw[warp]; it < it1; ++it) {
        const FTask t = ftask_unpack(f.TB[it]);
        const int c = t.blk;
        if (t.kind == FB_ROWS) {
            const int j = 32 * c + lane;
            const bool valid = j < N;
            const int jc = valid ? j : N - 1;
            const RoleJ B = load_role_j<VPHI>(s, jc);
            const int iSj = ft.colMask ? ((s.BINI[jc].x >> 9) & 0x1ff) : 0;
            const bool tm = t.tcol != kNoTmem;
            uint32_t ta = tq_addr(tbase, quarter, t.tcol);
            double2 *kr = f.KR + tri(t.a) + j;
            for (int i = t.a; i < t.b; i += 2, ta += 8) {
                const bool two = i + 1 < t.b;
                const int i2 = two ? i + 1 : i;
                const RoleI A1 = load_role_i<VPHI, false>(s, i);
                const RoleI A2 = load_role_i<VPHI, false>(s, i2);
                const double2 k1 = pair_kernel<VPHI, LOG, false>(A1, B, i - j, pc, s);
                const double2 k2 = pair_kernel<VPHI, LOG, false>(A2, B, i2 - j, pc, s);
                if (valid) {
                    kr[0] = k1;
                    if (two) kr[i + 1] = k2;
                }
                kr += 2 * i + 3;                                       // tri(i + 2) - tri(i)
                if (tm) {
                    // column copy: Kf of rows below iS[j] is not part of the column sums (coag_tables.h)
                    const double f1 = (i < iSj) ? 0.0 : k1.y, f2 = (i2 < iSj) ? 0.0 : k2.y;
                    const uint32_t v[8] = {dlo(k1.x), dhi(k1.x), dlo(f1), dhi(f1), dlo(k2.x), dhi(k2.x), dlo(f2), dhi(f2)};
                    tmem_st8(ta, v);
                }
            }
        } else {
            for (int tt = t.a + lane; tt < t.b; tt += 32) {
                int r = (int)((sqrtf(8.0f * (float)tt + 1.0f) - 1.0f) * 0.5f);
                r += (tri(r + 1) <= tt) ? 1 : 0;
                r -= (tri(r) > tt) ? 1 : 0;
                const int i = 32 * c + r, j = 32 * c + (tt - tri(r));
                const RoleI A = load_role_i<VPHI, true>(s, i);
                const RoleJ B = load_role_j<VPHI>(s, j);
                double2 k2 = pair_kernel<VPHI, LOG, true>(A, B, i - j, pc, s);
                if (i == j) { k2.x *= 0.5; k2.y *= 0.5; }
                f.KR[tri(i) + j] = k2;
            }
        }
    }
    tmem_wait_st();
}

// sum_e coef[e] W[idx[e]] of the calling lane's target: table of `len` entries (multiple of 4) at
// tensor-memory column `col` of the warp's quarter, coefficients then stage indices.  The loads of
// batch e + 4 are in flight while batch e is summed.
__device__ __forceinline__ double band_gather(uint32_t tbase, int quarter, int col, int len, const double *wst)
{
    const uint32_t tc = tq_addr(tbase, quarter, col), ti = tc + 2 * len;
    double acc0 = 0.0, acc1 = 0.0;
    uint32_t cf[8], ixs[4];
    tmem_ld8(tc, cf);
    tmem_ld4(ti, ixs);
    tmem_wait_ld();
    for (int e0 = 0; e0 < len; e0 += 4) {
        const double w0 = wst[ixs[0]], w1 = wst[ixs[1]], w2 = wst[ixs[2]], w3 = wst[ixs[3]];
        const double c0 = u2d(cf[0], cf[1]), c1 = u2d(cf[2], cf[3]), c2 = u2d(cf[4], cf[5]), c3 = u2d(cf[6], cf[7]);
        if (e0 + 4 < len) {
            tmem_ld8(tc + 2 * (e0 + 4), cf);
            tmem_ld4(ti + e0 + 4, ixs);
        }
        acc0 = fma(c0, w0, acc0);
        acc1 = fma(c1, w1, acc1);
        acc0 = fma(c2, w2, acc0);
        acc1 = fma(c3, w3, acc1);
        tmem_wait_ld();
    }
    return acc0 + acc1;
}

// ------------------------------------------------------------------------------------------ eval
// One rate evaluation: thread k < N passes y_k and gets drho_k/dt.  mk, rmk: m_k, 1/m_k of the thread's bin.
template <int NT>
__device__ __forceinline__ double fast_eval(const DevTables &tb, const FastTables &ft, const FSm &f, double y,
                                            double mk, double rmk, int tid, uint32_t tbase, int ppart,
                                            const CellGas &nx, double mu, double sigma_mol, ProlState &ps,
                                            RoleVals &rv, int2 myband, long long *sa_prof)
{
    PROF_T(tp0);
    const Smem &s = f.s;
    const int N = tb.N, Np = tb.Np;
    const int lane = tid & 31, warp = tid >> 5, quarter = warp & 3;
    const int k = tid;
    const bool live = k < N;

    // ---- phase 0
    double nk = 0.0;
    if (live) {
        nk = y * rmk;
        s.NN[k] = nk;
        s.YY[k] = make_double2(y, y * mk);
    }
    __syncthreads();
    PROF_ADD(2, tp0);
    PROF_T(tpA);

    // a third of the NEXT cell's prologue per evaluation (ppart 1, 2, 3; 4: all of it), by the warps
    // that own bins; the static schedule gives them less of the task work
    if (ppart && 32 * warp < N) {
        if (ppart == 1 || ppart == 4) ps = prologue_begin(tb, nx, mu, sigma_mol, k);
        prologue_newton(ps, ppart == 4 ? 6 : 2);
        if (ppart >= 3) rv = prologue_finish(tb, nx, mu, ps, rmk, k);
    }

    // ---- phase A: the warp's own task list
    const int it1 = ft.ew[warp + 1];
    for (int it = ft.ew[warp]; it < it1; ++it) {
        const FTask t = ftask_unpack(f.TE[it]);
        if (t.kind == FE_RECT) {
            // lane <-> target row i; columns [a, b) of every row, no predicate
            const int iv = min(32 * t.blk + lane, N - 1);
            const double2 *kr = f.KR + tri(iv);
            double a1 = 0.0, a2 = 0.0, f1 = 0.0, f2 = 0.0, b1 = 0.0, b2 = 0.0, g1 = 0.0, g2 = 0.0;
#pragma unroll 4
            for (int j = t.a; j < t.b; j += 2) {
                const double2 k2 = kr[j], k3 = kr[j + 1];
                const double2 yy = s.YY[j], yz = s.YY[j + 1];
                a1 = fma(k2.x, yy.x, a1); a2 = fma(k2.x, yy.y, a2);
                f1 = fma(k2.y, yy.x, f1); f2 = fma(k2.y, yy.y, f2);
                b1 = fma(k3.x, yz.x, b1); b2 = fma(k3.x, yz.y, b2);
                g1 = fma(k3.y, yz.x, g1); g2 = fma(k3.y, yz.y, g2);
            }
            double2 *pp = reinterpret_cast<double2 *>(s.PARTR) + 2 * (32 * t.slot + lane);
            pp[0] = make_double2(a1 + b1, a2 + b2);
            pp[1] = make_double2(f1 + g1, f2 + g2);
        } else if (t.kind == FE_RAG) {
            // the ragged rest of the block: row i takes columns a <= j < n_bulk[i]
            const int i = 32 * t.blk + lane, iv = min(i, N - 1);
            const int je = (i < N) ? (s.BINI[iv].x & 0x1ff) : 0;
            const double2 *kr = f.KR + tri(iv);
            double a1 = 0.0, a2 = 0.0, f1 = 0.0, f2 = 0.0, b1 = 0.0, b2 = 0.0, g1 = 0.0, g2 = 0.0;
            // (branch-free: the loads are unconditional -- past the end of a row they hit the next rows of
            //  the packed array -- and (y, y m) is replaced by 0 where the column does not count)
            int j = t.a;
#pragma unroll 4
            for (; j + 1 < t.b; j += 2) {
                const double2 k2 = kr[j], k3 = kr[j + 1];
                double2 yy = s.YY[j], yz = s.YY[j + 1];
                if (j >= je) { yy.x = 0.0; yy.y = 0.0; }
                if (j + 1 >= je) { yz.x = 0.0; yz.y = 0.0; }
                a1 = fma(k2.x, yy.x, a1); a2 = fma(k2.x, yy.y, a2);
                f1 = fma(k2.y, yy.x, f1); f2 = fma(k2.y, yy.y, f2);
                b1 = fma(k3.x, yz.x, b1); b2 = fma(k3.x, yz.y, b2);
                g1 = fma(k3.y, yz.x, g1); g2 = fma(k3.y, yz.y, g2);
            }
            if (j < t.b) {
                const double2 k2 = kr[j];
                double2 yy = s.YY[j];
                if (j >= je) { yy.x = 0.0; yy.y = 0.0; }
                a1 = fma(k2.x, yy.x, a1); a2 = fma(k2.x, yy.y, a2);
                f1 = fma(k2.y, yy.x, f1); f2 = fma(k2.y, yy.y, f2);
            }
            a1 += b1; a2 += b2; f1 += g1; f2 += g2;
            double2 *pp = reinterpret_cast<double2 *>(s.PARTR) + 2 * (32 * t.slot + lane);
            pp[0] = make_double2(a1, a2);
            pp[1] = make_double2(f1, f2);
        } else if (t.kind == FE_COLT) {
            // lane <-> impactor column j = 32 c + lane; rows [a, b) from the tensor-memory column copy
            uint32_t ta = tq_addr(tbase, quarter, t.tcol);
            double gc = 0.0, h = 0.0, gc2 = 0.0, h2 = 0.0;
            int i = t.a;
            auto quad = [&](const uint32_t (&v)[16], const double2 n01, const double2 n23) {
                gc = fma(u2d(v[0], v[1]), n01.x, gc);    h = fma(u2d(v[2], v[3]), n01.x, h);
                gc2 = fma(u2d(v[4], v[5]), n01.y, gc2);  h2 = fma(u2d(v[6], v[7]), n01.y, h2);
                gc = fma(u2d(v[8], v[9]), n23.x, gc);    h = fma(u2d(v[10], v[11]), n23.x, h);
                gc2 = fma(u2d(v[12], v[13]), n23.y, gc2); h2 = fma(u2d(v[14], v[15]), n23.y, h2);
            };
            for (; i + 7 <= t.b; i += 8, ta += 32) {          // two quads per wait
                uint32_t v[16], w[16];
                tmem_ld16(ta, v);
                tmem_ld16(ta + 16, w);
                const double2 n01 = *reinterpret_cast<const double2 *>(s.NN + i);
                const double2 n23 = *reinterpret_cast<const double2 *>(s.NN + i + 2);
                const double2 n45 = *reinterpret_cast<const double2 *>(s.NN + i + 4);
                const double2 n67 = *reinterpret_cast<const double2 *>(s.NN + i + 6);
                tmem_wait_ld();
                quad(v, n01, n23);
                quad(w, n45, n67);
            }
            for (; i + 3 <= t.b; i += 4, ta += 16) {
                uint32_t v[16];
                tmem_ld16(ta, v);
                const double2 n01 = *reinterpret_cast<const double2 *>(s.NN + i);
                const double2 n23 = *reinterpret_cast<const double2 *>(s.NN + i + 2);
                tmem_wait_ld();
                quad(v, n01, n23);
            }
            if (i < t.b) {          // one or two rows left (an odd last row was stored twice; NN[N] = 0)
                uint32_t v[8];
                tmem_ld8(ta, v);
                const double2 n01 = *reinterpret_cast<const double2 *>(s.NN + i);
                tmem_wait_ld();
                gc = fma(u2d(v[0], v[1]), n01.x, gc);    h = fma(u2d(v[2], v[3]), n01.x, h);
                gc2 = fma(u2d(v[4], v[5]), n01.y, gc2);  h2 = fma(u2d(v[6], v[7]), n01.y, h2);
            }
            reinterpret_cast<double2 *>(s.PARTC)[32 * t.slot + lane] = make_double2(gc + gc2, h + h2);
        } else if (t.kind == FE_COLS) {
            // the same sums from the shared-memory copy: diagonal blocks (rows i >= j) and overflow rows
            // (branch-free: every lane loads a valid address of the packed array -- for i < j that is some
            //  other pair's entry -- and the multiplier n_i is masked to 0 where the pair does not count)
            const int j = 32 * t.blk + lane, jv = min(j, N - 1);
            const int iSj = (j < N) ? ((s.BINI[jv].x >> 9) & 0x1ff) : 0x7fffffff;
            const int jm = (j < N) ? j : 0x7fffffff;
            const double2 *kp = f.KR + tri(t.a) + jv;
            double gc = 0.0, h = 0.0, gc2 = 0.0, h2 = 0.0;
            int i = t.a;
#pragma unroll 2
            for (; i + 1 < t.b; i += 2) {
                const double2 k2 = kp[0], k3 = kp[i + 1];
                const double2 nn = make_double2(s.NN[i], s.NN[i + 1]);
                kp += 2 * i + 3;
                gc = fma(k2.x, (i >= jm) ? nn.x : 0.0, gc);
                h = fma(k2.y, (i >= iSj) ? nn.x : 0.0, h);
                gc2 = fma(k3.x, (i + 1 >= jm) ? nn.y : 0.0, gc2);
                h2 = fma(k3.y, (i + 1 >= iSj) ? nn.y : 0.0, h2);
            }
            if (i < t.b) {
                const double2 k2 = kp[0];
                const double ni = s.NN[i];
                gc = fma(k2.x, (i >= jm) ? ni : 0.0, gc);
                h = fma(k2.y, (i >= iSj) ? ni : 0.0, h);
            }
            gc += gc2; h += h2;
            reinterpret_cast<double2 *>(s.PARTC)[32 * t.slot + lane] = make_double2(gc, h);
        } else {
            // band products of rows i = 32 blk + lane: W[d][i] = n_i n_{i-d} (K p_coag, K p_frag), d < bandD
            const int i = 32 * t.blk + lane, iv = min(i, N - 1);
            const double ni = s.NN[iv];
            const double2 *kr = f.KR + tri(iv) + iv;
            double *wc = s.WST + iv, *wf = wc + (size_t)tb.bandD * Np;
            const int nd = (i < N) ? min(tb.bandD, i + 1) : 0;
#pragma unroll
            for (int dd = 0; dd < 8; ++dd) {
                if (dd < nd) {
                    const double2 k2 = kr[-dd];
                    const double w = ni * s.NN[iv - dd];
                    wc[dd * Np] = w * k2.x;
                    wf[dd * Np] = w * k2.y;
                }
            }
        }
    }
    PROF_ADD(3, tpA);
#ifdef CUDISC_PROF
    if (lane == 0 && sa_prof) sa_prof[16 + warp] += clock64() - tpA;
#endif
    __syncthreads();
    PROF_ADD(4, tpA);
    PROF_T(tpB);

    // ---- phase B (combine), three groups of warps side by side:
    //   R (warp w < nw, bin 32 w + lane)        row partials -> deposits into bins k-1, k, k+1
    //   C (warp nw + w, bin 32 w + lane)        column partials -> loss frequency G_k; fragment source of
    //                                           l-bin k (its band entries gathered here), suffix scan of
    //                                           S_l / B_l (Eq. 67 via l-bins)
    //   band (warps bgWarp[g])                  band sums of the density targets 32 g + lane
    // G_k and the scanned value travel through NN[k] and YY[k].y, dead by now.
    const int nw = ft.nwBins;
    double d0 = 0.0, dm1 = 0.0, dp1 = 0.0, cFA = 0.0;
    if (warp < nw) {
        uint32_t cb[16];
        tmem_ld16(tq_addr(tbase, quarter, fast_binc_col_r(warp)), cb);
        double a1 = 0.0, a2 = 0.0, f1 = 0.0, f2 = 0.0;
        const double2 *pp = reinterpret_cast<const double2 *>(s.PARTR) + 2 * (32 * ft.rpBase[warp] + lane);
        const int np = ft.rpCnt[warp];
        for (int p = 0; p < np; ++p) {
            const double2 u = pp[64 * p], v = pp[64 * p + 1];
            a1 += u.x; a2 += u.y; f1 += v.x; f2 += v.y;
        }
        tmem_wait_ld();
        const double cA1 = u2d(cb[2 * FBC_A1], cb[2 * FBC_A1 + 1]), cA2 = u2d(cb[2 * FBC_A2], cb[2 * FBC_A2 + 1]);
        const double cB1 = u2d(cb[2 * FBC_B1], cb[2 * FBC_B1 + 1]), cF1 = u2d(cb[2 * FBC_F1], cb[2 * FBC_F1 + 1]);
        const double cF2 = u2d(cb[2 * FBC_F2], cb[2 * FBC_F2 + 1]), cG1 = u2d(cb[2 * FBC_G1], cb[2 * FBC_G1 + 1]);
        cFA = u2d(cb[2 * FBC_FA], cb[2 * FBC_FA + 1]);
        if (live) {
            dm1 = nk * (cG1 * f1 - cF2 * f2);
            d0 = nk * ((cA1 * a1 + cA2 * a2) + (cF1 * f1 + cF2 * f2));
            dp1 = nk * (cB1 * a1 - cA2 * a2);
        }
    }
    double *wtot = s.RED, *eUp = s.RED + 16, *eDn = s.RED + 32;
    if (warp < nw) {
        if (lane == 0) eDn[warp] = dm1;
        if (lane == 31) eUp[warp] = dp1;
    }
    const double up = __shfl_up_sync(0xffffffffu, dp1, 1);
    const double dn = __shfl_down_sync(0xffffffffu, dm1, 1);
    if (warp >= nw && warp < 2 * nw) {
        const int g = warp - nw, kc = 32 * g + lane;
        uint32_t fb[2];
        tmem_ld2(tq_addr(tbase, quarter, fast_binc_col_c(nw, warp)), fb);
        auto colsum = [&](int j, double &gj, double &hj) {
            const int c = j >> 5, np = ft.cpCnt[c];
            const double2 *pc2 = reinterpret_cast<const double2 *>(s.PARTC) + 32 * ft.cpBase[c] + (j & 31);
            gj = 0.0; hj = 0.0;
#pragma unroll 4
            for (int r = 0; r < np; ++r) {
                const double2 u = pc2[32 * r];
                gj += u.x; hj += u.y;
            }
        };
        double sl = band_gather(tbase, quarter, ft.sgCol[g], ft.sgLen[g], s.WST);
        if (kc < N) {
            const int2 bi = s.BINI[kc];
            double gc, h;
            colsum(kc, gc, h);
            s.NN[kc] = gc + h;                             // G_k
            for (int j = bi.y & 0xffff; j < (bi.y >> 16); ++j) {
                double gj, hj = h;
                if (j != kc) colsum(j, gj, hj);
                sl = fma(tb.sS * s.YY[j].x, hj, sl);
            }
        }
        double sv = (kc < N) ? sl * u2d(fb[0], fb[1]) : 0.0;
        double suf = sv;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double v = __shfl_down_sync(0xffffffffu, suf, o);
            if (lane + o < 32) suf += v;
        }
        if (lane == 0) wtot[g] = suf;
        if (kc < N) s.YY[kc].y = suf;
    }
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int gh = q ? myband.y : myband.x;
        if (gh >= 0) {
            const double v = band_gather(tbase, quarter, ft.bgCol[gh], ft.bgLen[gh], s.WST);
            const int kt = 32 * (gh >> 1) + lane;
            if (kt < N) ((gh & 1) ? s.BANDV2 : s.BANDV)[kt] = v;
        }
    }
#ifdef CUDISC_PROF
    if (lane == 0 && sa_prof) sa_prof[32 + warp] += clock64() - tpB;
#endif
    __syncthreads();

    double d = 0.0;
    if (live) {
        double suf = s.YY[k].y;
        for (int w = warp + 1; w < nw; ++w) suf += wtot[w];
        const double prev = (lane > 0) ? up : (warp > 0 ? eUp[warp - 1] : 0.0);
        const double next = (lane < 31) ? dn : (warp + 1 < nw ? eDn[warp + 1] : 0.0);
        d = d0;
        if (k > 0) d += prev;
        if (k < N - 1) d += next;
        d += s.BANDV[k] + s.BANDV2[k];
        d = fma(-y, s.NN[k], d);
        d = fma(cFA, suf, d);
    }
    PROF_ADD(5, tpB);
    return d;
}

template <int NT, int MODE>
__global__ void __launch_bounds__(NT, 1)
coag_fast_kernel(const DevTables tb, const FastTables ft, const GasArgs gs, const StepArgs sa_in)
{
    StepArgs sa = sa_in;
    if (MODE == MODE_STEP && !apply_ctrl(sa)) return;
    extern __shared__ __align__(16) double smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, quarter = warp & 3;
    const int N = tb.N, Np = tb.Np;
    const FSm f = fast_carve(smem_raw, ft);
    const Smem &s = f.s;
    PairConst pc;
    const bool has_vphi = gs.vphi != nullptr;
    pc.c15vf2 = 1.5 * gs.v_frag * gs.v_frag;
    pc.Vg2 = 0.0;
    const int k = tid;
    const bool live = k < N;
    const int nw = ft.nwBins;

    // ---- per-CTA constants
    for (int q = tid; q < 64; q += NT) s.EXPT[q] = tb.exptab[q];
    if (tb.logGrid) for (int q = tid; q < N; q += NT) s.DTAB[q] = tb.dtab[q];
    for (int q = tid; q < N; q += NT) s.BINI[q] = tb.bini[q];
    for (int q = tid; q < ft.bw[16]; q += NT) f.TB[q] = ft.buildTasks[q];
    for (int q = tid; q < ft.ew[16]; q += NT) f.TE[q] = ft.evalTasks[q];
    for (int q = N + tid; q < Np + 8; q += NT) s.NN[q] = 0.0;      // rows past the grid weigh 0 in the column pass
    const double mk = live ? tb.binc[BC_M * Np + k] : 0.0, rmk = live ? tb.binc[BC_RM * Np + k] : 0.0;

    uint32_t *slot = reinterpret_cast<uint32_t *>(s.RED);
    if (tid < 32) tmem_alloc_all(slot);
    tmem_fence_before();
    __syncthreads();
    tmem_fence_after();
    const uint32_t tbase = *slot;
    // per-bin constants of the combine step
    if (warp < nw) {
        uint32_t v[16];
#pragma unroll
        for (int u = 0; u < 16; ++u) v[u] = 0u;
        if (live) {
            const int src[kFastBinc] = {BC_A1, BC_A2, BC_B1, BC_F1, BC_F2, BC_G1, BC_FA};
#pragma unroll
            for (int u = 0; u < kFastBinc; ++u) {
                const double c = tb.binc[src[u] * Np + k];
                v[2 * u] = dlo(c); v[2 * u + 1] = dhi(c);
            }
        }
        const uint32_t t0 = tq_addr(tbase, quarter, fast_binc_col_r(warp));
        const uint32_t v0[8] = {v[0], v[1], v[2], v[3], v[4], v[5], v[6], v[7]};
        const uint32_t v1[8] = {v[8], v[9], v[10], v[11], v[12], v[13], v[14], v[15]};
        tmem_st8(t0, v0);
        tmem_st8(t0 + 8, v1);
    } else if (warp < 2 * nw) {
        const int kc = tid - 32 * nw;
        const double c = kc < N ? tb.binc[BC_FIB * Np + kc] : 0.0;
        tmem_st2(tq_addr(tbase, quarter, fast_binc_col_c(nw, warp)), dlo(c), dhi(c));
    }
    // band tables: each group by the warp that gathers it (tables are [len][32], lane <-> target)
    auto upload = [&](int col, int len, int off) {
        const uint32_t tc = tq_addr(tbase, quarter, col), ti = tc + 2 * len;
        for (int e0 = 0; e0 < len; e0 += 4) {
            uint32_t v[8], ix[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const double c = ft.bandCoef[off + (e0 + u) * 32 + lane];
                v[2 * u] = dlo(c); v[2 * u + 1] = dhi(c);
                ix[u] = ft.bandIdx[off + (e0 + u) * 32 + lane];
            }
            tmem_st8(tc + 2 * e0, v);
            tmem_st4(ti + e0, ix);
        }
    };
    for (int gh = 0; gh < 2 * nw; ++gh)
        if (ft.bgWarp[gh] == warp) upload(ft.bgCol[gh], ft.bgLen[gh], ft.bgOff[gh]);
    if (warp >= nw && warp < 2 * nw) upload(ft.sgCol[warp - nw], ft.sgLen[warp - nw], ft.sgOff[warp - nw]);
    tmem_wait_st();
    tmem_fence_before();
    __syncthreads();
    tmem_fence_after();
    // the (at most two) density band halves this warp gathers in the combine phase
    int2 myband = make_int2(-1, -1);
    for (int gh = 0; gh < 2 * nw; ++gh)
        if (ft.bgWarp[gh] == warp) { if (myband.x < 0) myband.x = gh; else myband.y = gh; }

    // frozen inputs of a cell, fetched one cell ahead: the per-cell scalars at the
    // start of the previous cell (its evaluations run the next prologue piece by piece), the per-bin
    // velocities two evaluations before its end
    CellGas nx = {1.0, 1.0, 1.0, 1.0};
    double nvR = 0.0, nvZ = 0.0, nvP = 0.0;
    auto stage_gas = [&](int cell) {        // cp.async of the per-cell scalars into RED[80 .. 83]
        if (cell >= sa.C || tid >= 4) return;
        const double *src = tid == 0 ? gs.T : (tid == 1 ? gs.rho_g : (tid == 2 ? gs.Omega : gs.alpha));
        if (src) cp_async8(s.RED + 80 + tid, src + cell);
    };
    auto take_gas = [&]() {
        nx.T = s.RED[80]; nx.rho_g = s.RED[81]; nx.Om = s.RED[82];
        nx.alpha = gs.alpha ? s.RED[83] : gs.alpha_const;
    };
    auto fetch_vel = [&](int cell) {
        if (cell >= sa.C || !live) return;
        const size_t g = (size_t)cell * N + k;
        nvR = __ldg(gs.vR + g); nvZ = __ldg(gs.vZ + g);
        if (has_vphi) nvP = __ldg(gs.vphi + g);
    };
    stage_gas(blockIdx.x);
    cp_async_wait_all();
    __syncthreads();
    take_gas();
    fetch_vel(blockIdx.x);
    RoleVals rv;
    rv.Vg2 = 0.0;
    ProlState ps = {2.0, 0.0, 0.0, 0.0};
    bool rv_valid = false;

    long long *sa_prof = sa.prof ? sa.prof + 48 * (size_t)blockIdx.x : nullptr;
    (void)sa_prof;
    int err_cell = -1;          // cell whose warp error maxima wait in RED[64 ..) for the next barrier
    auto flush_err = [&]() {
        if (MODE == MODE_STEP && tid == 0 && err_cell >= 0) {
            unsigned long long m = 0ull;
            for (int w = 0; w < nw; ++w) {
                const unsigned long long v = reinterpret_cast<const unsigned long long *>(s.RED)[64 + w];
                m = v > m ? v : m;
            }
            sa.err[err_cell] = __longlong_as_double((long long)m);
        }
    };
    for (int cell = blockIdx.x; cell < sa.C; cell += gridDim.x) {
        PROF_T(tc0);
        const size_t row = (size_t)cell * N;
        if (!rv_valid) rv = prologue_compute(tb, nx, gs.mu, gs.sigma_mol, rmk, k);
        prologue_store(tb, rv, nvR, nvZ, nvP, has_vphi, false, s, k);
        if (tid == 0) s.RED[95] = rv.Vg2;
        __syncthreads();
        pc.Vg2 = s.RED[95];
        flush_err();
        PROF_ADD(0, tc0);
        PROF_T(tb0);
        // state and FSAL derivative of the cell (thread <-> bin) and the next cell's gas scalars: asynchronous
        // copies into (y, y m) -- free during the build -- and RED, landed by the post-build barrier
        if (live) {
            cp_async8(&s.YY[k].x, sa.rho + row + k);
            if (MODE == MODE_STEP && sa.have_k1) cp_async8(&s.YY[k].y, sa.k_fsal + row + k);
        }
        stage_gas(cell + gridDim.x);
        if (has_vphi) {
            if (tb.logGrid) fast_build<true, true>(tb, ft, f, pc, tbase, warp, lane);
            else fast_build<true, false>(tb, ft, f, pc, tbase, warp, lane);
        } else {
            if (tb.logGrid) fast_build<false, true>(tb, ft, f, pc, tbase, warp, lane);
            else fast_build<false, false>(tb, ft, f, pc, tbase, warp, lane);
        }
        cp_async_wait_all();
        double y0 = 0.0, k1 = 0.0;
        if (live) {                                   // the thread's own copies are complete
            y0 = s.YY[k].x;
            if (MODE == MODE_STEP && sa.have_k1) k1 = s.YY[k].y;
        }
        if (MODE == MODE_STEP && warp < nw) {
            double ws = y0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) ws += __shfl_xor_sync(0xffffffffu, ws, o);
            if (lane == 0) s.RED[48 + warp] = ws;
        }
        tmem_fence_before();
        __syncthreads();
        tmem_fence_after();
        take_gas();
        PROF_ADD(1, tb0);

        const bool more = cell + (int)gridDim.x < sa.C;
        if (MODE == MODE_OTF) {
            fetch_vel(cell + gridDim.x);
            const double d = fast_eval<NT>(tb, ft, f, y0, mk, rmk, tid, tbase, more ? 4 : 0, nx, gs.mu,
                                           gs.sigma_mol, ps, rv, myband, sa_prof);
            rv_valid = more;
            if (live) sa.out[row + k] = d;
            __syncthreads();
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
            if (st == 2) fetch_vel(cell + gridDim.x);
            if (st == 3) {
                yn = y0 + h * ((2.0 / 9.0) * k1 + (1.0 / 3.0) * k2 + (4.0 / 9.0) * k3);
                ys = yn;
            }
            const double d = fast_eval<NT>(tb, ft, f, ys, mk, rmk, tid, tbase, more ? st : 0, nx, gs.mu,
                                           gs.sigma_mol, ps, rv, myband, sa_prof);
            if (st == 3) rv_valid = more;
            if (st == 0) k1 = d;
            if (st == 1) k2 = d;
            if (st == 2) k3 = d;
            if (st == 3) k4 = d;
        }
        // error norm (R10) and write-back.  sum_k y0_k: warp sums taken before the post-build
        // barrier; max_k: warp maxima here, combined by thread 0 after the next block barrier (the scaled
        // errors are >= 0 or NaN, so the unsigned order of their bit patterns is the NaN-propagating max)
        PROF_T(ttail);
        double ysum = 0.0;
        for (int w = 0; w < nw; ++w) ysum += s.RED[48 + w];
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
        if (warp < nw) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const unsigned long long v = __shfl_xor_sync(0xffffffffu, eb, o);
                eb = v > eb ? v : eb;
            }
            if (lane == 0) reinterpret_cast<unsigned long long *>(s.RED)[64 + warp] = eb;
        }
        err_cell = cell;
        PROF_ADD(7, ttail);
        PROF_ADD(6, tc0);
    }
    tmem_fence_before();
    __syncthreads();
    flush_err();
    if (tid < 32) tmem_dealloc_all(tbase);
}

template <int MODE>
cudaError_t launch_fast_mode(const LaunchCfg &lc, const DevTables &tb, const FastTables &ft, const GasArgs &gs,
                             const StepArgs &sa, cudaStream_t st)
{
    auto fn = coag_fast_kernel<kThreads, MODE>;
    static bool attr_done[64] = {false};    // the attribute is per device (and per instantiation)
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !attr_done[dev]) {
        e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, lc.smem_optin);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) attr_done[dev] = true;
    }
    fn<<<lc.grid, kThreads, lc.smem_bytes, st>>>(tb, ft, gs, sa);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_fast(int mode, const LaunchCfg &lc, const DevTables &tb, const FastTables &ft,
                        const GasArgs &gs, const StepArgs &sa, cudaStream_t st)
{
    if (mode == MODE_OTF) return launch_fast_mode<MODE_OTF>(lc, tb, ft, gs, sa, st);
    return launch_fast_mode<MODE_STEP>(lc, tb, ft, gs, sa, st);
}

}  // namespace cudisc
