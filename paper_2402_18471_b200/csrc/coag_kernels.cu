// coag_kernels.cu -- __global__ entry points of libcudisc_coag.so (sm_100a, FP64) and their launchers.
//
// One persistent CTA per SM walks the cells c = blockIdx.x, blockIdx.x + gridDim.x, ...
// Every mode shares the device routines of coag_device.cuh:
//   MODE_KERNEL : prologue + pair build                -> K_out [C][2][P] in HBM      (cudisc_coag_kernel)
//   MODE_RATES  : K planes from HBM -> K store, eval   -> drho_dt                     (cudisc_coag_rates)
//   MODE_OTF    : prologue + pair build -> K store, eval -> drho_dt                   (cudisc_coag_rates_otf)
//   MODE_STEP   : prologue + pair build -> K store, BS3(2) stages (3 or 4 evals)      (cudisc_coag_step)
//   MODE_STEPK  : K planes from HBM -> K store, BS3(2) stages                         (cudisc_coag_step_cached)
// Thread k < N owns bin k: its density, stage values and derivatives live in registers.
#include "coag_launch.h"

namespace cudisc {


// ------------------------------------------------------------------------------------------ build
// K_ij p_coag, K_ij p_frag of every pair of the cell into the K store (or, MODE_KERNEL, to HBM).
//   rows item {c, ia, ib}: lanes <-> columns j = 32 c + lane (values of grain j stay in registers),
//       rows i in [ia, ib), all >= 32 c + 32 (no diagonal pair), two rows per iteration (an odd last
//       row is computed twice);
//   list item {c, t0, t1}: pairs of diagonal block c (rows 32 c .. 32 c + 31) by triangular index
//       t = r (r + 1) / 2 + s, i = 32 c + r, j = 32 c + s; lanes <-> t.
template <int MODE, bool SLAB, bool VPHI, bool LOG>
__device__ __forceinline__ void build_items(const DevTables &tb, const Smem &s, const KStore<SLAB> &ks,
                                            const PairConst &pc, double *kout, int lane)
{
    const int N = tb.N, P = tb.P;
    // the first item of every warp is fixed (item = warp; the counter starts at the warp count):
    // no pile-up of all warps on one shared-memory atomic at the start of the phase
    bool first = true;
    for (;;) {
        const int it = first ? (int)(threadIdx.x >> 5) : next_item(&s.CTR[0], lane);
        first = false;
        if (it >= tb.nBuildItems) break;
        const uint32_t item = s.ITB[it];
        const int c = (item >> 28) & 7, ia = (item >> 14) & 0x3fff, ib = item & 0x3fff;
        if ((item >> 31) == IT_BUILD_ROWS) {
            const int j = 32 * c + lane;
            const bool valid = j < N;
            const RoleJ B = load_role_j<VPHI>(s, valid ? j : N - 1);
            for (int i = ia; i < ib; i += 2) {
                const int i2 = min(i + 1, ib - 1);
                const RoleI A1 = load_role_i<VPHI, false>(s, i);
                const RoleI A2 = load_role_i<VPHI, false>(s, i2);
                const double2 k1 = pair_kernel<VPHI, LOG, false>(A1, B, i - j, pc, s);
                const double2 k2 = pair_kernel<VPHI, LOG, false>(A2, B, i2 - j, pc, s);
                if (valid) {
                    const int p1 = tri(i) + j, p2 = tri(i2) + j;
                    if (MODE == MODE_KERNEL) {
                        kout[p1] = k1.x; kout[P + p1] = k1.y;
                        kout[p2] = k2.x; kout[P + p2] = k2.y;
                    } else {
                        ks.st(p1, k1);
                        ks.st(p2, k2);
                    }
                }
            }
        } else {
            for (int t = ia + lane; t < ib; t += 32) {
                int r = (int)((sqrtf(8.0f * (float)t + 1.0f) - 1.0f) * 0.5f);
                r += (tri(r + 1) <= t) ? 1 : 0;
                r -= (tri(r) > t) ? 1 : 0;
                const int i = 32 * c + r, j = 32 * c + (t - tri(r));
                const RoleI A = load_role_i<VPHI, true>(s, i);
                const RoleJ B = load_role_j<VPHI>(s, j);
                double2 k2 = pair_kernel<VPHI, LOG, true>(A, B, i - j, pc, s);
                const int p = tri(i) + j;
                if (MODE == MODE_KERNEL) {
                    kout[p] = k2.x; kout[P + p] = k2.y;
                } else {
                    if (i == j) { k2.x *= 0.5; k2.y *= 0.5; }
                    ks.st(p, k2);
                }
            }
        }
    }
}

template <int MODE, bool SLAB>
__device__ __forceinline__ void build_cell(const DevTables &tb, const Smem &s, const KStore<SLAB> &ks,
                                           const PairConst &pc, bool has_vphi, double *kout, int lane)
{
    // warp-uniform dispatch: the inner loops are compiled for their case
    if (has_vphi) {
        if (tb.logGrid) build_items<MODE, SLAB, true, true>(tb, s, ks, pc, kout, lane);
        else build_items<MODE, SLAB, true, false>(tb, s, ks, pc, kout, lane);
    } else {
        if (tb.logGrid) build_items<MODE, SLAB, false, true>(tb, s, ks, pc, kout, lane);
        else build_items<MODE, SLAB, false, false>(tb, s, ks, pc, kout, lane);
    }
}

// ------------------------------------------------------------------------------------------ eval
// One rate evaluation of the current cell: thread k < N passes y_k and gets drho_k/dt.
// Three block barriers; every partial sum has its own slot and every combination a fixed order.
constexpr int kRedMbar = 88;     // Smem::RED slot that holds the mbarrier of the refill

// The same for a store of (Kc, Kf) pairs (cudisc_coag_step_cached: three evaluations per load, and the pair layout
// makes an evaluation 20 % faster than the planar one): 8-byte LDGSTS copies, plane 0 -> .x, plane 1 -> .y of
// every pair, by all threads; completed by cp.async.wait_all + a block barrier.
__device__ __forceinline__ void refill_pairs(double2 *ksm, const double *planes, int P, int tid, int nt)
{
    for (int p = tid; p < P; p += nt) {
        const uint32_t dst = smem_addr(ksm + p);
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" :: "r"(dst), "l"(planes + p) : "memory");
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" :: "r"(dst + 8), "l"(planes + P + p) : "memory");
    }
}

// kin_next: planes of the cell whose kernel the K store takes NEXT (modes that read K from HBM, last evaluation of
// a cell), or nullptr: the refill starts as soon as the last read of K is behind the block, under the combine phase.
template <int NT, bool SLAB, bool PLANAR>
__device__ __forceinline__ double eval_rates(const DevTables &tb, const Smem &s, const KStore<SLAB, PLANAR> &ks,
                                             double y, int tid, uint32_t tbase,
                                             bool pre, const CellGas &nx, double mu, double sigma_mol,
                                             RoleVals &rv, const double *kin_next = nullptr)
{
    const int N = tb.N, Np = tb.Np;
    const int lane = tid & 31, warp = tid >> 5;
    const int k = tid;
    const bool live = k < N;

    // ---- phase 0: number densities and the (y, y m) pairs
    double nk = 0.0;
    if (live) {
        nk = y * s.BINC[BC_RM * Np + k];
        s.NN[k] = nk;
        s.YY[k] = make_double2(y, y * s.BINC[BC_M * Np + k]);
        if (!tb.bandD) {                           // second band slot: only split groups write it
            s.BANDV2[k] = 0.0;
            s.BANDV2[N + k] = 0.0;
        }
    }
    if (tid == 0) { s.CTR[1] = NT / 32; s.CTR[2] = 0; }
    __syncthreads();

    // per-bin values of the NEXT cell (inputs were fetched an evaluation ago): the bin-owning warps
    // compute them here, in registers, while the other warps start on the items
    if (pre && 32 * warp < N) rv = prologue_compute(tb, nx, mu, sigma_mol, live ? s.BINC[BC_RM * Np + k] : 0.0, k);

    // ---- phase A: band gathers from tensor memory (tasks fixed per warp: a warp only reaches the
    //      tensor-memory lanes of its quarter), then row sums, column sums (and, without
    //      tensor-memory tables, band gathers) pulled by warps
    if (tb.bandTmem && !tb.bandD) {
#pragma unroll 1
        for (int q = 0; q < 2; ++q) {
            const int task = s.SCHED[SC_BTASK + 2 * warp + q];
            if (task >= 0) break;                                  // valid bit = sign bit
            const int g = (task >> 16) & 0xff, e0b = (task >> 8) & 0xff, e1b = task & 0xff;
            const int t = 32 * g + lane, Lp = tb.bandLp;
            const uint32_t tc = tmem_warp_addr(tbase, g, 0), ti = tc + 2 * Lp;
            const double *kd = reinterpret_cast<const double *>(ks.sm);
            double acc0 = 0.0, acc1 = 0.0;
            for (int e0 = e0b; e0 < e1b; e0 += 8) {
                uint32_t cf[16], ixs[8];
                tmem_ld16(tc + 2 * e0, cf);
                tmem_ld8(ti + e0, ixs);
                tmem_wait_ld();
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int i = ixs[u] & 0xff, j = (ixs[u] >> 8) & 0xff;
                    const int p2 = 2 * (tri(i) + j) + (int)((ixs[u] >> 16) & 1);
                    const double kv = SLAB ? ((ixs[u] >> 16) & 1 ? ks.ld(p2 >> 1).y : ks.ld(p2 >> 1).x)
                                           : (PLANAR ? kd[(p2 & 1) * tb.P + (p2 >> 1)] : kd[p2]);
                    const double c = __hiloint2double((int)cf[2 * u + 1], (int)cf[2 * u]);
                    if (u & 1) acc1 = fma(c * s.NN[i], s.NN[j] * kv, acc1);
                    else acc0 = fma(c * s.NN[i], s.NN[j] * kv, acc0);
                }
            }
            if (t < 2 * N) (((task >> 30) & 1) ? s.BANDV2 : s.BANDV)[t] = acc0 + acc1;
        }
    }
    // band gathers from the staged products (tensor-memory coefficients and stage indices): run by the
    // owning warp after its first item, when the (short, first-claimed) W items are done
    auto band_from_stage = [&]() {
#pragma unroll 1
        for (int q = 0; q < 2; ++q) {
            const int task = s.SCHED[SC_BTASK + 2 * warp + q];
            if (task >= 0) break;                                  // valid bit = sign bit
            while (*reinterpret_cast<volatile int *>(&s.CTR[2]) < tb.nWItems) { }
            __threadfence_block();
            const int g = (task >> 16) & 0xff, e0b = (task >> 8) & 0xff, e1b = task & 0xff;
            const int t = 32 * g + lane, Lp = tb.bandLp;
            const uint32_t tc = tmem_warp_addr(tbase, g, 0), ti = tc + 2 * Lp;
            double acc0 = 0.0, acc1 = 0.0;
            for (int e0 = e0b; e0 < e1b; e0 += 8) {
                uint32_t cf[16], ixs[8];
                tmem_ld16(tc + 2 * e0, cf);
                tmem_ld8(ti + e0, ixs);
                tmem_wait_ld();
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const double c = __hiloint2double((int)cf[2 * u + 1], (int)cf[2 * u]);
                    if (u & 1) acc1 = fma(c, s.WST[ixs[u]], acc1);
                    else acc0 = fma(c, s.WST[ixs[u]], acc0);
                }
            }
            if (t < 2 * N) s.BANDV[t] = acc0 + acc1;
        }
    };
    const bool stage_band = tb.bandTmem && tb.bandD && s.SCHED[SC_BTASK + 2 * warp] < 0;
    bool band_done = !stage_band;
    bool first = true;
    for (;;) {
        const int it = first ? NT / 32 - 1 - warp : next_item(&s.CTR[1], lane);
        first = false;
        if (it >= tb.nEvalItems) break;
        const uint32_t item = s.ITE[it];
        const int kind = item >> 30, ix = (item >> 26) & 15, iy = (item >> 23) & 7;
        const int iz = (item >> 9) & 0x1ff, iw = item & 0x1ff;
        if (kind == IT_ROW) {
            // lane <-> target row i of block ix, impactors j of chunk iy, j < n_bulk[i]
            const int i = 32 * ix + lane;
            const int jb = kRowChunk * iy;
            int je = 0;
            if (i < N) je = min(jb + kRowChunk, s.BINI[i].x & 0x1ff);
            const int jmax = iw;                             // max of je over the block (host)
            const int base = tri(i);
            double a1 = 0.0, a2 = 0.0, f1 = 0.0, f2 = 0.0, b1 = 0.0, b2 = 0.0, g1 = 0.0, g2 = 0.0;
#pragma unroll 4
            for (int j = jb; j < jmax; j += 2) {
                if (j < je) {
                    const double2 k2 = ks.ld(base + j);
                    const double2 yy = s.YY[j];
                    a1 = fma(k2.x, yy.x, a1); a2 = fma(k2.x, yy.y, a2);
                    f1 = fma(k2.y, yy.x, f1); f2 = fma(k2.y, yy.y, f2);
                }
                if (j + 1 < je) {
                    const double2 k2 = ks.ld(base + j + 1);
                    const double2 yy = s.YY[j + 1];
                    b1 = fma(k2.x, yy.x, b1); b2 = fma(k2.x, yy.y, b2);
                    g1 = fma(k2.y, yy.x, g1); g2 = fma(k2.y, yy.y, g2);
                }
            }
            const int first = s.SCHED[SC_ROWFIRST + iy];
            if (i < N && i >= first) {
                double2 *pp = reinterpret_cast<double2 *>(s.PARTR) + 2 * (s.SCHED[SC_ROWOFF + iy] - first + i);
                pp[0] = make_double2(a1 + b1, a2 + b2);
                pp[1] = make_double2(f1 + g1, f2 + g2);
            }
        } else if (kind == IT_COL) {
            // lane <-> impactor column j of block ix, target rows i in [iz, iw) of range iy
            const int j = 32 * ix + lane;
            if (j < min(N, iw)) {
                const int iSj = (s.BINI[j].x >> 9) & 0x1ff;
                double gc = 0.0, h = 0.0, gc2 = 0.0, h2 = 0.0;
                int i = max(iz, j);
                if ((iw - i) & 1) {
                    const double2 k2 = ks.ld(tri(i) + j);
                    const double ni = s.NN[i];
                    gc = fma(k2.x, ni, gc);
                    if (i >= iSj) h = fma(k2.y, ni, h);
                    ++i;
                }
#pragma unroll 4
                for (; i < iw; i += 2) {
                    const double2 k2 = ks.ld(tri(i) + j), k3 = ks.ld(tri(i + 1) + j);
                    const double ni = s.NN[i], ni1 = s.NN[i + 1];
                    gc = fma(k2.x, ni, gc);
                    if (i >= iSj) h = fma(k2.y, ni, h);
                    gc2 = fma(k3.x, ni1, gc2);
                    if (i + 1 >= iSj) h2 = fma(k3.y, ni1, h2);
                }
                reinterpret_cast<double2 *>(s.PARTC)[s.SCHED[SC_COLOFF + iy] + j] = make_double2(gc + gc2, h + h2);
            }
        } else if (kind == IT_W) {
            // band products of rows i = 32 ix + lane: W[d][i] = n_i n_{i-d} (K p_coag, K p_frag), d < bandD
            const int i = 32 * ix + lane;
            if (i < N) {
                const double ni = s.NN[i];
                const int base = tri(i);
                double *wc = s.WST + i, *wf = wc + (size_t)tb.bandD * Np;
                for (int dd = 0; dd < tb.bandD && dd <= i; ++dd) {
                    const double2 k2 = ks.ld(base + i - dd);
                    const double w = ni * s.NN[i - dd];
                    wc[dd * Np] = w * k2.x;
                    wf[dd * Np] = w * k2.y;
                }
            }
            __syncwarp();
            if (lane == 0) { __threadfence_block(); atomicAdd(&s.CTR[2], 1); }
        } else {
            // band gather from global tables (fallback): lane <-> target t of group ix
            const int t = 32 * ix + lane;
            const int cnt = (t < 2 * N) ? __ldg(tb.band_cnt + t) : 0;
            double acc = 0.0;
            for (int e = 0; e < iw; ++e) {
                if (e < cnt) {
                    const uint32_t ixe = __ldcg(tb.band_idx + (size_t)e * tb.bandW + t);
                    const double cf = __ldcg(tb.band_coef + (size_t)e * tb.bandW + t);
                    const int i = ixe & 0xff, j = (ixe >> 8) & 0xff;
                    const double2 k2 = ks.ld(tri(i) + j);
                    const double kv = (ixe >> 16) & 1 ? k2.y : k2.x;
                    acc = fma(cf * s.NN[i], s.NN[j] * kv, acc);
                }
            }
            if (t < 2 * N) s.BANDV[t] = acc;
        }
        if (!band_done) { band_from_stage(); band_done = true; }
    }
    if (!band_done) band_from_stage();
    __syncthreads();
    if (kin_next) {
        if (PLANAR) {
            if (tid == 0) refill_bulk(ks.sm, kin_next, tb.P, reinterpret_cast<uint64_t *>(s.RED + kRedMbar));
        } else if (!SLAB) {
            refill_pairs(ks.sm, kin_next, tb.P, tid, NT);
        }
    }

    // ---- phase B: combine partials in fixed order.  Two warp groups work side by side:
    //   group R (thread k, bin k)            row partials -> deposits into bins k-1, k, k+1
    //   group C (thread k + 32 nw, bin k)    column partials -> loss frequency G_k, fragment source,
    //                                        warp suffix scan of S_l / B_l (Eq. 67 via l-bins)
    // and meet at one barrier; G_k and the scanned value travel through NN[k] and YY[k].y, dead by now.
    const int nw = (N + 31) >> 5;
    double d0 = 0.0, dm1 = 0.0, dp1 = 0.0;
    if (live) {
        const int nb = s.BINI[k].x & 0x1ff;
        double a1 = 0.0, a2 = 0.0, f1 = 0.0, f2 = 0.0;
        // (straight-line: slot bases are kernel constants, the loads of all chunks issue together)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            if (nb > kRowChunk * c) {
                const double2 *pp = reinterpret_cast<const double2 *>(s.PARTR) + 2 * (tb.rowBase[c] + k);
                const double2 u = pp[0], v = pp[1];
                a1 += u.x; a2 += u.y; f1 += v.x; f2 += v.y;
            }
        }
        const double *bc = s.BINC + k;
        const double cA2 = bc[BC_A2 * Np], cF2 = bc[BC_F2 * Np];
        dm1 = nk * (bc[BC_G1 * Np] * f1 - cF2 * f2);
        d0 = nk * ((bc[BC_A1 * Np] * a1 + cA2 * a2) + (bc[BC_F1 * Np] * f1 + cF2 * f2));
        dp1 = nk * (bc[BC_B1 * Np] * a1 - cA2 * a2);
    }
    double *wtot = s.RED, *eUp = s.RED + 16, *eDn = s.RED + 32;
    if (warp < nw) {
        if (lane == 0) eDn[warp] = dm1;
        if (lane == 31) eUp[warp] = dp1;
    }
    const double up = __shfl_up_sync(0xffffffffu, dp1, 1);
    const double dn = __shfl_down_sync(0xffffffffu, dm1, 1);
    if (warp >= nw && warp < 2 * nw) {
        const int kc = tid - 32 * nw;                      // bin of this group-C thread
        double sv = 0.0;
        if (kc < N) {
            const int2 bi = s.BINI[kc];
            // column sums of bin j over the row ranges that hold rows >= j (fixed order)
            auto colsum = [&](int j, int rfirst, double &gj, double &hj) {
                gj = 0.0; hj = 0.0;
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    if (r >= rfirst && r < tb.nRng) {
                        const double2 u = reinterpret_cast<const double2 *>(s.PARTC)[tb.colOff[r] + j];
                        gj += u.x; hj += u.y;
                    }
                }
            };
            double gc, h;
            colsum(kc, bi.x >> 18, gc, h);
            s.NN[kc] = gc + h;                             // G_k
            // fragment source of l-bin k, scaled by 1/B_k
            double sl = s.BANDV[N + kc] + (tb.bandD ? 0.0 : s.BANDV2[N + kc]);
            for (int j = bi.y & 0xffff; j < (bi.y >> 16); ++j) {
                double gj, hj = h;
                if (j != kc) colsum(j, s.BINI[j].x >> 18, gj, hj);
                sl = fma(tb.sS * s.YY[j].x, hj, sl);
            }
            sv = sl * s.BINC[BC_FIB * Np + kc];
        }
        // inclusive suffix sum over the bins of the warp; the warp totals are added after the barrier
        double suf = sv;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double v = __shfl_down_sync(0xffffffffu, suf, o);
            if (lane + o < 32) suf += v;
        }
        if (lane == 0) wtot[warp - nw] = suf;
        if (kc < N) s.YY[kc].y = suf;
    }
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
        d += s.BANDV[k] + (tb.bandD ? 0.0 : s.BANDV2[k]);
        d = fma(-y, s.NN[k], d);
        d = fma(s.BINC[BC_FA * Np + k], suf, d);
    }
    return d;
}

template <int NT, int MODE, bool SLAB, bool VINT>
__global__ void __launch_bounds__(NT, 1)
coag_cells_kernel(const DevTables tb, const GasArgs gs, const StepArgs sa_in)
{
    StepArgs sa = sa_in;
    if ((MODE == MODE_STEP || MODE == MODE_STEPK) && !apply_ctrl(sa)) return;
    extern __shared__ __align__(16) double smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31;
    const int N = tb.N, P = tb.P;
    constexpr bool PLANAR = MODE == MODE_RATES && !SLAB;
    KStore<SLAB, PLANAR> ks;
    ks.sm = reinterpret_cast<double2 *>(smem_raw);
    ks.Psm = sa.Psm;
    ks.P = P;
    ks.gl = reinterpret_cast<double2 *>(sa.kslab) + (size_t)blockIdx.x * (size_t)(P - sa.Psm);
    const Smem s = carve(smem_raw + 2 * (size_t)sa.Psm, tb.Np, tb.partRowSlots, tb.partColSlots,
                         tb.nBuildItems, tb.nEvalItems, tb.bandD);
    PairConst pc;
    const bool has_vphi = gs.vphi != nullptr;
    constexpr bool has_h = VINT;        // vertically integrated kernel: its own instantiation
    pc.c15vf2 = 1.5 * gs.v_frag * gs.v_frag;
    pc.Vg2 = 0.0;

    // per-CTA constants in shared memory
    for (int q = tid; q < 64; q += NT) s.EXPT[q] = tb.exptab[q];
    if (tb.logGrid) for (int q = tid; q < N; q += NT) s.DTAB[q] = tb.dtab[q];
    for (int q = tid; q < kBinC * tb.Np; q += NT) s.BINC[q] = tb.binc[q];
    for (int q = tid; q < N; q += NT) s.BINI[q] = tb.bini[q];
    for (int q = tid; q < tb.nBuildItems; q += NT) s.ITB[q] = tb.buildItems[q];
    for (int q = tid; q < tb.nEvalItems; q += NT) s.ITE[q] = tb.evalItems[q];
    if (tid < kSched) s.SCHED[tid] = tb.sched[tid];
    // band tables -> tensor memory (grid-only constants, once per CTA)
    uint32_t tbase = 0;
    const bool use_tmem = MODE != MODE_KERNEL && tb.bandTmem;
    if (use_tmem) {
        uint32_t *slot = reinterpret_cast<uint32_t *>(s.RED);
        if (tid < 32) tmem_alloc_all(slot);
        tmem_fence_before();
        __syncthreads();
        tmem_fence_after();
        tbase = *slot;
        const int warp = tid >> 5;
        if (32 * warp < 2 * N) {
            const int t = 32 * warp + lane, Lp = tb.bandLp;
            const int cnt = tb.band_cnt[t];                        // band_cnt is padded to bandW >= 32 groups
            for (int e0 = 0; e0 < Lp; e0 += 8) {
                uint32_t v[8];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = e0 + u;
                    const double c = e < cnt ? tb.band_coef[(size_t)e * tb.bandW + t] : 0.0;
                    v[2 * u] = (uint32_t)__double2loint(c); v[2 * u + 1] = (uint32_t)__double2hiint(c);
                }
                tmem_st8(tmem_warp_addr(tbase, warp, 2 * e0), v);
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = e0 + 4 + u;
                    const double c = e < cnt ? tb.band_coef[(size_t)e * tb.bandW + t] : 0.0;
                    v[2 * u] = (uint32_t)__double2loint(c); v[2 * u + 1] = (uint32_t)__double2hiint(c);
                }
                tmem_st8(tmem_warp_addr(tbase, warp, 2 * e0 + 8), v);
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int e = e0 + u;
                    v[u] = e < cnt ? tb.band_idx[(size_t)e * tb.bandW + t] : 0u;
                }
                tmem_st8(tmem_warp_addr(tbase, warp, 2 * Lp + e0), v);
            }
            tmem_wait_st();
        }
        tmem_fence_before();
    }
    __syncthreads();
    if (use_tmem) tmem_fence_after();

    const int k = tid;
    const bool live = k < N;

    // frozen inputs of a cell, fetched one cell ahead: the loads of cell c + grid
    // are issued before the last rate evaluation of cell c
    CellGas nx = {1.0, 1.0, 1.0, 1.0};
    double nvR = 0.0, nvZ = 0.0, nvP = 0.0;
    auto fetch = [&](int cell) {
        if (MODE == MODE_RATES || MODE == MODE_STEPK || cell >= sa.C) return;
        nx.T = __ldg(gs.T + cell); nx.rho_g = __ldg(gs.rho_g + cell); nx.Om = __ldg(gs.Omega + cell);
        nx.alpha = gs.alpha ? __ldg(gs.alpha + cell) : gs.alpha_const;
        if (live) {
            const size_t g = (size_t)cell * N + k;
            nvR = __ldg(gs.vR + g); nvZ = __ldg(gs.vZ + g);
            if (has_vphi) nvP = __ldg(gs.vphi + g);
            if (has_h) nvP = __ldg(gs.hd + g);
        }
    };
    fetch(blockIdx.x);
    // refill of a PLANAR K store by bulk copies: mbarrier in RED, phase bit per cell
    uint64_t *kbar = reinterpret_cast<uint64_t *>(s.RED + kRedMbar);
    uint32_t kph = 0u;
    const bool kin_tma = PLANAR && (reinterpret_cast<uintptr_t>(sa.Kin) & 15) == 0;
    if (PLANAR) {
        if (tid == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" :: "r"(smem_addr(kbar)), "r"(1) : "memory");
            asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        }
        __syncthreads();
    }
    RoleVals rv;
    rv.Vg2 = 0.0;
    bool rv_valid = false;       // rv holds the next cell's values (computed during the last evaluation)

    for (int cell = blockIdx.x; cell < sa.C; cell += gridDim.x) {
        const size_t row = (size_t)cell * N;

        // ---------------- K store for this cell
        if (MODE == MODE_RATES || MODE == MODE_STEPK) {
            // The planes of this cell.  Everything fits in shared memory: the refill that the CTA started behind the
            // last read of its previous cell's kernel, i.e. under that cell's combine phase (eval_rates), lands here --
            // bulk copies completing on the mbarrier (PLANAR store; planes that are not 16-byte aligned take a plain
            // copy) or LDGSTS copies (store of pairs).  Slab: a flat, coalesced copy of both planes, 16 loads in
            // flight per thread.
            // Then the N diagonal entries are halved in place.
            const double *k0 = sa.Kin + (size_t)cell * 2 * P, *k1 = k0 + P;
            if (PLANAR) {
                if (kin_tma) {
                    if (cell == (int)blockIdx.x && tid == 0) refill_bulk(ks.sm, k0, P, kbar);
                    mbar_wait_parity(kbar, kph);
                    kph ^= 1u;
                } else {
                    double *dstp = reinterpret_cast<double *>(ks.sm);
                    for (int p = tid; p < 2 * P; p += NT) dstp[p] = __ldcs(k0 + p);
                }
            } else if (!SLAB) {
                if (cell == (int)blockIdx.x) refill_pairs(ks.sm, k0, P, tid, NT);
                asm volatile("cp.async.wait_all;\n" ::: "memory");
            } else {
                for (int p0 = tid; p0 < P; p0 += 8 * NT) {
                    double a[8], b[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int p = p0 + u * NT;
                        a[u] = p < P ? __ldcs(k0 + p) : 0.0;
                        b[u] = p < P ? __ldcs(k1 + p) : 0.0;
                    }
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int p = p0 + u * NT;
                        if (p < P) ks.st(p, make_double2(a[u], b[u]));
                    }
                }
            }
            __syncthreads();
            if (live) {
                const int p = tri(k) + k;
                const double2 v = ks.ld(p);
                ks.st(p, make_double2(0.5 * v.x, 0.5 * v.y));
            }
            // The K store of a cell fills the shared memory, so the next cell's planes cannot be staged there while
            // this one is evaluated: they are pulled into L2 meanwhile (asynchronous bulk prefetch, 8 KB per thread), and
            // the refill then reads them at L2 speed.  In flight over the chip: one cell per CTA (27 MB at 150 bins).
            if (cell + (int)gridDim.x < sa.C && (reinterpret_cast<uintptr_t>(sa.Kin) & 15) == 0) {
                const char *nxt = reinterpret_cast<const char *>(sa.Kin + (size_t)(cell + gridDim.x) * 2 * P);
                const size_t bytes = 16 * (size_t)P;
                constexpr size_t kChunk = 8192;
                for (size_t off = (size_t)tid * kChunk; off < bytes; off += (size_t)NT * kChunk) {
                    const uint32_t n = (uint32_t)(bytes - off < kChunk ? bytes - off : kChunk);
                    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(nxt + off), "r"(n) : "memory");
                }
            }
        } else {
            if (!rv_valid) rv = prologue_compute(tb, nx, gs.mu, gs.sigma_mol, live ? s.BINC[BC_RM * tb.Np + k] : 0.0, k);
            prologue_store(tb, rv, nvR, nvZ, nvP, has_vphi, has_h, s, k);
            // V_g^2 through shared memory: only the bin-owning warps hold the pre-computed values
            if (tid == 0) { s.CTR[0] = NT / 32; s.RED[95] = rv.Vg2; }
            __syncthreads();
            pc.Vg2 = s.RED[95];
        }
        // state (thread <-> bin): in flight during the build
        double y0 = 0.0, k1 = 0.0;
        if (MODE != MODE_KERNEL && live) {
            y0 = sa.rho[row + k];
            if ((MODE == MODE_STEP || MODE == MODE_STEPK) && sa.have_k1) k1 = sa.k_fsal[row + k];
        }
        if constexpr (MODE != MODE_RATES && MODE != MODE_STEPK)
            build_cell<MODE, SLAB>(tb, s, ks, pc, has_vphi,
                                   MODE == MODE_KERNEL ? sa.out + (size_t)cell * 2 * P : nullptr, lane);
        if (MODE == MODE_KERNEL) fetch(cell + gridDim.x);
        __syncthreads();
        // vertically integrated kernel: every K_ij / sqrt(2 pi (h_i^2 + h_j^2)); p_frag is
        // unchanged, so both planes take the factor.  A separate sweep keeps the pair loops as they are.
        if (MODE != MODE_RATES && MODE != MODE_STEPK && has_h) {
            for (int i = tid >> 5; i < N; i += NT / 32) {
                const double hi2 = s.V5[i];
                const int base = tri(i);
                for (int j = lane; j <= i; j += 32) {
                    const double f = 1.0 / sqrt((2.0 * kPiD) * (hi2 + s.V5[j]));
                    if (MODE == MODE_KERNEL) {
                        double *o = sa.out + (size_t)cell * 2 * P;
                        o[base + j] *= f; o[P + base + j] *= f;
                    } else {
                        const double2 v = ks.ld(base + j);
                        ks.st(base + j, make_double2(v.x * f, v.y * f));
                    }
                }
            }
            __syncthreads();
        }
        if (MODE == MODE_KERNEL) continue;

        if (MODE == MODE_RATES || MODE == MODE_OTF) {
            fetch(cell + gridDim.x);
            const double *kn = (MODE == MODE_RATES && kin_tma && cell + (int)gridDim.x < sa.C)
                                   ? sa.Kin + (size_t)(cell + gridDim.x) * 2 * P : nullptr;
            const double d = eval_rates<NT, SLAB, PLANAR>(tb, s, ks, y0, tid, tbase, false, nx, gs.mu, gs.sigma_mol, rv, kn);
            if (live) sa.out[row + k] = d;
            __syncthreads();
            continue;
        }

        // ---------------- Bogacki-Shampine 3(2), PAPER.md:478 (tableau: Bogacki & Shampine 1989)
        const double h = sa.dt;
        double k2 = 0.0, k3 = 0.0, k4 = 0.0, yn = y0;
#pragma unroll 1
        for (int st = sa.have_k1 ? 1 : 0; st < 4; ++st) {
            double ys = y0;
            if (st == 1) ys = y0 + 0.5 * h * k1;
            if (st == 2) ys = y0 + 0.75 * h * k2;
            if (st == 2) fetch(cell + gridDim.x);
            if (st == 3) {
                yn = y0 + h * ((2.0 / 9.0) * k1 + (1.0 / 3.0) * k2 + (4.0 / 9.0) * k3);
                ys = yn;
            }
            const bool pre = MODE == MODE_STEP && st == 3 && cell + (int)gridDim.x < sa.C;
            const double *kn = (MODE == MODE_STEPK && st == 3 && cell + (int)gridDim.x < sa.C)
                                   ? sa.Kin + (size_t)(cell + gridDim.x) * 2 * P : nullptr;
            const double d = eval_rates<NT, SLAB, PLANAR>(tb, s, ks, ys, tid, tbase, pre, nx, gs.mu,
                                                  gs.sigma_mol, rv, kn);
            if (st == 3) rv_valid = pre;
            if (st == 0) k1 = d;
            if (st == 1) k2 = d;
            if (st == 2) k3 = d;
            if (st == 3) k4 = d;
        }

        // error norm (R10) and write-back
        const double atol = sa.atol_factor * block_sum<NT>(y0, s.RED + 48, tid);
        double emax = 0.0;
        if (live) {
            const double e = h * ((-5.0 / 72.0) * k1 + (1.0 / 12.0) * k2 + (1.0 / 9.0) * k3 - (1.0 / 8.0) * k4);
            const double sc = atol + sa.rtol * fmax(fabs(y0), fabs(yn));
            emax = (e == 0.0) ? 0.0 : fabs(e) / sc;      // R10: a bin with no error estimate (empty cell: 0/0) counts 0
            sa.rho_out[row + k] = yn;
            sa.k_out[row + k] = k4;
        }
        emax = block_nanmax<NT>(emax, s.RED + 64, tid);
        if (tid == 0) sa.err[cell] = emax;
    }
    if (use_tmem) {
        tmem_fence_before();
        __syncthreads();
        if (tid < 32) tmem_dealloc_all(tbase);
    }
}

// ------------------------------------------------------------------------------------------ launch
template <int MODE, bool SLAB, bool VINT>
static cudaError_t launch_vint(const LaunchCfg &lc, const DevTables &tb, const GasArgs &gs,
                               const StepArgs &sa, cudaStream_t st)
{
    constexpr int NT = kThreads;
    auto fn = coag_cells_kernel<NT, MODE, SLAB, VINT>;
    static bool attr_done[64] = {false};    // the attribute is per device (and per instantiation)
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !attr_done[dev]) {
        e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, lc.smem_optin);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) attr_done[dev] = true;
    }
    fn<<<lc.grid, NT, lc.smem_bytes, st>>>(tb, gs, sa);
    return cudaGetLastError();
}

template <int MODE, bool SLAB>
static cudaError_t launch_mode(const LaunchCfg &lc, const DevTables &tb, const GasArgs &gs,
                               const StepArgs &sa, cudaStream_t st)
{
    // the modes that read K from HBM never see a gas state
    if (MODE != MODE_RATES && MODE != MODE_STEPK && gs.hd) return launch_vint<MODE, SLAB, true>(lc, tb, gs, sa, st);
    return launch_vint<MODE, SLAB, false>(lc, tb, gs, sa, st);
}

template <bool SLAB>
static cudaError_t launch_slab(int mode, const LaunchCfg &lc, const DevTables &tb, const GasArgs &gs,
                               const StepArgs &sa, cudaStream_t st)
{
    switch (mode) {
    case MODE_KERNEL: return launch_mode<MODE_KERNEL, SLAB>(lc, tb, gs, sa, st);
    case MODE_RATES: return launch_mode<MODE_RATES, SLAB>(lc, tb, gs, sa, st);
    case MODE_STEPK: return launch_mode<MODE_STEPK, SLAB>(lc, tb, gs, sa, st);
    case MODE_OTF: return launch_mode<MODE_OTF, SLAB>(lc, tb, gs, sa, st);
    default: return launch_mode<MODE_STEP, SLAB>(lc, tb, gs, sa, st);
    }
}

cudaError_t launch_cells(int mode, const LaunchCfg &lc, const DevTables &tb, const GasArgs &gs,
                         const StepArgs &sa, cudaStream_t st)
{
    // SLAB: part of the K store lives in the per-CTA global slab (n_bins too large for shared memory)
    return sa.Psm < tb.P ? launch_slab<true>(mode, lc, tb, gs, sa, st)
                         : launch_slab<false>(mode, lc, tb, gs, sa, st);
}

int cells_occupancy(int smem_bytes, int smem_optin)
{
    auto fn = coag_cells_kernel<kThreads, MODE_STEP, true, false>;
    if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin) != cudaSuccess)
        return 0;
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, fn, kThreads, (size_t)smem_bytes) != cudaSuccess)
        return 0;
    return n;
}

// ------------------------------------------------------------------------------------------ peaks
// FP64 FMA peak: 8 independent chains per thread, no memory traffic.
__global__ void __launch_bounds__(256) dfma_peak_kernel(double *out, int n_iter, double a, double b)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5,
           x6 = x0 + 6, x7 = x0 + 7;
#pragma unroll 1
    for (int it = 0; it < n_iter; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    const double r = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (r == 123.456) out[0] = r;   // never true for the constants used; keeps the chains alive
}

__global__ void __launch_bounds__(256) copy_peak_kernel(const double2 *__restrict__ src,
                                                        double2 *__restrict__ dst, size_t n)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += stride) dst[q] = src[q];
}

// global error norm of a step: max over cells, NaN wins (one block; C doubles are L2-resident)
__global__ void __launch_bounds__(1024) err_max_kernel(const double *__restrict__ err, int n, double *out)
{
    __shared__ double red[64];
    double v = 0.0;
    for (int q = threadIdx.x; q < n; q += 1024) v = nanmax(v, err[q]);
    v = block_nanmax<1024>(v, red, threadIdx.x);   // 32 warps -> 32 slots
    if (threadIdx.x == 0) out[0] = v;
}

// Controller step (R10): E = max_c E_c; accept iff E <= 1; next size h clamp(0.9 E^(-1/3), 0.2, 5)
// (5 for E == 0); the last step is cut to land on t_span and a cut step does not shrink the next size.
__global__ void __launch_bounds__(1024) ctrl_kernel(const double *__restrict__ err, int n, CtrlState *cs,
                                                    double *log)
{
    __shared__ double red[64];
    if (cs->done) return;
    double v = 0.0;
    for (int q = threadIdx.x; q < n; q += 1024) v = nanmax(v, err[q]);
    v = block_nanmax<1024>(v, red, threadIdx.x);
    if (threadIdx.x != 0) return;
    CtrlState c = *cs;
    const double E = v, h = c.h;
    const int slot = c.n_acc + c.n_rej;
    if (!(E == E) || isinf(E)) {
        c.status = 1; c.done = 1;
        *cs = c;
        return;
    }
    double f = 5.0;
    if (E > 0.0) f = 0.9 * pow(E, -1.0 / 3.0);
    f = fmin(5.0, fmax(0.2, f));
    const double sug = h * f;
    if (E <= 1.0) {
        c.cur ^= 1; c.have_k1 = 1;
        c.t = c.cut ? c.t_span : c.t + h;
        c.dt_last = h; c.err_last = E;
        if (log) log[slot] = h;
        c.n_acc++;
        c.dt = c.cut ? fmax(sug, c.dt) : sug;
    } else {
        if (log) log[slot] = -h;
        c.n_rej++;
        c.dt = sug;
    }
    if (c.t >= c.t_span || c.n_acc >= c.max_acc || c.n_acc + c.n_rej >= c.max_steps) c.done = 1;
    const double left = c.t_span - c.t;
    c.cut = c.dt >= left;
    c.h = c.cut ? left : c.dt;
    *cs = c;
}

cudaError_t launch_ctrl(const double *err, int n, CtrlState *cs, double *log, cudaStream_t st)
{
    ctrl_kernel<<<1, 1024, 0, st>>>(err, n, cs, log);
    return cudaGetLastError();
}

cudaError_t launch_err_max(const double *err, int n, double *out, cudaStream_t st)
{
    err_max_kernel<<<1, 1024, 0, st>>>(err, n, out);
    return cudaGetLastError();
}

cudaError_t launch_dfma_peak(int grid, int n_iter, double *out, cudaStream_t st)
{
    dfma_peak_kernel<<<grid, 256, 0, st>>>(out, n_iter, 0.999999, 1e-6);
    return cudaGetLastError();
}

cudaError_t launch_copy_peak(int grid, const void *src, void *dst, size_t n16, cudaStream_t st)
{
    copy_peak_kernel<<<grid, 256, 0, st>>>((const double2 *)src, (double2 *)dst, n16);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------ static scratch
// The per-CTA overflow slab of the K store for callers that may not allocate (cudisc_coag_rates_otf_noalloc):
// a file-scope array, so every GPU that loads the library holds kStaticSlabBytes of it until the process exits.
// In host code `g_static_slab` is only a stand-in for the symbol, not a device address: the address comes from
// cudaGetSymbolAddress, looked up once per device with that device current, and goes to the kernel in
// StepArgs::kslab.  All calls share the array; the kernel writes every slab pair of a cell before it reads it,
// so nothing has to be cleared between calls -- but two launches that overlap on the GPU would race on it.
static __device__ __align__(256) unsigned char g_static_slab[kStaticSlabBytes];

cudaError_t launch_cells_static_slab(int mode, const LaunchCfg &lc, const DevTables &tb, const GasArgs &gs,
                                     const StepArgs &sa_in, cudaStream_t st)
{
    static void *addr[64] = {nullptr};      // per device
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (!addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_slab);
        if (e != cudaSuccess) return e;
        addr[dev] = p;
    }
    StepArgs sa = sa_in;
    sa.kslab = reinterpret_cast<double *>(addr[dev]);
    return launch_cells(mode, lc, tb, gs, sa, st);
}

}  // namespace cudisc
