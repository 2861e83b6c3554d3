// coag_api.cu -- the C ABI of include/cudisc_coag.h: handles, argument checks, table upload,
// launch configuration.  No arithmetic of the method lives here (tables: coag_tables.cpp,
// kernels: coag_kernels.cu / coag_device.cuh).
#include "../../include/cudisc_coag.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "coag_v3.h"
#include "coag_launch.h"
#include "coag_tables.h"

using namespace cudisc;

namespace {

constexpr unsigned kBinsMagic = 0xC0A6B125u;
constexpr unsigned kGridMagic = 0xC0A66D1Du;
constexpr int kMaxBins = 256;
// cudisc_coag_kernel on the stencil kernel's build: what the whole prologue of the next cell costs a bin-owning warp, in
// the units of the build cost model of coag_v3_host.cpp (one row of 32 pairs = 95)
constexpr double kOwnerCostKernelMode = 1300.0;

thread_local char g_err[512] = "";
std::atomic<long long> g_launches{0};

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int cuda_fail(cudaError_t e, const char *what)
{
    return fail(CUDISC_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

}  // namespace

struct cudisc_bins_s {
    unsigned magic;
    HostTables ht;
    cudisc_params p;
    // device copy (lazy)
    bool on_device;
    int device;
    void *dev_blob;
    DevTables dt;
    V3Tables v3;            // stencil cell kernel tables (v3.on == 0: not applicable to this grid)
    V3Tables v3k;           // the same kernel's build alone (cudisc_coag_kernel): run lists with the prologue on the bin owners
};

struct cudisc_grid_s {
    unsigned magic;
    int n_r, n_z, C;
    cudisc_bins bins;
    bool gas_bound;
    cudisc_gas_state gs;
    bool fsal_valid;
    const void *fsal_rho, *fsal_K;   // the state array (and kernel planes, NULL = built on the fly) k_fsal belongs to
    double *k_fsal;     // [C x N]
    double *kslab;      // per-CTA overflow of the K store
    double *stage_rho;  // [C x N] staging of cudisc_coag_step_host (lazy)
    double *stage_err;  // [C]
    cudaStream_t pipe[2];      // internal streams of the sliced end-to-end step
    cudaEvent_t pipe_ev[3];
    double *trial_rho, *trial_k, *trial_err, *d_log;   // cudisc_coag_integrate (lazy, all or nothing)
    CtrlState *d_ctrl, *h_ctrl;                        // controller state: device, pinned host mirror
    int log_cap;
    int num_sms, smem_optin, grid_ctas, Psm, smem_bytes;
    bool fast;          // cudisc_coag_step / rates_otf run on the tensor-memory kernel
    int fast_ctas;
};

namespace {

bool bins_ok(cudisc_bins b) { return b && b->magic == kBinsMagic; }
bool grid_ok(cudisc_grid g) { return g && g->magic == kGridMagic && bins_ok(g->bins); }

int check_params(const cudisc_params &p)
{
    if (!(p.eta < 2.0)) return fail(CUDISC_ERR_INVALID, "eta must be < 2 (got %g)", p.eta);
    if (!(p.chi_im > 0.0)) return fail(CUDISC_ERR_INVALID, "chi_im must be > 0 (got %g)", p.chi_im);
    return CUDISC_OK;
}

int make_bins(const std::vector<double> &m, const std::vector<double> &me, const std::vector<double> &a,
              double rho_m, const cudisc_params &p, cudisc_bins *out)
{
    cudisc_bins b = new (std::nothrow) cudisc_bins_s();
    if (!b) return fail(CUDISC_ERR_INVALID, "out of host memory");
    std::string why = build_tables(m, me, a, rho_m, p.eta, p.chi_im, p.readings, b->ht);
    if (!why.empty()) { delete b; return fail(CUDISC_ERR_INVALID, "%s", why.c_str()); }
    b->magic = kBinsMagic;
    b->p = p;
    b->on_device = false;
    b->device = -1;
    b->dev_blob = nullptr;
    *out = b;
    return CUDISC_OK;
}

// ---- work-item lists and band ELL (host), then one blob upload
struct Blob {
    std::vector<unsigned char> bytes;
    size_t add(const void *src, size_t n)
    {
        size_t off = (bytes.size() + 15) & ~(size_t)15;
        bytes.resize(off + n);
        if (n) memcpy(bytes.data() + off, src, n);
        return off;
    }
    template <class T> size_t add(const std::vector<T> &v) { return add(v.data(), v.size() * sizeof(T)); }
};

// Everything the kernels need besides the K store, built on the host from the grid-only tables:
// work items, packed slot offsets, band ELL / tensor-memory tasks, per-bin constants.  No CUDA calls.
struct Schedule {
    DevTables d;                       // scalars only; pointers are set after the upload
    std::vector<uint32_t> buildItems, evalItems, bidx;
    std::vector<int> sched, cnt;
    std::vector<double> binc, bcoef, dtab, exptab;
    std::vector<int2> bini;
};

void build_schedule(const HostTables &t, Schedule &S)
{
    const int N = t.N;
    DevTables d;
    memset(&d, 0, sizeof(d));
    d.N = N; d.Np = (N + 1) & ~1; d.P = N * (N + 1) / 2;
    d.rho_m = t.rho_m; d.sS = t.sS;

    const int nblk = (N + 31) / 32;

    // ---- build items (all about equal: small items for balance), packed (coag_device.cuh)
    std::vector<uint32_t> buildItems;
    constexpr int kRowsPerItem = 24, kPairsPerItem = 96;
    for (int c = 0; c < nblk; ++c)
        for (int ia = 32 * c + 32; ia < N; ia += kRowsPerItem)
            buildItems.push_back(pack_build(IT_BUILD_ROWS, c, ia, std::min(N, ia + kRowsPerItem)));
    for (int c = 0; c < nblk; ++c) {
        const int rows = std::min(32 * c + 32, N) - 32 * c;          // rows 32 c .. 32 c + rows - 1
        const int last = rows * (rows + 1) / 2;
        for (int a = 0; a < last; a += kPairsPerItem)
            buildItems.push_back(pack_build(IT_BUILD_LIST, c, a, std::min(last, a + kPairsPerItem)));
    }

    // ---- eval items: row / column passes, heaviest first.  Partial sums go to packed slots:
    //      row chunk c holds rows i >= rowFirst[c], column range r holds columns j < R1[r]
    const int nchRow = std::min(4, std::max(1, (N + kRowChunk - 1) / kRowChunk));
    const int nRng = std::min(4, std::max(1, (N + 63) / 64));
    const int rngLen = (N + nRng - 1) / nRng;
    std::vector<int> sched(kSched, 0);
    int rowSlots = 0, colSlots = 0;
    for (int c = 0; c < nchRow; ++c) {
        int first = N;
        for (int i = 0; i < N; ++i)
            if (t.n_bulk[i] > kRowChunk * c) { first = i; break; }
        sched[SC_ROWFIRST + c] = first;
        sched[SC_ROWOFF + c] = rowSlots;
        rowSlots += N - first;
    }
    for (int r = 0; r < nRng; ++r) {
        sched[SC_COLOFF + r] = colSlots;
        colSlots += std::min(N, (r + 1) * rngLen);
    }
    d.partRowSlots = rowSlots; d.partColSlots = colSlots;
    for (int c = 0; c < 4; ++c) {
        d.rowBase[c] = c < nchRow ? sched[SC_ROWOFF + c] - sched[SC_ROWFIRST + c] : 0;
        d.colOff[c] = c < nRng ? sched[SC_COLOFF + c] : 0;
    }
    struct Cost { uint32_t item; long cost; };
    std::vector<Cost> work;
    for (int blk = 0; blk < nblk; ++blk)
        for (int cw = 0; cw < nchRow; ++cw) {
            int jmax = 0;
            for (int i = blk * 32; i < std::min(N, blk * 32 + 32); ++i)
                jmax = std::max(jmax, std::min(kRowChunk * cw + kRowChunk, t.n_bulk[i]));
            // the item must exist (and write zeros) whenever a row of the block owns a slot of chunk cw
            if (std::min(N, blk * 32 + 32) <= sched[SC_ROWFIRST + cw]) continue;
            jmax = std::max(jmax, kRowChunk * cw);
            work.push_back({pack_eval(IT_ROW, blk, cw, 0, jmax), 5L * (jmax - kRowChunk * cw) + 20});
        }
    for (int cb = 0; cb < nblk; ++cb)
        for (int r = 0; r < nRng; ++r) {
            const int i0 = r * rngLen, i1 = std::min(N, (r + 1) * rngLen);
            if (i1 <= 32 * cb) continue;
            work.push_back({pack_eval(IT_COL, cb, r, i0, i1), 5L * (i1 - std::max(i0, 32 * cb)) + 20});
        }
    std::stable_sort(work.begin(), work.end(), [](const Cost &x, const Cost &y) { return x.cost > y.cost; });
    d.nchRow = nchRow; d.nRng = nRng; d.rngLen = rngLen;

    // per-bin constants
    std::vector<double> binc((size_t)kBinC * d.Np, 0.0);
    std::vector<int2> bini(d.Np, make_int2(0, 0));
    for (int k = 0; k < N; ++k) {
        binc[(size_t)BC_M * d.Np + k] = t.m[k];   binc[(size_t)BC_RM * d.Np + k] = t.rm[k];
        binc[(size_t)BC_A1 * d.Np + k] = t.cA1[k]; binc[(size_t)BC_A2 * d.Np + k] = t.cA2[k];
        binc[(size_t)BC_B1 * d.Np + k] = t.cB1[k];
        binc[(size_t)BC_F1 * d.Np + k] = t.cF1[k]; binc[(size_t)BC_F2 * d.Np + k] = t.cF2[k];
        binc[(size_t)BC_G1 * d.Np + k] = t.cG1[k];
        binc[(size_t)BC_FA * d.Np + k] = t.fA[k];  binc[(size_t)BC_FIB * d.Np + k] = t.finvB[k];
        // n_bulk <= 256 and iS <= 256 need 9 bits each; first column range r with R1[r] > k
        bini[k] = make_int2(t.n_bulk[k] | (t.iS[k] << 9) | ((k / rngLen) << 18),
                            t.jS_lo[k] | (t.jS_hi[k] << 16));
    }

    // per-offset tables of a log grid: sigma_ij = a_i^2 pi (1 + q^-d)^2, (St_i - St_j)/(St_i + St_j)
    // = (1 - q^-d)/(1 + q^-d) with q^-d = a_0 / a_d (Epstein Stokes numbers are proportional to a)
    std::vector<double> dtab(2 * (size_t)N, 0.0), exptab(64);
    {
        const double q = std::pow(t.a[N - 1] / t.a[0], 1.0 / (double)(N - 1));
        bool lg = true;
        for (int k = 0; k + 1 < N; ++k)
            if (std::fabs(t.a[k + 1] / t.a[k] - q) > 1e-12 * q) lg = false;
        d.logGrid = lg ? 1 : 0;
        for (int dd = 0; dd < N; ++dd) {
            const double r = t.a[0] / t.a[dd];
            dtab[2 * dd] = 3.14159265358979323846 * (1.0 + r) * (1.0 + r);
            dtab[2 * dd + 1] = (1.0 - r) / (1.0 + r);
        }
        for (int qq = 0; qq < 64; ++qq) exptab[qq] = std::exp2((double)qq / 64.0);
    }

    // band ELL: entries of target t at [e][t], e < band_cnt[t]
    const int W = (2 * N + 31) & ~31;
    std::vector<int> cnt(W, 0);
    for (const BandEntry &be : t.band) cnt[be.target]++;
    int L = 0;
    for (int q = 0; q < W; ++q) L = std::max(L, cnt[q]);
    std::vector<uint32_t> bidx((size_t)L * W, 0u);
    std::vector<double> bcoef((size_t)L * W, 0.0);
    std::vector<int> fill(W, 0);
    for (const BandEntry &be : t.band) {     // t.band is sorted by (target, i, j, plane): fixed order
        const int e2 = fill[be.target]++;
        bidx[(size_t)e2 * W + be.target] = (uint32_t)be.i | ((uint32_t)be.j << 8) | ((uint32_t)be.plane << 16);
        bcoef[(size_t)e2 * W + be.target] = be.coef;
    }
    d.bandW = W; d.bandL = L;
    // band tables in tensor memory when they fit: target group g sits in the tensor-memory lanes of
    // quarter g % 4 (columns 128 (g / 4) ...), readable by warps w with w % 4 == g % 4: its gather
    // is a task of the least loaded warp of that quarter.
    //   bandD > 0 (band pairs within bandD of the diagonal and the stage fits): the products
    //     n_i n_j K of the band pairs are staged once per evaluation (W items) and the indices address
    //     the stage: plane * bandD * Np + (i - j) * Np + i;
    //   bandD == 0: indices address the K store; a long list is cut in two tasks (two BANDV slots).
    const int nGroups = (2 * N + 31) / 32;
    d.bandLp = (L + 7) & ~7;
    d.bandTmem = (d.bandLp <= kBandTmemMax && nGroups <= kThreads / 32) ? 1 : 0;
    int bandD = 0;
    for (const BandEntry &be : t.band) bandD = std::max(bandD, be.i - be.j + 1);
    if (!d.bandTmem || t.band.empty() || (size_t)2 * bandD * d.Np * sizeof(double) > 16384) bandD = 0;
    std::vector<uint32_t> evalItems;
    {
        constexpr int nWarps = kThreads / 32;
        int load[nWarps] = {0}, ntask[nWarps] = {0};
        // the bin-owning warps also compute the next cell's per-bin values during the last evaluation
        for (int w = 0; w < nWarps; ++w) load[w] = (32 * w < N) ? 12 : 0;
        for (int tg = 0; tg < nGroups && d.bandTmem; ++tg) {
            int cmax = 0;
            for (int q = tg * 32; q < std::min(W, tg * 32 + 32); ++q) cmax = std::max(cmax, cnt[q]);
            const int Lg = (cmax + 7) & ~7;        // a group without entries still gets a task: it zeroes BANDV
            const int half = (!bandD && Lg > 16) ? ((Lg / 2 + 7) & ~7) : Lg;
            const int cuts[3] = {0, half, Lg};
            for (int h = 0; h < 2; ++h) {
                if (h == 1 && cuts[1] == cuts[2]) break;
                int best = -1;
                for (int w = tg % 4; w < nWarps; w += 4)
                    if (ntask[w] < 2 && (best < 0 || load[w] < load[best])) best = w;
                if (best < 0) { d.bandTmem = 0; break; }
                sched[SC_BTASK + 2 * best + ntask[best]] =
                    (int)(0x80000000u | ((uint32_t)h << 30) | ((uint32_t)tg << 16) |
                          ((uint32_t)cuts[h] << 8) | (uint32_t)cuts[h + 1]);
                ntask[best]++;
                load[best] += cuts[h + 1] - cuts[h] + 4;
            }
        }
        if (!d.bandTmem) {
            bandD = 0;
            for (int q = 0; q < 2 * nWarps; ++q) sched[SC_BTASK + q] = 0;
            for (int tg = 0; tg < nGroups; ++tg) {
                int cmax = 0;
                for (int q = tg * 32; q < std::min(W, tg * 32 + 32); ++q) cmax = std::max(cmax, cnt[q]);
                evalItems.push_back(pack_eval(IT_BAND, tg, 0, 0, cmax));
            }
        }
    }
    d.bandD = bandD; d.nWItems = 0;
    if (bandD) {
        for (uint32_t &ix : bidx) {                 // padding entries (coef 0) point at stage slot 0
            const int i = ix & 0xff, j = (ix >> 8) & 0xff, plane = (ix >> 16) & 1;
            ix = (uint32_t)(plane * bandD * d.Np + (i - j) * d.Np + i);
        }
        for (int blk = 0; blk < nblk; ++blk) evalItems.push_back(pack_eval(IT_W, blk, 0, 0, 0));
        d.nWItems = nblk;
    }
    for (const Cost &c : work) evalItems.push_back(c.item);
    d.nBuildItems = (int)buildItems.size(); d.nEvalItems = (int)evalItems.size();

    S.d = d;
    S.buildItems = std::move(buildItems); S.evalItems = std::move(evalItems); S.bidx = std::move(bidx);
    S.sched = std::move(sched); S.cnt = std::move(cnt);
    S.binc = std::move(binc); S.bcoef = std::move(bcoef); S.dtab = std::move(dtab); S.exptab = std::move(exptab);
    S.bini = std::move(bini);
}

int upload_tables(cudisc_bins b)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (b->on_device && b->device == dev) return CUDISC_OK;
    if (b->on_device) { cudaFree(b->dev_blob); b->on_device = false; b->dev_blob = nullptr; }

    const HostTables &t = b->ht;
    Schedule S;
    build_schedule(t, S);
    DevTables d = S.d;
    const std::vector<uint32_t> &buildItems = S.buildItems, &evalItems = S.evalItems, &bidx = S.bidx;
    const std::vector<int> &sched = S.sched, &cnt = S.cnt;
    const std::vector<double> &binc = S.binc, &bcoef = S.bcoef, &dtab = S.dtab, &exptab = S.exptab;
    const std::vector<int2> &bini = S.bini;

    int optin = 0;
    e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaDeviceGetAttribute");
    V3Host V;
    v3_build(t, d.logGrid, optin, V);
    Blob bl;
    const size_t o_a = bl.add(t.a), o_binc = bl.add(binc), o_bini = bl.add(bini);
    const size_t o_cnt = bl.add(cnt), o_bidx = bl.add(bidx), o_bcoef = bl.add(bcoef);
    const size_t o_bI = bl.add(buildItems), o_eI = bl.add(evalItems);
    const size_t o_dt = bl.add(dtab), o_ex = bl.add(exptab), o_sc = bl.add(sched);

    void *blob = nullptr;
    e = cudaMalloc(&blob, bl.bytes.size());
    if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc(tables)");
    e = cudaMemcpy(blob, bl.bytes.data(), bl.bytes.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(blob); return cuda_fail(e, "cudaMemcpy(tables)"); }
    const unsigned char *base = (const unsigned char *)blob;
    d.a = (const double *)(base + o_a);
    d.binc = (const double *)(base + o_binc); d.bini = (const int2 *)(base + o_bini);
    d.band_cnt = (const int *)(base + o_cnt);
    d.band_idx = (const uint32_t *)(base + o_bidx); d.band_coef = (const double *)(base + o_bcoef);
    d.buildItems = (const uint32_t *)(base + o_bI); d.evalItems = (const uint32_t *)(base + o_eI);
    d.dtab = (const double2 *)(base + o_dt); d.exptab = (const double *)(base + o_ex);
    d.sched = (const int *)(base + o_sc);
    b->dt = d;
    b->v3 = V.t;
    {
        V3Host Vk;
        v3_build(t, d.logGrid, optin, Vk, kOwnerCostKernelMode, true);
        b->v3k = Vk.t;
        if (!V.t.on) b->v3k.on = 0;
    }
    b->dev_blob = blob;
    b->device = dev;
    b->on_device = true;
    return CUDISC_OK;
}

GasArgs gas_args(const cudisc_gas_state &gs, const cudisc_params &p)
{
    GasArgs g;
    g.T = gs.T; g.rho_g = gs.rho_gas; g.Omega = gs.Omega; g.alpha = gs.alpha;
    g.vR = gs.v_R; g.vZ = gs.v_Z; g.vphi = gs.v_phi; g.hd = gs.h_dust;
    g.alpha_const = p.alpha; g.mu = p.mu; g.v_frag = p.v_frag; g.sigma_mol = p.sigma_mol;
    return g;
}

int check_gas(const cudisc_gas_state *gs)
{
    if (!gs) return fail(CUDISC_ERR_INVALID, "gas_state is NULL");
    if (!gs->T || !gs->rho_gas || !gs->Omega || !gs->v_R || !gs->v_Z)
        return fail(CUDISC_ERR_INVALID, "gas_state: T, rho_gas, Omega, v_R and v_Z must be non-NULL");
    if (gs->v_phi && gs->h_dust)
        return fail(CUDISC_ERR_UNSUPPORTED, "gas_state: v_phi and h_dust cannot both be given");
    return CUDISC_OK;
}

int check_pair(cudisc_grid g, cudisc_bins b)
{
    if (!grid_ok(g)) return fail(CUDISC_ERR_HANDLE, "bad grid handle");
    if (!bins_ok(b)) return fail(CUDISC_ERR_HANDLE, "bad bins handle");
    if (g->bins != b) return fail(CUDISC_ERR_HANDLE, "grid was created for a different bins handle");
    return CUDISC_OK;
}

// Launch over the cells [c0, c1) of the grid (default: all): cells are independent, so a range is the same
// launch with every per-cell pointer advanced by c0.
int run(cudisc_grid g, int mode, GasArgs ga, StepArgs sa, cudisc_stream stream, int c0 = 0, int c1 = -1)
{
    int rc = upload_tables(g->bins);
    if (rc) return rc;
    if (c1 < 0) c1 = g->C;
    sa.C = c1 - c0;
    if (c0 > 0) {
        const size_t N = (size_t)g->bins->ht.N, P2 = 2 * (size_t)g->bins->dt.P;
        auto adv = [&](const double *&p, size_t stride) { if (p) p += (size_t)c0 * stride; };
        auto advw = [&](double *&p, size_t stride) { if (p) p += (size_t)c0 * stride; };
        adv(ga.T, 1); adv(ga.rho_g, 1); adv(ga.Omega, 1); adv(ga.alpha, 1);
        adv(ga.vR, N); adv(ga.vZ, N); adv(ga.vphi, N); adv(ga.hd, N);
        adv(sa.rho, N); adv(sa.k_fsal, N); advw(sa.rho_out, N); advw(sa.k_out, N); advw(sa.err, 1);
        adv(sa.Kin, P2);
        if (sa.out) sa.out += (size_t)c0 * (mode == MODE_KERNEL ? P2 : N);
    }
    sa.Psm = g->Psm;
    sa.kslab = g->kslab;
    LaunchCfg lc{std::min(g->grid_ctas, std::max(1, sa.C)), g->smem_bytes, g->smem_optin};
    cudaError_t e;
    if (g->fast && mode == MODE_KERNEL && g->bins->v3k.on && !ga.hd && !ga.vphi) {
        LaunchCfg lf{std::min(g->fast_ctas, std::max(1, sa.C)), g->bins->v3k.smemBytes, g->smem_optin};
        e = launch_v3(mode, lf, g->bins->dt, g->bins->v3k, ga, sa, (cudaStream_t)stream);
    } else if (g->fast && (mode == MODE_OTF || mode == MODE_STEP || mode == MODE_RATES || mode == MODE_STEPK) && !ga.hd &&
               !ga.vphi) {
        LaunchCfg lf{std::min(g->fast_ctas, std::max(1, sa.C)), g->bins->v3.smemBytes, g->smem_optin};
        e = launch_v3(mode, lf, g->bins->dt, g->bins->v3, ga, sa, (cudaStream_t)stream);
    } else {
        e = launch_cells(mode, lc, g->bins->dt, ga, sa, (cudaStream_t)stream);
    }
    if (e != cudaSuccess) return cuda_fail(e, "kernel launch");
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return CUDISC_OK;
}

}  // namespace

// =============================================================================================
extern "C" {

int cudisc_bins_create(int n_bins, double a_min, double a_max, double rho_m, cudisc_params p,
                       cudisc_bins *out)
{
    if (!out) return fail(CUDISC_ERR_INVALID, "out is NULL");
    *out = nullptr;
    if (n_bins > kMaxBins) return fail(CUDISC_ERR_UNSUPPORTED, "n_bins %d > %d", n_bins, kMaxBins);
    int rc = check_params(p);
    if (rc) return rc;
    std::vector<double> m, me, a;
    std::string why = build_log_grid(n_bins, a_min, a_max, rho_m, m, me, a);
    if (!why.empty()) return fail(CUDISC_ERR_INVALID, "%s", why.c_str());
    return make_bins(m, me, a, rho_m, p, out);
}

int cudisc_bins_create_general(int n_bins, const double *m_centres, const double *m_edges,
                               double rho_m, cudisc_params p, cudisc_bins *out)
{
    if (!out) return fail(CUDISC_ERR_INVALID, "out is NULL");
    *out = nullptr;
    if (!m_centres || !m_edges) return fail(CUDISC_ERR_INVALID, "mass arrays are NULL");
    if (n_bins < 2) return fail(CUDISC_ERR_INVALID, "n_bins < 2");
    if (n_bins > kMaxBins) return fail(CUDISC_ERR_UNSUPPORTED, "n_bins %d > %d", n_bins, kMaxBins);
    if (!(rho_m > 0.0)) return fail(CUDISC_ERR_INVALID, "rho_m <= 0");
    int rc = check_params(p);
    if (rc) return rc;
    std::vector<double> m(m_centres, m_centres + n_bins), me(m_edges, m_edges + n_bins + 1), a(n_bins);
    const double pi = 3.14159265358979323846;
    for (int k = 0; k < n_bins; ++k) a[k] = std::cbrt(3.0 * m[k] / (4.0 * pi * rho_m));
    return make_bins(m, me, a, rho_m, p, out);
}

int cudisc_bins_destroy(cudisc_bins b)
{
    if (!bins_ok(b)) return fail(CUDISC_ERR_HANDLE, "bad bins handle");
    if (b->on_device) cudaFree(b->dev_blob);
    b->magic = 0;
    delete b;
    return CUDISC_OK;
}

int cudisc_bins_query(cudisc_bins b, int *n_bins, double *m_centres, double *m_edges,
                      double *a_centres, int *n_bulk, int *n_band)
{
    if (!bins_ok(b)) return fail(CUDISC_ERR_HANDLE, "bad bins handle");
    const HostTables &t = b->ht;
    if (n_bins) *n_bins = t.N;
    if (m_centres) memcpy(m_centres, t.m.data(), sizeof(double) * t.N);
    if (m_edges) memcpy(m_edges, t.me.data(), sizeof(double) * (t.N + 1));
    if (a_centres) memcpy(a_centres, t.a.data(), sizeof(double) * t.N);
    if (n_bulk) memcpy(n_bulk, t.n_bulk.data(), sizeof(int) * t.N);
    if (n_band) *n_band = (int)t.band.size();
    return CUDISC_OK;
}

int cudisc_bins_expand_outcomes(cudisc_bins b, long long *n_entries, int *target, int *i, int *j,
                                int *plane, double *coef, double *frag_A, double *frag_invB)
{
    if (!bins_ok(b)) return fail(CUDISC_ERR_HANDLE, "bad bins handle");
    std::vector<BandEntry> ex;
    expand_outcomes(b->ht, ex);
    if (n_entries) *n_entries = (long long)ex.size();
    for (size_t e = 0; e < ex.size(); ++e) {
        if (target) target[e] = ex[e].target;
        if (i) i[e] = ex[e].i;
        if (j) j[e] = ex[e].j;
        if (plane) plane[e] = ex[e].plane;
        if (coef) coef[e] = ex[e].coef;
    }
    if (frag_A) memcpy(frag_A, b->ht.fA.data(), sizeof(double) * b->ht.N);
    if (frag_invB) memcpy(frag_invB, b->ht.finvB.data(), sizeof(double) * b->ht.N);
    return CUDISC_OK;
}

int cudisc_bins_schedule_check(cudisc_bins b, long long *out)
{
    if (!bins_ok(b)) return fail(CUDISC_ERR_HANDLE, "bad bins handle");
    if (!out) return fail(CUDISC_ERR_INVALID, "out is NULL");
    const HostTables &t = b->ht;
    Schedule S;
    build_schedule(t, S);
    const DevTables &d = S.d;
    const int N = d.N, Np = d.Np;
    long long bad[6] = {0, 0, 0, 0, 0, 0};
    auto tri_h = [](int i) { return i * (i + 1) / 2; };
    // ---- build items
    std::vector<int> built((size_t)N * N, 0);
    for (uint32_t item : S.buildItems) {
        const int c = (item >> 28) & 7, ia = (item >> 14) & 0x3fff, ib = item & 0x3fff;
        if ((item >> 31) == IT_BUILD_ROWS) {
            for (int i = ia; i < ib; ++i)
                for (int lane = 0; lane < 32; ++lane) {
                    const int j = 32 * c + lane;
                    if (j >= N) continue;
                    if (i >= N || j >= i) { ++bad[0]; continue; }      // rows items never hold the diagonal
                    built[(size_t)i * N + j]++;
                }
        } else {
            for (int tt = ia; tt < ib; ++tt) {
                int r = (int)((std::sqrt(8.0 * tt + 1.0) - 1.0) * 0.5);
                while (tri_h(r + 1) <= tt) ++r;
                while (tri_h(r) > tt) --r;
                const int i = 32 * c + r, j = 32 * c + (tt - tri_h(r));
                if (i >= N || j > i) { ++bad[0]; continue; }
                built[(size_t)i * N + j]++;
            }
        }
    }
    for (int i = 0; i < N; ++i)
        for (int j = 0; j <= i; ++j) bad[0] += built[(size_t)i * N + j] != 1;
    // ---- eval items
    std::vector<int> rowcov((size_t)N * N, 0), colcov((size_t)N * N, 0);
    std::vector<int> rowslot(std::max(1, d.partRowSlots), 0), colslot(std::max(1, d.partColSlots), 0);
    int nW = 0;
    for (uint32_t item : S.evalItems) {
        const int kind = item >> 30, ix = (item >> 26) & 15, iy = (item >> 23) & 7;
        const int iz = (item >> 9) & 0x1ff, iw = item & 0x1ff;
        if (kind == IT_ROW) {
            const int first = S.sched[SC_ROWFIRST + iy];
            for (int lane = 0; lane < 32; ++lane) {
                const int i = 32 * ix + lane;
                if (i >= N) continue;
                const int jb = kRowChunk * iy, je = std::min(jb + kRowChunk, t.n_bulk[i]);
                for (int j = jb; j < iw; ++j)
                    if (j < je) rowcov[(size_t)i * N + j]++;
                if (je > iw) ++bad[1];                                 // host bound too small
                if (i >= first) {
                    const int slot = S.sched[SC_ROWOFF + iy] + i - first;
                    if (slot < 0 || slot >= d.partRowSlots || slot != d.rowBase[iy] + i) ++bad[3];
                    else if (rowslot[slot]++) ++bad[3];
                }
            }
        } else if (kind == IT_COL) {
            for (int lane = 0; lane < 32; ++lane) {
                const int j = 32 * ix + lane;
                if (j >= std::min(N, iw)) continue;
                for (int i = std::max(iz, j); i < iw; ++i) colcov[(size_t)i * N + j]++;
                const int slot = S.sched[SC_COLOFF + iy] + j;
                if (slot < 0 || slot >= d.partColSlots || slot != d.colOff[iy] + j) ++bad[3];
                else if (colslot[slot]++) ++bad[3];
            }
        } else if (kind == IT_W) {
            ++nW;
        }
    }
    for (int i = 0; i < N; ++i)
        for (int j = 0; j <= i; ++j) {
            bad[1] += rowcov[(size_t)i * N + j] != (j < t.n_bulk[i] ? 1 : 0);
            bad[2] += colcov[(size_t)i * N + j] != 1;
        }
    // slots the combine step (phase B) reads must have been written
    for (int k = 0; k < N; ++k) {
        for (int c = 0; c < 4; ++c)
            if (t.n_bulk[k] > kRowChunk * c && !(c < d.nchRow && rowslot[d.rowBase[c] + k] == 1)) ++bad[3];
        for (int r = k / d.rngLen; r < d.nRng; ++r)
            if (colslot[d.colOff[r] + k] != 1) ++bad[3];
    }
    // ---- band
    long long entries = 0;
    for (int q = 0; q < d.bandW; ++q) entries += S.cnt[q];
    if (entries != (long long)t.band.size()) ++bad[4];
    if (d.bandD) {
        if (nW != d.nWItems || nW != (N + 31) / 32) ++bad[4];
        for (uint32_t ix : S.bidx)
            if (ix >= (uint32_t)(2 * d.bandD * Np)) ++bad[4];
    } else {
        for (uint32_t ix : S.bidx) {
            const int i = ix & 0xff, j = (ix >> 8) & 0xff;
            if (i >= N || j > i) ++bad[4];
        }
    }
    if (d.bandTmem) {
        const int nGroups = (2 * N + 31) / 32;
        std::vector<int> covered(nGroups, 0);
        for (int w = 0; w < kThreads / 32; ++w)
            for (int q = 0; q < 2; ++q) {
                const int task = S.sched[SC_BTASK + 2 * w + q];
                if (task >= 0) continue;
                const int g = (task >> 16) & 0xff, e0 = (task >> 8) & 0xff, e1 = task & 0xff;
                if (g >= nGroups || (g & 3) != (w & 3) || e0 > e1 || e1 > d.bandLp || (e0 & 7) || (e1 & 7)) { ++bad[5]; continue; }
                covered[g] += (e1 - e0) + 1000;                        // entries + one per task
            }
        for (int g = 0; g < nGroups; ++g) {
            int cmax = 0;
            for (int q = 32 * g; q < std::min(d.bandW, 32 * g + 32); ++q) cmax = std::max(cmax, S.cnt[q]);
            const int Lg = (cmax + 7) & ~7, ntask = covered[g] / 1000, ent = covered[g] % 1000;
            if (ntask < 1 || ntask > 2 || ent != Lg) ++bad[5];
        }
    }
    // ---- the static run lists of the stencil cell kernel, when this grid takes it (coag_v3.h): same counters
    V3Host V;
    v3_build(t, d.logGrid, 232448, V);
    if (V.t.on) v3_check(t, V, bad);
    if (V.t.on) {       // the build-only run lists of cudisc_coag_kernel: every pair built exactly once
        V3Host Vk;
        v3_build(t, d.logGrid, 232448, Vk, kOwnerCostKernelMode, true);
        if (Vk.t.on) {
            long long bk[6] = {0, 0, 0, 0, 0, 0};
            v3_check(t, Vk, bk);
            bad[0] += bk[0];
        }
    }
    for (int q = 0; q < 6; ++q) out[q] = bad[q];
    out[6] = (long long)S.buildItems.size() + (long long)S.evalItems.size();
    out[7] = (long long)(smem_vec_doubles(Np, d.partRowSlots, d.partColSlots, d.nBuildItems + d.nEvalItems, d.bandD)
                         * sizeof(double));
    return CUDISC_OK;
}

int cudisc_bins_fast_path(cudisc_bins b, int *on, long long *smem_bytes, int *tmem_cols_used)
{
    if (!bins_ok(b)) return fail(CUDISC_ERR_HANDLE, "bad bins handle");
    Schedule S;
    build_schedule(b->ht, S);
    V3Host V;
    v3_build(b->ht, S.d.logGrid, 232448, V);
    if (on) *on = V.t.on;
    if (smem_bytes) *smem_bytes = V.t.on ? (long long)V.t.smemBytes : 0;
    if (tmem_cols_used) {
        int used = 0;
        if (V.t.on) {
            for (int w = 0; w < kV3Warps; ++w)
                for (int r = 0; r < kV3ColRuns; ++r)
                    if (V.t.col[w][r]) used += 32 * v3_unpack_col(V.t.col[w][r]).n;
        }
        *tmem_cols_used = used;
    }
    return CUDISC_OK;
}

int cudisc_grid_create(int n_r, int n_z, cudisc_bins b, cudisc_grid *out)
{
    if (!out) return fail(CUDISC_ERR_INVALID, "out is NULL");
    *out = nullptr;
    if (!bins_ok(b)) return fail(CUDISC_ERR_HANDLE, "bad bins handle");
    if (n_r < 1 || n_z < 1) return fail(CUDISC_ERR_INVALID, "n_r and n_z must be >= 1");
    if ((long long)n_r * n_z > (1ll << 30)) return fail(CUDISC_ERR_UNSUPPORTED, "too many cells");
    int rc = upload_tables(b);
    if (rc) return rc;
    int dev = 0, sms = 0, optin = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return cuda_fail(e, "device query");

    cudisc_grid g = new (std::nothrow) cudisc_grid_s();
    if (!g) return fail(CUDISC_ERR_INVALID, "out of host memory");
    g->magic = kGridMagic;
    g->n_r = n_r; g->n_z = n_z; g->C = n_r * n_z;
    g->bins = b;
    g->gas_bound = false; g->fsal_valid = false;
    g->fsal_rho = g->fsal_K = nullptr;
    g->k_fsal = nullptr; g->kslab = nullptr;
    g->stage_rho = nullptr; g->stage_err = nullptr;
    g->pipe[0] = g->pipe[1] = nullptr;
    g->pipe_ev[0] = g->pipe_ev[1] = g->pipe_ev[2] = nullptr;
    g->trial_rho = g->trial_k = g->trial_err = g->d_log = nullptr;
    g->d_ctrl = nullptr; g->h_ctrl = nullptr; g->log_cap = 0;
    g->num_sms = sms; g->smem_optin = optin;

    const DevTables &d = b->dt;
    const size_t vec_bytes = smem_vec_doubles(d.Np, d.partRowSlots, d.partColSlots, d.nBuildItems + d.nEvalItems, d.bandD) * sizeof(double);
    if (vec_bytes + 16 * 64 > (size_t)optin) {
        delete g;
        return fail(CUDISC_ERR_UNSUPPORTED, "n_bins %d needs %zu B of shared memory", d.N, vec_bytes);
    }
    const int fit = (int)(((size_t)optin - vec_bytes) / 16);
    g->Psm = std::min(d.P, fit);
    g->smem_bytes = (int)(vec_bytes + (size_t)g->Psm * 16);
    int per_sm = cells_occupancy(g->smem_bytes, optin);
    if (per_sm < 1) { delete g; return fail(CUDISC_ERR_CUDA, "kernel does not fit on an SM"); }
    g->grid_ctas = std::max(1, std::min(g->C, sms * per_sm));
    g->fast = b->v3.on && b->v3.smemBytes <= optin && !getenv("CUDISC_NO_FAST");
    g->fast_ctas = std::max(1, std::min(g->C, sms));

    const size_t row_bytes = (size_t)g->C * d.N * sizeof(double);
    e = cudaMalloc((void **)&g->k_fsal, row_bytes);
    if (e == cudaSuccess && d.P > g->Psm)
        e = cudaMalloc((void **)&g->kslab, (size_t)g->grid_ctas * (size_t)(d.P - g->Psm) * 16);
    if (e != cudaSuccess) {
        if (g->k_fsal) cudaFree(g->k_fsal);
        delete g;
        return cuda_fail(e, "cudaMalloc(grid)");
    }
    *out = g;
    return CUDISC_OK;
}


int cudisc_grid_bind_gas(cudisc_grid g, const cudisc_gas_state *gs)
{
    if (!grid_ok(g)) return fail(CUDISC_ERR_HANDLE, "bad grid handle");
    int rc = check_gas(gs);
    if (rc) return rc;
    g->gs = *gs;
    g->gas_bound = true;
    g->fsal_valid = false;
    return CUDISC_OK;
}

int cudisc_grid_reset_fsal(cudisc_grid g)
{
    if (!grid_ok(g)) return fail(CUDISC_ERR_HANDLE, "bad grid handle");
    g->fsal_valid = false;
    return CUDISC_OK;
}

int cudisc_grid_destroy(cudisc_grid g)
{
    if (!g || g->magic != kGridMagic) return fail(CUDISC_ERR_HANDLE, "bad grid handle");
    if (g->k_fsal) cudaFree(g->k_fsal);
    if (g->kslab) cudaFree(g->kslab);
    if (g->stage_rho) cudaFree(g->stage_rho);
    if (g->stage_err) cudaFree(g->stage_err);
    for (int q = 0; q < 2; ++q) if (g->pipe[q]) cudaStreamDestroy(g->pipe[q]);
    for (int q = 0; q < 3; ++q) if (g->pipe_ev[q]) cudaEventDestroy(g->pipe_ev[q]);
    if (g->trial_rho) cudaFree(g->trial_rho);
    if (g->trial_k) cudaFree(g->trial_k);
    if (g->trial_err) cudaFree(g->trial_err);
    if (g->d_ctrl) cudaFree(g->d_ctrl);
    if (g->d_log) cudaFree(g->d_log);
    if (g->h_ctrl) cudaFreeHost(g->h_ctrl);
    g->magic = 0;
    delete g;
    return CUDISC_OK;
}

int cudisc_coag_kernel(cudisc_grid g, cudisc_bins b, const cudisc_gas_state *gs, cudisc_params p,
                       double *K_out, cudisc_stream stream)
{
    int rc = check_pair(g, b);
    if (rc) return rc;
    rc = check_gas(gs);
    if (rc) return rc;
    if (!K_out) return fail(CUDISC_ERR_INVALID, "K_out is NULL");
    StepArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.out = K_out;
    return run(g, 0, gas_args(*gs, p), sa, stream);
}

int cudisc_coag_rates(cudisc_grid g, cudisc_bins b, const double *K, const double *rho_dust,
                      double *drho_dt, cudisc_stream stream)
{
    int rc = check_pair(g, b);
    if (rc) return rc;
    if (!K || !rho_dust || !drho_dt) return fail(CUDISC_ERR_INVALID, "NULL array argument");
    if (rho_dust == drho_dt) return fail(CUDISC_ERR_INVALID, "rho_dust and drho_dt may not alias");
    StepArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.Kin = K; sa.rho = rho_dust; sa.out = drho_dt;
    GasArgs ga;
    memset(&ga, 0, sizeof(ga));
    return run(g, 1, ga, sa, stream);
}

int cudisc_coag_rates_otf(cudisc_grid g, cudisc_bins b, const double *rho_dust, double *drho_dt,
                          cudisc_stream stream)
{
    int rc = check_pair(g, b);
    if (rc) return rc;
    if (!g->gas_bound) return fail(CUDISC_ERR_INVALID, "no gas state bound (cudisc_grid_bind_gas)");
    if (!rho_dust || !drho_dt) return fail(CUDISC_ERR_INVALID, "NULL array argument");
    if (rho_dust == drho_dt) return fail(CUDISC_ERR_INVALID, "rho_dust and drho_dt may not alias");
    StepArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.rho = rho_dust; sa.out = drho_dt;
    return run(g, 2, gas_args(g->gs, b->p), sa, stream);
}

int cudisc_coag_rates_otf_noalloc(cudisc_grid g, cudisc_bins b, const double *rho_dust, double *drho_dt,
                                  cudisc_stream stream)
{
    static_assert(kStaticSlabBytes == CUDISC_STATIC_SCRATCH_BYTES, "header and kernel file disagree on the scratch size");
    int rc = check_pair(g, b);
    if (rc) return rc;
    if (!g->gas_bound) return fail(CUDISC_ERR_INVALID, "no gas state bound (cudisc_grid_bind_gas)");
    if (!rho_dust || !drho_dt) return fail(CUDISC_ERR_INVALID, "NULL array argument");
    if (rho_dust == drho_dt) return fail(CUDISC_ERR_INVALID, "rho_dust and drho_dt may not alias");
    // nothing on this path may allocate: the tables must be on the current device already
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (!b->on_device || b->device != dev)
        return fail(CUDISC_ERR_INVALID, "tables of this mass grid are not on the current device (create the grid there first)");
    const DevTables &d = b->dt;
    const int ctas = std::min(g->grid_ctas, std::max(1, g->C));
    const size_t need = d.P > g->Psm ? (size_t)ctas * (size_t)(d.P - g->Psm) * 16 : 0;
    if (need > kStaticSlabBytes)
        return fail(CUDISC_ERR_UNSUPPORTED,
                    "n_bins %d on %d CTAs needs %zu B of scratch, the static array holds %zu B: use cudisc_coag_rates_otf",
                    d.N, ctas, need, (size_t)kStaticSlabBytes);
    StepArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.rho = rho_dust; sa.out = drho_dt;
    sa.C = g->C;
    sa.Psm = g->Psm;
    LaunchCfg lc{ctas, g->smem_bytes, g->smem_optin};
    e = launch_cells_static_slab(MODE_OTF, lc, d, gas_args(g->gs, b->p), sa, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "kernel launch (static scratch)");
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return CUDISC_OK;
}

int cudisc_coag_step(cudisc_grid g, cudisc_bins b, double *rho_dust, double dt, double *err_out,
                     cudisc_stream stream)
{
    int rc = check_pair(g, b);
    if (rc) return rc;
    if (!g->gas_bound) return fail(CUDISC_ERR_INVALID, "no gas state bound (cudisc_grid_bind_gas)");
    if (!rho_dust || !err_out) return fail(CUDISC_ERR_INVALID, "NULL array argument");
    StepArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.rho = rho_dust; sa.rho_out = rho_dust;
    sa.k_fsal = g->k_fsal; sa.k_out = g->k_fsal;
    sa.err = err_out;
    sa.dt = dt; sa.rtol = b->p.rtol; sa.atol_factor = b->p.atol_factor;
    // the saved derivative belongs to one state array and one kernel source: anything else recomputes k1
    if (g->fsal_rho != rho_dust || g->fsal_K != nullptr) g->fsal_valid = false;
    sa.have_k1 = g->fsal_valid ? 1 : 0;
    rc = run(g, 3, gas_args(g->gs, b->p), sa, stream);
    if (rc == CUDISC_OK) { g->fsal_valid = true; g->fsal_rho = rho_dust; g->fsal_K = nullptr; }
    return rc;
}

int cudisc_coag_step_cached(cudisc_grid g, cudisc_bins b, const double *K, double *rho_dust, double dt,
                            double *err_out, cudisc_stream stream)
{
    int rc = check_pair(g, b);
    if (rc) return rc;
    if (!K || !rho_dust || !err_out) return fail(CUDISC_ERR_INVALID, "NULL array argument");
    StepArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.Kin = K;
    sa.rho = rho_dust; sa.rho_out = rho_dust;
    sa.k_fsal = g->k_fsal; sa.k_out = g->k_fsal;
    sa.err = err_out;
    sa.dt = dt; sa.rtol = b->p.rtol; sa.atol_factor = b->p.atol_factor;
    if (g->fsal_rho != rho_dust || g->fsal_K != K) g->fsal_valid = false;
    sa.have_k1 = g->fsal_valid ? 1 : 0;
    GasArgs ga;
    memset(&ga, 0, sizeof(ga));
    rc = run(g, 4, ga, sa, stream);
    if (rc == CUDISC_OK) { g->fsal_valid = true; g->fsal_rho = rho_dust; g->fsal_K = K; }
    return rc;
}

int cudisc_coag_step_host(cudisc_grid g, cudisc_bins b, double *rho_host, double dt,
                          double *err_host, cudisc_stream stream)
{
    int rc = check_pair(g, b);
    if (rc) return rc;
    if (!g->gas_bound) return fail(CUDISC_ERR_INVALID, "no gas state bound (cudisc_grid_bind_gas)");
    if (!rho_host || !err_host) return fail(CUDISC_ERR_INVALID, "NULL array argument");
    const size_t N = (size_t)b->ht.N;
    const size_t row_bytes = (size_t)g->C * N * sizeof(double);
    const size_t err_bytes = (size_t)g->C * sizeof(double);
    cudaError_t e = cudaSuccess;
    if (!g->stage_rho) {                           // all or nothing
        e = cudaMalloc((void **)&g->stage_rho, row_bytes);
        if (e == cudaSuccess) e = cudaMalloc((void **)&g->stage_err, err_bytes);
        for (int q = 0; q < 2 && e == cudaSuccess; ++q) e = cudaStreamCreateWithFlags(&g->pipe[q], cudaStreamNonBlocking);
        for (int q = 0; q < 3 && e == cudaSuccess; ++q) e = cudaEventCreateWithFlags(&g->pipe_ev[q], cudaEventDisableTiming);
        if (e != cudaSuccess) {
            if (g->stage_rho) cudaFree(g->stage_rho);
            if (g->stage_err) cudaFree(g->stage_err);
            for (int q = 0; q < 2; ++q) if (g->pipe[q]) { cudaStreamDestroy(g->pipe[q]); g->pipe[q] = nullptr; }
            for (int q = 0; q < 3; ++q) if (g->pipe_ev[q]) { cudaEventDestroy(g->pipe_ev[q]); g->pipe_ev[q] = nullptr; }
            g->stage_rho = g->stage_err = nullptr;
            return cuda_fail(e, "staging buffers / streams");
        }
    }
    // Cells are independent: the grid is cut in slices that alternate between two internal streams, so the
    // host->device copy of slice s + 1 and the device->host copy of slice s - 1 run under the kernel of
    // slice s (copy engines and SMs in parallel).  Both streams start after `stream` and `stream` waits
    // for both.
    cudaStream_t st = (cudaStream_t)stream;
    if (g->fsal_rho != g->stage_rho || g->fsal_K != nullptr) g->fsal_valid = false;
    StepArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.rho = g->stage_rho; sa.rho_out = g->stage_rho;
    sa.k_fsal = g->k_fsal; sa.k_out = g->k_fsal;
    sa.err = g->stage_err;
    sa.dt = dt; sa.rtol = b->p.rtol; sa.atol_factor = b->p.atol_factor;
    sa.have_k1 = g->fsal_valid ? 1 : 0;
    const GasArgs ga = gas_args(g->gs, b->p);
    const int min_cells = 8 * g->num_sms;                        // keep every SM busy within a slice
    // (the per-CTA overflow slab of the general kernel is indexed by CTA: no two launches in flight then)
    const int n_slices = g->kslab ? 1 : std::max(1, std::min(4, g->C / std::max(1, min_cells)));
    e = cudaEventRecord(g->pipe_ev[0], st);
    for (int q = 0; q < 2 && e == cudaSuccess; ++q) e = cudaStreamWaitEvent(g->pipe[q], g->pipe_ev[0], 0);
    if (e != cudaSuccess) return cuda_fail(e, "step_host fork");
    for (int sl = 0; sl < n_slices; ++sl) {
        const int c0 = (int)((long long)g->C * sl / n_slices), c1 = (int)((long long)g->C * (sl + 1) / n_slices);
        cudaStream_t ps = g->pipe[sl & 1];
        e = cudaMemcpyAsync(g->stage_rho + (size_t)c0 * N, rho_host + (size_t)c0 * N,
                            (size_t)(c1 - c0) * N * sizeof(double), cudaMemcpyHostToDevice, ps);
        if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync(H2D)");
        rc = run(g, MODE_STEP, ga, sa, (cudisc_stream)ps, c0, c1);
        if (rc) return rc;
        e = cudaMemcpyAsync(rho_host + (size_t)c0 * N, g->stage_rho + (size_t)c0 * N,
                            (size_t)(c1 - c0) * N * sizeof(double), cudaMemcpyDeviceToHost, ps);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(err_host + c0, g->stage_err + c0, (size_t)(c1 - c0) * sizeof(double),
                                cudaMemcpyDeviceToHost, ps);
        if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync(D2H)");
    }
    for (int q = 0; q < 2 && e == cudaSuccess; ++q) {
        e = cudaEventRecord(g->pipe_ev[1 + q], g->pipe[q]);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(st, g->pipe_ev[1 + q], 0);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(e, "step_host join");
    g->fsal_valid = true; g->fsal_rho = g->stage_rho; g->fsal_K = nullptr;
    return CUDISC_OK;
}

double cudisc_controller_next_dt(double E, double h)
{
    double f = 5.0;
    if (E > 0.0) f = 0.9 * std::pow(E, -1.0 / 3.0);
    f = std::min(5.0, std::max(0.2, f));
    return h * f;
}

}  // extern "C"

namespace {

void free_integrate(cudisc_grid g)
{
    if (g->trial_rho) cudaFree(g->trial_rho);
    if (g->trial_k) cudaFree(g->trial_k);
    if (g->trial_err) cudaFree(g->trial_err);
    if (g->d_ctrl) cudaFree(g->d_ctrl);
    if (g->d_log) cudaFree(g->d_log);
    if (g->h_ctrl) cudaFreeHost(g->h_ctrl);
    g->trial_rho = g->trial_k = g->trial_err = g->d_log = nullptr;
    g->d_ctrl = nullptr; g->h_ctrl = nullptr;
    g->log_cap = 0;
}

// Adaptive sub-cycling driven from the device: every trial is one step launch that reads its
// size and buffer roles from the controller state, plus one controller launch; trials are enqueued in
// batches of kBatch without a host round trip (launches after the end are no-ops) and the host reads the
// 96-byte state once per batch.
int integrate_impl(cudisc_grid g, cudisc_bins b, double *rho_dust, double t_span, int max_accepted,
                   double dt_try, int max_steps, double *dt_log, cudisc_integrate_info *info,
                   cudisc_stream stream)
{
    constexpr int kBatch = 32;
    const size_t row_bytes = (size_t)g->C * b->ht.N * sizeof(double);
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaSuccess;
    if (!g->trial_rho || g->log_cap < max_steps) {
        free_integrate(g);                  // all or nothing: a partial failure leaves no dangling pointer
        e = cudaMalloc((void **)&g->trial_rho, row_bytes);
        if (e == cudaSuccess) e = cudaMalloc((void **)&g->trial_k, row_bytes);
        if (e == cudaSuccess) e = cudaMalloc((void **)&g->trial_err, (size_t)g->C * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void **)&g->d_ctrl, sizeof(CtrlState));
        if (e == cudaSuccess) e = cudaMalloc((void **)&g->d_log, (size_t)max_steps * sizeof(double));
        if (e == cudaSuccess) e = cudaMallocHost((void **)&g->h_ctrl, sizeof(CtrlState));
        if (e != cudaSuccess) { free_integrate(g); return cuda_fail(e, "cudaMalloc(integrate)"); }
        g->log_cap = max_steps;
    }
    CtrlState c;
    memset(&c, 0, sizeof(c));
    c.t = 0.0; c.t_span = t_span; c.dt = dt_try;
    c.cut = dt_try >= t_span; c.h = c.cut ? t_span : dt_try;
    if (g->fsal_rho != rho_dust || g->fsal_K != nullptr) g->fsal_valid = false;
    c.cur = 0; c.have_k1 = g->fsal_valid ? 1 : 0;
    c.max_acc = max_accepted; c.max_steps = max_steps;
    *g->h_ctrl = c;
    e = cudaMemcpyAsync(g->d_ctrl, g->h_ctrl, sizeof(CtrlState), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);       // h_ctrl is reused for the read-backs
    if (e != cudaSuccess) return cuda_fail(e, "integrate setup");

    StepArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.rho = rho_dust; sa.rho_out = g->trial_rho;           // buffer pair 0 / 1 (roles swap with ctrl->cur)
    sa.k_fsal = g->k_fsal; sa.k_out = g->trial_k;
    sa.err = g->trial_err;
    sa.rtol = b->p.rtol; sa.atol_factor = b->p.atol_factor;
    sa.ctrl = g->d_ctrl;
    const GasArgs ga = gas_args(g->gs, b->p);
    int enq = 0;
    for (;;) {
        const int n = std::min(kBatch, max_steps - enq);
        for (int q = 0; q < n; ++q) {
            int rc = run(g, MODE_STEP, ga, sa, stream);
            if (rc) return rc;
            e = launch_ctrl(g->trial_err, g->C, g->d_ctrl, g->d_log, st);
            if (e != cudaSuccess) return cuda_fail(e, "controller launch");
            g_launches.fetch_add(1, std::memory_order_relaxed);
        }
        enq += n;
        e = cudaMemcpyAsync(g->h_ctrl, g->d_ctrl, sizeof(CtrlState), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(e, "integrate batch");
        if (g->h_ctrl->done || enq >= max_steps) break;
    }
    c = *g->h_ctrl;
    const int n_trials = c.n_acc + c.n_rej;
    if (dt_log && n_trials > 0) {
        e = cudaMemcpyAsync(dt_log, g->d_log, (size_t)n_trials * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(e, "integrate log copy");
    }
    if (c.cur) {                                            // state ended in the second buffer pair
        e = cudaMemcpyAsync(rho_dust, g->trial_rho, row_bytes, cudaMemcpyDeviceToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(e, "integrate copy-back");
        std::swap(g->k_fsal, g->trial_k);
    }
    if (c.n_acc > 0) { g->fsal_valid = true; g->fsal_rho = rho_dust; g->fsal_K = nullptr; }
    if (info) {
        info->t_done = c.t; info->dt_last = c.dt_last; info->dt_next = c.dt; info->err_last = c.err_last;
        info->n_accepted = c.n_acc; info->n_rejected = c.n_rej;
    }
    if (c.status) return fail(CUDISC_ERR_INVALID, "non-finite error norm at t = %g s (dt = %g s)", c.t, c.h);
    return CUDISC_OK;
}

}  // namespace

extern "C" {

int cudisc_coag_integrate(cudisc_grid g, cudisc_bins b, double *rho_dust, double t_span, double dt_try,
                          int max_steps, double *dt_log, cudisc_integrate_info *info, cudisc_stream stream)
{
    int rc = check_pair(g, b);
    if (rc) return rc;
    if (!g->gas_bound) return fail(CUDISC_ERR_INVALID, "no gas state bound (cudisc_grid_bind_gas)");
    if (!rho_dust) return fail(CUDISC_ERR_INVALID, "NULL array argument");
    if (!(t_span > 0.0) || !(dt_try > 0.0) || max_steps < 1)
        return fail(CUDISC_ERR_INVALID, "need t_span > 0, dt_try > 0, max_steps >= 1");
    return integrate_impl(g, b, rho_dust, t_span, 0x7fffffff, dt_try, max_steps, dt_log, info, stream);
}

int cudisc_coag_integrate_steps(cudisc_grid g, cudisc_bins b, double *rho_dust, int n_accepted, double dt_try,
                                int max_steps, double *dt_log, cudisc_integrate_info *info, cudisc_stream stream)
{
    int rc = check_pair(g, b);
    if (rc) return rc;
    if (!g->gas_bound) return fail(CUDISC_ERR_INVALID, "no gas state bound (cudisc_grid_bind_gas)");
    if (!rho_dust) return fail(CUDISC_ERR_INVALID, "NULL array argument");
    if (n_accepted < 1 || !(dt_try > 0.0) || max_steps < n_accepted)
        return fail(CUDISC_ERR_INVALID, "need n_accepted >= 1, dt_try > 0, max_steps >= n_accepted");
    return integrate_impl(g, b, rho_dust, 1.0e300, n_accepted, dt_try, max_steps, dt_log, info, stream);
}

int cudisc_microbench_dfma(int n_iter, double *dfma_per_s, double *elapsed_ms)
{
    if (!dfma_per_s) return fail(CUDISC_ERR_INVALID, "dfma_per_s is NULL");
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_fail(e, "device query");
    if (n_iter <= 0) n_iter = 20000;
    const int grid = sms * 8;
    double *out = nullptr;
    cudaEvent_t e0, e1;
    e = cudaMalloc((void **)&out, 64);
    if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc");
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {        // rep 0 = warm-up
        cudaEventRecord(e0, 0);
        e = launch_dfma_peak(grid, n_iter, out, 0);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        cudaEventRecord(e1, 0);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    if (e != cudaSuccess) return cuda_fail(e, "dfma microbenchmark");
    const double n = (double)grid * 256.0 * 64.0 * (double)n_iter;
    *dfma_per_s = n / ((double)best * 1e-3);
    if (elapsed_ms) *elapsed_ms = best;
    return CUDISC_OK;
}

int cudisc_microbench_copy(long long n_bytes, double *bytes_per_s, double *elapsed_ms)
{
    if (!bytes_per_s) return fail(CUDISC_ERR_INVALID, "bytes_per_s is NULL");
    if (n_bytes <= 0) n_bytes = 1ll << 30;
    n_bytes &= ~15ll;
    if (n_bytes < 16) return fail(CUDISC_ERR_INVALID, "n_bytes too small");
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_fail(e, "device query");
    void *src = nullptr, *dst = nullptr;
    e = cudaMalloc(&src, (size_t)n_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&dst, (size_t)n_bytes);
    if (e == cudaSuccess) e = cudaMemset(src, 1, (size_t)n_bytes);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 6 && e == cudaSuccess; ++rep) {
        cudaEventRecord(e0, 0);
        e = launch_copy_peak(sms * 16, src, dst, (size_t)n_bytes / 16, 0);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        cudaEventRecord(e1, 0);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (src) cudaFree(src);
    if (dst) cudaFree(dst);
    if (e != cudaSuccess) return cuda_fail(e, "copy microbenchmark");
    *bytes_per_s = 2.0 * (double)n_bytes / ((double)best * 1e-3);
    if (elapsed_ms) *elapsed_ms = best;
    return CUDISC_OK;
}

long long cudisc_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
/* internal: the other translation units of the library report their launches here */
void cudisc_count_launch_(void) { g_launches.fetch_add(1, std::memory_order_relaxed); }
const char *cudisc_last_error(void) { return g_err; }
const char *cudisc_version(void) { return "cudisc-coag-b200 0.1 (sm_100a)"; }

}  // extern "C"
