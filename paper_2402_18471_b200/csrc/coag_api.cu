// coag_api.cu -- the C ABI of include/cudisc_coag.h: handles, argument checks, table upload,
// launch configuration.  No arithmetic of the method lives here (tables: coag_tables.cpp,
// kernels: coag_kernels.cu / coag_device.cuh).
#include "../../include/cudisc_coag.h"

#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "coag_launch.h"
#include "coag_tables.h"

using namespace cudisc;

namespace {

constexpr unsigned kBinsMagic = 0xC0A6B125u;
constexpr unsigned kGridMagic = 0xC0A66D1Du;
constexpr int kMaxBins = 256;

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
};

struct cudisc_grid_s {
    unsigned magic;
    int n_r, n_z, C;
    cudisc_bins bins;
    bool gas_bound;
    cudisc_gas_state gs;
    bool fsal_valid;
    double *k_fsal;     // [C x N]
    double *kslab;      // per-CTA overflow of the K store
    double *stage_rho;  // [C x N] staging of cudisc_coag_step_host (lazy)
    double *stage_err;  // [C]
    int num_sms, smem_optin, grid_ctas, Psm, smem_bytes;
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
    std::string why = build_tables(m, me, a, rho_m, p.eta, p.chi_im, b->ht);
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

int upload_tables(cudisc_bins b)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (b->on_device && b->device == dev) return CUDISC_OK;
    if (b->on_device) { cudaFree(b->dev_blob); b->on_device = false; b->dev_blob = nullptr; }

    const HostTables &t = b->ht;
    const int N = t.N;
    DevTables d;
    memset(&d, 0, sizeof(d));
    d.N = N; d.Np = (N + 1) & ~1; d.P = N * (N + 1) / 2;
    d.rho_m = t.rho_m; d.sS = t.sS;

    // row-pass items: (block of 32 rows, chunk of 32 impactors), heaviest first
    std::vector<uint32_t> itemsA, itemsB;
    int nchA = 1;
    const int nblk = (N + 31) / 32;
    for (int blk = 0; blk < nblk; ++blk) {
        int mx = 0;
        for (int i = blk * 32; i < std::min(N, blk * 32 + 32); ++i) mx = std::max(mx, t.n_bulk[i]);
        const int nch = (mx + 31) / 32;
        nchA = std::max(nchA, nch);
        for (int c = 0; c < nch; ++c) itemsA.push_back((uint32_t)blk | ((uint32_t)c << 16));
    }
    // column-pass items: (block of 32 columns cb, chunk r of 32 rows starting at the diagonal block)
    const int nchB = nblk;
    for (int cb = 0; cb < nblk; ++cb)
        for (int r = 0; cb * 32 + r * 32 < N; ++r) itemsB.push_back((uint32_t)cb | ((uint32_t)r << 16));
    d.nItemsA = (int)itemsA.size(); d.nItemsB = (int)itemsB.size();
    d.nchA = nchA; d.nchB = nchB;
    d.partStride = std::max(std::max(4 * nchA, 2 * nchB), 12);

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

    Blob bl;
    const size_t o_m = bl.add(t.m), o_rm = bl.add(t.rm), o_a = bl.add(t.a);
    const size_t o_cA1 = bl.add(t.cA1), o_cA2 = bl.add(t.cA2), o_cB1 = bl.add(t.cB1), o_cB2 = bl.add(t.cB2);
    const size_t o_cF1 = bl.add(t.cF1), o_cF2 = bl.add(t.cF2), o_cG1 = bl.add(t.cG1), o_cG2 = bl.add(t.cG2);
    const size_t o_nb = bl.add(t.n_bulk), o_iS = bl.add(t.iS), o_lj = bl.add(t.lj);
    const size_t o_jlo = bl.add(t.jS_lo), o_jhi = bl.add(t.jS_hi);
    const size_t o_fA = bl.add(t.fA), o_fB = bl.add(t.finvB);
    const size_t o_cnt = bl.add(cnt), o_bidx = bl.add(bidx), o_bcoef = bl.add(bcoef);
    const size_t o_iA = bl.add(itemsA), o_iB = bl.add(itemsB);

    void *blob = nullptr;
    e = cudaMalloc(&blob, bl.bytes.size());
    if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc(tables)");
    e = cudaMemcpy(blob, bl.bytes.data(), bl.bytes.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(blob); return cuda_fail(e, "cudaMemcpy(tables)"); }
    const unsigned char *base = (const unsigned char *)blob;
    d.m = (const double *)(base + o_m); d.rm = (const double *)(base + o_rm); d.a = (const double *)(base + o_a);
    d.cA1 = (const double *)(base + o_cA1); d.cA2 = (const double *)(base + o_cA2);
    d.cB1 = (const double *)(base + o_cB1); d.cB2 = (const double *)(base + o_cB2);
    d.cF1 = (const double *)(base + o_cF1); d.cF2 = (const double *)(base + o_cF2);
    d.cG1 = (const double *)(base + o_cG1); d.cG2 = (const double *)(base + o_cG2);
    d.n_bulk = (const int *)(base + o_nb); d.iS = (const int *)(base + o_iS); d.lj = (const int *)(base + o_lj);
    d.jS_lo = (const int *)(base + o_jlo); d.jS_hi = (const int *)(base + o_jhi);
    d.fA = (const double *)(base + o_fA); d.finvB = (const double *)(base + o_fB);
    d.band_cnt = (const int *)(base + o_cnt);
    d.band_idx = (const uint32_t *)(base + o_bidx); d.band_coef = (const double *)(base + o_bcoef);
    d.itemsA = (const uint32_t *)(base + o_iA); d.itemsB = (const uint32_t *)(base + o_iB);
    b->dt = d;
    b->dev_blob = blob;
    b->device = dev;
    b->on_device = true;
    return CUDISC_OK;
}

GasArgs gas_args(const cudisc_gas_state &gs, const cudisc_params &p)
{
    GasArgs g;
    g.T = gs.T; g.rho_g = gs.rho_gas; g.Omega = gs.Omega; g.alpha = gs.alpha;
    g.vR = gs.v_R; g.vZ = gs.v_Z; g.vphi = gs.v_phi;
    g.alpha_const = p.alpha; g.mu = p.mu; g.v_frag = p.v_frag; g.sigma_mol = p.sigma_mol;
    return g;
}

int check_gas(const cudisc_gas_state *gs)
{
    if (!gs) return fail(CUDISC_ERR_INVALID, "gas_state is NULL");
    if (!gs->T || !gs->rho_gas || !gs->Omega || !gs->v_R || !gs->v_Z)
        return fail(CUDISC_ERR_INVALID, "gas_state: T, rho_gas, Omega, v_R and v_Z must be non-NULL");
    return CUDISC_OK;
}

int check_pair(cudisc_grid g, cudisc_bins b)
{
    if (!grid_ok(g)) return fail(CUDISC_ERR_HANDLE, "bad grid handle");
    if (!bins_ok(b)) return fail(CUDISC_ERR_HANDLE, "bad bins handle");
    if (g->bins != b) return fail(CUDISC_ERR_HANDLE, "grid was created for a different bins handle");
    return CUDISC_OK;
}

int run(cudisc_grid g, int mode, const GasArgs &ga, StepArgs sa, cudisc_stream stream)
{
    int rc = upload_tables(g->bins);
    if (rc) return rc;
    sa.C = g->C;
    sa.Psm = g->Psm;
    sa.kslab = g->kslab;
    LaunchCfg lc{g->grid_ctas, g->smem_bytes, g->smem_optin};
    cudaError_t e = launch_cells(mode, lc, g->bins->dt, ga, sa, (cudaStream_t)stream);
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
    g->k_fsal = nullptr; g->kslab = nullptr;
    g->stage_rho = nullptr; g->stage_err = nullptr;
    g->num_sms = sms; g->smem_optin = optin;

    const DevTables &d = b->dt;
    const size_t vec_bytes = smem_vec_doubles(d.Np, d.partStride) * sizeof(double);
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
    sa.have_k1 = g->fsal_valid ? 1 : 0;
    rc = run(g, 3, gas_args(g->gs, b->p), sa, stream);
    if (rc == CUDISC_OK) g->fsal_valid = true;
    return rc;
}

int cudisc_coag_step_host(cudisc_grid g, cudisc_bins b, double *rho_host, double dt,
                          double *err_host, cudisc_stream stream)
{
    int rc = check_pair(g, b);
    if (rc) return rc;
    if (!rho_host || !err_host) return fail(CUDISC_ERR_INVALID, "NULL array argument");
    const size_t row_bytes = (size_t)g->C * b->ht.N * sizeof(double);
    const size_t err_bytes = (size_t)g->C * sizeof(double);
    cudaError_t e = cudaSuccess;
    if (!g->stage_rho) {
        e = cudaMalloc((void **)&g->stage_rho, row_bytes);
        if (e == cudaSuccess) e = cudaMalloc((void **)&g->stage_err, err_bytes);
        if (e != cudaSuccess) {
            if (g->stage_rho) { cudaFree(g->stage_rho); g->stage_rho = nullptr; }
            return cuda_fail(e, "cudaMalloc(staging)");
        }
    }
    cudaStream_t st = (cudaStream_t)stream;
    e = cudaMemcpyAsync(g->stage_rho, rho_host, row_bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpyAsync(H2D)");
    rc = cudisc_coag_step(g, b, g->stage_rho, dt, g->stage_err, stream);
    if (rc) return rc;
    e = cudaMemcpyAsync(rho_host, g->stage_rho, row_bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(err_host, g->stage_err, err_bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(e, "step_host copies");
    return CUDISC_OK;
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
const char *cudisc_last_error(void) { return g_err; }
const char *cudisc_version(void) { return "cudisc-coag-b200 0.1 (sm_100a)"; }

}  // extern "C"
