// hydro.cu -- vertical hydrostatic equilibrium of the gas (cuDisc section 3.5; PAPER.md:242-274,
// Eqs. 32-37) for sm_100a: cudisc_hydro_create / cudisc_hydrostatic / cudisc_hydro_destroy.
//
// This is the step that produces the rho_gas the coagulation path consumes.  It is
// HBM-bound: 8 B read (c_s^2) and 8 B written (rho_g) per cell.  One CTA owns one radial column at a
// time (columns are contiguous in memory: j, the Z index, runs fastest), four consecutive cells per thread:
//   * the column of c_s^2 arrives in shared memory by a 1-D bulk copy (cp.async.bulk, the TMA engine)
//     completing on an mbarrier; the copy of the CTA's NEXT column is in flight while it works;
//   * per cell the pressure ratio of Eq. 34 (IEEE divide in the paper's operation order, exp); Eq. 36 as a
//     product inside the thread, a multiplicative scan over the lanes and one over the warps, all in a fixed
//     order; omega = P / c_s^2; sum_k omega V by a block reduction (Eq. 37);
//   * the normalised densities leave through a bulk store from shared memory.
// (Round 1 of this kernel gave a whole column to one warp: 14 warps per SM, one latency chain per 128 cells,
//  0.13 of the HBM rate.)
// Written from the paper; shares nothing with oracle/.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <new>
#include <vector>

#include "../../include/cudisc_coag.h"

extern "C" void cudisc_count_launch_(void);

namespace {

constexpr unsigned kHydroMagic = 0x48594452u;

struct HydroGeom {
    int n_r, n_z;
    const double *Rc, *dR3, *RdR;     // [n_r]  centre radius, d(R^3)_i, (R dR)_i = d(R^2)_i / 2
    const double *sj, *dtan3;         // [n_z]  sqrt(1 + tan^2 theta^c_j) (r = R^c s), d(tan theta)_j / 3
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" :: "r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile("{\n.reg .pred p;\nWAIT_%=:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 "@!p bra WAIT_%=;\n}\n" :: "r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_load(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 :: "r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_store(void *dst_gmem, const void *src_smem, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n"
                 :: "l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.commit_group;\n" ::: "memory");
}
__device__ __forceinline__ void bulk_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;\n" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

// One CTA per radial column at a time, 4 consecutive cells per thread (blockDim = ceil(n_z / 4) rounded up to a
// warp, <= 1024).  TMA = true (n_z even, 16-byte aligned arrays): the column of c_s^2 arrives in shared memory by a
// 1-D bulk copy completing on an mbarrier, the CTA's NEXT column in flight meanwhile, and the densities leave
// through a bulk store; else plain loads / stores.  The product of Eq. 36 is taken in a fixed order: within the
// thread, then a multiplicative scan over the lanes, then over the warps.
constexpr int kHU = 4;

template <bool TMA>
__global__ void __launch_bounds__(1024) hydro_kernel(const HydroGeom gm, const double *__restrict__ cs2,
                                                     const double *__restrict__ Sigma, double GM,
                                                     double *__restrict__ rho)
{
    extern __shared__ __align__(16) double hs[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const int n_z = gm.n_z, nzp = (n_z + 1) & ~1;
    double *buf0 = hs, *buf1 = hs + nzp;
    double *edge = hs + 2 * nzp;                 // [2][32] last 1/r, 1/c_s^2 of every warp
    double *wtot = edge + 64;                    // [32] warp products
    double *wsum = wtot + 32;                    // [32] warp sums of omega V
    uint64_t *bar = reinterpret_cast<uint64_t *>(wsum + 32);
    const uint32_t bytes = (uint32_t)n_z * 8u;
    if (TMA && tid == 0) {
        mbar_init(bar, 1); mbar_init(bar + 1, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        if ((int)blockIdx.x < gm.n_r) { mbar_expect_tx(bar, bytes); bulk_load(buf0, cs2 + (size_t)blockIdx.x * n_z, bytes, bar); }
    }
    __syncthreads();
    uint32_t ph0 = 0u, ph1 = 0u;
    int b = 0;
    const int j0 = kHU * tid;
    for (int i = blockIdx.x; i < gm.n_r; i += gridDim.x, b ^= 1) {
        double *c = b ? buf1 : buf0;             // column buffer: c_s^2 in, rho out
        if (TMA) {
            const int inext = i + gridDim.x;
            if (tid == 0) {
                bulk_store_wait_read();          // the previous column's store has read the other buffer
                if (inext < gm.n_r) {
                    fence_async_smem();
                    mbar_expect_tx(bar + (b ^ 1), bytes);
                    bulk_load(b ? buf0 : buf1, cs2 + (size_t)inext * n_z, bytes, bar + (b ^ 1));
                }
            }
            mbar_wait(bar + b, b ? ph1 : ph0);
            if (b) ph1 ^= 1u; else ph0 ^= 1u;
        }
        const double *cin = TMA ? c : cs2 + (size_t)i * n_z;
        const double Rc = gm.Rc[i], dR3 = gm.dR3[i];
        double cj[kHU], inv_r[kHU], inv_c[kHU], p[kHU];
        bool act[kHU];
#pragma unroll
        for (int u = 0; u < kHU; ++u) {
            const int j = j0 + u;
            act[u] = j < n_z;
            cj[u] = act[u] ? cin[j] : 1.0;
            const double r = __dmul_rn(Rc, act[u] ? gm.sj[j] : 1.0);
            inv_r[u] = __drcp_rn(r);             // == 1.0 / r, correctly rounded
            inv_c[u] = __drcp_rn(cj[u]);
        }
        // the previous cell's 1/r, 1/c_s^2 of the thread's first cell: the neighbour lane, or the last lane of
        // the previous warp through shared memory
        double pr = __shfl_up_sync(0xffffffffu, inv_r[kHU - 1], 1), pc = __shfl_up_sync(0xffffffffu, inv_c[kHU - 1], 1);
        if (lane == 31) { edge[warp] = inv_r[kHU - 1]; edge[32 + warp] = inv_c[kHU - 1]; }
        __syncthreads();
        if (lane == 0 && warp > 0) { pr = edge[warp - 1]; pc = edge[32 + warp - 1]; }
        double q = 1.0;                          // running product inside the thread
#pragma unroll
        for (int u = 0; u < kHU; ++u) {
            const double r_prev = u ? inv_r[u - 1] : pr, c_prev = u ? inv_c[u - 1] : pc;
            double ratio = 1.0;
            if (act[u] && j0 + u > 0) {
                const double avg = __dmul_rn(0.5, __dadd_rn(inv_c[u], c_prev));                    // Eq. 35
                ratio = exp(__dmul_rn(__dmul_rn(GM, avg), __dsub_rn(inv_r[u], r_prev)));         // Eq. 34
            }
            q *= ratio;
            p[u] = q;
        }
        // Eq. 36: exclusive multiplicative scan of the thread products over the lanes, then over the warps
        double incl = q;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl *= v;
        }
        double excl = __shfl_up_sync(0xffffffffu, incl, 1);
        if (lane == 0) excl = 1.0;
        if (lane == 31) wtot[warp] = incl;
        __syncthreads();
        double carry = 1.0;
        for (int w = 0; w < warp; ++w) carry *= wtot[w];
        carry *= excl;
        double part = 0.0;
#pragma unroll
        for (int u = 0; u < kHU; ++u) {
            if (act[u]) {
                const int j = j0 + u;
                const double omega = __dmul_rn(__dmul_rn(p[u], carry), inv_c[u]);     // P / c_s^2 (one extra rounding)
                part = fma(omega, dR3 * gm.dtan3[j], part);                                        // Eq. 1
                p[u] = omega;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        if (lane == 0) wsum[warp] = part;
        __syncthreads();
        double tot = 0.0;
        for (int w = 0; w < nwarps; ++w) tot += wsum[w];
        const double norm = __ddiv_rn(__dmul_rn(Sigma[i], gm.RdR[i]), tot);                        // Eq. 37
        double *o = TMA ? c : rho + (size_t)i * n_z;
#pragma unroll
        for (int u = 0; u < kHU; ++u)
            if (act[u]) o[j0 + u] = __dmul_rn(p[u], norm);
        if (TMA) {
            fence_async_smem();
            __syncthreads();
            if (tid == 0) bulk_store(rho + (size_t)i * n_z, c, bytes);
        } else {
            __syncthreads();                     // edge / wtot / wsum are free for the next column
        }
    }
    if (TMA && tid == 0) bulk_store_wait_read();
}

thread_local char h_err[256] = "";
int hfail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(h_err, sizeof(h_err), fmt, ap);
    va_end(ap);
    return code;
}

}  // namespace

struct cudisc_hydro_s {
    unsigned magic;
    int n_r, n_z, sms, smem_optin;
    double *blob;
    HydroGeom gm;
};

extern "C" {

const char *cudisc_hydro_last_error(void) { return h_err; }

int cudisc_hydro_create(int n_r, int n_z, const double *R_edges, const double *tan_edges,
                        const double *R_centres, const double *tan_centres, cudisc_hydro *out)
{
    if (!out) return hfail(CUDISC_ERR_INVALID, "out is NULL");
    *out = nullptr;
    if (n_r < 1 || n_z < 1) return hfail(CUDISC_ERR_INVALID, "n_r and n_z must be >= 1");
    if (n_z > 4096) return hfail(CUDISC_ERR_UNSUPPORTED, "n_z %d > 4096", n_z);
    if (!R_edges || !tan_edges || !R_centres || !tan_centres) return hfail(CUDISC_ERR_INVALID, "NULL grid array");
    for (int i = 0; i < n_r; ++i)
        if (!(R_edges[i] >= 0.0) || !(R_edges[i] < R_centres[i]) || !(R_centres[i] < R_edges[i + 1]))
            return hfail(CUDISC_ERR_INVALID, "radial grid not monotone at i = %d", i);
    for (int j = 0; j < n_z; ++j)
        if (!(tan_edges[j] <= tan_centres[j]) || !(tan_centres[j] <= tan_edges[j + 1]) || !(tan_edges[j] < tan_edges[j + 1]))
            return hfail(CUDISC_ERR_INVALID, "polar grid not monotone at j = %d", j);
    std::vector<double> h((size_t)3 * n_r + 2 * n_z);
    for (int i = 0; i < n_r; ++i) {
        const double a = R_edges[i], b = R_edges[i + 1];
        h[i] = R_centres[i];
        h[n_r + i] = b * b * b - a * a * a;                  // d(R^3)_i, Eq. 1
        h[2 * n_r + i] = 0.5 * (b * b - a * a);              // (R dR)_i
    }
    for (int j = 0; j < n_z; ++j) {
        h[3 * n_r + j] = std::sqrt(1.0 + tan_centres[j] * tan_centres[j]);       // r_{i,j} = R^c_i * this
        h[3 * n_r + n_z + j] = (tan_edges[j + 1] - tan_edges[j]) / 3.0;
    }
    int dev = 0, sms = 0, optin = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return hfail(CUDISC_ERR_CUDA, "device query: %s", cudaGetErrorString(e));
    cudisc_hydro hh = new (std::nothrow) cudisc_hydro_s();
    if (!hh) return hfail(CUDISC_ERR_INVALID, "out of host memory");
    e = cudaMalloc((void **)&hh->blob, h.size() * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpy(hh->blob, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        if (hh->blob) cudaFree(hh->blob);
        delete hh;
        return hfail(CUDISC_ERR_CUDA, "geometry upload: %s", cudaGetErrorString(e));
    }
    hh->magic = kHydroMagic; hh->n_r = n_r; hh->n_z = n_z; hh->sms = sms; hh->smem_optin = optin;
    hh->gm.n_r = n_r; hh->gm.n_z = n_z;
    hh->gm.Rc = hh->blob; hh->gm.dR3 = hh->blob + n_r; hh->gm.RdR = hh->blob + 2 * n_r;
    hh->gm.sj = hh->blob + 3 * n_r; hh->gm.dtan3 = hh->blob + 3 * n_r + n_z;
    *out = hh;
    return CUDISC_OK;
}

int cudisc_hydro_destroy(cudisc_hydro h)
{
    if (!h || h->magic != kHydroMagic) return hfail(CUDISC_ERR_HANDLE, "bad hydro handle");
    cudaFree(h->blob);
    h->magic = 0;
    delete h;
    return CUDISC_OK;
}

int cudisc_hydrostatic(cudisc_hydro h, const double *cs2, const double *Sigma_g, double GM,
                       double *rho_gas_out, cudisc_stream stream)
{
    if (!h || h->magic != kHydroMagic) return hfail(CUDISC_ERR_HANDLE, "bad hydro handle");
    if (!cs2 || !Sigma_g || !rho_gas_out) return hfail(CUDISC_ERR_INVALID, "NULL array argument");
    if (cs2 == rho_gas_out) return hfail(CUDISC_ERR_INVALID, "cs2 and rho_gas_out may not alias");
    const int n_z = h->n_z, nzp = (n_z + 1) & ~1;
    const bool tma = (n_z % 2 == 0) && ((uintptr_t)cs2 % 16 == 0) && ((uintptr_t)rho_gas_out % 16 == 0);
    const int threads = std::min(1024, ((n_z + kHU - 1) / kHU + 31) & ~31);
    const size_t smem = (size_t)(2 * nzp + 64 + 32 + 32 + 2) * sizeof(double);
    // resident CTAs per SM: threads and shared memory (registers: 64 per thread)
    const int per_sm = std::max(1, std::min({2048 / threads, (int)((size_t)h->smem_optin / (smem + 1024)), 65536 / (64 * threads)}));
    const int blocks = std::max(1, std::min(h->n_r, per_sm * h->sms));
    cudaError_t e = cudaSuccess;
    {
        static bool attr_done[64] = {false};
        int dev = 0;
        e = cudaGetDevice(&dev);
        if (e == cudaSuccess && (dev < 0 || dev >= 64 || !attr_done[dev])) {
            e = cudaFuncSetAttribute(hydro_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin);
            if (e == cudaSuccess)
                e = cudaFuncSetAttribute(hydro_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin);
            if (e == cudaSuccess && dev >= 0 && dev < 64) attr_done[dev] = true;
        }
        if (e != cudaSuccess) return hfail(CUDISC_ERR_CUDA, "hydro attribute: %s", cudaGetErrorString(e));
    }
    if (tma) hydro_kernel<true><<<blocks, threads, smem, (cudaStream_t)stream>>>(h->gm, cs2, Sigma_g, GM, rho_gas_out);
    else hydro_kernel<false><<<blocks, threads, smem, (cudaStream_t)stream>>>(h->gm, cs2, Sigma_g, GM, rho_gas_out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return hfail(CUDISC_ERR_CUDA, "hydro launch: %s", cudaGetErrorString(e));
    cudisc_count_launch_();
    return CUDISC_OK;
}

}  // extern "C"
