// hydro.cu -- vertical hydrostatic equilibrium of the gas (cuDisc section 3.5; PAPER.md:242-274,
// Eqs. 32-37) for sm_100a: cudisc_hydro_create / cudisc_hydrostatic / cudisc_hydro_destroy.
//
// This is the step that produces the rho_gas the coagulation path consumes.  It is
// HBM-bound: 8 B read (c_s^2) and 8 B written (rho_g) per cell.  One warp owns one radial column at a
// time (columns are contiguous in memory: j, the Z index, runs fastest):
//   * the column of c_s^2 arrives in shared memory by a 1-D bulk copy (cp.async.bulk, the TMA engine)
//     completing on an mbarrier; the copy of the warp's NEXT column is in flight while it works;
//   * per 32 cells: the pressure ratios of Eq. 34 (IEEE sqrt / divide in the paper's operation order,
//     exp), a multiplicative inclusive scan over the lanes in a fixed order (Eq. 36) times the carry of
//     the previous 32, omega = P / c_s^2, the lane's share of sum_k omega V (Eq. 37);
//   * the normalised densities leave through a bulk store from shared memory.
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

// TMA = true: n_z even (16-byte columns): bulk copies through shared memory; else plain loads / stores.
// Four groups of 32 cells are in flight per warp (their ratios and lane scans are independent; only the
// carry of Eq. 36 chains them), which is what hides the divide / exp / shuffle latencies.
template <bool TMA>
__global__ void __launch_bounds__(512) hydro_kernel(const HydroGeom gm, const double *__restrict__ cs2,
                                                    const double *__restrict__ Sigma, double GM,
                                                    double *__restrict__ rho)
{
    extern __shared__ __align__(16) double hs[];
    constexpr int U = 4;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpb = blockDim.x >> 5;
    const int n_z = gm.n_z, nzp = (n_z + 1) & ~1;
    // per warp: two column buffers (the densities overwrite the sound speeds in place), 2 mbarriers
    double *in0 = hs + (size_t)wib * (2 * nzp + 2), *in1 = in0 + nzp;
    uint64_t *bar = reinterpret_cast<uint64_t *>(in1 + nzp);
    const int gw = blockIdx.x * wpb + wib, nw = gridDim.x * wpb;
    const uint32_t bytes = (uint32_t)n_z * 8u;
    if (TMA) {
        if (lane == 0) { mbar_init(bar, 1); mbar_init(bar + 1, 1); }
        __syncwarp();
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        if (lane == 0 && gw < gm.n_r) { mbar_expect_tx(bar, bytes); bulk_load(in0, cs2 + (size_t)gw * n_z, bytes, bar); }
    }
    uint32_t ph0 = 0u, ph1 = 0u;
    int buf = 0;
    for (int i = gw; i < gm.n_r; i += nw, buf ^= 1) {
        double *c;                                       // column buffer: c_s^2 in, rho out
        if (TMA) {
            const int inext = i + nw;
            bulk_store_wait_read();                      // the previous column's store has read the other buffer
            if (lane == 0 && inext < gm.n_r) {
                fence_async_smem();
                mbar_expect_tx(bar + (buf ^ 1), bytes);
                bulk_load(buf ? in0 : in1, cs2 + (size_t)inext * n_z, bytes, bar + (buf ^ 1));
            }
            mbar_wait(bar + buf, buf ? ph1 : ph0);
            if (buf) ph1 ^= 1u; else ph0 ^= 1u;
            c = buf ? in1 : in0;
            __syncwarp();
        } else {
            c = rho + (size_t)i * n_z;                   // results are staged in the output column
        }
        const double *cin = TMA ? c : cs2 + (size_t)i * n_z;
        const double Rc = gm.Rc[i], dR3 = gm.dR3[i];
        double carry = 1.0, part = 0.0, inv_r_last = 0.0, inv_c_last = 0.0;
        for (int j0 = 0; j0 < n_z; j0 += 32 * U) {
            double cj[U], inv_r[U], inv_c[U], p[U];
            bool act[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int j = j0 + 32 * u + lane;
                act[u] = j < n_z;
                cj[u] = act[u] ? cin[j] : 1.0;
                const double r = __dmul_rn(Rc, act[u] ? gm.sj[j] : 1.0);
                inv_r[u] = __ddiv_rn(1.0, r);
                inv_c[u] = __ddiv_rn(1.0, cj[u]);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                double inv_r_prev = __shfl_up_sync(0xffffffffu, inv_r[u], 1);
                double inv_c_prev = __shfl_up_sync(0xffffffffu, inv_c[u], 1);
                const double rl = u ? __shfl_sync(0xffffffffu, inv_r[u ? u - 1 : 0], 31) : inv_r_last;
                const double cl = u ? __shfl_sync(0xffffffffu, inv_c[u ? u - 1 : 0], 31) : inv_c_last;
                if (lane == 0) { inv_r_prev = rl; inv_c_prev = cl; }
                p[u] = 1.0;
                if (act[u] && j0 + 32 * u + lane > 0) {
                    const double avg = __dmul_rn(0.5, __dadd_rn(inv_c[u], inv_c_prev));                // Eq. 35
                    p[u] = exp(__dmul_rn(__dmul_rn(GM, avg), __dsub_rn(inv_r[u], inv_r_prev)));     // Eq. 34
                }
            }
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {                                                       // Eq. 36
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const double v = __shfl_up_sync(0xffffffffu, p[u], o);
                    if (lane >= o) p[u] *= v;
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                p[u] *= carry;
                carry = __shfl_sync(0xffffffffu, p[u], 31);
                if (act[u]) {
                    const int j = j0 + 32 * u + lane;
                    const double omega = __ddiv_rn(p[u], cj[u]);
                    const double V = dR3 * gm.dtan3[j];                                              // Eq. 1
                    part = fma(omega, V, part);
                    c[j] = omega;
                }
            }
            inv_r_last = __shfl_sync(0xffffffffu, inv_r[U - 1], 31);
            inv_c_last = __shfl_sync(0xffffffffu, inv_c[U - 1], 31);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        const double norm = __ddiv_rn(__dmul_rn(Sigma[i], gm.RdR[i]), part);                         // Eq. 37
        __syncwarp();
        for (int j = lane; j < n_z; j += 32) c[j] = __dmul_rn(c[j], norm);
        if (TMA) {
            fence_async_smem();
            __syncwarp();
            if (lane == 0) bulk_store(rho + (size_t)i * n_z, c, bytes);
        }
    }
    if (TMA) bulk_store_wait_read();
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
    const size_t per_warp = (size_t)(2 * nzp + 2) * sizeof(double);
    int wpb = 16;
    while (wpb > 1 && wpb * per_warp > (size_t)h->smem_optin - 1024) --wpb;
    const size_t smem = tma ? wpb * per_warp : 0;
    const int blocks = std::max(1, std::min((h->n_r + wpb - 1) / wpb, 8 * h->sms));
    cudaError_t e = cudaSuccess;
    if (tma) {
        static bool attr_done[64] = {false};
        int dev = 0;
        e = cudaGetDevice(&dev);
        if (e == cudaSuccess && (dev < 0 || dev >= 64 || !attr_done[dev])) {
            e = cudaFuncSetAttribute(hydro_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin);
            if (e == cudaSuccess && dev >= 0 && dev < 64) attr_done[dev] = true;
        }
        if (e != cudaSuccess) return hfail(CUDISC_ERR_CUDA, "hydro attribute: %s", cudaGetErrorString(e));
        hydro_kernel<true><<<blocks, 32 * wpb, smem, (cudaStream_t)stream>>>(h->gm, cs2, Sigma_g, GM, rho_gas_out);
    } else {
        hydro_kernel<false><<<blocks, 32 * wpb, 0, (cudaStream_t)stream>>>(h->gm, cs2, Sigma_g, GM, rho_gas_out);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return hfail(CUDISC_ERR_CUDA, "hydro launch: %s", cudaGetErrorString(e));
    cudisc_count_launch_();
    return CUDISC_OK;
}

}  // extern "C"
