// coag_kernels.cu -- __global__ entry points of libcudisc_coag.so (sm_100a, FP64) and their launchers.
//
// One persistent CTA per resident slot walks the cells c = blockIdx.x, blockIdx.x + gridDim.x, ...
// Every mode shares the device routines of coag_device.cuh:
//   MODE_KERNEL : prologue + pair build                -> K_out [C][2][P] in HBM      (cudisc_coag_kernel)
//   MODE_RATES  : K planes from HBM -> K store, eval   -> drho_dt                     (cudisc_coag_rates)
//   MODE_OTF    : prologue + pair build -> K store, eval -> drho_dt                   (cudisc_coag_rates_otf)
//   MODE_STEP   : prologue + pair build -> K store, BS3(2) stages (3 or 4 evals)      (cudisc_coag_step)
#include "coag_launch.h"

namespace cudisc {

enum { MODE_KERNEL = 0, MODE_RATES = 1, MODE_OTF = 2, MODE_STEP = 3 };

template <int NT, int MODE>
__global__ void __launch_bounds__(NT, 1)
coag_cells_kernel(const DevTables tb, const GasArgs gs, const StepArgs sa)
{
    extern __shared__ __align__(16) double smem_raw[];
    const int tid = threadIdx.x;
    const int N = tb.N, P = tb.P;
    KStore ks;
    ks.sm = reinterpret_cast<double2 *>(smem_raw);
    ks.Psm = sa.Psm;
    ks.gl = reinterpret_cast<double2 *>(sa.kslab) + (size_t)blockIdx.x * (size_t)(P - sa.Psm);
    const Smem s = carve(smem_raw + 2 * (size_t)sa.Psm, tb.Np, tb.partStride);
    const bool has_vphi = gs.vphi != nullptr;
    const double c15vf2 = 1.5 * gs.v_frag * gs.v_frag;

    for (int cell = blockIdx.x; cell < sa.C; cell += gridDim.x) {
        const size_t row = (size_t)cell * N;

        // ---------------- K store for this cell
        if (MODE == MODE_RATES) {
            const double *k0 = sa.Kin + (size_t)cell * 2 * P, *k1 = k0 + P;
            for (int p = tid; p < P; p += NT) {
                int i, j;
                pair_decode(p, i, j);
                const double h = (i == j) ? 0.5 : 1.0;
                ks.st(p, make_double2(h * __ldg(k0 + p), h * __ldg(k1 + p)));
            }
        } else {
            const double Vg2 = cell_prologue(tb, gs, cell, s, tid);
            __syncthreads();
            for (int p = tid; p < P; p += NT) {
                int i, j;
                pair_decode(p, i, j);
                double2 k2 = pair_kernel(s, i, j, Vg2, c15vf2, has_vphi);
                if (MODE == MODE_KERNEL) {
                    double *o = sa.out + (size_t)cell * 2 * P;
                    o[p] = k2.x;
                    o[P + p] = k2.y;
                } else {
                    if (i == j) { k2.x *= 0.5; k2.y *= 0.5; }
                    ks.st(p, k2);
                }
            }
        }
        if (MODE == MODE_KERNEL) { __syncthreads(); continue; }

        // ---------------- state
        for (int k = tid; k < N; k += NT) {
            s.Y[k] = sa.rho[row + k];
            if (MODE == MODE_STEP && sa.have_k1) s.K1[k] = sa.k_fsal[row + k];
        }
        __syncthreads();

        if (MODE == MODE_RATES || MODE == MODE_OTF) {
            eval_rates<NT>(tb, s, ks, s.Y, s.K1, tid);
            for (int k = tid; k < N; k += NT) sa.out[row + k] = s.K1[k];
            __syncthreads();
            continue;
        }

        // ---------------- Bogacki-Shampine 3(2), PAPER.md:478 (tableau: Bogacki & Shampine 1989)
        const double h = sa.dt;
        if (!sa.have_k1) eval_rates<NT>(tb, s, ks, s.Y, s.K1, tid);
        for (int k = tid; k < N; k += NT) s.YS[k] = s.Y[k] + 0.5 * h * s.K1[k];
        __syncthreads();
        eval_rates<NT>(tb, s, ks, s.YS, s.K2, tid);
        for (int k = tid; k < N; k += NT) s.YS[k] = s.Y[k] + 0.75 * h * s.K2[k];
        __syncthreads();
        eval_rates<NT>(tb, s, ks, s.YS, s.K3, tid);
        for (int k = tid; k < N; k += NT)
            s.YS[k] = s.Y[k] + h * ((2.0 / 9.0) * s.K1[k] + (1.0 / 3.0) * s.K2[k] + (4.0 / 9.0) * s.K3[k]);
        __syncthreads();
        eval_rates<NT>(tb, s, ks, s.YS, s.K4, tid);

        // error norm (R10) and write-back
        double part = 0.0;
        for (int k = tid; k < N; k += NT) part += s.Y[k];
        const double atol = sa.atol_factor * block_sum<NT>(part, s.RED, tid);
        double emax = 0.0;
        for (int k = tid; k < N; k += NT) {
            const double e = h * ((-5.0 / 72.0) * s.K1[k] + (1.0 / 12.0) * s.K2[k]
                                  + (1.0 / 9.0) * s.K3[k] - (1.0 / 8.0) * s.K4[k]);
            const double sc = atol + sa.rtol * fmax(fabs(s.Y[k]), fabs(s.YS[k]));
            emax = nanmax(emax, fabs(e) / sc);
            sa.rho_out[row + k] = s.YS[k];
            sa.k_out[row + k] = s.K4[k];
        }
        emax = block_nanmax<NT>(emax, s.RED, tid);
        if (tid == 0) sa.err[cell] = emax;
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------ launch
template <int MODE>
static cudaError_t launch_mode(const LaunchCfg &lc, const DevTables &tb, const GasArgs &gs,
                               const StepArgs &sa, cudaStream_t st)
{
    constexpr int NT = kThreads;
    auto fn = coag_cells_kernel<NT, MODE>;
    static bool attr_done = false;          // per process and per mode; same value every time
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             lc.smem_optin);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    fn<<<lc.grid, NT, lc.smem_bytes, st>>>(tb, gs, sa);
    return cudaGetLastError();
}

cudaError_t launch_cells(int mode, const LaunchCfg &lc, const DevTables &tb, const GasArgs &gs,
                         const StepArgs &sa, cudaStream_t st)
{
    switch (mode) {
    case MODE_KERNEL: return launch_mode<MODE_KERNEL>(lc, tb, gs, sa, st);
    case MODE_RATES: return launch_mode<MODE_RATES>(lc, tb, gs, sa, st);
    case MODE_OTF: return launch_mode<MODE_OTF>(lc, tb, gs, sa, st);
    default: return launch_mode<MODE_STEP>(lc, tb, gs, sa, st);
    }
}

int cells_occupancy(int smem_bytes, int smem_optin)
{
    auto fn = coag_cells_kernel<kThreads, MODE_STEP>;
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

}  // namespace cudisc
