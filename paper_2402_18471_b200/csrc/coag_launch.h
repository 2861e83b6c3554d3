// coag_launch.h -- internal interface between the C-ABI layer (coag_api.cu) and the kernels.
#pragma once
#include "coag_device.cuh"

namespace cudisc {

constexpr int kThreads = 512;   // threads per CTA of the cell kernels

// modes of the cell kernels
enum { MODE_KERNEL = 0, MODE_RATES = 1, MODE_OTF = 2, MODE_STEP = 3, MODE_STEPK = 4 };

struct LaunchCfg {
    int grid;            // persistent CTAs
    int smem_bytes;      // dynamic shared memory of this launch
    int smem_optin;      // device limit (cudaDevAttrMaxSharedMemoryPerBlockOptin)
};

// mode: 0 kernel, 1 rates (supplied K), 2 rates on the fly, 3 BS3(2) step
cudaError_t launch_cells(int mode, const LaunchCfg &lc, const DevTables &tb, const GasArgs &gs,
                         const StepArgs &sa, cudaStream_t st);
// launch_cells with the K-overflow slab in the library's file-scope scratch array instead of sa.kslab (no
// allocation anywhere on this path); the caller has checked lc.grid * (P - Psm) * 16 <= kStaticSlabBytes
constexpr size_t kStaticSlabBytes = (size_t)24 << 20;
cudaError_t launch_cells_static_slab(int mode, const LaunchCfg &lc, const DevTables &tb, const GasArgs &gs,
                                     const StepArgs &sa, cudaStream_t st);
// the stencil cell kernel (coag_v3.cu): MODE_OTF or MODE_STEP on a mass grid with vt.on
struct V3Tables;
cudaError_t launch_v3(int mode, const LaunchCfg &lc, const DevTables &tb, const V3Tables &vt,
                      const GasArgs &gs, const StepArgs &sa, cudaStream_t st);
// resident CTAs per SM of the cell kernels with `smem_bytes` of dynamic shared memory (0 on error)
int cells_occupancy(int smem_bytes, int smem_optin);
cudaError_t launch_dfma_peak(int grid, int n_iter, double *out, cudaStream_t st);
cudaError_t launch_copy_peak(int grid, const void *src, void *dst, size_t n16, cudaStream_t st);
// one controller update after a trial step (ctrl_kernel, coag_kernels.cu); log may be NULL
cudaError_t launch_ctrl(const double *err, int n, CtrlState *cs, double *log, cudaStream_t st);
// out[0] = NaN-propagating max of err[0..n)
cudaError_t launch_err_max(const double *err, int n, double *out, cudaStream_t st);

}  // namespace cudisc
