// coag_fast.h -- tables and task encoding of the tensor-memory ("fast") cell kernel (coag_fast.cu).
//
// The fast kernel keeps TWO copies of the cell's collision kernel on the SM:
//   row copy    shared memory, packed lower-triangular (Kc, Kf) at i (i + 1) / 2 + j: the row pass
//               (lane <-> target row i), the band products and the diagonal blocks read it;
//   column copy tensor memory, lane <-> impactor column j, four 32-bit columns per row i: the
//               column pass of all rows i >= 32 c + 32 of column block c reads it with tcgen05.ld
//               (~450 B/clk per SM measured against 128 B/clk of shared memory), so a rate
//               evaluation reads the shared-memory copy once instead of twice.
// A warp reaches only the 32 tensor-memory lanes of its quarter (warp % 4).  The work of a cell is
// deterministic, so the host deals it out STATICALLY: every warp owns a list of build tasks, a list of
// evaluation tasks and, for the combine phase, band gather groups (longest-processing-time-first over
// a cost model, tensor-memory tasks restricted to the warps of their quarter; coag_api.cu).  No atomics,
// no queue traffic, fixed summation order.  The encode / decode helpers below are the ONLY place the
// packing is written down: the device and the host-side schedule check both call them.
#pragma once
#include <stdint.h>

#include "coag_device.cuh"

namespace cudisc {

enum { FB_ROWS = 0, FB_LIST = 1 };                              // build task kinds
enum { FE_RECT = 0, FE_RAG = 1, FE_COLT = 2, FE_COLS = 3, FE_W = 4 };   // evaluation task kinds
constexpr int kNoTmem = 0x3ff;         // "no tensor-memory destination" in the tcol field
constexpr int kFastRowsBuild = 8;      // rows per build task
constexpr int kFastRowsColT = 32;      // rows per tensor-memory column task
constexpr int kFastRectCols = 40;      // columns per rectangular row-pass task
constexpr int kFastMaxBlk = 8;         // 32-bin blocks (n_bins <= 256)

struct FTask {
    int kind, blk, tcol, slot, a, b;
};

// x: kind[0:4) blk[4:8) tcol[8:18) slot[18:32)      y: a[0:16) b[16:32)
__host__ __device__ inline uint2 ftask_pack(int kind, int blk, int tcol, int slot, int a, int b)
{
    uint2 u;
    u.x = (uint32_t)kind | ((uint32_t)blk << 4) | ((uint32_t)tcol << 8) | ((uint32_t)slot << 18);
    u.y = (uint32_t)a | ((uint32_t)b << 16);
    return u;
}
__host__ __device__ inline FTask ftask_unpack(uint2 u)
{
    FTask t;
    t.kind = u.x & 15; t.blk = (u.x >> 4) & 15; t.tcol = (u.x >> 8) & 0x3ff; t.slot = (int)(u.x >> 18);
    t.a = u.y & 0xffff; t.b = (int)(u.y >> 16);
    return t;
}
//   FB_ROWS  blk = column block c, rows [a, b) (all >= 32 c + 32), tcol = tensor-memory column of row a
//            in the quarter of the warp that owns the task (kNoTmem: shared-memory copy only)
//   FB_LIST  blk = diagonal block c, triangular indices [a, b)
//   FE_RECT  blk = row block, columns [a, b) (a, b even; every row of the block has n_bulk >= b),
//            slot = row part p: sums to slots 32 p + lane
//   FE_RAG   blk = row block, columns [a, b), row i takes j < n_bulk[i] (predicated), slot = row part p
//   FE_COLT  blk = column block c, rows [a, b) from tensor-memory column tcol, slot = column part p
//   FE_COLS  blk = column block c, rows [a, b) from the shared-memory copy (diagonal blocks: i >= j;
//            overflow rows), slot = column part p
//   FE_W     blk = row block whose band products are staged

// shared-memory layout of the fast kernel: offsets in doubles from the start of dynamic shared memory
// (the K row copy sits at 0).  The build-time role vectors alias the partial-sum slots and the band stage.
enum { FO_YY = 0, FO_DTAB, FO_NN, FO_BANDV, FO_BANDV2, FO_BINI, FO_EXPT, FO_RED, FO_TB, FO_TE, FO_UNION,
       FO_PARTC, FO_WST, FO_B0, FO_B1, FO_J2, FO_J3, FO_V5, FO_END, kFastOff };

struct FastTables {
    int on;                        // 0: this mass grid runs on the general kernel
    int off[kFastOff];             // FO_*: array offsets; off[FO_END] = total doubles
    int bw[17], ew[17];            // warp w: build tasks [bw[w], bw[w+1]), evaluation tasks [ew[w], ew[w+1])
    int colMask;                   // 1: some tensor-memory rows lie below iS[j]: Kf is masked in the column copy
    int nwBins;                    // warps that own bins: ceil(N / 32)
    int nRowParts, nColParts;      // partial-sum parts: 32 slots each (row slots 4 doubles, column slots 2)
    int rpBase[kFastMaxBlk], rpCnt[kFastMaxBlk];   // row block b: parts [rpBase[b], + rpCnt[b])
    int cpBase[kFastMaxBlk], cpCnt[kFastMaxBlk];   // column block c: parts [cpBase[c], + cpCnt[c])
    // band gathers (combine phase).  Density targets: group g <-> bins 32 g + lane; its entry list is cut
    // in two halves h = 0, 1 (sums to BANDV / BANDV2), half 2 g + h gathered by warp bgWarp[2 g + h] from its
    // quarter's tensor-memory columns [bgCol, + 3 bgLen).  Fragment-source targets: group g <-> l-bins
    // 32 g + lane, gathered by the column-combine warp nwBins + g itself.
    int bgWarp[2 * kFastMaxBlk], bgCol[2 * kFastMaxBlk], bgLen[2 * kFastMaxBlk], bgOff[2 * kFastMaxBlk];
    int sgCol[kFastMaxBlk], sgLen[kFastMaxBlk], sgOff[kFastMaxBlk];
    const uint2 *buildTasks, *evalTasks;
    const double *bandCoef;        // tables [len][32] of every group at offset *Off (entries)
    const uint32_t *bandIdx;       // stage index plane * bandD * Np + (i - j) * Np + i
};

// Per-bin constants of the combine step live in tensor memory (shared memory is full at 150 bins).
// Row-combine group: warp w < nw owns bins 32 w + lane and holds FBC_* of its bins in the 16 columns
// [16 (w / 4), + 16) of its quarter; column-combine group: warp nw + w owns the same bins and holds
// 1 / B_k in the two columns [16 ceil(nw / 4) + 2 (warp / 4), + 2) of ITS quarter.  m_k and 1 / m_k stay
// in registers of the bin-owning threads.
enum { FBC_A1 = 0, FBC_A2, FBC_B1, FBC_F1, FBC_F2, FBC_G1, FBC_FA, kFastBinc };
__host__ __device__ inline int fast_binc_col_r(int warp) { return 16 * (warp >> 2); }
__host__ __device__ inline int fast_binc_col_c(int nw, int warp) { return 16 * ((nw + 3) >> 2) + 2 * (warp >> 2); }
__host__ __device__ inline int fast_binc_cols(int nw) { return 16 * ((nw + 3) >> 2) + 2 * (((2 * nw - 1) >> 2) + 1); }

// fills ft.off from the sizes already set in ft (nRowParts, nColParts, bw, ew)
inline void fast_layout(FastTables &ft, int P, int Np, int bandD)
{
    int q = 2 * P;
    auto take = [&](int what, int n) { ft.off[what] = q; q += (n + 1) & ~1; };
    take(FO_YY, 2 * Np); take(FO_DTAB, 2 * Np); take(FO_NN, Np + 8); take(FO_BANDV, Np); take(FO_BANDV2, Np);
    take(FO_BINI, Np); take(FO_EXPT, 64); take(FO_RED, 96);
    take(FO_TB, ft.bw[16]); take(FO_TE, ft.ew[16]);
    ft.off[FO_UNION] = q;
    ft.off[FO_PARTC] = q + 128 * ft.nRowParts;
    ft.off[FO_WST] = ft.off[FO_PARTC] + 64 * ft.nColParts;
    const int part = 128 * ft.nRowParts + 64 * ft.nColParts + 2 * bandD * Np;
    ft.off[FO_B0] = q + 10 * Np; ft.off[FO_B1] = q + 12 * Np; ft.off[FO_J2] = q + 14 * Np; ft.off[FO_J3] = q + 16 * Np;
    ft.off[FO_V5] = q + 18 * Np;
    const int build = 19 * Np;
    ft.off[FO_END] = q + (part > build ? part : build);
}

}  // namespace cudisc
