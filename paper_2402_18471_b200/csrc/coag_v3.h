// coag_v3.h -- tables of the stencil cell kernel (coag_v3.cu): cudisc_coag_step and cudisc_coag_rates_otf
// on mass grids whose near-diagonal ("band") outcomes form a shift-invariant stencil (every exact log grid).
//
// Layout of one cell's collision kernel on the SM:
//   row copy     shared memory, packed lower-triangular (Kc, Kf) at i (i + 1) / 2 + j, diagonal halved
//                (PAPER.md:436): read by the row pass (lane <-> target row i) and by the band stencil;
//   column copy  tensor memory, lane <-> impactor column j of a 32-column block c, four 32-bit columns per
//                row i >= 32 c (rows above the diagonal and Kf of rows i < iS[j] are stored as 0), in chunks
//                of 8 rows: read by the column pass with one tcgen05.ld.x32 per chunk.
// A warp reaches only the tensor-memory lanes of its quarter (warp % 4), so a chunk is built and later
// summed by the same warp.  All work of a cell is dealt out STATICALLY on the host (this file's V3Tables,
// passed to the kernel by value): per warp a few "runs" of column chunks, of row-pass columns and of band
// taps.  No queues, no atomics, fixed summation order.
//
// Band as a stencil.  coag_tables.cpp lists every outcome that the bulk row / column sums do not cover as
// gather entries (target, i, j, plane, coef).  On a grid with constant mass ratio coef / m_i depends only on
// (d = i - j, o = target - i, plane, kind) away from the grid ends, so the host folds the entries into
// "taps" (d, o, c0, c1, s1):
//   dens[t] += y_i n_{i-d} (c0 Kc + c1 Kf)[i][i-d],   S[t] += y_i n_{i-d} s1 Kf[i][i-d],   i = t - o,
// plus a short list of exception entries (grid ends) that carries the residual coefficients.  The host
// re-expands taps + exceptions and checks them against the gather entries (v3_build refuses the grid
// otherwise), so the stencil is an exact restatement of the table, not an approximation of it.
#pragma once
#include <stdint.h>

#include <string>
#include <vector>

#include "coag_tables.h"

namespace cudisc {

constexpr int kV3Warps = 16;
constexpr int kV3MaxBlk = 5;           // 32-bin blocks: n_bins <= 160 (shared memory decides first)
constexpr int kV3MaxTaps = 40;
constexpr int kV3ColRuns = 4;          // per warp
constexpr int kV3RowRuns = 3;          // per warp
constexpr int kV3MaxFold = 20;         // folded row pairs per diagonal block
constexpr int kV3Pad = 8;              // zero padding (entries) on both sides of NN and YY

struct V3Tap {
    double c0, c1, s1;                 // coefficients / m_i of plane 0 -> density, plane 1 -> density, plane 1 -> S
    int d, o;                          // pair (i, i - d) feeds target i + o
};

struct V3ColRun {                      // chunks [k0, k0 + n) of column block c: rows 32 c + 8 k ..
    short c, k0, n, tcol;              // tcol: first tensor-memory column (in the warp's quarter); n == 0: unused
    short slot, diag, pad0, pad1;      // column partial slot; diag: the run is the whole diagonal block of c
};

struct V3RowRun {                      // columns [ja, jb) of row block b -> row partial slot
    short b, ja, jb, slot;             // jb == ja: unused
};

struct V3Exc {                         // exception entry (global memory): coef * n_i * n_j * Kplane[i][j]
    double coef;
    int i, j, plane, pad;
};

struct V3ExcTarget {                   // exceptions [e0, e1) feed target `t` (kind 1: S target)
    short t, kind, e0, e1;
};

struct V3Tables {
    int on;                            // 0: this mass grid runs on the general kernel
    int N, nb, P;
    int nTaps, nExcT;
    // shared-memory byte offsets (coag_v3.cu); the row copy of K is the last array
    int oYY, oNN, oDTAB, oEXPT, oRED, oBAND, oGK, oNBULK, oUNION, oCOLP, oROWP, oK, smemBytes;
    int nColSlots, nRowSlots;
    int rpBase[kV3MaxBlk], rpCnt[kV3MaxBlk];     // row block b: row partial slots [rpBase, + rpCnt)
    int cpBase[kV3MaxBlk], cpCnt[kV3MaxBlk];     // column block c: column partial slots
    int cmin[kV3MaxBlk];                         // columns [0, cmin[b]) are bulk for EVERY row of block b
    short bincCol[kV3Warps];                     // tensor-memory column of the warp's per-bin constants (-1: none)
    V3ColRun col[kV3Warps][kV3ColRuns];
    V3RowRun row[kV3Warps][kV3RowRuns];
    short bandBlk[kV3Warps], bandT0[kV3Warps], bandT1[kV3Warps], bandSlot[kV3Warps];   // taps [T0, T1) of target block (-1: none)
    unsigned char foldA[kV3MaxBlk][kV3MaxFold], foldB[kV3MaxBlk][kV3MaxFold];       // diagonal block: local rows (0xff: none)
    short nFold[kV3MaxBlk];
    V3ExcTarget excT[8];
    V3Tap taps[kV3MaxTaps];
    const V3Exc *exc;                  // device
    const int *nbulk;                  // device [N]
    const int *iS;                     // device [N]
};

struct V3Host {
    V3Tables t;
    std::vector<V3Exc> exc;
    std::string why;                   // reason the grid does not take this kernel (t.on == 0)
};

// Builds the stencil, checks it against the gather entries and deals the work out.  smem_optin: device limit.
void v3_build(const HostTables &ht, int logGrid, int smem_optin, V3Host &out);

// Host-side check of the run lists and of the stencil (CPU tests, cudisc_bins_schedule_check): adds to
//   bad[0] pairs not built exactly once            bad[1] bulk pairs not in the row pass exactly once
//   bad[2] pairs not in the column pass exactly once   bad[3] tensor-memory / partial-slot clashes
//   bad[4] stencil + exceptions != gather entries (evaluated on pseudo-random n, K)   bad[5] band tasks
void v3_check(const HostTables &ht, const V3Host &v, long long bad[6]);

}  // namespace cudisc
