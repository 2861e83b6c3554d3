// coag_v3.h -- tables of the stencil cell kernel (coag_v3.cu): cudisc_coag_step and cudisc_coag_rates_otf
// on mass grids whose near-diagonal ("band") outcomes form a shift-invariant stencil (every exact log grid).
//
// Layout of one cell's collision kernel on the SM:
//   row copy     shared memory, packed lower-triangular (Kc, Kf) at i (i + 1) / 2 + j, diagonal halved
//                (PAPER.md:436): read by the row pass (lane <-> target row i) and by the band stage;
//   column copy  tensor memory, lane <-> impactor column j of a 32-column block c, four 32-bit columns per
//                row i >= 32 c (rows above the diagonal and Kf of rows i < iS[j] are stored as 0), in chunks
//                of 8 rows: read by the column pass with tcgen05.ld.
// A warp reaches only the tensor-memory lanes of its quarter (warp % 4), so a chunk is built and later
// summed by the same warp.  All work of a cell is dealt out STATICALLY on the host (this file's V3Tables,
// passed to the kernel by value): per warp a few "runs" of column chunks and of row-pass columns, packed
// one run per 32-bit word, copied to shared memory once per launch and decoded where a phase starts.  No queues,
// no atomics, fixed summation order.
//
// Band as a stencil.  coag_tables.cpp lists every outcome that the bulk row / column sums do not cover as
// gather entries (target, i, j, plane, coef).  On a grid with constant mass ratio coef / m_i depends only on
// (d = i - j, o = target - i, plane, kind) away from the grid ends.  Per evaluation one warp group
// stages  W[plane][d][i] = y_i n_{i-d} Kplane[i][i-d]   (y_i = m_i n_i; d < bandD) in shared memory, and
//   dens[t] = sum_taps c W[plane][d][t - o],   S[t] likewise,
// with warp-uniform coefficients from a small table in shared memory (one 16-byte entry per tap), plus a short
// list of exception entries at the grid ends that carries the residual coefficients.  The host re-expands taps + exceptions and checks them against
// the gather entries (v3_build refuses the grid otherwise; v3_check re-evaluates both on pseudo-random
// data), so the stencil is a restatement of the table, not an approximation of it.
#pragma once
#include <stdint.h>

#include <string>
#include <vector>

#include "coag_tables.h"

namespace cudisc {

constexpr int kV3Warps = 16;
constexpr int kV3MaxBlk = 5;           // 32-bin blocks: n_bins <= 160 (shared memory decides first)
constexpr int kV3NpMax = 32 * kV3MaxBlk;
constexpr int kV3MaxTaps = 40;         // density taps (one per plane); S taps: kV3MaxSTaps
constexpr int kV3MaxSTaps = 8;
constexpr int kV3ColRuns = 4;          // per warp
constexpr int kV3RowRuns = 3;          // per warp
constexpr int kV3MaxFold = 20;         // folded row pairs per diagonal block
constexpr int kV3MaxExc = 28;
constexpr int kV3MaxExcT = 8;          // targets with exception entries

// shared-memory byte offsets fixed at compile time (arrays sized for 160 bins); what follows them --
// band stage, partial-sum slots, row copy of K -- is laid out by the host (V3Tables::o*)
constexpr int kV3oRED = 0;                                   // double[128]: reductions and exchanges
constexpr int kV3oBINI = kV3oRED + 8 * 128;                  // int2[160]
constexpr int kV3oYY = kV3oBINI + 8 * kV3NpMax;              // double2[160]  (y, y m); .y: scanned suffix in the combine phase
constexpr int kV3oNN = kV3oYY + 16 * kV3NpMax;               // double[160 + 16]  n = y / m (zeros past the bins); G_k in the combine phase
constexpr int kV3oBANDV = kV3oNN + 8 * (kV3NpMax + 16);      // double[160]  band sums of the density targets
constexpr int kV3oHOT = kV3oBANDV + 8 * kV3NpMax;            // V3Hot: the small tables the loops index (copied from the parameters)
constexpr int kV3HotBytes = 1600;
constexpr int kV3oRUNS = kV3oHOT + kV3HotBytes;              // uint32[16][8]: the packed runs of every warp (4 column, 3 row, 1 unused)
constexpr int kV3oUNION = kV3oRUNS + 32 * kV3Warps;          // build: role vectors; evaluation: W stage, partial sums
constexpr int kV3BuildUnionBytes = 8 * 19 * kV3NpMax;
constexpr int kV3ColSlotBytes = 32 * 16;                     // (G, H) per lane
constexpr int kV3RowSlotBytes = 32 * 24;                     // deposits into bins i-1, i, i+1 (per unit n_i), [3][32]

// packed runs (one 32-bit word each; 0 = unused)
//   column run: c[0:3) k0[3:8) n[8:13) tcol[13:23) slot[23:28) diag[28] valid[31]
//   row run   : b[0:3) ja[3:11) jb[11:19) slot[19:24) valid[31]
inline uint32_t v3_pack_col(int c, int k0, int n, int tcol, int slot, int diag)
{
    return (uint32_t)c | ((uint32_t)k0 << 3) | ((uint32_t)n << 8) | ((uint32_t)tcol << 13) | ((uint32_t)slot << 23) |
           ((uint32_t)diag << 28) | 0x80000000u;
}
inline uint32_t v3_pack_row(int b, int ja, int jb, int slot)
{
    return (uint32_t)b | ((uint32_t)ja << 3) | ((uint32_t)jb << 11) | ((uint32_t)slot << 19) | 0x80000000u;
}
struct V3ColRun { int c, k0, n, tcol, slot, diag; };
struct V3RowRun { int b, ja, jb, slot; };
#if defined(__CUDACC__)
#define V3_HD __host__ __device__
#else
#define V3_HD
#endif
V3_HD inline V3ColRun v3_unpack_col(uint32_t w)
{
    V3ColRun r;
    r.c = w & 7; r.k0 = (w >> 3) & 31; r.n = (w >> 8) & 31; r.tcol = (w >> 13) & 1023; r.slot = (w >> 23) & 31;
    r.diag = (w >> 28) & 1;
    return r;
}
V3_HD inline V3RowRun v3_unpack_row(uint32_t w)
{
    V3RowRun r;
    r.b = w & 7; r.ja = (w >> 3) & 255; r.jb = (w >> 11) & 255; r.slot = (w >> 19) & 31;
    return r;
}

struct alignas(16) V3Tap {             // target t += c * W[off + t]   (off = plane, d and -o folded, in doubles)
    double c;
    int off, pad;
};

struct V3Exc {                         // exception entry: target += c * W[off]   (absolute stage index)
    double c;
    short off, t, kind, pad;           // kind 0: density target t, 1: S target t
};

struct V3ExcTarget {                   // entries [e0, e1) (at most 32) feed target t of `kind`
    short t, kind, e0, e1;
};

// The tables that loops index with a run-time subscript.  As kernel parameters such reads are indexed
// constant loads with several hundred cycles of latency each (measured), so the kernel copies this block
// to shared memory once and reads it there.
struct V3Hot {
    int rpBase[kV3MaxBlk], rpCnt[kV3MaxBlk];     // row block b: row partial slots [rpBase, + rpCnt)
    int cpBase[kV3MaxBlk], cpCnt[kV3MaxBlk];     // column block c: column partial slots
    int cmin[kV3MaxBlk];                         // columns [0, cmin[b]) are bulk for EVERY row of block b
    short nFold[kV3MaxBlk + 1];
    unsigned char foldA[kV3MaxBlk][kV3MaxFold], foldB[kV3MaxBlk][kV3MaxFold];   // diagonal block: local rows (0xff: none)
    V3Tap taps[kV3MaxTaps];            // density targets (padded to a multiple of 8 with zero coefficients)
    V3Tap staps[kV3MaxSTaps];          // S targets
    V3Exc exc[kV3MaxExc];              // sorted by (kind, t)
    V3ExcTarget excT[kV3MaxExcT];      // unused entries: t = -1
};
static_assert(sizeof(V3Hot) <= kV3HotBytes && sizeof(V3Hot) % 4 == 0, "V3Hot layout");

struct V3Tables {
    int on;                            // 0: this mass grid runs on the general kernel
    int N, nb, P, bandD;
    int wRow;                          // entries per (plane, d) row of the W stage; entry of bin i at wPad + i
    int wPad;
    int nTaps, nSTaps, nExc, nExcT;
    int nTapsR;                        // taps [0, nTapsR) go to combine group R, the rest to group D (multiples of 8)
    int nExcS;                         // exception entries of S targets (kind 1)
    int diagBulk;                      // 1: some row's bulk prefix reaches its diagonal pair (coarse grids), so the row pass
                                       //    reads diagonal pairs and a PLANAR row copy gets its diagonal halved in place
    int excLocal;                      // 1: every density exception reads stage entries of its target's own 32-bin block, so
                                       //    the warp that staged the block sums them right away (phase A)
    // shared-memory byte offsets laid out by the host (the fixed ones are kV3o*)
    int oWST, oCOLP, oROWP, oK, smemBytes;
    int oDTAB;                         // per-offset and exp tables of the pair kernel behind the row copy (0: no room, read through L1)
    int nColSlots, nRowSlots;
    uint32_t col[kV3Warps][kV3ColRuns];          // packed column runs
    uint32_t row[kV3Warps][kV3RowRuns];          // packed row runs
    V3Hot hot;
};

struct V3Host {
    V3Tables t;
    std::string why;                   // reason the grid does not take this kernel (t.on == 0)
};

// Builds the stencil, checks it against the gather entries and deals the work out.  smem_optin: device limit.
// ownerBuildCost >= 0: cost units that the bin-owning warps carry in the build phase besides their rows (default:
// the late start of the step / rates kernels); buildOnly: tables for cudisc_coag_kernel, whose build writes K to HBM
// and nothing to tensor memory (no tensor-memory capacity limit; only the build runs of the result are used).
void v3_build(const HostTables &ht, int logGrid, int smem_optin, V3Host &out, double ownerBuildCost = -1.0,
              bool buildOnly = false);

// Host-side check of the run lists and of the stencil (CPU tests, cudisc_bins_schedule_check): adds to
//   bad[0] pairs not built exactly once            bad[1] bulk pairs not in the row pass exactly once
//   bad[2] pairs not in the column pass exactly once   bad[3] tensor-memory / partial-slot / layout clashes
//   bad[4] stencil + exceptions != gather entries (evaluated on pseudo-random n, K)
void v3_check(const HostTables &ht, const V3Host &v, long long bad[6]);

}  // namespace cudisc
