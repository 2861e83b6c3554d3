// coag_v3_host.cpp -- host side of the stencil cell kernel (coag_v3.h): folds the band gather entries of
// coag_tables.cpp into a shift-invariant stencil + exceptions, proves the two equal, and deals the work of
// a cell out to the 16 warps (column chunks in tensor memory, row-pass columns, band taps).
#include "coag_v3.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <tuple>

namespace cudisc {

namespace {

// cost model (cycles of one warp; measured ratios on B200, only the ratios matter)
constexpr double kCBuildRow = 95.0, kCBuildFold = 120.0, kCBuildDiagCopy = 320.0, kCBuildOwnerLate = 250.0;
constexpr double kCColChunk = 600.0, kCColRun = 150.0;
constexpr double kCRowRect = 64.0, kCRowRag = 85.0, kCRowRun = 300.0;
constexpr double kCStage = 500.0;          // band stage of 32 bins (warps of combine group D)
constexpr double kCProlPiece = 2900.0;     // a third of the next cell's prologue, on the bin-owning warps

struct Key {
    int kind, d, plane, o;
    bool operator<(const Key &x) const { return std::tie(kind, d, plane, o) < std::tie(x.kind, x.d, x.plane, x.o); }
};

}  // namespace

void v3_build(const HostTables &ht, int logGrid, int smem_optin, V3Host &out, double ownerBuildCost, bool buildOnly)
{
    // what the bin-owning warps carry in the build phase besides their rows: a late start (step / rates kernels: they
    // assemble and finish the previous cell first) or the whole prologue of the next cell (cudisc_coag_kernel)
    const double ownerLate = ownerBuildCost >= 0.0 ? ownerBuildCost : kCBuildOwnerLate;
    V3Tables &t = out.t;
    memset(&t, 0, sizeof(t));
    out.why.clear();
    const int N = ht.N, nb = (N + 31) / 32, P = N * (N + 1) / 2, Np = 32 * nb;
    if (!logGrid) { out.why = "not an exact log grid"; return; }
    if (N < 40 || nb > kV3MaxBlk) { out.why = "n_bins outside [40, 160]"; return; }
    t.N = N; t.nb = nb; t.P = P;

    // ------------------------------------------------------------------ stencil of the band entries
    // entries that share (target, i, j, plane) are summed first (equal grains lose twice)
    std::map<std::tuple<int, int, int, int, int>, double> want, have;   // (kind, target, i, j, plane)
    int maxd = 0;
    for (const BandEntry &e : ht.band) {
        const int kind = e.target >= N, tb = e.target - kind * N;
        want[{kind, tb, e.i, e.j, e.plane}] += e.coef;
        maxd = std::max(maxd, e.i - e.j);
    }
    std::map<Key, std::vector<double>> ratio;
    for (auto &kv : want) {
        const int kind = std::get<0>(kv.first), tb = std::get<1>(kv.first), i = std::get<2>(kv.first);
        ratio[{kind, i - std::get<3>(kv.first), std::get<4>(kv.first), tb - i}].push_back(kv.second / ht.m[i]);
    }
    if (maxd >= 8) { out.why = "band wider than 8 diagonals"; return; }
    std::map<Key, double> cc;                      // class constant of the regular classes
    for (auto &kv : ratio) {
        if (kv.first.kind == 1 && kv.first.plane == 0) { out.why = "S entry on the coagulation plane"; return; }
        if (kv.second.size() < 8) continue;
        std::vector<double> v = kv.second;
        std::sort(v.begin(), v.end());
        cc[kv.first] = v[v.size() / 2];
    }
    int omin = 0, omax = 0;
    for (auto &kv : cc) { omin = std::min(omin, kv.first.o); omax = std::max(omax, kv.first.o); }
    const int D = maxd + 1;
    t.bandD = D;
    t.wPad = (omax + 1) & ~1;
    t.wRow = (t.wPad + N + (-omin) + 1) & ~1;
    if (2 * D * t.wRow > 32000) { out.why = "band stage too large"; return; }
    // the kernel zeroes the padding of the stage with 16 threads per (plane, d) row
    if (t.wRow - N > 16 || 2 * D > 32 * kV3Warps / 16) { out.why = "band stage padding too wide"; return; }
    t.nTaps = t.nSTaps = 0;
    for (auto &kv : cc) {                          // sorted by (kind, d, plane, o): fixed summation order
        const Key &k = kv.first;
        V3Tap tp;
        tp.c = kv.second; tp.pad = 0;
        tp.off = (k.plane * D + k.d) * t.wRow + t.wPad - k.o;
        if (k.kind == 0) {
            if (t.nTaps >= kV3MaxTaps) { out.why = "too many stencil taps"; return; }
            t.hot.taps[t.nTaps++] = tp;
        } else {
            if (t.nSTaps >= kV3MaxSTaps) { out.why = "too many S stencil taps"; return; }
            t.hot.staps[t.nSTaps++] = tp;
        }
        // what the tap adds at (kind, target, i, j, plane)
        for (int tg = 0; tg < N; ++tg) {
            const int i = tg - k.o, j = i - k.d;
            if (i < 0 || i >= N || j < 0) continue;
            have[{k.kind, tg, i, j, k.plane}] += kv.second * ht.m[i];
        }
    }
    // residuals against the table -> exception entries (coefficient per unit W = m_i n_i n_j K)
    std::vector<V3Exc> excs;
    auto residual = [&](const std::tuple<int, int, int, int, int> &key, double w, double h) {
        const int i = std::get<2>(key), j = std::get<3>(key), plane = std::get<4>(key);
        // coefficients are O(m_i): a difference of 1e-12 m_i is 1e-12 of the pair's own mass flux (the tables'
        // own rounding, e.g. of eps = (m_u - m) / (m_u - m_l), is of that size where eps is small)
        if (std::fabs(w - h) <= 1e-12 * ht.m[i]) return;
        V3Exc x;
        x.c = (w - h) / ht.m[i];
        x.off = (short)((plane * D + (i - j)) * t.wRow + t.wPad + i);
        x.kind = (short)std::get<0>(key); x.t = (short)std::get<1>(key); x.pad = 0;
        excs.push_back(x);
    };
    for (auto &kv : want) {
        auto it = have.find(kv.first);
        residual(kv.first, kv.second, it == have.end() ? 0.0 : it->second);
    }
    for (auto &kv : have)
        if (!want.count(kv.first)) residual(kv.first, 0.0, kv.second);
    if ((int)excs.size() > kV3MaxExc) { out.why = "too many stencil exceptions (" + std::to_string(excs.size()) + ")"; return; }
    std::stable_sort(excs.begin(), excs.end(), [](const V3Exc &x, const V3Exc &y) {
        return x.kind != y.kind ? x.kind < y.kind : x.t < y.t;
    });
    t.nExc = (int)excs.size();
    for (int q = 0; q < t.nExc; ++q) t.hot.exc[q] = excs[q];
    // the kernel walks taps in batches of 8: pad with entries that add nothing
    while (t.nTaps & 7) {
        if (t.nTaps >= kV3MaxTaps) { out.why = "too many stencil taps"; return; }
        V3Tap z; z.c = 0.0; z.off = t.wPad; z.pad = 0;
        t.hot.taps[t.nTaps++] = z;
    }
    t.diagBulk = 0;
    for (int i = 0; i < N; ++i)
        if (ht.n_bulk[i] > i) t.diagBulk = 1;
    t.nTapsR = (2 * t.nTaps / 5) & ~7;
    t.nExcS = 0; t.excLocal = 1;
    for (int q = 0; q < t.nExc; ++q) {
        const V3Exc &x = t.hot.exc[q];
        if (x.kind == 1) { t.nExcS++; continue; }
        const int i = (x.off % t.wRow) - t.wPad;
        if ((i >> 5) != (x.t >> 5)) t.excLocal = 0;
    }
    // exception entries by target: one warp sums the (at most 32) entries of a target with a fixed shuffle tree
    t.nExcT = 0;
    for (int q = 0; q < kV3MaxExcT; ++q) { t.hot.excT[q].t = -1; t.hot.excT[q].kind = 0; t.hot.excT[q].e0 = t.hot.excT[q].e1 = 0; }
    for (int q = 0; q < t.nExc;) {
        int e = q;
        while (e < t.nExc && t.hot.exc[e].kind == t.hot.exc[q].kind && t.hot.exc[e].t == t.hot.exc[q].t) ++e;
        if (t.nExcT >= kV3MaxExcT || e - q > 32) { out.why = "too many stencil exception targets"; return; }
        V3ExcTarget &x = t.hot.excT[t.nExcT++];
        x.t = t.hot.exc[q].t; x.kind = t.hot.exc[q].kind; x.e0 = (short)q; x.e1 = (short)e;
        q = e;
    }

    // ------------------------------------------------------------------ column chunks -> warps
    if (3 * nb > kV3Warps) { out.why = "too many bins for the three combine groups"; return; }
    int cap[4];
    for (int q = 0; q < 4; ++q) cap[q] = buildOnly ? 1 << 20 : 512 / 32;     // (build only: nothing goes to tensor memory)
    // diagonal blocks: folded row pairs
    double diagCost[kV3MaxBlk];
    for (int c = 0; c < nb; ++c) {
        const int R = std::min(32, N - 32 * c);
        std::vector<int> left;
        for (int r = R - 1; r >= 0; --r) left.push_back(r);     // longest first
        int nf = 0;
        while (!left.empty()) {
            const int rA = left.front();
            left.erase(left.begin());
            int rB = 0xff;
            for (size_t q = 0; q < left.size(); ++q)
                if (left[q] + 1 <= 32 - (rA + 1)) { rB = left[q]; left.erase(left.begin() + q); break; }
            if (nf >= kV3MaxFold) { out.why = "diagonal block needs too many folded rows"; return; }
            t.hot.foldA[c][nf] = (unsigned char)rA; t.hot.foldB[c][nf] = (unsigned char)rB;
            ++nf;
        }
        t.hot.nFold[c] = (short)nf;
        diagCost[c] = kCBuildFold * nf + kCBuildDiagCopy * ((R + 7) / 8) / 4.0;
    }
    struct Chunk { int c, k, rows; };
    std::vector<Chunk> off;
    double total = 0.0;
    for (int c = 0; c < nb; ++c) {
        total += diagCost[c];
        const int nch = (N - 32 * c + 7) / 8;
        for (int k = 4; k < nch; ++k) {
            const int rows = std::min(8, N - (32 * c + 8 * k));
            off.push_back({c, k, rows});
            total += kCBuildRow * rows;
        }
    }
    total += ownerLate * nb;
    const double T = total / kV3Warps;
    std::vector<std::vector<Chunk>> mine(kV3Warps);
    double load[kV3Warps] = {0};
    int qfill[4] = {0, 0, 0, 0};
    int diagWarp[kV3MaxBlk];
    // the bin-owning warps join the build late: they assemble and finish the previous cell first (coag_v3.cu)
    for (int w = 0; w < nb; ++w) load[w] = ownerLate;
    for (int c = 0; c < nb; ++c) {
        const int w = kV3Warps - 1 - c;                 // away from the bin-owning warps
        diagWarp[c] = w;
        load[w] += diagCost[c];
        qfill[w & 3] += (std::min(32, N - 32 * c) + 7) / 8;
    }
    {
        size_t next = 0;
        for (int w = 0; w < kV3Warps && next < off.size(); ++w)
            while (next < off.size() && qfill[w & 3] < cap[w & 3] &&
                   load[w] + 0.5 * kCBuildRow * off[next].rows <= T) {
                mine[w].push_back(off[next]);
                load[w] += kCBuildRow * off[next].rows;
                qfill[w & 3]++;
                ++next;
            }
        for (; next < off.size(); ++next) {             // leftovers: least loaded warp with room
            int best = -1;
            for (int w = 0; w < kV3Warps; ++w)
                if (qfill[w & 3] < cap[w & 3] && (best < 0 || load[w] < load[best])) best = w;
            if (best < 0) { out.why = "column copy exceeds tensor memory"; return; }
            mine[best].push_back(off[next]);
            load[best] += kCBuildRow * off[next].rows;
            qfill[best & 3]++;
        }
    }
    // runs, tensor-memory columns, column partial slots (contiguous per column block)
    std::vector<std::vector<V3ColRun>> cr(kV3Warps);
    int tcolNext[4] = {0, 0, 0, 0};
    for (int w = 0; w < kV3Warps; ++w) {
        for (int c = 0; c < nb; ++c)
            if (diagWarp[c] == w) {
                const int n = (std::min(32, N - 32 * c) + 7) / 8;
                cr[w].push_back({c, 0, n, buildOnly ? 0 : tcolNext[w & 3], 0, 1});
                tcolNext[w & 3] += 32 * n;
            }
        std::sort(mine[w].begin(), mine[w].end(), [](const Chunk &x, const Chunk &y) {
            return x.c != y.c ? x.c < y.c : x.k < y.k;
        });
        for (const Chunk &ch : mine[w]) {
            if (!cr[w].empty() && !cr[w].back().diag && cr[w].back().c == ch.c && cr[w].back().k0 + cr[w].back().n == ch.k)
                cr[w].back().n++;
            else
                cr[w].push_back({ch.c, ch.k, 1, buildOnly ? 0 : tcolNext[w & 3], 0, 0});
            tcolNext[w & 3] += 32;
        }
        if ((int)cr[w].size() > kV3ColRuns) { out.why = "too many column runs on a warp"; return; }
    }
    for (int q = 0; q < 4; ++q)
        if (!buildOnly && tcolNext[q] > 512) { out.why = "column copy exceeds tensor memory"; return; }
    {
        int slot = 0;
        for (int c = 0; c < nb; ++c) {
            t.hot.cpBase[c] = slot;
            for (int w = 0; w < kV3Warps; ++w)
                for (V3ColRun &r : cr[w])
                    if (r.c == c) r.slot = slot++;
            t.hot.cpCnt[c] = slot - t.hot.cpBase[c];
        }
        t.nColSlots = slot;
        if (slot > 32) { out.why = "too many column partial slots"; return; }
    }
    for (int w = 0; w < kV3Warps; ++w)
        for (size_t q = 0; q < cr[w].size(); ++q)
            t.col[w][q] = v3_pack_col(cr[w][q].c, cr[w][q].k0, cr[w][q].n, cr[w][q].tcol, cr[w][q].slot, cr[w][q].diag);

    // ------------------------------------------------------------------ evaluation: row columns
    double pre[kV3Warps];
    for (int w = 0; w < kV3Warps; ++w) {
        pre[w] = w < nb ? kCProlPiece + kCStage : 0.0;
        for (const V3ColRun &r : cr[w]) pre[w] += kCColRun + kCColChunk * r.n;
    }
    struct Col { int b, j; double cost; };
    std::vector<Col> cols;
    double rowTotal = 0.0;
    for (int b = 0; b < nb; ++b) {
        int cmin = 1 << 30, cmax = 0;
        for (int i = 32 * b; i < std::min(N, 32 * b + 32); ++i) {
            cmin = std::min(cmin, ht.n_bulk[i]); cmax = std::max(cmax, ht.n_bulk[i]);
        }
        t.hot.cmin[b] = cmin;
        for (int j = 0; j < cmax; ++j) {
            cols.push_back({b, j, j < cmin ? kCRowRect : kCRowRag});
            rowTotal += cols.back().cost;
        }
    }
    {
        // water level L with sum_w max(0, L - pre[w] - run overhead) = row work (bisection)
        double lo = 0.0, hi = 0.0;
        for (int w = 0; w < kV3Warps; ++w) hi = std::max(hi, pre[w]);
        hi += rowTotal + kCRowRun;
        for (int it = 0; it < 60; ++it) {
            const double L = 0.5 * (lo + hi);
            double room = 0.0;
            for (int w = 0; w < kV3Warps; ++w) room += std::max(0.0, L - pre[w] - kCRowRun);
            (room < rowTotal ? lo : hi) = L;
        }
        const double level = hi;
        size_t next = 0;
        std::vector<std::vector<V3RowRun>> rr(kV3Warps);
        auto left_in_block = [&](size_t q) {            // columns of cols[q]'s block from q on
            size_t e = q;
            while (e < cols.size() && cols[e].b == cols[q].b) ++e;
            return (int)(e - q);
        };
        auto give = [&](int w, double budget) {
            while (next < cols.size()) {
                const bool same = !rr[w].empty() && rr[w].back().b == cols[next].b;
                if (budget <= 0.0 && !(same && left_in_block(next) <= 5)) break;    // a short block tail stays with its run
                if (!same) {
                    if ((int)rr[w].size() >= kV3RowRuns) return;
                    if (budget < 8.0 * cols[next].cost + (rr[w].empty() ? 0.0 : kCRowRun)) return;   // not worth a run
                    rr[w].push_back({cols[next].b, cols[next].j, cols[next].j, 0});
                    if (rr[w].size() > 1) budget -= kCRowRun;
                }
                rr[w].back().jb++;
                budget -= cols[next].cost;
                ++next;
            }
        };
        for (int w = 0; w < kV3Warps; ++w) give(w, level - pre[w] - kCRowRun);
        for (int w = kV3Warps - 1; w >= 0 && next < cols.size(); --w) give(w, 1e30);   // rounding leftovers
        if (next < cols.size()) { out.why = "row pass does not fit the run lists"; return; }
        int slotCount = 0;
        for (int b = 0; b < nb; ++b) {
            t.hot.rpBase[b] = slotCount;
            for (int w = 0; w < kV3Warps; ++w)
                for (V3RowRun &r : rr[w])
                    if (r.b == b && r.jb > r.ja) r.slot = slotCount++;
            t.hot.rpCnt[b] = slotCount - t.hot.rpBase[b];
        }
        t.nRowSlots = slotCount;
        if (slotCount > 32) { out.why = "too many row partial slots"; return; }
        for (int w = 0; w < kV3Warps; ++w)
            for (size_t q = 0; q < rr[w].size(); ++q)
                if (rr[w][q].jb > rr[w][q].ja) t.row[w][q] = v3_pack_row(rr[w][q].b, rr[w][q].ja, rr[w][q].jb, rr[w][q].slot);
    }

    // ------------------------------------------------------------------ shared-memory layout (bytes)
    {
        const int wst = 8 * 2 * D * t.wRow;
        t.oWST = kV3oUNION;
        t.oCOLP = t.oWST + ((wst + 15) & ~15);
        t.oROWP = t.oCOLP + kV3ColSlotBytes * t.nColSlots;
        const int evalBytes = t.oROWP + kV3RowSlotBytes * t.nRowSlots - kV3oUNION;
        t.oK = kV3oUNION + ((std::max(kV3BuildUnionBytes, evalBytes) + 15) & ~15);
        t.smemBytes = t.oK + 16 * P;
        t.oDTAB = 0;
        if (t.smemBytes + 16 * N + 512 <= smem_optin) { t.oDTAB = t.smemBytes; t.smemBytes += 16 * N + 512; }   // + exp table
    }
    if (t.smemBytes > smem_optin) { out.why = "kernel of a cell does not fit shared memory"; return; }
    t.on = 1;
}

void v3_check(const HostTables &ht, const V3Host &v, long long bad[6])
{
    const V3Tables &t = v.t;
    const int N = ht.N, nb = t.nb, D = t.bandD;
    std::vector<int> built((size_t)N * N, 0), rowc((size_t)N * N, 0), colc((size_t)N * N, 0);
    std::vector<int> tmap(4 * 512, 0), cslot(std::max(1, t.nColSlots), 0), rslot(std::max(1, t.nRowSlots), 0);
    auto claim = [&](int q, int col, int n) {
        for (int u = col; u < col + n; ++u) {
            if (u < 0 || u >= 512 || tmap[q * 512 + u]++) ++bad[3];
        }
    };
    for (int w = 0; w < kV3Warps; ++w) {
        for (int r = 0; r < kV3ColRuns; ++r) {
            if (!t.col[w][r]) continue;
            const V3ColRun run = v3_unpack_col(t.col[w][r]);          // the decode the device uses
            if (run.n == 0) { ++bad[3]; continue; }
            claim(w & 3, run.tcol, 32 * run.n);
            if (run.slot < t.hot.cpBase[run.c] || run.slot >= t.hot.cpBase[run.c] + t.hot.cpCnt[run.c] || cslot[run.slot]++) ++bad[3];
            // column pass: rows of the chunks x the 32 columns of the block
            for (int i = 32 * run.c + 8 * run.k0; i < std::min(N, 32 * run.c + 8 * (run.k0 + run.n)); ++i)
                for (int j = 32 * run.c; j < std::min(N, 32 * run.c + 32); ++j)
                    if (i >= j) colc[(size_t)i * N + j]++;
            if (run.diag) {
                if (run.k0 != 0 || run.n != (std::min(32, N - 32 * run.c) + 7) / 8) ++bad[0];
                for (int fi = 0; fi < t.hot.nFold[run.c]; ++fi)
                    for (int lane = 0; lane < 32; ++lane) {
                        const int rA = t.hot.foldA[run.c][fi], rB = t.hot.foldB[run.c][fi];
                        int r2, q;
                        if (lane <= rA) { r2 = rA; q = lane; }
                        else if (rB != 0xff && lane - rA - 1 <= rB) { r2 = rB; q = lane - rA - 1; }
                        else continue;
                        const int i = 32 * run.c + r2, j = 32 * run.c + q;
                        if (i >= N || j > i) { ++bad[0]; continue; }
                        built[(size_t)i * N + j]++;
                    }
            } else {
                if (run.k0 < 4) ++bad[0];
                for (int i = 32 * run.c + 8 * run.k0; i < std::min(N, 32 * run.c + 8 * (run.k0 + run.n)); ++i)
                    for (int j = 32 * run.c; j < 32 * run.c + 32; ++j) {
                        if (j >= N || j >= i) { ++bad[0]; continue; }
                        built[(size_t)i * N + j]++;
                    }
            }
        }
        for (int r = 0; r < kV3RowRuns; ++r) {
            if (!t.row[w][r]) continue;
            const V3RowRun run = v3_unpack_row(t.row[w][r]);
            if (run.jb <= run.ja) { ++bad[3]; continue; }
            if (run.slot < t.hot.rpBase[run.b] || run.slot >= t.hot.rpBase[run.b] + t.hot.rpCnt[run.b] || rslot[run.slot]++) ++bad[3];
            for (int i = 32 * run.b; i < std::min(N, 32 * run.b + 32); ++i)
                for (int j = run.ja; j < run.jb; ++j) {
                    if (j < t.hot.cmin[run.b] && j >= ht.n_bulk[i]) ++bad[1];      // the rectangle must be bulk
                    if (j < ht.n_bulk[i]) rowc[(size_t)i * N + j]++;
                }
        }
    }
    for (int p = 0; p < t.nColSlots; ++p) bad[3] += cslot[p] != 1;
    for (int p = 0; p < t.nRowSlots; ++p) bad[3] += rslot[p] != 1;
    for (int i = 0; i < N; ++i)
        for (int j = 0; j <= i; ++j) {
            bad[0] += built[(size_t)i * N + j] != 1;
            bad[1] += rowc[(size_t)i * N + j] != (j < ht.n_bulk[i] ? 1 : 0);
            bad[2] += colc[(size_t)i * N + j] != 1;
        }
    // layout: stage, slots and role vectors below the row copy; the band pairs are all inside the stage
    if (t.oWST != kV3oUNION || t.oCOLP < t.oWST + 8 * 2 * D * t.wRow || t.oROWP != t.oCOLP + kV3ColSlotBytes * t.nColSlots ||
        t.oROWP + kV3RowSlotBytes * t.nRowSlots > t.oK || kV3oUNION + kV3BuildUnionBytes > t.oK ||
        t.smemBytes != t.oK + 16 * t.P + (t.oDTAB ? 16 * N + 512 : 0) || (t.oDTAB && t.oDTAB != t.oK + 16 * t.P)) ++bad[3];
    for (int i = 0; i < N; ++i)
        for (int j = ht.n_bulk[i]; j <= i; ++j)
            if (i - j >= D) ++bad[4];
    // stencil + exceptions against the gather entries on pseudo-random n and K, through the stage layout
    {
        std::vector<double> n(N), Kc((size_t)N * N), Kf((size_t)N * N);
        unsigned long long sd = 88172645463325252ull;
        auto rnd = [&]() { sd ^= sd << 13; sd ^= sd >> 7; sd ^= sd << 17; return 0.5 + (double)(sd >> 11) / 9007199254740992.0; };
        for (int i = 0; i < N; ++i) n[i] = rnd() / ht.m[i];
        for (size_t q = 0; q < Kc.size(); ++q) { Kc[q] = rnd(); Kf[q] = rnd(); }
        std::vector<double> ref(2 * N, 0.0), refAbs(2 * N, 0.0), got(2 * N, 0.0);
        for (const BandEntry &e : ht.band) {
            const double x = e.coef * n[e.i] * n[e.j] * (e.plane ? Kf : Kc)[(size_t)e.i * N + e.j];
            ref[e.target] += x; refAbs[e.target] += std::fabs(x);
        }
        std::vector<double> W((size_t)2 * D * t.wRow, 0.0);
        for (int p = 0; p < 2; ++p)
            for (int d = 0; d < D; ++d)
                for (int i = d; i < N; ++i)
                    W[(size_t)(p * D + d) * t.wRow + t.wPad + i] = ht.m[i] * n[i] * n[i - d] * (p ? Kf : Kc)[(size_t)i * N + i - d];
        auto at = [&](long idx) -> double {
            if (idx < 0 || idx >= (long)W.size()) { ++bad[4]; return 0.0; }
            return W[(size_t)idx];
        };
        for (int tg = 0; tg < N; ++tg) {
            for (int q = 0; q < t.nTaps; ++q) got[tg] += t.hot.taps[q].c * at((long)t.hot.taps[q].off + tg);
            for (int q = 0; q < t.nSTaps; ++q) got[N + tg] += t.hot.staps[q].c * at((long)t.hot.staps[q].off + tg);
        }
        for (int q = 0; q < t.nExc; ++q) {
            if (t.hot.exc[q].t < 0 || t.hot.exc[q].t >= N) { ++bad[4]; continue; }
            got[t.hot.exc[q].kind * N + t.hot.exc[q].t] += t.hot.exc[q].c * at(t.hot.exc[q].off);
        }
        for (int q = 0; q < 2 * N; ++q)
            if (std::fabs(got[q] - ref[q]) > 1e-12 * refAbs[q]) ++bad[4];
        // every exception entry inside exactly one target range of its own (kind, t)
        std::vector<int> cov(std::max(1, t.nExc), 0);
        for (int x = 0; x < t.nExcT; ++x)
            for (int e = t.hot.excT[x].e0; e < t.hot.excT[x].e1; ++e) {
                if (e < 0 || e >= t.nExc || t.hot.exc[e].t != t.hot.excT[x].t || t.hot.exc[e].kind != t.hot.excT[x].kind) { ++bad[4]; continue; }
                cov[e]++;
            }
        for (int e = 0; e < t.nExc; ++e) bad[4] += cov[e] != 1;
    }
}

}  // namespace cudisc
