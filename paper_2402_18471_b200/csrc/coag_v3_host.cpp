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
constexpr double kCBuildRow = 95.0, kCBuildFold = 120.0, kCBuildDiagCopy = 320.0;
constexpr double kCColChunk = 70.0, kCColRun = 90.0;
constexpr double kCRowRect = 24.0, kCRowRag = 32.0, kCRowRun = 110.0;
constexpr double kCTap = 50.0, kCBandTask = 150.0, kCExcTarget = 260.0;
constexpr double kCProlPiece = 700.0;     // a third of the next cell's prologue, on the bin-owning warps

struct Key {
    int kind, d, plane, o;
    bool operator<(const Key &x) const { return std::tie(kind, d, plane, o) < std::tie(x.kind, x.d, x.plane, x.o); }
};

}  // namespace

void v3_build(const HostTables &ht, int logGrid, int smem_optin, V3Host &out)
{
    V3Tables &t = out.t;
    memset(&t, 0, sizeof(t));
    out.exc.clear();
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
    if (maxd >= kV3Pad) { out.why = "band wider than the stencil padding"; return; }
    std::map<Key, double> cc;                      // class constant of the regular classes
    for (auto &kv : ratio) {
        if (kv.first.kind == 1 && kv.first.plane == 0) { out.why = "S entry on the coagulation plane"; return; }
        if (kv.second.size() < 8) continue;
        std::vector<double> v = kv.second;
        std::sort(v.begin(), v.end());
        cc[kv.first] = v[v.size() / 2];
    }
    std::map<std::pair<int, int>, V3Tap> tapmap;   // (d, o)
    for (auto &kv : cc) {
        const Key &k = kv.first;
        if (std::abs(k.o) >= kV3Pad) { out.why = "stencil offset beyond the padding"; return; }
        V3Tap &tp = tapmap[{k.d, k.o}];
        tp.d = k.d; tp.o = k.o;
        if (k.kind == 0 && k.plane == 0) tp.c0 = kv.second;
        else if (k.kind == 0) tp.c1 = kv.second;
        else tp.s1 = kv.second;
    }
    if ((int)tapmap.size() > kV3MaxTaps) { out.why = "too many stencil taps"; return; }
    // residuals: what the taps add at (kind, target, i, j, plane), against what the table says
    for (auto &kv : tapmap) {
        const V3Tap &tp = kv.second;
        for (int tg = 0; tg < N; ++tg) {
            const int i = tg - tp.o, j = i - tp.d;
            if (i < 0 || i >= N || j < 0) continue;
            if (tp.c0 != 0.0) have[{0, tg, i, j, 0}] += tp.c0 * ht.m[i];
            if (tp.c1 != 0.0) have[{0, tg, i, j, 1}] += tp.c1 * ht.m[i];
            if (tp.s1 != 0.0) have[{1, tg, i, j, 1}] += tp.s1 * ht.m[i];
        }
    }
    std::map<std::pair<int, int>, std::vector<V3Exc>> excBy;   // (kind, target)
    auto residual = [&](const std::tuple<int, int, int, int, int> &key, double w, double h) {
        const int i = std::get<2>(key);
        // coefficients are O(m_i): a difference of 1e-12 m_i is 1e-12 of the pair's own mass flux (the tables'
        // own rounding, e.g. of eps = (m_u - m) / (m_u - m_l), is of that size where eps is small)
        if (std::fabs(w - h) <= 1e-12 * ht.m[i]) return;
        V3Exc x;
        x.coef = w - h; x.i = i; x.j = std::get<3>(key); x.plane = std::get<4>(key); x.pad = 0;
        excBy[{std::get<0>(key), std::get<1>(key)}].push_back(x);
    };
    for (auto &kv : want) {
        auto it = have.find(kv.first);
        residual(kv.first, kv.second, it == have.end() ? 0.0 : it->second);
    }
    for (auto &kv : have)
        if (!want.count(kv.first)) residual(kv.first, 0.0, kv.second);
    if (excBy.size() > 8) {
        out.why = "too many targets with stencil exceptions:";
        for (auto &kv : excBy) out.why += " " + std::to_string(kv.first.first) + "/" + std::to_string(kv.first.second) + "x" + std::to_string(kv.second.size());
        return;
    }
    t.nExcT = 0;
    for (auto &kv : excBy) {
        V3ExcTarget &x = t.excT[t.nExcT++];
        x.kind = (short)kv.first.first; x.t = (short)kv.first.second;
        x.e0 = (short)out.exc.size();
        out.exc.insert(out.exc.end(), kv.second.begin(), kv.second.end());
        x.e1 = (short)out.exc.size();
    }
    t.nTaps = 0;
    for (auto &kv : tapmap) t.taps[t.nTaps++] = kv.second;     // sorted by (d, o)

    // ------------------------------------------------------------------ column chunks -> warps
    // tensor-memory columns already taken in each quarter: per-bin constants of the two combine groups
    if (2 * nb > kV3Warps) { out.why = "too many bins for the two combine groups"; return; }
    int used[4] = {0, 0, 0, 0};
    for (int w = 0; w < kV3Warps; ++w) {
        t.bincCol[w] = -1;
        if (w < nb) { t.bincCol[w] = (short)used[w & 3]; used[w & 3] += 16; }
        else if (w < 2 * nb) { t.bincCol[w] = (short)used[w & 3]; used[w & 3] += 2; }
    }
    int cap[4];
    for (int q = 0; q < 4; ++q) cap[q] = (512 - used[q]) / 32;
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
            t.foldA[c][nf] = (unsigned char)rA; t.foldB[c][nf] = (unsigned char)rB;
            ++nf;
        }
        t.nFold[c] = (short)nf;
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
    const double T = total / kV3Warps;
    std::vector<std::vector<Chunk>> mine(kV3Warps);
    double load[kV3Warps] = {0};
    int qfill[4] = {0, 0, 0, 0};
    int diagWarp[kV3MaxBlk];
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
    int tcolNext[4];
    for (int q = 0; q < 4; ++q) tcolNext[q] = used[q];
    for (int w = 0; w < kV3Warps; ++w) {
        int nr = 0;
        for (int c = 0; c < nb; ++c)
            if (diagWarp[c] == w) {
                if (nr >= kV3ColRuns) { out.why = "too many column runs on a warp"; return; }
                const int n = (std::min(32, N - 32 * c) + 7) / 8;
                V3ColRun &r = t.col[w][nr++];
                r.c = (short)c; r.k0 = 0; r.n = (short)n; r.diag = 1;
                r.tcol = (short)tcolNext[w & 3];
                tcolNext[w & 3] += 32 * n;
            }
        std::sort(mine[w].begin(), mine[w].end(), [](const Chunk &x, const Chunk &y) {
            return x.c != y.c ? x.c < y.c : x.k < y.k;
        });
        for (size_t q = 0; q < mine[w].size(); ++q) {
            const Chunk &ch = mine[w][q];
            if (nr > 0 && !t.col[w][nr - 1].diag && t.col[w][nr - 1].c == ch.c &&
                t.col[w][nr - 1].k0 + t.col[w][nr - 1].n == ch.k) {
                t.col[w][nr - 1].n++;
            } else {
                if (nr >= kV3ColRuns) { out.why = "too many column runs on a warp"; return; }
                V3ColRun &r = t.col[w][nr++];
                r.c = (short)ch.c; r.k0 = (short)ch.k; r.n = 1; r.diag = 0;
                r.tcol = (short)tcolNext[w & 3];
            }
            tcolNext[w & 3] += 32;
        }
    }
    for (int q = 0; q < 4; ++q)
        if (tcolNext[q] > 512) { out.why = "column copy exceeds tensor memory"; return; }
    {
        int slot = 0;
        for (int c = 0; c < nb; ++c) {
            t.cpBase[c] = slot;
            for (int w = 0; w < kV3Warps; ++w)
                for (int r = 0; r < kV3ColRuns; ++r)
                    if (t.col[w][r].n > 0 && t.col[w][r].c == c) t.col[w][r].slot = (short)slot++;
            t.cpCnt[c] = slot - t.cpBase[c];
        }
        t.nColSlots = slot;
    }

    // ------------------------------------------------------------------ evaluation: band taps and row columns
    double pre[kV3Warps];
    for (int w = 0; w < kV3Warps; ++w) {
        pre[w] = w < nb ? kCProlPiece : 0.0;
        for (int r = 0; r < kV3ColRuns; ++r)
            if (t.col[w][r].n > 0) pre[w] += kCColRun + kCColChunk * t.col[w][r].n;
        t.bandBlk[w] = -1; t.bandT0[w] = t.bandT1[w] = t.bandSlot[w] = 0;
    }
    {
        // two band tasks per target block (halves of the tap list), each to the least loaded free warp
        const int half = (t.nTaps + 1) / 2;
        for (int g = 0; g < nb; ++g)
            for (int h = 0; h < 2; ++h) {
                int best = -1;
                for (int w = 0; w < kV3Warps; ++w)
                    if (t.bandBlk[w] < 0 && (best < 0 || pre[w] < pre[best])) best = w;
                if (best < 0) { out.why = "no warp left for a band task"; return; }
                t.bandBlk[best] = (short)g;
                t.bandT0[best] = (short)(h ? half : 0); t.bandT1[best] = (short)(h ? t.nTaps : half);
                t.bandSlot[best] = (short)h;
                double cst = kCBandTask + kCTap * (t.bandT1[best] - t.bandT0[best]);
                if (h == 0)
                    for (int x = 0; x < t.nExcT; ++x)
                        if (t.excT[x].t / 32 == g) cst += kCExcTarget;
                pre[best] += cst;
            }
    }
    struct Col { int b, j; double cost; };
    std::vector<Col> cols;
    double rowTotal = 0.0;
    for (int b = 0; b < nb; ++b) {
        int cmin = 1 << 30, cmax = 0;
        for (int i = 32 * b; i < std::min(N, 32 * b + 32); ++i) {
            cmin = std::min(cmin, ht.n_bulk[i]); cmax = std::max(cmax, ht.n_bulk[i]);
        }
        t.cmin[b] = cmin;
        for (int j = 0; j < cmax; ++j) {
            cols.push_back({b, j, j < cmin ? kCRowRect : kCRowRag});
            rowTotal += cols.back().cost;
        }
    }
    {
        double sumPre = 0.0;
        for (int w = 0; w < kV3Warps; ++w) sumPre += pre[w];
        // water level: warps whose preload already exceeds it take no row work
        double level = (sumPre + rowTotal) / kV3Warps;
        for (int it = 0; it < 8; ++it) {
            double room = 0.0; int n = 0;
            for (int w = 0; w < kV3Warps; ++w)
                if (pre[w] < level) { room += level - pre[w]; ++n; }
            if (n == 0) break;
            level += (rowTotal + kCRowRun * n - room) / n;
        }
        size_t next = 0;
        int slotCount = 0;
        std::vector<std::vector<V3RowRun>> rr(kV3Warps);
        auto give = [&](int w, double budget) {
            while (next < cols.size() && budget > 0.0) {
                if (rr[w].empty() || rr[w].back().b != cols[next].b) {
                    if ((int)rr[w].size() >= kV3RowRuns) return;
                    V3RowRun r;
                    r.b = (short)cols[next].b; r.ja = r.jb = (short)cols[next].j; r.slot = 0;
                    rr[w].push_back(r);
                    budget -= kCRowRun;
                }
                rr[w].back().jb++;
                budget -= cols[next].cost;
                ++next;
            }
        };
        for (int w = 0; w < kV3Warps; ++w) give(w, level - pre[w]);
        for (int w = kV3Warps - 1; w >= 0 && next < cols.size(); --w) give(w, 1e30);   // rounding leftovers
        if (next < cols.size()) { out.why = "row pass does not fit the run lists"; return; }
        for (int b = 0; b < nb; ++b) {
            t.rpBase[b] = slotCount;
            for (int w = 0; w < kV3Warps; ++w)
                for (V3RowRun &r : rr[w])
                    if (r.b == b && r.jb > r.ja) r.slot = (short)slotCount++;
            t.rpCnt[b] = slotCount - t.rpBase[b];
        }
        t.nRowSlots = slotCount;
        for (int w = 0; w < kV3Warps; ++w)
            for (size_t q = 0; q < rr[w].size(); ++q) t.row[w][q] = rr[w][q];
    }

    // ------------------------------------------------------------------ shared-memory layout (bytes)
    {
        int q = 0;
        auto take = [&](int bytes) { const int o = q; q += (bytes + 15) & ~15; return o; };
        t.oYY = take(16 * (Np + 2 * kV3Pad));
        t.oNN = take(8 * (Np + 2 * kV3Pad + 8));
        t.oDTAB = take(16 * Np);
        t.oEXPT = take(8 * 64);
        t.oRED = take(8 * 128);
        t.oBAND = take(8 * 4 * Np);                 // [slot][kind][Np]
        t.oGK = take(8 * 2 * Np);                   // G_k, scanned suffix
        t.oNBULK = take(8 * Np);                   // int2 per bin: n_bulk | iS << 9, jS_lo | jS_hi << 16
        t.oUNION = q;
        const int roles = 8 * 19 * Np;
        t.oCOLP = t.oUNION;
        t.oROWP = t.oCOLP + 512 * t.nColSlots;
        const int parts = 512 * t.nColSlots + 1024 * t.nRowSlots;
        q += (std::max(roles, parts) + 15) & ~15;
        t.oK = q;
        t.smemBytes = q + 16 * P;
    }
    if (t.smemBytes > smem_optin) { out.why = "kernel of a cell does not fit shared memory"; return; }
    t.on = 1;
}

void v3_check(const HostTables &ht, const V3Host &v, long long bad[6])
{
    const V3Tables &t = v.t;
    const int N = ht.N, nb = t.nb, Np = 32 * nb;
    std::vector<int> built((size_t)N * N, 0), rowc((size_t)N * N, 0), colc((size_t)N * N, 0);
    std::vector<int> tmap(4 * 512, 0), cslot(std::max(1, t.nColSlots), 0), rslot(std::max(1, t.nRowSlots), 0);
    auto claim = [&](int q, int col, int n) {
        for (int u = col; u < col + n; ++u) {
            if (u < 0 || u >= 512 || tmap[q * 512 + u]++) ++bad[3];
        }
    };
    for (int w = 0; w < kV3Warps; ++w) {
        if (w < nb) claim(w & 3, t.bincCol[w], 16);
        else if (w < 2 * nb) claim(w & 3, t.bincCol[w], 2);
        for (int r = 0; r < kV3ColRuns; ++r) {
            const V3ColRun &run = t.col[w][r];
            if (run.n == 0) continue;
            claim(w & 3, run.tcol, 32 * run.n);
            if (run.slot < t.cpBase[run.c] || run.slot >= t.cpBase[run.c] + t.cpCnt[run.c] || cslot[run.slot]++) ++bad[3];
            // column pass: rows of the chunks x the 32 columns of the block
            for (int i = 32 * run.c + 8 * run.k0; i < std::min(N, 32 * run.c + 8 * (run.k0 + run.n)); ++i)
                for (int j = 32 * run.c; j < std::min(N, 32 * run.c + 32); ++j)
                    if (i >= j) colc[(size_t)i * N + j]++;
            if (run.diag) {
                if (run.k0 != 0 || run.n != (std::min(32, N - 32 * run.c) + 7) / 8) ++bad[0];
                for (int fi = 0; fi < t.nFold[run.c]; ++fi)
                    for (int lane = 0; lane < 32; ++lane) {
                        const int rA = t.foldA[run.c][fi], rB = t.foldB[run.c][fi];
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
            const V3RowRun &run = t.row[w][r];
            if (run.jb == run.ja) continue;
            if (run.slot < t.rpBase[run.b] || run.slot >= t.rpBase[run.b] + t.rpCnt[run.b] || rslot[run.slot]++) ++bad[3];
            for (int i = 32 * run.b; i < std::min(N, 32 * run.b + 32); ++i)
                for (int j = run.ja; j < run.jb; ++j) {
                    if (j < t.cmin[run.b] && j >= ht.n_bulk[i]) ++bad[1];      // the rectangle must be bulk
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
    if (t.oROWP + 1024 * t.nRowSlots > t.oK || t.oUNION + 8 * 19 * Np > t.oK) ++bad[3];
    // band tasks: both halves of every block, taps covered once
    for (int g = 0; g < nb; ++g) {
        std::vector<int> cov(std::max(1, t.nTaps), 0);
        int slots = 0;
        for (int w = 0; w < kV3Warps; ++w)
            if (t.bandBlk[w] == g) {
                slots |= 1 << t.bandSlot[w];
                for (int q = t.bandT0[w]; q < t.bandT1[w]; ++q) cov[q]++;
            }
        if (slots != 3) ++bad[5];
        for (int q = 0; q < t.nTaps; ++q) bad[5] += cov[q] != 1;
    }
    // stencil + exceptions against the gather entries on pseudo-random n and K
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
        for (int q = 0; q < t.nTaps; ++q)
            for (int tg = 0; tg < N; ++tg) {
                const int i = tg - t.taps[q].o, j = i - t.taps[q].d;
                if (i < 0 || i >= N || j < 0) continue;
                const double w = ht.m[i] * n[i] * n[j];
                got[tg] += w * (t.taps[q].c0 * Kc[(size_t)i * N + j] + t.taps[q].c1 * Kf[(size_t)i * N + j]);
                got[N + tg] += w * t.taps[q].s1 * Kf[(size_t)i * N + j];
            }
        for (int x = 0; x < t.nExcT; ++x)
            for (int e = t.excT[x].e0; e < t.excT[x].e1; ++e) {
                const V3Exc &ex = v.exc[e];
                got[t.excT[x].kind * N + t.excT[x].t] += ex.coef * n[ex.i] * n[ex.j] * (ex.plane ? Kf : Kc)[(size_t)ex.i * N + ex.j];
            }
        for (int q = 0; q < 2 * N; ++q)
            if (std::fabs(got[q] - ref[q]) > 1e-12 * refAbs[q]) ++bad[4];
    }
}

}  // namespace cudisc
