#include "gp_schedule.h"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <functional>
#include <queue>

namespace gpb {
namespace {

struct Shape {
    int M, Mm, nbt, NB, NBm;
    bool predict;
    // block id spaces: L [0, NB*NB), V [offV, offV + NBm*NB), S [offS, ...)
    int64_t offV, offS, nblocks;
    Shape(int M_, int Mm_, int nbt_, bool predict_) : M(M_), Mm(Mm_), nbt(nbt_), predict(predict_) {
        NB = M * nbt;
        NBm = Mm * nbt;
        offV = (int64_t)NB * NB;
        offS = offV + (int64_t)NBm * NB;
        nblocks = offS + (int64_t)NBm * NBm;
    }
    int64_t idL(int gr, int gc) const { return (int64_t)gr * NB + gc; }
    int64_t idV(int gr, int gc) const { return offV + (int64_t)gr * NB + gc; }
    int64_t idS(int gr, int gc) const { return offS + (int64_t)gr * NBm + gc; }
    int finL(int gr, int gc) const {
        const int K = gc / nbt, bk = gc % nbt;
        return (gr / nbt == K) ? K + 1 + bk : K + 1 + (bk > 0 ? 1 : 0);
    }
    int finV(int gc) const { return gc / nbt + 1 + (gc % nbt > 0 ? 1 : 0); }
};

// versions an UPD item adds to its output block: one per tile column it covers (at least one)
inline int upd_versions(int q0, int q1, int nbt) { return (q1 - q0) / nbt > 1 ? (q1 - q0) / nbt : 1; }

// The waits and writes of an item, mirroring gp_exec.cuh exactly.
template <class FW, class FR>
void item_effects(const Shape& s, const SchedItem& it, FW&& wait, FR&& write) {
    const int gr = (int)it.gr, gc = (int)it.gc, q0 = (int)(it.q & 0xffffu), q1 = (int)(it.q >> 16);
    const int nbt = s.nbt;
    switch (it.op) {
        case S_UPD_L:
            wait(s.idL(gr, gc), q0 / nbt + q0 % nbt);
            for (int q = q0; q < q1; ++q) { wait(s.idL(gr, q), s.finL(gr, q)); wait(s.idL(gc, q), s.finL(gc, q)); }
            // an update that spans several tile columns (merged SYRK/GEMM tile tasks) counts as one version per column
            for (int c = 0; c < upd_versions(q0, q1, nbt); ++c) write(s.idL(gr, gc));
            break;
        case S_TRSM_L:
            wait(s.idL(gr, gc), s.finL(gr, gc) - 1);
            wait(s.idL(gc, gc), s.finL(gc, gc));
            write(s.idL(gr, gc));
            break;
        case S_POTRF:
            wait(s.idL(gc, gc), s.finL(gc, gc) - 1);
            write(s.idL(gc, gc));
            break;
        case S_ROW_L:
            for (int jj = 0; jj < nbt; ++jj) {
                wait(s.idL(gr, gc + jj), gc / nbt);
                wait(s.idL(gc + jj, gc + jj), s.finL(gc + jj, gc + jj));
            }
            for (int jj = 0; jj < nbt; ++jj) {
                if (jj > 0) write(s.idL(gr, gc + jj));
                write(s.idL(gr, gc + jj));
            }
            break;
        case S_UPD_V:
            wait(s.idV(gr, gc), q0 / nbt);
            for (int q = q0; q < q1; ++q) wait(s.idV(gr, q), s.finV(q));
            for (int c = 0; c < upd_versions(q0, q1, nbt); ++c) write(s.idV(gr, gc));
            break;
        case S_ROW_V:
            for (int jj = 0; jj < nbt; ++jj) wait(s.idV(gr, gc + jj), gc / nbt);
            for (int jj = 0; jj < nbt; ++jj) {
                if (jj > 0) write(s.idV(gr, gc + jj));
                write(s.idV(gr, gc + jj));
            }
            break;
        case S_UPD_S:
            wait(s.idS(gr, gc), q0 / nbt);
            for (int q = q0; q < q1; ++q) { wait(s.idV(gr, q), s.finV(q)); wait(s.idV(gc, q), s.finV(q)); }
            for (int c = 0; c < upd_versions(q0, q1, nbt); ++c) write(s.idS(gr, gc));
            break;
        default: break;
    }
}

// cost model in microseconds (B200, FP64 DMMA path; only the ratios matter)
struct Cost {
    double per_q, fixed, potrf;
    explicit Cost(int blk) {
        if (blk >= 128) { per_q = 17.6; fixed = 2.5; potrf = 40.0; }     // potrf: the r02 diagonal block (38 us measured)
        else if (blk >= 64) { per_q = 2.6; fixed = 3.0; potrf = 16.0; }     // per_q: n = 8192 runs at <= 3.05 us per 64^3 product all in
        else { per_q = 0.8; fixed = 2.5; potrf = 7.0; }
    }
    double of(const SchedItem& it, int nbt) const {
        const int q0 = (int)(it.q & 0xffffu), q1 = (int)(it.q >> 16);
        switch (it.op) {
            case S_UPD_L: case S_UPD_V: case S_UPD_S: return fixed + per_q * (q1 - q0);
            case S_TRSM_L: return fixed + per_q;
            case S_POTRF: return potrf;
            case S_ROW_L: case S_ROW_V: {
                double c = 0.0;
                for (int jj = 0; jj < nbt; ++jj) c += (jj > 0 ? fixed + per_q * jj : 0.0) + fixed + per_q;
                return c;
            }
            default: return 1.0;
        }
    }
};

inline SchedItem mk(uint32_t op, int gr, int gc, int q0 = 0, int q1 = 0) {
    SchedItem it;
    it.op = op; it.gr = (uint32_t)gr; it.gc = (uint32_t)gc; it.q = (uint32_t)q0 | ((uint32_t)q1 << 16);
    return it;
}

// `task` receives, per item, the index of the paper's tile task it belongs to:
// the scheduler keeps the block items of one tile task together so that they share operand panels in L2.
constexpr int kMergeTail = 2;

constexpr int kMergeColumns = 4;     // tile columns per trailing-update item (1..4 measured in round 1: 33.9 / 34.2 / 34.4 / 34.5
                                     // TFLOP/s at n = 32768; more than 4 gains nothing).  A constant of the build, not a run-time knob.
constexpr int merge_columns() { return kMergeColumns; }

void program_order_cholesky(int M, int nbt, std::vector<SchedItem>& v, std::vector<int32_t>& task) {
    int32_t tid = 0;
    const int merge = merge_columns();
    auto emit = [&](const SchedItem& it) { v.push_back(it); task.push_back(tid); };
    for (int J = 0; J < M; ++J) {
        const int qt = J * nbt;
        // POTRF tile task = right-looking block Cholesky of the diagonal tile; its items are
        // on the critical path and are scheduled one by one
        for (int jj = 0; jj < nbt; ++jj) {
            emit(mk(S_POTRF, qt + jj, qt + jj)); ++tid;
            for (int ii = jj + 1; ii < nbt; ++ii) { emit(mk(S_TRSM_L, qt + ii, qt + jj)); ++tid; }
            for (int kk = jj + 1; kk < nbt; ++kk)
                for (int ii = kk; ii < nbt; ++ii) { emit(mk(S_UPD_L, qt + ii, qt + kk, qt + jj, qt + jj + 1)); ++tid; }
        }
        // TRSM tile tasks: one chain per block row
        for (int I = J + 1; I < M; ++I) {
            for (int bi = 0; bi < nbt; ++bi) emit(mk(S_ROW_L, I * nbt + bi, qt));
            ++tid;
        }
        // SYRK and GEMM tile tasks.  The updates of tile (I,K) by the tile columns
        // 0..K-1 are the paper's K separate tile tasks; here consecutive columns are MERGED in groups of
        // `merge` into one work item per block (contraction depth merge * t), except the last kMergeTail
        // columns, which gate the panel of step K and stay single.  A group is emitted in the step of its last
        // column.  Same arithmetic in the same order per block; half the C traffic and half the per-item
        // prologue/epilogue (the contraction path alone runs 34.9 TFLOP/s at depth 1024, 35.7 at 4096).
        for (int K = J + 1; K < M; ++K) {
            int c0 = J, c1 = J;                                  // group of columns [c0, c1] that ends at this step, if any
            const int nmerge = K - kMergeTail;                   // columns 0 .. nmerge-1 are merged
            if (merge > 1 && J < nmerge) {
                const int g0 = (J / merge) * merge, g1 = std::min(g0 + merge - 1, nmerge - 1);
                if (J != g1) continue;                           // this column waits for the end of its group
                c0 = g0; c1 = g1;
            }
            for (int I = K; I < M; ++I) {
                for (int bk = 0; bk < nbt; ++bk)
                    for (int bi = (I == K ? bk : 0); bi < nbt; ++bi)
                        emit(mk(S_UPD_L, I * nbt + bi, K * nbt + bk, c0 * nbt, (c1 + 1) * nbt));
                ++tid;
            }
        }
    }
}

void program_order_predict(int M, int Mm, int nbt, bool with_sigma, std::vector<SchedItem>& v, std::vector<int32_t>& task) {
    int32_t tid = 0;
    const int merge = merge_columns();
    auto emit = [&](const SchedItem& it) { v.push_back(it); task.push_back(tid); };
    for (int J = 0; J < M; ++J) {
        const int qt = J * nbt;
        for (int A = 0; A < Mm; ++A) {                                                            // V^T_{A,J} = (..) L_JJ^-T
            for (int ba = 0; ba < nbt; ++ba) emit(mk(S_ROW_V, A * nbt + ba, qt));
            ++tid;
        }
        // V^T_{A,P} -= V^T_{A,J} L_{P,J}^T: consecutive tile columns J merged as in the factorisation, the last
        // kMergeTail columns before P (which gate the solve of column P) stay single
        for (int P = J + 1; P < M; ++P) {
            int c0 = J, c1 = J;
            const int nmerge = P - kMergeTail;
            if (merge > 1 && J < nmerge) {
                const int g0 = (J / merge) * merge, g1 = std::min(g0 + merge - 1, nmerge - 1);
                if (J != g1) continue;
                c0 = g0; c1 = g1;
            }
            for (int A = 0; A < Mm; ++A) {
                for (int bk = 0; bk < nbt; ++bk)
                    for (int ba = 0; ba < nbt; ++ba) emit(mk(S_UPD_V, A * nbt + ba, P * nbt + bk, c0 * nbt, (c1 + 1) * nbt));
                ++tid;
            }
        }
        if (!with_sigma) continue;                                                                // variances only: no W
        // Sigma_{A,B} -= V^T_{A,J} V^T_{B,J}^T: every group of `merge` columns in one item (nothing waits for Sigma)
        {
            const int g0 = (J / merge) * merge, g1 = std::min(g0 + merge - 1, M - 1);
            if (J != g1) continue;
            for (int B = 0; B < Mm; ++B)
                for (int A = B; A < Mm; ++A) {
                    for (int bb = 0; bb < nbt; ++bb)
                        for (int ba = (A == B ? bb : 0); ba < nbt; ++ba)
                            emit(mk(S_UPD_S, A * nbt + ba, B * nbt + bb, g0 * nbt, (g1 + 1) * nbt));
                    ++tid;
                }
        }
    }
}

// `base`: versions every block already carries when the program starts (0 for a whole factorisation; J for the panel
// step of tile column J, whose blocks have received J trailing updates from outside the executor).
void schedule(const Shape& s, std::vector<SchedItem>& prog, const std::vector<int32_t>& task, int workers, int blk,
              std::vector<SchedItem>& out, SchedStats* stats, bool simulate, int base = 0) {
    const int N = (int)prog.size();
    if (!simulate || N == 0) { out = prog; return; }
    const Cost cost(blk);
    // 1. writers of every block version
    std::vector<int32_t> wcount(s.nblocks + 1, 0);
    for (int i = 0; i < N; ++i) item_effects(s, prog[i], [](int64_t, int) {}, [&](int64_t b) { ++wcount[b + 1]; });
    for (int64_t b = 0; b < s.nblocks; ++b) wcount[b + 1] += wcount[b];
    std::vector<int32_t> writer(wcount[s.nblocks]);
    {
        std::vector<int32_t> fill(wcount.begin(), wcount.end() - 1);
        for (int i = 0; i < N; ++i) item_effects(s, prog[i], [](int64_t, int) {}, [&](int64_t b) { writer[fill[b]++] = i; });
    }
    // 2. dependency lists (CSR), deduplicated
    std::vector<int64_t> dep_off(N + 1, 0);
    std::vector<int32_t> deps;
    deps.reserve((size_t)N * 4);
    std::vector<int32_t> tmp;
    for (int i = 0; i < N; ++i) {
        tmp.clear();
        item_effects(s, prog[i],
                     [&](int64_t b, int need) {
                         if (need - base > 0) {
                             const int32_t w = writer[wcount[b] + need - base - 1];
                             if (w != i) tmp.push_back(w);
                         }
                     },
                     [](int64_t) {});
        std::sort(tmp.begin(), tmp.end());
        tmp.erase(std::unique(tmp.begin(), tmp.end()), tmp.end());
        deps.insert(deps.end(), tmp.begin(), tmp.end());
        dep_off[i + 1] = (int64_t)deps.size();
    }
    // 3. bottom levels (critical path to the end) in reverse program order
    std::vector<float> dur(N), bottom(N);
    double work = 0.0;
    for (int i = 0; i < N; ++i) { dur[i] = (float)cost.of(prog[i], s.nbt); bottom[i] = dur[i]; work += dur[i]; }
    for (int i = N - 1; i >= 0; --i)
        for (int64_t e = dep_off[i]; e < dep_off[i + 1]; ++e) {
            const int d = deps[e];
            bottom[d] = std::max(bottom[d], dur[d] + bottom[i]);
        }
    // successor CSR
    std::vector<int64_t> suc_off(N + 1, 0);
    for (int64_t e = 0; e < (int64_t)deps.size(); ++e) ++suc_off[deps[e] + 1];
    for (int i = 0; i < N; ++i) suc_off[i + 1] += suc_off[i];
    std::vector<int32_t> sucs(deps.size());
    {
        std::vector<int64_t> fill(suc_off.begin(), suc_off.end() - 1);
        for (int i = 0; i < N; ++i)
            for (int64_t e = dep_off[i]; e < dep_off[i + 1]; ++e) sucs[fill[deps[e]]++] = i;
    }
    // 4. list scheduling.  Priority = the critical-path length of the item's TILE TASK (the maximum over
    // its block items), ties by program order: ready items of one tile task leave the queue together,
    // so the ~148 items in flight belong to two or three tile tasks and share their operand panels in L2
    // (ordering single items by their own bottom level interleaves dozens of tile tasks: 572 GB of DRAM
    // traffic per factorisation at n = 32768 instead of ~150 GB, profiles/r01b).
    std::vector<float> prio(N);
    {
        const int32_t ntask = N > 0 ? task[N - 1] + 1 : 0;
        std::vector<float> tmax(ntask, 0.f);
        for (int i = 0; i < N; ++i) tmax[task[i]] = std::max(tmax[task[i]], bottom[i]);
        for (int i = 0; i < N; ++i) prio[i] = tmax[task[i]];
    }
    std::vector<int32_t> missing(N);
    using PR = std::pair<float, int32_t>;                       // (task priority, -item) max-heap
    std::priority_queue<PR> ready;
    for (int i = 0; i < N; ++i) {
        missing[i] = (int32_t)(dep_off[i + 1] - dep_off[i]);
        if (missing[i] == 0) ready.push(PR(prio[i], -i));
    }
    using EV = std::pair<double, int32_t>;                      // (finish time, item) min-heap
    std::priority_queue<EV, std::vector<EV>, std::greater<EV>> running;
    out.clear();
    out.reserve(N);
    int idle = workers;
    double now = 0.0, makespan = 0.0;
    while ((int)out.size() < N) {
        while (idle > 0 && !ready.empty()) {
            const int i = -ready.top().second;
            ready.pop();
            out.push_back(prog[i]);
            running.push(EV(now + dur[i], i));
            --idle;
        }
        if (running.empty()) break;   // cannot happen for a valid DAG
        // advance to the next completion (and everything finishing at the same instant)
        now = running.top().first;
        while (!running.empty() && running.top().first <= now) {
            const int i = running.top().second;
            running.pop();
            ++idle;
            for (int64_t e = suc_off[i]; e < suc_off[i + 1]; ++e) {
                const int sc = sucs[e];
                if (--missing[sc] == 0) ready.push(PR(prio[sc], -sc));
            }
        }
        makespan = now;
    }
    while (!running.empty()) { makespan = std::max(makespan, running.top().first); running.pop(); }
    if (stats) {
        stats->makespan_us = makespan;
        stats->work_us = work;
        stats->edges = (int64_t)deps.size();
        float cp = 0.f;
        for (int i = 0; i < N; ++i) cp = std::max(cp, bottom[i]);
        stats->critical_path_us = cp;
    }
}

}  // namespace

void build_cholesky_schedule(int M, int nbt, int workers, std::vector<SchedItem>& out, int blk, SchedStats* stats, bool simulate) {
    std::vector<SchedItem> prog;
    std::vector<int32_t> task;
    program_order_cholesky(M, nbt, prog, task);
    schedule(Shape(M, 0, nbt, false), prog, task, workers, blk, out, stats, simulate);
}

// The FP64 part of step J of the factorisation alone (gp_cholesky_tiled_mixed): the POTRF tile task of the diagonal
// tile (J, J) and the TRSM tile tasks of the tiles below it, for blocks that already carry J versions.
void build_panel_schedule(int M, int nbt, int J, int workers, std::vector<SchedItem>& out, int blk, SchedStats* stats) {
    std::vector<SchedItem> prog;
    std::vector<int32_t> task;
    int32_t tid = 0;
    auto emit = [&](const SchedItem& it) { prog.push_back(it); task.push_back(tid); };
    const int qt = J * nbt;
    for (int jj = 0; jj < nbt; ++jj) {
        emit(mk(S_POTRF, qt + jj, qt + jj)); ++tid;
        for (int ii = jj + 1; ii < nbt; ++ii) { emit(mk(S_TRSM_L, qt + ii, qt + jj)); ++tid; }
        for (int kk = jj + 1; kk < nbt; ++kk)
            for (int ii = kk; ii < nbt; ++ii) { emit(mk(S_UPD_L, qt + ii, qt + kk, qt + jj, qt + jj + 1)); ++tid; }
    }
    // The TRSM tile tasks below the diagonal tile.  Inside the whole factorisation they are one chain per block row
    // (S_ROW_L), and the trailing updates of other columns fill the gaps; here the panel is ALONE on the chip, and
    // (M - J - 1) nbt chains of ~0.6 ms on 148 workers leave up to half of them idle in the last wave (panel 0 of
    // n = 32768: 248 chains, 1.9 ms for 1.0 ms of work).  So a block row is emitted left-looking block by block:
    // L(r, q) = (K(r, q) - sum_{p<q} L(r, p) L(q, p)^T) inv(L(q, q))^T as one update item and one solve item, same
    // arithmetic and order as the chain, same version counts.
    for (int I = J + 1; I < M; ++I) {
        for (int bi = 0; bi < nbt; ++bi) {
            const int r = I * nbt + bi;
            for (int jj = 0; jj < nbt; ++jj) {
                if (jj > 0) emit(mk(S_UPD_L, r, qt + jj, qt, qt + jj));
                emit(mk(S_TRSM_L, r, qt + jj));
            }
        }
        ++tid;
    }
    schedule(Shape(M, 0, nbt, false), prog, task, workers, blk, out, stats, true, J);
}

bool validate_panel_schedule(const std::vector<SchedItem>& items, int M, int nbt, int J) {
    const Shape s(M, 0, nbt, false);
    std::vector<int32_t> ver(s.nblocks, 0);
    for (int gr = J * nbt; gr < s.NB; ++gr)
        for (int gc = J * nbt; gc < (J + 1) * nbt && gc <= gr; ++gc) ver[s.idL(gr, gc)] = J;
    bool ok = true;
    for (const SchedItem& it : items) {
        item_effects(s, it, [&](int64_t b, int need) { if (ver[b] < need) ok = false; }, [&](int64_t b) { ++ver[b]; });
        if (!ok) return false;
    }
    for (int gr = J * nbt; gr < s.NB; ++gr)
        for (int gc = J * nbt; gc < (J + 1) * nbt && gc <= gr; ++gc)
            if (ver[s.idL(gr, gc)] != s.finL(gr, gc)) return false;
    return true;
}

void build_predict_schedule(int M, int Mm, int nbt, int workers, std::vector<SchedItem>& out, int blk, SchedStats* stats, bool simulate,
                            bool with_sigma) {
    std::vector<SchedItem> prog;
    std::vector<int32_t> task;
    program_order_predict(M, Mm, nbt, with_sigma, prog, task);
    schedule(Shape(M, Mm, nbt, true), prog, task, workers, blk, out, stats, simulate);
}

bool validate_schedule(const std::vector<SchedItem>& items, int M, int Mm, int nbt, bool predict, const char** why, bool with_sigma) {
    const Shape s(M, predict ? Mm : 0, nbt, predict);
    std::vector<int32_t> ver(s.nblocks, 0);
    static const char* kWait = "an item waits for a version no earlier item produces";
    static const char* kFinal = "a block does not end at its final version";
    static const char* kCount = "wrong number of items";
    static const char* kInside = "an item waits for a version that a merged update passes without stopping at it";
    // A merged update raises its block's counter by several versions in steps that are not ordered among the
    // eight consumer warps (gp_exec.cuh), so the versions strictly inside such a write are never a state in
    // which the block is complete: nothing may wait for exactly one of them.  `interior` marks them.
    std::vector<int64_t> multi_blocks;
    std::vector<int32_t> multi_lo, multi_hi;          // versions lo < v < hi of block multi_blocks[k] are interior
    {
        std::vector<int32_t> v2(s.nblocks, 0);
        for (const SchedItem& it : items) {
            int64_t blk_written = -1;
            int count = 0;
            item_effects(s, it, [](int64_t, int) {}, [&](int64_t b) { if (b == blk_written || blk_written < 0) { blk_written = b; ++count; } });
            const bool is_upd = it.op == S_UPD_L || it.op == S_UPD_V || it.op == S_UPD_S;
            if (is_upd && count > 1) { multi_blocks.push_back(blk_written); multi_lo.push_back(v2[blk_written]); multi_hi.push_back(v2[blk_written] + count); }
            item_effects(s, it, [](int64_t, int) {}, [&](int64_t b) { ++v2[b]; });
        }
    }
    std::vector<int64_t> order(multi_blocks.size());
    for (size_t k = 0; k < order.size(); ++k) order[k] = (int64_t)k;
    std::sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return multi_blocks[a] < multi_blocks[b]; });
    auto is_interior = [&](int64_t b, int need) {
        auto lo = std::lower_bound(order.begin(), order.end(), b, [&](int64_t k, int64_t blk) { return multi_blocks[k] < blk; });
        for (; lo != order.end() && multi_blocks[*lo] == b; ++lo)
            if (need > multi_lo[*lo] && need < multi_hi[*lo]) return true;
        return false;
    };
    bool ok = true, inside = false;
    for (const SchedItem& it : items) {
        item_effects(s, it, [&](int64_t b, int need) { if (ver[b] < need) ok = false; if (need > 0 && is_interior(b, need)) inside = true; },
                     [&](int64_t b) { ++ver[b]; });
        if (!ok) { if (why) *why = kWait; return false; }
        if (inside) { if (why) *why = kInside; return false; }
    }
    if (!predict) {
        for (int gr = 0; gr < s.NB; ++gr)
            for (int gc = 0; gc <= gr; ++gc)
                if (ver[s.idL(gr, gc)] != s.finL(gr, gc)) { if (why) *why = kFinal; return false; }
    } else {
        for (int gr = 0; gr < s.NBm; ++gr) {
            for (int gc = 0; gc < s.NB; ++gc)
                if (ver[s.idV(gr, gc)] != s.finV(gc)) { if (why) *why = kFinal; return false; }
            for (int gc = 0; gc <= gr; ++gc)
                if (ver[s.idS(gr, gc)] != (with_sigma ? M : 0)) { if (why) *why = kFinal; return false; }
        }
    }
    std::vector<SchedItem> prog;
    std::vector<int32_t> task;
    if (predict) program_order_predict(M, Mm, nbt, with_sigma, prog, task); else program_order_cholesky(M, nbt, prog, task);
    if (prog.size() != items.size()) { if (why) *why = kCount; return false; }
    return true;
}

uint64_t schedule_fingerprint(const std::vector<SchedItem>& items) {
    uint64_t h = 1469598103934665603ull;                         // FNV-1a over the item words
    for (const SchedItem& it : items)
        for (uint32_t w : {it.op, it.gr, it.gc, it.q})
            for (int b = 0; b < 4; ++b) { h ^= (w >> (8 * b)) & 0xffu; h *= 1099511628211ull; }
    return h;
}

}  // namespace gpb
