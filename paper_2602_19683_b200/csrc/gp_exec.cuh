// gp_exec.cuh -- the persistent tile-task executor (step a6) and the block kernels it runs.
//
// The paper drives its tile DAG from the host: one HPX task per tile operation, a round-robin
// CUDA stream, and a cudaStreamSynchronize inside every task.  Here the
// whole DAG runs inside ONE kernel launch: `sched_width` persistent CTAs pull work items in a
// fixed, topologically sorted order from a global ticket counter and synchronise through
// per-block version counters in global memory (release/acquire), so nothing returns to the host.
//
// Each CTA is warp-specialised (the sm_100a shape of a persistent GEMM, with DMMA in place of
// tcgen05 because FP64 has no tcgen05 kind):
//   * warp 8, the PRODUCER: takes the next ticket, decodes the item, polls its dependencies,
//     hands a job descriptor to the consumers through a small mbarrier-guarded queue and streams
//     the operands with TMA (cp.async.bulk.tensor, 128-byte swizzle) into a ring of k-stages.
//     It runs ahead of the consumers by the depth of the ring, ACROSS items: ticket, dependency
//     polling and the first stages of item i+1 overlap the main loop of item i.
//   * warps 0-7, the CONSUMERS: wait for a filled stage, LDS.64 + DMMA (gp_gemm.cuh), release the
//     stage; at the end of a job each warp stores its part of C and bumps the block's version
//     counter on its own (a version = kConsumerWarps increments) -- no CTA-wide barrier anywhere
//     on the GEMM path.
//
// Work items are block-level (b x b, b = 128 for tiles that are multiples of 128) pieces of the
// paper's tile tasks (readings A3/A4):
//   UPD   C(gr,gc) -= sum_{q in [q0,q1)} A(gr,q) B(gc,q)^T      SYRK / GEMM tiles (q-range = one to four
//                                                                consecutive tile columns, one version
//                                                                each), POTRF sub-updates
//   TRSM  C(gr,gc)  = C(gr,gc) invD(gc)^T                        panel solve with the inverted
//                                                                diagonal block
//   POTRF L(q,q)    = chol(C(q,q)), invD(q) = L(q,q)^-1          diagonal block
//   ROW   the left-looking chain of one block row through one tile column (TRSM tile task)
// on three matrices: L (lower-packed tiles), V^T (general tiles) and Sigma (dense).
//
// Deadlock freedom: the item list is a topological order of the DAG and tickets are handed out
// in list order.  A CTA holds up to three tickets at once (the item its consumers run, a short item
// that is already completely streamed into the ring behind it, and the one its producer is polling
// for), but it works through them IN ticket order, and a producer only polls for item k after it
// has handed over every earlier ticket of its CTA.  So consider the unfinished item with the lowest
// ticket: every dependency of it has a lower ticket and is therefore finished, its producer's poll
// succeeds, and every earlier ticket of the same CTA is finished, so its consumers reach it: it
// completes.  By induction every item completes.
// Versions: a merged update raises its block's counter by several versions in steps that are not
// ordered among the eight consumer warps, so the versions strictly INSIDE such a write are never a
// state in which the block is complete; no item may wait for one of them, and
// validate_schedule (gp_schedule.cpp) rejects a schedule in which one does.
#pragma once
#include "gp_diag.cuh"
#include "gp_gemm.cuh"

namespace gpb {

enum Op : uint32_t {
    OP_UPD_L = 0, OP_TRSM_L = 1, OP_POTRF = 2, OP_ROW_L = 3,
    OP_UPD_V = 4, OP_ROW_V = 5, OP_UPD_S = 6,
};

struct Item {              // 16 bytes
    uint32_t op;
    uint32_t gr;           // block row of the output
    uint32_t gc;           // block column of the output (ROW_*: first block column of the tile column)
    uint32_t q;            // q0 | (q1 << 16): contraction block range (UPD_*)
};

constexpr int kMaxPeers = 7;

struct ExecParams {
    double* L;             // lower-packed tiles (n x n)
    double* Vt;            // general tiles (m x n), or nullptr
    double* S;             // dense m x m, or nullptr
    double* invD;          // NB blocks of b x b: inverses of the diagonal blocks of L
    int* verL;             // NB x NB version counters (one version = kConsumerWarps increments)
    int* verV;             // NBm x NB
    int* verS;             // NBm x NBm
    const Item* items;
    unsigned int* ticket;
    int* d_info;
    int nitems;
    int t;                 // tile edge
    int nbt;               // blocks per tile edge (t / b): ADDRESSING only (the storage tile of the API)
    int snbt;              // blocks per SCHEDULING tile: the tile tasks of Fig. 1 are formed over virtual tiles of snbt x snbt
                           // blocks, chosen by the library for the problem size and independent of the storage tile
                           // (gp_api.cu, pick_sched_blocks); version counting, ROW chains and column merging use this one
    int NB;                // n / b
    int NBm;               // m / b
    int Mt;                // n / t (tiles per row of V^T)
    int64_t m;             // leading dimension of Sigma
    int s_row0;            // block row of V^T that row 0 of S corresponds to (0 except for the sharded block rows of Sigma)
    int L_final;           // 1: L is an input that is final everywhere (predictor), no waits on it
    int no_deps;           // 1: skip every dependency wait (contraction microbenchmark only)
    unsigned long long* stats;   // 8 per worker CTA, see gp_exec_stats in include/gp_b200.h
    // Fused panel broadcast ("broadcast ... fused as the epilogue of the TRSM kernel"): every block of L
    // that a job FINISHES (POTRF of a diagonal block, the solve of a block below it) is also stored at the same offset of
    // npeers other tile arrays -- the copies of L the other ranks hold, mapped into this GPU's address space (NVLink peer
    // memory; in the one-GPU emulation other buffers of the same device).  The transfer rides on the panel step block by
    // block instead of following it as a separate collective.  0 peers: nothing changes.
    double* peerL[kMaxPeers];
    int npeers;
};

enum JobKind : int { JOB_GEMM_SUB = 0, JOB_GEMM_SET = 1, JOB_POTRF = 2, JOB_EXIT = 3 };

struct __align__(16) Job {   // 32 bytes, producer -> consumers
    double* C;             // output block (POTRF: the diagonal block of L)
    int* sig;              // version counter of the output block
    int ldc;
    int nk;                // k-stages of GemmCfg::kStageDepth
    int kind;
    int arg;               // POTRF: diagonal block index q; GEMM: versions the job adds to the block (>= 1)
};

// Shared-memory carve-up (dynamic, base rounded up to 1024 B for the TMA swizzle)
template <int BLK>
struct ExecSmem {
    static constexpr int kRing = GemmCfg<BLK>::kRingBytes;
    static constexpr int kPotrf = DiagSmem<BLK>::kBytes;
    static constexpr int kWork = kRing > kPotrf ? kRing : kPotrf;       // POTRF factors inside the idle ring
    static constexpr int kFull = kWork;                                  // uint64 full[kStages]
    static constexpr int kEmpty = kFull + 8 * kStages;
    static constexpr int kJobFull = kEmpty + 8 * kStages;
    static constexpr int kJobEmpty = kJobFull + 8 * kJobSlots;
    static constexpr int kJobs = (kJobEmpty + 8 * kJobSlots + 15) / 16 * 16;
    static constexpr int kTotal = kJobs + (int)sizeof(Job) * kJobSlots;
    static constexpr int kBytes = kTotal + 1024;                         // slack for the manual alignment
};

template <int BLK>
constexpr int exec_smem_bytes() { return ExecSmem<BLK>::kBytes; }

// ---------------------------------------------------------------------------------------------
// The producer warp.
// ---------------------------------------------------------------------------------------------
template <int BLK>
struct Producer {
    using Cfg = GemmCfg<BLK>;
    using SM = ExecSmem<BLK>;
    const ExecParams& p;
    const CUtensorMap *mapL, *mapV, *mapD;
    char* ring;
    uint64_t *full, *empty, *job_full, *job_empty;
    Job* jobs;
    int lane;
    int stage = 0, phase = 0, slot = 0, jphase = 0;
    long long poll_cycles = 0;

    __device__ Producer(const ExecParams& p_, const CUtensorMap* l, const CUtensorMap* v, const CUtensorMap* d, char* base)
        : p(p_), mapL(l), mapV(v), mapD(d), ring(base),
          full(reinterpret_cast<uint64_t*>(base + SM::kFull)), empty(reinterpret_cast<uint64_t*>(base + SM::kEmpty)),
          job_full(reinterpret_cast<uint64_t*>(base + SM::kJobFull)), job_empty(reinterpret_cast<uint64_t*>(base + SM::kJobEmpty)),
          jobs(reinterpret_cast<Job*>(base + SM::kJobs)), lane(threadIdx.x & 31) {}

    // ---- addressing ---------------------------------------------------------------------------
    __device__ __forceinline__ double* blkL(int gr, int gc) const {
        const int I = gr / p.nbt, J = gc / p.nbt;
        return p.L + ((size_t)I * (I + 1) / 2 + J) * (size_t)p.t * p.t + (size_t)(gr % p.nbt) * BLK * p.t +
               (size_t)(gc % p.nbt) * BLK;
    }
    __device__ __forceinline__ double* blkV(int gr, int gc) const {
        const int I = gr / p.nbt, J = gc / p.nbt;
        return p.Vt + ((size_t)I * p.Mt + J) * (size_t)p.t * p.t + (size_t)(gr % p.nbt) * BLK * p.t +
               (size_t)(gc % p.nbt) * BLK;
    }
    __device__ __forceinline__ double* blkS(int gr, int gc) const { return p.S + (size_t)(gr - p.s_row0) * BLK * p.m + (size_t)gc * BLK; }
    // TMA coordinates {inner element, row} of block (gr, gc) in the [tiles*t, t] view of L / V^T
    __device__ __forceinline__ int2 crdL(int gr, int gc) const {
        const int I = gr / p.nbt, J = gc / p.nbt;
        return make_int2((gc % p.nbt) * BLK, (I * (I + 1) / 2 + J) * p.t + (gr % p.nbt) * BLK);
    }
    __device__ __forceinline__ int2 crdV(int gr, int gc) const {
        const int I = gr / p.nbt, J = gc / p.nbt;
        return make_int2((gc % p.nbt) * BLK, (I * p.Mt + J) * p.t + (gr % p.nbt) * BLK);
    }
    // number of writes after which block (gr,gc) of L is final
    __device__ __forceinline__ int finL(int gr, int gc) const {
        const int K = gc / p.snbt, bk = gc % p.snbt;
        return (gr / p.snbt == K) ? K + 1 + bk : K + 1 + (bk > 0 ? 1 : 0);
    }
    __device__ __forceinline__ int finV(int gc) const { return gc / p.snbt + 1 + (gc % p.snbt > 0 ? 1 : 0); }

    // ---- dependency polling: wait w of the current job is handled by lane w % 32 ------------------
    __device__ __forceinline__ void poll(const int* addr, int need) {
        if (addr != nullptr && need > 0) {
            const int target = need * kConsumerWarps;
            [[maybe_unused]] unsigned spins = 0;
            while (ld_acquire(addr) < target) {
                GPB_SPIN_GUARD(spins, "dependency poll", target, ld_acquire(addr))
                __nanosleep(40);
            }
        }
    }
    __device__ __forceinline__ void deps_done(long long t0) {
        __syncwarp();
        fence_proxy_async_global();      // acquired generic-proxy writes -> visible to the TMA reads issued below
        if (lane == 0) poll_cycles += clock64() - t0;
    }

    // ---- job hand-off and operand streaming ------------------------------------------------------
    // Lane 0 alone runs the mbarrier / TMA protocol (its stage, phase, slot, jphase are the only live
    // copies); the other lanes help with dependency polling and L2 prefetch and meet lane 0 again at
    // the __syncwarp() of the next job's deps_done().
    __device__ __forceinline__ void push_job(double* C, int* sig, int ldc, int nk, int kind, int arg) {
        if (lane != 0) return;
        mbar_wait(&job_empty[slot], (uint32_t)(jphase ^ 1), 1);
        Job j;
        j.C = C; j.sig = sig; j.ldc = ldc; j.nk = nk; j.kind = kind; j.arg = arg;
        jobs[slot] = j;
        mbar_arrive(&job_full[slot]);
        if (++slot == kJobSlots) { slot = 0; jphase ^= 1; }
    }
    // `C`/`ldc` (may be null): the block the consumers will read in their epilogue.  Its rows are pulled into
    // L2 with cp.async.bulk.prefetch.L2 at the start of this call; the caller passes it with the block that is
    // streamed two blocks (16 stages) before the end of the job -- early enough to hide the HBM latency, late
    // enough not to be evicted again (at job start, ~140 us earlier, it was).
    __device__ __forceinline__ void stream(const CUtensorMap* mA, int2 a, const CUtensorMap* mB, int2 b, int nk,
                                           const double* C = nullptr, int ldc = 0) {
        if (lane != 0) return;
        const int kpre = 0;                    // the caller picks the block at which the prefetch is due
        for (int kt = 0; kt < nk; ++kt) {
            mbar_wait(&empty[stage], (uint32_t)(phase ^ 1), 2);
            char* dst = ring + (size_t)stage * Cfg::kStageBytes;
            mbar_arrive_expect_tx(&full[stage], (uint32_t)Cfg::kStageBytes);
#pragma unroll
            for (int sub = 0; sub < Cfg::kSub; ++sub) {
                tma_load_2d(dst + sub * Cfg::kSubBytes, mA, a.x + (kt * Cfg::kSub + sub) * kBK, a.y, &full[stage]);
                tma_load_2d(dst + Cfg::kOperandBytes + sub * Cfg::kSubBytes, mB, b.x + (kt * Cfg::kSub + sub) * kBK, b.y, &full[stage]);
            }
            if (++stage == kStages) { stage = 0; phase ^= 1; }
            if (kt == kpre && C != nullptr) {
#pragma unroll 1
                for (int r = 0; r < BLK; ++r) l2_prefetch_bulk(C + (size_t)r * ldc, BLK * 8);
            }
        }
    }

    // C(gr,gc) -= A(gr,q0:q1) B(gc,q0:q1)^T on (matC, matA, matB) given by op
    __device__ void update(uint32_t op, int gr, int gc, int q0, int q1) {
        const int nq = q1 - q0;
        const long long t0 = clock64();
        if (!p.no_deps) {
            // waits: 0: own block; 1..nq: A panel; 1+nq..2nq: B panel
            for (int w = lane; w < 1 + 2 * nq; w += 32) {
                const int* addr = nullptr;
                int need = 0;
                if (op == OP_UPD_L) {
                    if (w == 0) { addr = p.verL + (size_t)gr * p.NB + gc; need = q0 / p.snbt + q0 % p.snbt; }
                    else if (w <= nq) { const int q = q0 + w - 1; addr = p.verL + (size_t)gr * p.NB + q; need = finL(gr, q); }
                    else { const int q = q0 + w - 1 - nq; addr = p.verL + (size_t)gc * p.NB + q; need = finL(gc, q); }
                } else if (op == OP_UPD_V) {
                    if (w == 0) { addr = p.verV + (size_t)gr * p.NB + gc; need = q0 / p.snbt; }
                    else if (w <= nq) { const int q = q0 + w - 1; addr = p.verV + (size_t)gr * p.NB + q; need = finV(q); }
                    else if (!p.L_final) { const int q = q0 + w - 1 - nq; addr = p.verL + (size_t)gc * p.NB + q; need = finL(gc, q); }
                } else {  // OP_UPD_S
                    if (w == 0) { addr = p.verS + (size_t)gr * p.NBm + gc; need = q0 / p.snbt; }
                    else if (w <= nq) { const int q = q0 + w - 1; addr = p.verV + (size_t)gr * p.NB + q; need = finV(q); }
                    else { const int q = q0 + w - 1 - nq; addr = p.verV + (size_t)gc * p.NB + q; need = finV(q); }
                }
                poll(addr, need);
            }
        }
        deps_done(t0);
        const int nk = nq * BLK / Cfg::kStageDepth;
        // merged tile columns: one job, one version per column.  The panels are streamed block by block (a block
        // is contiguous in the TMA view of its storage tile; a run of blocks need not be: the scheduling tile is
        // independent of the storage tile), and the C block is prefetched into L2 two blocks before the end.
        const int ncol = nq > p.snbt ? nq / p.snbt : 1;
        const int qpre = nq > 2 ? q1 - 2 : q0;
        if (op == OP_UPD_L) {
            double* C = blkL(gr, gc);
            push_job(C, p.verL + (size_t)gr * p.NB + gc, p.t, nk, JOB_GEMM_SUB, ncol);
            for (int q = q0; q < q1; ++q) stream(mapL, crdL(gr, q), mapL, crdL(gc, q), BLK / Cfg::kStageDepth, q == qpre ? C : nullptr, p.t);
        } else if (op == OP_UPD_V) {
            double* C = blkV(gr, gc);
            push_job(C, p.verV + (size_t)gr * p.NB + gc, p.t, nk, JOB_GEMM_SUB, ncol);
            for (int q = q0; q < q1; ++q) stream(mapV, crdV(gr, q), mapL, crdL(gc, q), BLK / Cfg::kStageDepth, q == qpre ? C : nullptr, p.t);
        } else {
            double* C = blkS(gr, gc);
            push_job(C, p.verS + (size_t)gr * p.NBm + gc, (int)p.m, nk, JOB_GEMM_SUB, ncol);
            for (int q = q0; q < q1; ++q) stream(mapV, crdV(gr, q), mapV, crdV(gc, q), BLK / Cfg::kStageDepth, q == qpre ? C : nullptr, (int)p.m);
        }
    }

    // C(gr,gc) = C(gr,gc) invD(gc)^T   (is_v: C is a block of V^T, else of L)
    __device__ void trsm(bool is_v, int gr, int gc) {
        const long long t0 = clock64();
        if (!p.no_deps) {
            if (lane == 0) {
                if (is_v) poll(p.verV + (size_t)gr * p.NB + gc, finV(gc) - 1);
                else poll(p.verL + (size_t)gr * p.NB + gc, finL(gr, gc) - 1);
            } else if (lane == 1 && !(is_v && p.L_final)) {
                poll(p.verL + (size_t)gc * p.NB + gc, finL(gc, gc));
            }
        }
        deps_done(t0);
        const int2 d = make_int2(0, gc * BLK);
        if (is_v) {
            push_job(blkV(gr, gc), p.verV + (size_t)gr * p.NB + gc, p.t, BLK / Cfg::kStageDepth, JOB_GEMM_SET, 1);
            stream(mapV, crdV(gr, gc), mapD, d, BLK / Cfg::kStageDepth);
        } else {
            push_job(blkL(gr, gc), p.verL + (size_t)gr * p.NB + gc, p.t, BLK / Cfg::kStageDepth, JOB_GEMM_SET, 1);
            stream(mapL, crdL(gr, gc), mapD, d, BLK / Cfg::kStageDepth);
        }
    }

    __device__ void row_chain(bool is_v, int gr, int qt) {
        for (int jj = 0; jj < p.snbt; ++jj) {
            if (jj > 0) update(is_v ? OP_UPD_V : OP_UPD_L, gr, qt + jj, qt, qt + jj);
            trsm(is_v, gr, qt + jj);
        }
    }

    // The consumers factor the block inside the operand ring: no TMA may be in flight into it, so
    // the producer hands the job over and then waits for the block's final version before it streams again.
    __device__ void potrf(int q) {
        const long long t0 = clock64();
        int* ver = p.verL + (size_t)q * p.NB + q;
        if (lane == 0 && !p.no_deps) poll(ver, finL(q, q) - 1);
        deps_done(t0);
        push_job(blkL(q, q), ver, p.t, 0, JOB_POTRF, q);
        const long long t1 = clock64();
        if (lane == 0) poll(ver, finL(q, q));
        __syncwarp();
        if (lane == 0) poll_cycles += clock64() - t1;
    }

    __device__ void run(const Item& it) {
        switch (it.op) {
            case OP_UPD_L: case OP_UPD_V: case OP_UPD_S:
                update(it.op, (int)it.gr, (int)it.gc, (int)(it.q & 0xffffu), (int)(it.q >> 16)); break;
            case OP_TRSM_L: trsm(false, (int)it.gr, (int)it.gc); break;
            case OP_POTRF: potrf((int)it.gc); break;
            case OP_ROW_L: row_chain(false, (int)it.gr, (int)it.gc); break;
            case OP_ROW_V: row_chain(true, (int)it.gr, (int)it.gc); break;
            default: break;
        }
    }
};

// ---------------------------------------------------------------------------------------------
// The consumer warps.
// ---------------------------------------------------------------------------------------------
template <int BLK>
__device__ void consumer_loop(const ExecParams& p, char* base) {
    using Cfg = GemmCfg<BLK>;
    using SM = ExecSmem<BLK>;
    uint64_t* full = reinterpret_cast<uint64_t*>(base + SM::kFull);
    uint64_t* empty = reinterpret_cast<uint64_t*>(base + SM::kEmpty);
    uint64_t* job_full = reinterpret_cast<uint64_t*>(base + SM::kJobFull);
    uint64_t* job_empty = reinterpret_cast<uint64_t*>(base + SM::kJobEmpty);
    const Job* jobs = reinterpret_cast<const Job*>(base + SM::kJobs);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    WarpTile<BLK> w;
    w.init(warp, lane);
    int stage = 0, phase = 0, slot = 0, jphase = 0;
    int pending = -1;                      // ring stage consumed but not yet released
    const bool keeper = (threadIdx.x == 0) && p.stats != nullptr;     // consumer-side statistics
    long long job_wait = 0;
    unsigned int njobs = 0;
    for (;;) {
        const long long tj = clock64();
        mbar_wait(&job_full[slot], (uint32_t)jphase, 3);
        if (keeper) job_wait += clock64() - tj;
        const Job j = jobs[slot];
        __syncwarp();
        if (lane == 0) mbar_arrive(&job_empty[slot]);
        if (++slot == kJobSlots) { slot = 0; jphase ^= 1; }
        if (j.kind == JOB_EXIT) break;
        ++njobs;
        if (j.kind == JOB_POTRF) {
            // every earlier stage has been consumed by this warp; the barrier inside makes that true for all warps
            cbar();
            potrf_block<BLK>(reinterpret_cast<double*>(base), j.C, j.ldc, p.invD + (size_t)j.arg * BLK * BLK, p.d_info, j.arg * BLK);
            fence_proxy_async_global();      // L(q,q), invD(q): read by other CTAs' TMA
            fence_proxy_async_shared();      // the ring is about to be overwritten by TMA again
            cbar();
            if (p.npeers > 0) {              // the finished diagonal block goes to the other ranks' copies of L
                const size_t off = (size_t)(j.C - p.L);
                for (int k = 0; k < p.npeers; ++k) {
                    double* dst = p.peerL[k] + off;
                    for (int idx = threadIdx.x; idx < BLK * BLK / 2; idx += kConsumerThreads) {
                        const int r = idx / (BLK / 2), c2 = idx % (BLK / 2);
                        __stcg(reinterpret_cast<double2*>(dst + (size_t)r * j.ldc) + c2, __ldcg(reinterpret_cast<const double2*>(j.C + (size_t)r * j.ldc) + c2));
                    }
                }
            }
            if (threadIdx.x == 0) red_release_add(j.sig, kConsumerWarps);
            continue;
        }
        double acc[Cfg::MI][Cfg::NJ][2];
#pragma unroll
        for (int i = 0; i < Cfg::MI; ++i)
#pragma unroll
            for (int jj = 0; jj < Cfg::NJ; ++jj) acc[i][jj][0] = acc[i][jj][1] = 0.0;
        for (int kt = 0; kt < j.nk; ++kt) {
            mbar_wait(&full[stage], (uint32_t)phase, 4);
            // Deferred release: the stage consumed one step ago is handed back only now.  Releasing a
            // stage right behind its last LDS.64 is NOT safe -- the arrive does not wait for loads
            // still in flight and the TMA refill then races them (measured: 11 of 80 runs of config 2
            // came out wrong at 1e-5; 0 of 80 with either a fence.acq_rel.cta before the arrive or
            // this deferral, which costs nothing but one stage of ring depth).  By now every DMMA of
            // the previous stage has issued, so every load of it has returned.  `pending` carries
            // across jobs; a stage still pending at a POTRF or at EXIT is simply not needed.
            if (pending >= 0) {
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[pending]);
            }
            pending = stage;
            consume_stage<BLK>(base + (size_t)stage * Cfg::kStageBytes, w, acc);
            if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        store_tile<BLK>(j.C, j.ldc, j.kind, w, acc);
        if (j.kind == JOB_GEMM_SET && p.npeers > 0) {       // a solved block of L is final: the other ranks' copies get it too
            const size_t off = (size_t)(j.C - p.L);
            for (int k = 0; k < p.npeers; ++k) store_tile<BLK>(p.peerL[k] + off, j.ldc, JOB_GEMM_SET, w, acc);
        }
        fence_proxy_async_global();          // this warp's part of C: read by TMA later
        __syncwarp();
        if (lane == 0) red_release_add(j.sig, j.arg);   // versions this job adds (tile columns it covered)
    }
    if (keeper) {
        unsigned long long* st = p.stats + 8 * (size_t)blockIdx.x;
        st[4] = (unsigned long long)job_wait;
        st[5] = 0;
        st[6] = (unsigned long long)njobs;
    }
}

// The persistent executor kernel.
template <int BLK>
__global__ void __launch_bounds__(kThreads, 1)
exec_kernel(const __grid_constant__ ExecParams p, const __grid_constant__ CUtensorMap mapL, const __grid_constant__ CUtensorMap mapV,
            const __grid_constant__ CUtensorMap mapD) {
    extern __shared__ char smem_raw[];
    using SM = ExecSmem<BLK>;
    char* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        uint64_t* full = reinterpret_cast<uint64_t*>(base + SM::kFull);
        uint64_t* empty = reinterpret_cast<uint64_t*>(base + SM::kEmpty);
        uint64_t* job_full = reinterpret_cast<uint64_t*>(base + SM::kJobFull);
        uint64_t* job_empty = reinterpret_cast<uint64_t*>(base + SM::kJobEmpty);
        for (int s = 0; s < kStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], kConsumerWarps); }
        for (int s = 0; s < kJobSlots; ++s) { mbar_init(&job_full[s], 1); mbar_init(&job_empty[s], kConsumerWarps); }
        fence_mbar_init();
    }
    __syncthreads();
    if (warp < kConsumerWarps) {
        reg_alloc<kConsumerRegs>();
        consumer_loop<BLK>(p, base);
        return;
    }
    reg_dealloc<kProducerRegs>();
    if (warp != kConsumerWarps) return;     // the rest of the producer warpgroup only gives its registers away
    // ---- producer warp ----
    const long long t_start = clock64();
    if (lane == 0) { tma_prefetch_desc(&mapL); tma_prefetch_desc(&mapV); tma_prefetch_desc(&mapD); }
    Producer<BLK> prod(p, &mapL, &mapV, &mapD, base);
    unsigned long long nrun = 0;
    for (;;) {
        unsigned int tk = 0;
        if (lane == 0) tk = atomicAdd(p.ticket, 1u);
        tk = __shfl_sync(0xffffffffu, tk, 0);
        if (tk >= (unsigned int)p.nitems) break;
        const int4 raw = __ldg(reinterpret_cast<const int4*>(p.items) + tk);
        Item it;
        it.op = (uint32_t)raw.x; it.gr = (uint32_t)raw.y; it.gc = (uint32_t)raw.z; it.q = (uint32_t)raw.w;
        prod.run(it);
        ++nrun;
    }
    prod.push_job(nullptr, nullptr, 0, 0, JOB_EXIT, 0);
    if (lane == 0 && p.stats != nullptr) {
        unsigned int smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        unsigned long long* st = p.stats + 8 * (size_t)blockIdx.x;
        st[0] = (unsigned long long)prod.poll_cycles;
        st[1] = (unsigned long long)(clock64() - t_start);
        st[2] = nrun;
        st[3] = smid;
    }
}

// Batched inverse of the diagonal blocks of L (used by gp_solve and gp_predict_full_cov, which
// receive only L): one CTA of kConsumerThreads per diagonal block.
// `fill` (may be null): a vector of gridDim.x * BLK doubles whose block q is overwritten with the "not yet computed" pattern
// of the solve kernels (gp_kernels.cuh: kSolvePending), so that gp_solve needs no extra launch for it.
template <int BLK>
__global__ void __launch_bounds__(kConsumerThreads, 1) trtri_diag_kernel(const double* __restrict__ L, int t, int nbt,
                                                                          double* __restrict__ invD, double* __restrict__ fill) {
    extern __shared__ __align__(16) double smem[];
    const int q = blockIdx.x;
    if (fill != nullptr && threadIdx.x < BLK) fill[(size_t)q * BLK + threadIdx.x] = __longlong_as_double(kSolvePending);
    const int I = q / nbt;
    const double* G = L + ((size_t)I * (I + 1) / 2 + I) * (size_t)t * t + (size_t)(q % nbt) * BLK * t + (size_t)(q % nbt) * BLK;
    trtri_block<BLK>(smem, G, t, invD + (size_t)q * BLK * BLK);
}

}  // namespace gpb
