// gp_exec.cuh -- the persistent tile-task executor (step a6) and the block kernels it runs.
//
// The paper drives its tile DAG from the host: one HPX task per tile operation, a round-robin
// CUDA stream, and a cudaStreamSynchronize inside every task.  Here the
// whole DAG runs inside ONE kernel launch: `sched_width` persistent CTAs pull work items in a
// fixed, topologically sorted order from a global ticket counter and synchronise through
// per-block version counters in global memory (release/acquire), so a dependent item starts
// ~1 us after its producer finishes and nothing returns to the host.
//
// Work items are block-level (b x b, b = 128 for tiles that are multiples of 128) pieces of the
// paper's tile tasks (readings A3/A4):
//   UPD   C(gr,gc) -= sum_{q in [q0,q1)} A(gr,q) B(gc,q)^T      SYRK / GEMM tiles (q-range = one
//                                                                tile column J), POTRF sub-updates
//   TRSM  C(gr,gc)  = C(gr,gc) invD(gc)^T                        panel solve with the inverted
//                                                                diagonal block
//   POTRF L(q,q)    = chol(C(q,q)), invD(q) = L(q,q)^-1          diagonal block
//   ROW   the left-looking chain of one block row through one tile column (TRSM tile task)
// on three matrices: L (lower-packed tiles), V^T (general tiles) and Sigma (dense).
//
// Deadlock freedom: the item list is a topological order of the DAG and tickets are handed out
// in list order to CTAs that are already running, so every item a CTA waits for was claimed
// earlier by a CTA that is running or finished.
#pragma once
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

struct ExecParams {
    double* L;             // lower-packed tiles (n x n)
    double* Vt;            // general tiles (m x n), or nullptr
    double* S;             // dense m x m, or nullptr
    double* invD;          // NB blocks of b x b: inverses of the diagonal blocks of L
    int* verL;             // NB x NB version counters
    int* verV;             // NBm x NB
    int* verS;             // NBm x NBm
    const Item* items;
    unsigned int* ticket;
    int* d_info;
    int nitems;
    int t;                 // tile edge
    int nbt;               // blocks per tile edge (t / b)
    int NB;                // n / b
    int NBm;               // m / b
    int Mt;                // n / t (tiles per row of V^T)
    int64_t m;             // rows of Sigma (leading dimension)
    int L_final;           // 1: L is an input that is final everywhere (predictor), no waits on it
    unsigned long long* stats;   // per worker CTA: {cycles waiting on dependencies, cycles total, items run, SM id}
};

__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}

template <int BLK>
struct Exec {
    const ExecParams& p;
    double* smem;
    long long* wait_cycles;   // shared-memory accumulator owned by thread 0
    __device__ Exec(const ExecParams& p_, double* smem_, long long* wc) : p(p_), smem(smem_), wait_cycles(wc) {}

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
    __device__ __forceinline__ double* blkS(int gr, int gc) const {
        return p.S + (size_t)gr * BLK * p.m + (size_t)gc * BLK;
    }
    // number of writes after which block (gr,gc) of L is final
    __device__ __forceinline__ int finL(int gr, int gc) const {
        const int K = gc / p.nbt, bk = gc % p.nbt;
        return (gr / p.nbt == K) ? K + 1 + bk : K + 1 + (bk > 0 ? 1 : 0);
    }
    __device__ __forceinline__ int finV(int gc) const { return gc / p.nbt + 1 + (gc % p.nbt > 0 ? 1 : 0); }

    // ---- dependency waits: lane i of warp 0 polls wait i, then the CTA barrier publishes it
    struct Waits {
        const int* addr;   // this lane's counter (nullptr = none)
        int need;
    };
    __device__ __forceinline__ void wait_all(const int* addr, int need) const {
        const long long t0 = clock64();
        if (addr != nullptr) {
            while (ld_acquire(addr) < need) __nanosleep(64);
        }
        __syncthreads();
        if (threadIdx.x == 0) *wait_cycles += clock64() - t0;
    }
    __device__ __forceinline__ void signal(int* counter) const {
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            atomicAdd(counter, 1);
        }
    }

    // C(gr,gc) -= A(gr,q0:q1) B(gc,q0:q1)^T on (matC, matA, matB) given by op
    __device__ void update(uint32_t op, int gr, int gc, int q0, int q1) const {
        const int tid = threadIdx.x;
        const int nq = q1 - q0;
        // waits: lane 0: own block; lanes 1..nq: A panel; lanes 1+nq..2nq: B panel
        const int* addr = nullptr;
        int need = 0;
        if (tid < 1 + 2 * nq) {
            if (op == OP_UPD_L) {
                if (tid == 0) { addr = p.verL + (size_t)gr * p.NB + gc; need = q0 / p.nbt + q0 % p.nbt; }
                else if (tid <= nq) { const int q = q0 + tid - 1; addr = p.verL + (size_t)gr * p.NB + q; need = finL(gr, q); }
                else { const int q = q0 + tid - 1 - nq; addr = p.verL + (size_t)gc * p.NB + q; need = finL(gc, q); }
            } else if (op == OP_UPD_V) {
                if (tid == 0) { addr = p.verV + (size_t)gr * p.NB + gc; need = q0 / p.nbt; }
                else if (tid <= nq) { const int q = q0 + tid - 1; addr = p.verV + (size_t)gr * p.NB + q; need = finV(q); }
                else if (!p.L_final) { const int q = q0 + tid - 1 - nq; addr = p.verL + (size_t)gc * p.NB + q; need = finL(gc, q); }
            } else {  // OP_UPD_S
                if (tid == 0) { addr = p.verS + (size_t)gr * p.NBm + gc; need = q0 / p.nbt; }
                else if (tid <= nq) { const int q = q0 + tid - 1; addr = p.verV + (size_t)gr * p.NB + q; need = finV(q); }
                else { const int q = q0 + tid - 1 - nq; addr = p.verV + (size_t)gc * p.NB + q; need = finV(q); }
            }
        }
        wait_all(addr, need);
        const int K = nq * BLK;
        if (op == OP_UPD_L) {
            gemm_nt_block<BLK>(blkL(gr, gc), p.t, blkL(gr, q0), p.t, blkL(gc, q0), p.t, K, kSub, smem);
            signal(p.verL + (size_t)gr * p.NB + gc);
        } else if (op == OP_UPD_V) {
            gemm_nt_block<BLK>(blkV(gr, gc), p.t, blkV(gr, q0), p.t, blkL(gc, q0), p.t, K, kSub, smem);
            signal(p.verV + (size_t)gr * p.NB + gc);
        } else {
            gemm_nt_block<BLK>(blkS(gr, gc), (int)p.m, blkV(gr, q0), p.t, blkV(gc, q0), p.t, K, kSub, smem);
            signal(p.verS + (size_t)gr * p.NBm + gc);
        }
    }

    // C(gr,gc) = C(gr,gc) invD(gc)^T   (is_v: C is a block of V^T, else of L)
    __device__ void trsm(bool is_v, int gr, int gc) const {
        const int tid = threadIdx.x;
        const int* addr = nullptr;
        int need = 0;
        if (tid == 0) {
            if (is_v) { addr = p.verV + (size_t)gr * p.NB + gc; need = finV(gc) - 1; }
            else { addr = p.verL + (size_t)gr * p.NB + gc; need = finL(gr, gc) - 1; }
        } else if (tid == 1 && !(is_v && p.L_final)) {
            addr = p.verL + (size_t)gc * p.NB + gc; need = finL(gc, gc);
        }
        wait_all(addr, need);
        double* C = is_v ? blkV(gr, gc) : blkL(gr, gc);
        gemm_nt_block<BLK>(C, p.t, C, p.t, p.invD + (size_t)gc * BLK * BLK, BLK, BLK, kSet, smem);
        signal(is_v ? p.verV + (size_t)gr * p.NB + gc : p.verL + (size_t)gr * p.NB + gc);
    }

    __device__ void row_chain(bool is_v, int gr, int qt) const {
        for (int jj = 0; jj < p.nbt; ++jj) {
            if (jj > 0) update(is_v ? OP_UPD_V : OP_UPD_L, gr, qt + jj, qt, qt + jj);
            trsm(is_v, gr, qt + jj);
        }
    }

    __device__ void potrf(int q) const;

    __device__ void run(const Item& it) const {
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
// Diagonal block kernels (shared-memory resident, BLK x BLK, padded stride BLK+1).
// POTRF: unblocked right-looking Cholesky of the block; then the inverse of the
// lower-triangular factor in place, so that TRSM becomes a DMMA product.
// ---------------------------------------------------------------------------------------------
template <int BLK>
__device__ void chol_lower_smem(double* S, int* d_info, int col0) {
    constexpr int SP = BLK + 1;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    for (int j = 0; j < BLK; ++j) {
        const double d = S[j * SP + j];
        if (!(d > 0.0) && tid == 0) atomicCAS(d_info, 0, col0 + j + 1);
        const double ljj = sqrt(d);
        for (int r = j + 1 + tid; r < BLK; r += kThreads) S[r * SP + j] = S[r * SP + j] / ljj;
        __syncthreads();
        if (tid == 0) S[j * SP + j] = ljj;
        for (int c = j + 1 + warp; c < BLK; c += kThreads / 32) {
            const double lc = S[c * SP + j];
            for (int r = c + lane; r < BLK; r += 32) S[r * SP + c] = fma(-S[r * SP + j], lc, S[r * SP + c]);
        }
        __syncthreads();
    }
}

// In-place inverse of the lower-triangular matrix in S (stride BLK+1): from X L = I,
//   X[j][j] = 1/L[j][j],  X[i][j] = -(sum_{k=j+1..i} X[i][k] L[k][j]) / L[j][j],  j = BLK-1..0.
// Two threads per row split the sum (even/odd k).
template <int BLK>
__device__ void inv_lower_smem(double* S) {
    constexpr int SP = BLK + 1;
    const int tid = threadIdx.x;
    const int i = tid >> 1, half = tid & 1;
    for (int j = BLK - 1; j >= 0; --j) {
        double s = 0.0;
        if (i < BLK && i > j) {
            for (int k = j + 1 + half; k <= i; k += 2) s = fma(S[i * SP + k], S[k * SP + j], s);
        }
        s += __shfl_xor_sync(0xffffffffu, s, 1);
        const double rd = 1.0 / S[j * SP + j];
        __syncthreads();
        if (i < BLK && half == 0) {
            if (i > j) S[i * SP + j] = -s * rd;
            else if (i == j) S[j * SP + j] = rd;
        }
        __syncthreads();
    }
}

template <int BLK>
__device__ void load_lower_to_smem(double* S, const double* __restrict__ G, int ld) {
    constexpr int SP = BLK + 1;
    for (int idx = threadIdx.x; idx < BLK * BLK; idx += kThreads) {
        const int r = idx / BLK, c = idx % BLK;
        S[r * SP + c] = (c <= r) ? __ldcg(G + (size_t)r * ld + c) : 0.0;
    }
    __syncthreads();
}

template <int BLK>
__device__ void Exec<BLK>::potrf(int q) const {
    const int* addr = nullptr;
    int need = 0;
    if (threadIdx.x == 0) { addr = p.verL + (size_t)q * p.NB + q; need = finL(q, q) - 1; }
    wait_all(addr, need);
    constexpr int SP = BLK + 1;
    double* S = smem;
    double* G = blkL(q, q);
    load_lower_to_smem<BLK>(S, G, p.t);
    chol_lower_smem<BLK>(S, p.d_info, q * BLK);
    for (int idx = threadIdx.x; idx < BLK * BLK; idx += kThreads) {
        const int r = idx / BLK, c = idx % BLK;
        if (c <= r) __stcg(G + (size_t)r * p.t + c, S[r * SP + c]);
    }
    inv_lower_smem<BLK>(S);
    double* inv = p.invD + (size_t)q * BLK * BLK;
    for (int idx = threadIdx.x; idx < BLK * BLK; idx += kThreads) {
        const int r = idx / BLK, c = idx % BLK;
        __stcg(inv + idx, S[r * SP + c]);      // strict upper part of S is still the zeros loaded above
    }
    signal(p.verL + (size_t)q * p.NB + q);
}

// The persistent executor kernel.
template <int BLK>
__global__ void __launch_bounds__(kThreads, 1) exec_kernel(const __grid_constant__ ExecParams p) {
    extern __shared__ __align__(16) double smem[];
    __shared__ unsigned int s_ticket;
    __shared__ long long s_wait;
    if (threadIdx.x == 0) s_wait = 0;
    const long long t_start = clock64();
    unsigned long long nrun = 0;
    Exec<BLK> ex(p, smem, &s_wait);
    for (;;) {
        if (threadIdx.x == 0) s_ticket = atomicAdd(p.ticket, 1u);
        __syncthreads();
        const unsigned int tk = s_ticket;
        if (tk >= (unsigned int)p.nitems) break;
        const int4 raw = __ldg(reinterpret_cast<const int4*>(p.items) + tk);
        Item it;
        it.op = (uint32_t)raw.x; it.gr = (uint32_t)raw.y; it.gc = (uint32_t)raw.z; it.q = (uint32_t)raw.w;
        ex.run(it);
        ++nrun;
        // run() always ends with signal(), whose barrier also protects s_ticket and the ring
    }
    if (threadIdx.x == 0 && p.stats != nullptr) {
        unsigned int smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        unsigned long long* st = p.stats + 4 * (size_t)blockIdx.x;
        st[0] = (unsigned long long)s_wait;
        st[1] = (unsigned long long)(clock64() - t_start);
        st[2] = nrun;
        st[3] = smid;
    }
}

// Batched inverse of the diagonal blocks of L (used by gp_solve and gp_predict_full_cov, which
// receive only L): one CTA per diagonal block.
template <int BLK>
__global__ void __launch_bounds__(kThreads, 1) trtri_diag_kernel(const double* __restrict__ L, int t, int nbt,
                                                                  double* __restrict__ invD) {
    extern __shared__ __align__(16) double smem[];
    constexpr int SP = BLK + 1;
    const int q = blockIdx.x;
    const int I = q / nbt;
    const double* G = L + ((size_t)I * (I + 1) / 2 + I) * (size_t)t * t + (size_t)(q % nbt) * BLK * t + (size_t)(q % nbt) * BLK;
    load_lower_to_smem<BLK>(smem, G, t);
    inv_lower_smem<BLK>(smem);
    double* inv = invD + (size_t)q * BLK * BLK;
    for (int idx = threadIdx.x; idx < BLK * BLK; idx += kThreads) {
        const int r = idx / BLK, c = idx % BLK;
        inv[idx] = smem[r * SP + c];
    }
}

template <int BLK>
constexpr int exec_smem_bytes() {
    return GemmCfg<BLK>::kSmemBytes > BLK * (BLK + 1) * 8 ? GemmCfg<BLK>::kSmemBytes : BLK * (BLK + 1) * 8;
}

}  // namespace gpb
