// gp_diag.cuh -- the diagonal block (steps a2/a3 at block level): POTRF of a BLK x BLK block in
// shared memory and the inverse of its lower-triangular factor, so that every TRSM below it is a
// DMMA product with invD.
//
// This is the serial spine of the tile DAG: n/BLK of these run one after another on the critical
// path.  The first version factored and inverted column by column with two CTA barriers per column
// (512 barriers, ~250 us per 128-block: at n = 8192 the 64 diagonal blocks WERE the factorisation
// time).  Now the block is processed in panels of 32 columns:
//   * the 32 x 32 diagonal piece is factored AND inverted by one warp entirely in registers
//     (lane r holds row r; columns travel by shuffles; no barrier at all), as north_star suggests
//     for small POTRF/TRSM tiles;
//   * the panel below it becomes a product with that small inverse, X = A21 inv(L11)^T, and the
//     trailing part gets A22 -= X X^T: both spread over all consumer threads, one barrier each;
//   * the inverse of the whole block is assembled from the 32 x 32 inverses by recursive halving,
//     inv([[A,0],[B,C]]) = [[inv A,0],[-inv(C) B inv(A), inv C]], in place, 4 x 4 register tiles.
// 19 barriers for BLK = 128 instead of 512; the sqrt + division of every column became one refined
// rsqrt, and the dependent FMA chains of the triangular inverse are split four ways.
#pragma once
#include "gp_gemm.cuh"

namespace gpb {

__device__ __forceinline__ void cbar() { named_bar_sync<1, kConsumerThreads>(); }

template <int BLK>
struct DiagSmem {
    static constexpr int SP = BLK + 1;               // padded row stride of the working block
    static constexpr int NP = BLK / 32;              // 32-column panels
    static constexpr int TP = 33;                    // row stride of the 32 x 32 scratch blocks
    static constexpr int kT = BLK * SP;              // NP inverses of the diagonal 32 x 32 pieces
    static constexpr int kU = kT + NP * 32 * TP;     // one 32 x 32 temporary
    static constexpr int kDoubles = kU + (BLK >= 128 ? 64 * 65 : 2 * 32 * TP);   // scratch for the inner products of inv_blocked
    static constexpr int kBytes = kDoubles * 8;
};

// One warp, registers only.  Lane r holds row r of the 32 x 32 piece at (c0, c0) of S.
// FACTOR: Cholesky of the piece first (result written back to S); then always the inverse of the
// lower-triangular piece into T (32 x 33, explicit zeros above the diagonal).
template <bool FACTOR>
__device__ __forceinline__ void diag32_warp(double* S, int SP, int c0, double* T, int* d_info, int global_col0) {
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    double a[32];
#pragma unroll
    for (int c = 0; c < 32; ++c) a[c] = S[(c0 + lane) * SP + c0 + c];
    double rdiag = 0.0;                                      // lane j: 1 / L[j][j]
    if (FACTOR) {
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            const double d = __shfl_sync(full, a[j], j);
            if (!(d > 0.0) && lane == 0) atomicCAS(d_info, 0, global_col0 + c0 + j + 1);
            // the column chain is latency-bound: one rsqrt (refined once) replaces sqrt + division
            double r = rsqrt(d);
            r = fma(r * 0.5, fma(-d * r, r, 1.0), r);           // Newton step: full double accuracy of 1/sqrt(d)
            const double ljj = d * r;
            if (lane == j) rdiag = r;
            a[j] = (lane == j) ? ljj : a[j] * r;            // column j of L (rows above j hold junk that is never used)
#pragma unroll
            for (int c = j + 1; c < 32; ++c) {
                const double lc = __shfl_sync(full, a[j], c);   // L[c][j]
                a[c] = fma(-a[j], lc, a[c]);                    // meaningful for rows r >= c
            }
        }
#pragma unroll
        for (int c = 0; c < 32; ++c)
            if (c <= lane) S[(c0 + lane) * SP + c0 + c] = a[c];
    } else {
        double dl = 1.0;
#pragma unroll
        for (int c = 0; c < 32; ++c)
            if (lane == c) dl = a[c];
        rdiag = 1.0 / dl;
    }
    // W L = I, row r of W in lane r:  w[r] = 1/L[r][r],  w[c] = -(sum_{k=c+1..r} w[k] L[k][c]) / L[c][c]
    // (four partial sums: the chain of dependent FMAs is what costs, not their number)
    double w[32];
#pragma unroll
    for (int c = 0; c < 32; ++c) w[c] = 0.0;
#pragma unroll
    for (int c = 31; c >= 0; --c) {
        const double rc = __shfl_sync(full, rdiag, c);
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
        for (int k = c + 1; k < 32; ++k) {
            const double lkc = __shfl_sync(full, a[c], k);      // L[k][c]; w[k] = 0 for k > r
            if (((k - c) & 3) == 1) s0 = fma(w[k], lkc, s0);
            else if (((k - c) & 3) == 2) s1 = fma(w[k], lkc, s1);
            else if (((k - c) & 3) == 3) s2 = fma(w[k], lkc, s2);
            else s3 = fma(w[k], lkc, s3);
        }
        const double s = (s0 + s1) + (s2 + s3);
        w[c] = (lane == c) ? rc : (lane > c ? -s * rc : 0.0);
    }
#pragma unroll
    for (int c = 0; c < 32; ++c) T[lane * DiagSmem<32>::TP + c] = w[c];
}

// X = A21 inv(L11)^T for the rows below panel kb:  X[r][c] = sum_{k<=c} A21[r][k] Tinv[c][k].
// Two threads per row (16 columns each); every thread reads its whole input row before anyone writes.
template <int BLK>
__device__ __forceinline__ void panel_solve(double* S, const double* Tinv, int c0) {
    using DS = DiagSmem<BLK>;
    const int rows = BLK - c0 - 32;
    for (int task0 = 0; task0 < 2 * rows; task0 += kConsumerThreads) {
        const int task = task0 + (int)threadIdx.x;
        const bool on = task < 2 * rows;
        const int r = c0 + 32 + (on ? task >> 1 : 0), h = task & 1;
        double in[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) in[k] = S[r * DS::SP + c0 + k];
        cbar();
        if (on) {
#pragma unroll
            for (int cc = 0; cc < 16; ++cc) {
                const int c = 16 * h + cc;
                double x = 0.0;
#pragma unroll
                for (int k = 0; k < 32; ++k)
                    if (k <= 16 + cc) x = fma(in[k], Tinv[c * DS::TP + k], x);   // Tinv is zero above its diagonal
                S[r * DS::SP + c0 + c] = x;
            }
        }
        cbar();
    }
}

// A22 -= X X^T on the lower part of the trailing block, 4 x 4 patches, patch list = lower triangle of patches.
template <int BLK>
__device__ __forceinline__ void trailing_update(double* S, int c0) {
    using DS = DiagSmem<BLK>;
    const int base = c0 + 32, P = (BLK - base) / 4, npatch = P * (P + 1) / 2;
    for (int pidx = threadIdx.x; pidx < npatch; pidx += kConsumerThreads) {
        int pi = (int)((sqrtf(8.0f * (float)pidx + 1.0f) - 1.0f) * 0.5f);
        while ((pi + 1) * (pi + 2) / 2 <= pidx) ++pi;
        while (pi * (pi + 1) / 2 > pidx) --pi;
        const int pj = pidx - pi * (pi + 1) / 2;
        const int r0 = base + 4 * pi, q0 = base + 4 * pj;
        double acc[4][4];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
#pragma unroll 8
        for (int k = 0; k < 32; ++k) {
            double xr[4], xc[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) { xr[i] = S[(r0 + i) * DS::SP + c0 + k]; xc[i] = S[(q0 + i) * DS::SP + c0 + k]; }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fma(xr[i], xc[j], acc[i][j]);
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (q0 + j <= r0 + i) S[(r0 + i) * DS::SP + q0 + j] -= acc[i][j];
    }
}

// Blocked Cholesky of the lower part of S (BLK x BLK, stride SP), diagonal 32 x 32 inverses left in T.
template <int BLK>
__device__ void chol_blocked(double* smem, int* d_info, int global_col0) {
    using DS = DiagSmem<BLK>;
    double* S = smem;
    double* T = smem + DS::kT;
    for (int kb = 0; kb < DS::NP; ++kb) {
        const int c0 = 32 * kb;
        if ((threadIdx.x >> 5) == 0) diag32_warp<true>(S, DS::SP, c0, T + kb * 32 * DS::TP, d_info, global_col0);
        cbar();
        if (kb + 1 < DS::NP) {
            panel_solve<BLK>(S, T + kb * 32 * DS::TP, c0);      // ends with a barrier
            trailing_update<BLK>(S, c0);
            cbar();
        }
    }
}

// Small dense products on shared-memory blocks for the inverse: OUT (R x C, stride so) = sgn * A (R x K, stride sa)
// * B (K x C, stride sb), 4 x 4 outputs per thread, threads [t0, t0 + R*C/16).
template <int R, int C, int K>
__device__ __forceinline__ void small_gemm(double* OUT, int so, const double* A, int sa, const double* B, int sb, double sgn, int t0) {
    const int t = (int)threadIdx.x - t0;
    if (t < 0 || t >= (R / 4) * (C / 4)) return;
    const int r0 = 4 * (t / (C / 4)), q0 = 4 * (t % (C / 4));
    double acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
#pragma unroll 4
    for (int k = 0; k < K; ++k) {
        double x[4], y[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) { x[i] = A[(r0 + i) * sa + k]; y[i] = B[k * sb + q0 + i]; }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j] = fma(x[i], y[j], acc[i][j]);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) OUT[(r0 + i) * so + q0 + j] = sgn * acc[i][j];
}

// In-place inverse of the lower-triangular S given the inverses T of its diagonal 32 x 32 pieces, by
// recursive halving:  inv([[A,0],[B,C]]) = [[inv A, 0], [-inv(C) B inv(A), inv C]].
//   level 32: the blocks (1,0) and (3,2) (independent, half the threads each):  W = -T_i (L_i,i-1 T_i-1)
//   level 64: the 64 x 64 block (2:4, 0:2):  W = -inv(C) (B inv(A)) with inv(A), inv(C) the 64 x 64 inverses
//             just completed (their diagonal pieces live in T, so they are first copied into S).
// Every W overwrites the L block it replaces; U is scratch for the inner product.
template <int BLK>
__device__ void inv_blocked(double* smem) {
    using DS = DiagSmem<BLK>;
    double* S = smem;
    double* T = smem + DS::kT;
    double* U = smem + DS::kU;                       // 64 x 65 when BLK = 128, else 32 x 33
    constexpr int SP = DS::SP, TP = DS::TP;
    if (DS::NP == 1) return;
    // ---- level 32: pairs (2p+1, 2p) ----
    constexpr int NPAIR = DS::NP / 2;
    constexpr int TPB = kConsumerThreads / (NPAIR > 0 ? NPAIR : 1);   // threads per pair (>= 64 needed: 32*32/16)
#pragma unroll
    for (int pr = 0; pr < NPAIR; ++pr)              // U_pr = L_(2p+1,2p) * T_2p
        small_gemm<32, 32, 32>(U + pr * 32 * TP, TP, S + (32 * (2 * pr + 1)) * SP + 32 * (2 * pr), SP, T + (2 * pr) * 32 * TP, TP, 1.0, pr * TPB);
    cbar();
#pragma unroll
    for (int pr = 0; pr < NPAIR; ++pr)              // W = -T_(2p+1) * U_pr
        small_gemm<32, 32, 32>(S + (32 * (2 * pr + 1)) * SP + 32 * (2 * pr), SP, T + (2 * pr + 1) * 32 * TP, TP, U + pr * 32 * TP, TP, -1.0, pr * TPB);
    cbar();
    if (DS::NP == 4) {
        // the diagonal pieces of the two 64 x 64 inverses into S (their strict upper parts are zero already)
        for (int idx = threadIdx.x; idx < 4 * 32 * 32; idx += kConsumerThreads) {
            const int kb = idx >> 10, r = (idx >> 5) & 31, c = idx & 31;
            S[(32 * kb + r) * SP + 32 * kb + c] = T[kb * 32 * TP + r * TP + c];
        }
        cbar();
        // U = B * inv(A):  B = S[64:128, 0:64],  inv(A) = S[0:64, 0:64]   (64 x 64 x 64, all 256 threads)
        small_gemm<64, 64, 64>(U, 65, S + 64 * SP, SP, S, SP, 1.0, 0);
        cbar();
        // W = -inv(C) * U,  inv(C) = S[64:128, 64:128]
        small_gemm<64, 64, 64>(S + 64 * SP, SP, S + 64 * SP + 64, SP, U, 65, -1.0, 0);
        cbar();
    }
}

template <int BLK>
__device__ void load_lower_to_smem(double* S, const double* __restrict__ G, int ld) {
    constexpr int SP = BLK + 1;
    constexpr int PER = BLK * BLK / kConsumerThreads;    // elements per thread (4, 16 or 64)
    constexpr int BATCH = PER < 16 ? PER : 16;           // loads in flight per thread
    for (int b0 = 0; b0 < PER; b0 += BATCH) {
        double v[BATCH];
#pragma unroll
        for (int u = 0; u < BATCH; ++u) {
            const int idx = (b0 + u) * kConsumerThreads + threadIdx.x;
            const int r = idx / BLK, c = idx % BLK;
            v[u] = (c <= r) ? __ldcg(G + (size_t)r * ld + c) : 0.0;
        }
#pragma unroll
        for (int u = 0; u < BATCH; ++u) {
            const int idx = (b0 + u) * kConsumerThreads + threadIdx.x;
            S[(idx / BLK) * SP + idx % BLK] = v[u];
        }
    }
    cbar();
}

// inv (global, BLK x BLK row-major, zeros above the diagonal) <- the inverse assembled in shared memory
template <int BLK>
__device__ void store_inverse(const double* smem, double* __restrict__ inv) {
    using DS = DiagSmem<BLK>;
    const double* S = smem;
    const double* T = smem + DS::kT;
    for (int idx = threadIdx.x; idx < BLK * BLK; idx += kConsumerThreads) {
        const int r = idx / BLK, c = idx % BLK;
        double v = 0.0;
        if ((r >> 5) == (c >> 5)) v = T[(r >> 5) * 32 * DS::TP + (r & 31) * DS::TP + (c & 31)];
        else if (c < r) v = S[r * DS::SP + c];
        __stcg(inv + idx, v);
    }
}

// POTRF job, all consumer threads: G = diagonal block (q,q) of L in global memory (leading
// dimension t), inv = invD(q).  smem is the (idle) operand ring.
template <int BLK>
__device__ void potrf_block(double* smem, double* __restrict__ G, int t, double* __restrict__ inv, int* d_info, int col0) {
    constexpr int SP = BLK + 1;
    load_lower_to_smem<BLK>(smem, G, t);
    chol_blocked<BLK>(smem, d_info, col0);
    for (int idx = threadIdx.x; idx < BLK * BLK; idx += kConsumerThreads) {
        const int r = idx / BLK, c = idx % BLK;
        if (c <= r) __stcg(G + (size_t)r * t + c, smem[r * SP + c]);
    }
    inv_blocked<BLK>(smem);
    store_inverse<BLK>(smem, inv);
}

// inverse only (L given): the diagonal 32 x 32 inverses by one warp each, then the block assembly
template <int BLK>
__device__ void trtri_block(double* smem, const double* __restrict__ G, int t, double* __restrict__ inv) {
    using DS = DiagSmem<BLK>;
    load_lower_to_smem<BLK>(smem, G, t);
    const int warp = threadIdx.x >> 5;
    for (int kb = warp; kb < DS::NP; kb += kConsumerWarps)
        diag32_warp<false>(smem, DS::SP, 32 * kb, smem + DS::kT + kb * 32 * DS::TP, nullptr, 0);
    cbar();
    inv_blocked<BLK>(smem);
    store_inverse<BLK>(smem, inv);
}

}  // namespace gpb
