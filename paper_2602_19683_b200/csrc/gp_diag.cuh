// gp_diag.cuh -- the diagonal block (steps a2/a3 at block level): POTRF of a BLK x BLK block in
// shared memory and the inverse of its lower-triangular factor, so that every TRSM below it is a
// DMMA product with invD.
//
// This is the serial spine of the tile DAG: n/BLK of these run one after another on the critical
// path, so what matters here is LATENCY, not throughput.  History of the 128-block:
//   r01a  column by column, two CTA barriers per column: ~250 us (at n = 8192 the 64 diagonal blocks WERE the
//         factorisation time);
//   r01d  panels of 32 columns, the 32 x 32 diagonal piece factored and inverted by one warp in registers with
//         shuffles, DFMA 4 x 4 register tiles for everything else: 80 us -- and the probe of round 2 showed
//         where that went: 25 000 cycles per 32 x 32 piece, because every one of its ~1000 shuffle -> FMA pairs
//         paid the full shuffle latency (__shfl_sync cannot be batched by the compiler), and 34 000 cycles in
//         the DFMA products of the inverse;
//   r02   (this file) a tiny tiled Cholesky over the 32 x 32 pieces of the block with LOOK-AHEAD:
//     * the diagonal piece is factored by one warp, lane r = row r, but a finished column travels through a
//       64-double shared-memory line (one STS per lane, then broadcast loads that the compiler batches)
//       instead of 31 - j shuffles: ~200 cycles per column, all of it the pivot's rsqrt chain;
//     * its inverse is a forward substitution with lane c = column c of the identity: no cross-lane traffic at
//       all, L read from shared memory as broadcasts, the newest unknown enters each sum last so the
//       dependent chain is one FMA + one multiply per row;
//     * every product (panel solve X = A21 inv(L11)^T, trailing update A22 -= X X^T, the recursive-halving
//       assembly of the block inverse) is DMMA.8x8x4 on 16 x 16 macro-blocks straight out of the working
//       block, whose row stride (BLK + 4 doubles, = 4 mod 16) makes the fragment loads of both the A B^T and
//       the A B forms bank-conflict-free;
//     * per panel only  factor -> inverse -> panel solve -> update of the NEXT diagonal piece  is serial; the
//       rest of the trailing update, the store of the finished columns of L and the first level of the inverse
//       run on warps 1-7 while warp 0 already factors the next piece.
#pragma once
#include "gp_gemm.cuh"

namespace gpb {

__device__ __forceinline__ void cbar() { named_bar_sync<1, kConsumerThreads>(); }

template <int BLK>
struct DiagSmem {
    static constexpr int SP = BLK + 4;               // row stride of the working block: = 4 (mod 16) doubles
    static constexpr int NP = BLK / 32;              // 32-column panels
    static constexpr int TP = 36;                    // row stride of the 32 x 32 scratch blocks, = 4 (mod 16)
    static constexpr int UW = BLK >= 128 ? 64 : 32;  // edge of the scratch block of the inverse assembly
    static constexpr int UP = UW + 4;
    static constexpr int kT = BLK * SP;              // NP inverses of the diagonal 32 x 32 pieces
    static constexpr int kU = kT + NP * 32 * TP;     // scratch for the inner products of inv_blocked
    static constexpr int kCol = kU + UW * UP;        // 2 x 32: the column a factoring warp broadcasts (double-buffered)
    static constexpr int kRd = kCol + 64;            // NP x 32: reciprocals of the diagonal of L
    static constexpr int kDoubles = kRd + NP * 32;
    static constexpr int kBytes = kDoubles * 8;
};

// ---- DMMA products on 16 x 16 macro-blocks of shared-memory matrices ----------------------------------------------
// Fragment conventions of mma.m8n8k4.f64 (gp_gemm.cuh): lane (g = lane / 4, t = lane % 4) supplies A[g][t] and
// B[k = t][n = g] and holds C[g][2t], C[g][2t + 1].
struct Acc16 {
    double v[2][2][2];
    __device__ __forceinline__ void zero() {
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 2; ++j) v[i][j][0] = v[i][j][1] = 0.0;
    }
};

// acc += A(16 x [k0,k1)) * B^T (B_TRANS: B is 16 x K row-major, the "A B^T" form) or * B (B is K x 16 row-major)
template <bool B_TRANS>
__device__ __forceinline__ void mm16(Acc16& acc, const double* A, int lda, const double* B, int ldb, int k0, int k1, int g, int t) {
#pragma unroll 4
    for (int k = k0; k < k1; k += 4) {
        const double a0 = A[g * lda + k + t], a1 = A[(g + 8) * lda + k + t];
        double b0, b1;
        if (B_TRANS) { b0 = B[g * ldb + k + t]; b1 = B[(g + 8) * ldb + k + t]; }
        else { b0 = B[(k + t) * ldb + g]; b1 = B[(k + t) * ldb + g + 8]; }
        dmma884(acc.v[0][0][0], acc.v[0][0][1], a0, b0);
        dmma884(acc.v[0][1][0], acc.v[0][1][1], a0, b1);
        dmma884(acc.v[1][0][0], acc.v[1][0][1], a1, b0);
        dmma884(acc.v[1][1][0], acc.v[1][1][1], a1, b1);
    }
}

// C (16 x 16 at stride ldc) -= acc   /   C = sgn * acc
__device__ __forceinline__ void sub16(double* C, int ldc, const Acc16& acc, int g, int t) {
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            double2* p = reinterpret_cast<double2*>(C + (8 * i + g) * ldc + 8 * j + 2 * t);
            double2 c = *p;
            c.x -= acc.v[i][j][0];
            c.y -= acc.v[i][j][1];
            *p = c;
        }
}
__device__ __forceinline__ void set16(double* C, int ldc, const Acc16& acc, double sgn, int g, int t) {
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j)
            *reinterpret_cast<double2*>(C + (8 * i + g) * ldc + 8 * j + 2 * t) = make_double2(sgn * acc.v[i][j][0], sgn * acc.v[i][j][1]);
}

// ---- the 32 x 32 diagonal piece, one warp -----------------------------------------------------------------------------
// Cholesky of the piece at (c0, c0) of S, in place (lower part), reciprocals of its diagonal into rd[0..32).
// Lane r holds row r.  Column j, once scaled, is published through col[j & 1][.] and read back as broadcasts.
__device__ __forceinline__ void factor32_warp(double* S, int SP, int c0, double* col, double* rd, int* d_info, int global_col0) {
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    double a[32];
#pragma unroll
    for (int c = 0; c < 32; c += 2) {
        const double2 v = *reinterpret_cast<const double2*>(S + (c0 + lane) * SP + c0 + c);
        a[c] = v.x;
        a[c + 1] = v.y;
    }
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        const double d = __shfl_sync(full, a[j], j);
        if (!(d > 0.0) && lane == 0) atomicCAS(d_info, 0, global_col0 + c0 + j + 1);
        // the column chain is latency-bound: one rsqrt (refined once) replaces sqrt + division
        double r = rsqrt(d);
        r = fma(r * 0.5, fma(-d * r, r, 1.0), r);           // Newton step: full double accuracy of 1/sqrt(d)
        const double lj = (lane == j) ? d * r : a[j] * r;   // L[lane][j]  (rows above j hold junk that is never used)
        a[j] = lj;
        double* cj = col + 32 * (j & 1);
        cj[lane] = lj;
        if (lane == j) rd[j] = r;
        __syncwarp();
#pragma unroll
        for (int c = j + 1; c < 32; ++c) a[c] = fma(-lj, cj[c], a[c]);      // meaningful for rows r >= c
    }
#pragma unroll
    for (int c = 0; c < 32; ++c)
        if (c <= lane) S[(c0 + lane) * SP + c0 + c] = a[c];
    __syncwarp();
}

// T (32 x TP, zeros above the diagonal) <- inverse of the lower-triangular piece at (c0, c0) of S.
// Lane c solves L x = e_c:  x[i] = (delta_ic - sum_{k<i} L[i][k] x[k]) / L[i][i].  For the chain to be short
// the term with the newest unknown x[i-1] is added last.
template <bool HAVE_RD>
__device__ __forceinline__ void invert32_warp(const double* S, int SP, int c0, double* rd, double* T) {
    const int lane = threadIdx.x & 31;
    if (!HAVE_RD) {
        rd[lane] = 1.0 / S[(c0 + lane) * SP + c0 + lane];
        __syncwarp();
    }
    double x[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) {
        const double* Li = S + (c0 + i) * SP + c0;
        double s0 = (lane == i) ? 1.0 : 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
        for (int k = 0; k + 1 < i; ++k) {                      // everything but the newest unknown
            if ((k & 3) == 0) s0 = fma(-Li[k], x[k], s0);
            else if ((k & 3) == 1) s1 = fma(-Li[k], x[k], s1);
            else if ((k & 3) == 2) s2 = fma(-Li[k], x[k], s2);
            else s3 = fma(-Li[k], x[k], s3);
        }
        double s = (s0 + s1) + (s2 + s3);
        if (i > 0) s = fma(-Li[i - 1], x[i - 1], s);
        x[i] = s * rd[i];                                      // rows above the lane's column come out as exact zeros
    }
#pragma unroll
    for (int i = 0; i < 32; ++i) T[i * DiagSmem<32>::TP + lane] = x[i];
    __syncwarp();
}

// ---- panel solve X = A21 inv(L11)^T ------------------------------------------------------------------------------------
// Unit u = rows [base + 16u, base + 16u + 16) of the panel, all 32 columns, in place: the warp reads its 16 rows
// completely into A fragments before it stores (no other warp touches them).  inv(L11) is lower triangular:
// column block nb of the result needs k < 8 nb + 8 only.
template <int BLK>
__device__ __forceinline__ void panel_unit(double* S, const double* Tinv, int c0, int u) {
    using DS = DiagSmem<BLK>;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    double* A = S + (c0 + 32 + 16 * u) * DS::SP + c0;
    double af[2][8];
#pragma unroll
    for (int ks = 0; ks < 8; ++ks) {
        af[0][ks] = A[g * DS::SP + 4 * ks + t];
        af[1][ks] = A[(g + 8) * DS::SP + 4 * ks + t];
    }
    double acc[2][4][2];
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int nb = 0; nb < 4; ++nb) acc[h][nb][0] = acc[h][nb][1] = 0.0;
#pragma unroll
    for (int ks = 0; ks < 8; ++ks)
#pragma unroll
        for (int nb = 0; nb < 4; ++nb)
            if (4 * ks < 8 * nb + 8) {
                const double b = Tinv[(8 * nb + g) * DS::TP + 4 * ks + t];
                dmma884(acc[0][nb][0], acc[0][nb][1], af[0][ks], b);
                dmma884(acc[1][nb][0], acc[1][nb][1], af[1][ks], b);
            }
    __syncwarp();                                              // every lane's A fragments are in registers
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int nb = 0; nb < 4; ++nb)
            *reinterpret_cast<double2*>(A + (8 * h + g) * DS::SP + 8 * nb + 2 * t) = make_double2(acc[h][nb][0], acc[h][nb][1]);
}

// ---- trailing update A22 -= X X^T on 16 x 16 macro-blocks (i, j), j <= i, of the rows below the panel -------------------
template <int BLK>
__device__ __forceinline__ void update_unit(double* S, int c0, int i, int j) {
    using DS = DiagSmem<BLK>;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int base = c0 + 32;
    Acc16 acc;
    acc.zero();
    mm16<true>(acc, S + (base + 16 * i) * DS::SP + c0, DS::SP, S + (base + 16 * j) * DS::SP + c0, DS::SP, 0, 32, g, t);
    // a diagonal macro-block also rewrites its strict upper part, which nothing reads as data
    sub16(S + (base + 16 * i) * DS::SP + base + 16 * j, DS::SP, acc, g, t);
}

// store columns [c0, c0 + 32) of the finished factor (rows c0 .. BLK-1, lower part) to global memory; threads [t0, t0 + nt)
template <int BLK>
__device__ __forceinline__ void store_L_panel(const double* S, double* __restrict__ G, int ldg, int c0, int t0, int nt) {
    using DS = DiagSmem<BLK>;
    const int rows = BLK - c0;
    for (int idx = (int)threadIdx.x - t0; idx < rows * 16; idx += nt) {
        const int r = c0 + (idx >> 4), c = c0 + 2 * (idx & 15);
        if (c > r) continue;
        const double2 v = *reinterpret_cast<const double2*>(S + r * DS::SP + c);
        if (c + 1 <= r) __stcg(reinterpret_cast<double2*>(G + (size_t)r * ldg + c), v);
        else __stcg(G + (size_t)r * ldg + c, v.x);
    }
}

// ---- inverse of the whole block by recursive halving -------------------------------------------------------------------
//   inv([[A,0],[B,C]]) = [[inv A, 0], [-inv(C) B inv(A), inv C]]
// level 32: the pieces (2p+1, 2p):  W = -T_(2p+1) (L_(2p+1,2p) T_(2p)),  one warp per 16 x 16 macro-block;
// level 64: the 64 x 64 block (2:4, 0:2) from the two 64 x 64 inverses just completed.
// Every W overwrites the L block it replaces, so L must have left for global memory first.
template <int BLK>
__device__ __forceinline__ void inv_pair_first(double* smem, int pr, int mb) {        // U_pr = L_(2p+1,2p) T_2p, macro-block mb of 4
    using DS = DiagSmem<BLK>;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const double* S = smem;
    const double* T = smem + DS::kT;
    double* U = smem + DS::kU + pr * 32 * DS::TP;            // 32 x TP per pair (UW * UP >= 2 * 32 * TP)
    const int mi = mb >> 1, mj = mb & 1;
    Acc16 acc;
    acc.zero();
    // T_2p is lower triangular: T[k][n] = 0 for k < n
    mm16<false>(acc, S + (32 * (2 * pr + 1) + 16 * mi) * DS::SP + 32 * (2 * pr), DS::SP, T + (2 * pr) * 32 * DS::TP + 16 * mj, DS::TP,
                16 * mj, 32, g, t);
    set16(U + 16 * mi * DS::TP + 16 * mj, DS::TP, acc, 1.0, g, t);
}
template <int BLK>
__device__ __forceinline__ void inv_pair_second(double* smem, int pr, int mb) {       // W = -T_(2p+1) U_pr into S
    using DS = DiagSmem<BLK>;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    double* S = smem;
    const double* T = smem + DS::kT;
    const double* U = smem + DS::kU + pr * 32 * DS::TP;
    const int mi = mb >> 1, mj = mb & 1;
    Acc16 acc;
    acc.zero();
    // T_(2p+1) is lower triangular: rows 16 mi .. 16 mi + 15 need k < 16 mi + 16
    mm16<false>(acc, T + (2 * pr + 1) * 32 * DS::TP + 16 * mi * DS::TP, DS::TP, U + 16 * mj, DS::TP, 0, 16 * mi + 16, g, t);
    set16(S + (32 * (2 * pr + 1) + 16 * mi) * DS::SP + 32 * (2 * pr) + 16 * mj, DS::SP, acc, -1.0, g, t);
}

// pairs_done: bit p set = the level-32 piece of pair p has already been assembled (look-ahead of chol_blocked)
template <int BLK>
__device__ void inv_blocked(double* smem, unsigned pairs_done = 0u) {
    using DS = DiagSmem<BLK>;
    double* S = smem;
    double* T = smem + DS::kT;
    double* U = smem + DS::kU;
    constexpr int SP = DS::SP, TP = DS::TP, UP = DS::UP;
    if (DS::NP == 1) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    constexpr int NPAIR = DS::NP / 2;
    // ---- level 32: 4 macro-blocks per pair, warp w -> pair w / 4, macro-block w % 4 ----
    {
        const int pr = warp >> 2, mb = warp & 3;
        const bool mine = pr < NPAIR && !((pairs_done >> pr) & 1u);
        if (mine) inv_pair_first<BLK>(smem, pr, mb);
        cbar();
        if (mine) inv_pair_second<BLK>(smem, pr, mb);
        cbar();
    }
    if (DS::NP == 4) {
        // the diagonal pieces of the two 64 x 64 inverses into S, zeros into the pieces above them
        for (int idx = threadIdx.x; idx < 4 * 32 * 32; idx += kConsumerThreads) {
            const int kb = idx >> 10, r = (idx >> 5) & 31, c = idx & 31;
            S[(32 * kb + r) * SP + 32 * kb + c] = T[kb * 32 * TP + r * TP + c];
            if ((kb & 1) == 0) S[(32 * kb + r) * SP + 32 * (kb + 1) + c] = 0.0;
        }
        cbar();
        // U = B inv(A):  B = S[64:128, 0:64],  inv(A) = S[0:64, 0:64] lower triangular (k >= n only); 16 macro-blocks, 2 per warp
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const int mb = 2 * warp + q, mi = mb >> 2, mj = mb & 3;
            Acc16 acc;
            acc.zero();
            mm16<false>(acc, S + (64 + 16 * mi) * SP, SP, S + 16 * mj, SP, 16 * mj, 64, g, t);
            set16(U + 16 * mi * UP + 16 * mj, UP, acc, 1.0, g, t);
        }
        cbar();
        // W = -inv(C) U,  inv(C) = S[64:128, 64:128] lower triangular (k <= m only)
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const int mb = 2 * warp + q, mi = mb >> 2, mj = mb & 3;
            Acc16 acc;
            acc.zero();
            mm16<false>(acc, S + (64 + 16 * mi) * SP + 64, SP, U + 16 * mj, UP, 0, 16 * mi + 16, g, t);
            set16(S + (64 + 16 * mi) * SP + 16 * mj, SP, acc, -1.0, g, t);
        }
        cbar();
    }
}

// ---- blocked Cholesky with look-ahead ---------------------------------------------------------------------------------
// Lower part of S (BLK x BLK, stride SP) -> L, the finished columns stored to G as they complete, the inverses of the
// diagonal 32 x 32 pieces left in T.  Returns the mask of level-32 inverse pairs already assembled (inv_blocked).
//   per panel kb:  [ warp 0: factor + invert piece kb  ||  warps 1-7: rest of the trailing update of panel kb-1, store of
//                    the columns of panel kb-1, (last panel of a 128-block) the level-32 inverse piece (1,0) ]
//                  barrier;  panel solve;  barrier;  update of piece kb+1;  barrier
// prof (probe builds only): clock64 stamps of thread 0 in [0, 16) and of thread 32 in [16, 32).
template <int BLK>
__device__ unsigned chol_blocked(double* smem, double* __restrict__ G, int ldg, int* d_info, int global_col0, long long* prof = nullptr) {
    using DS = DiagSmem<BLK>;
    double* S = smem;
    double* T = smem + DS::kT;
    double* col = smem + DS::kCol;
    double* rd = smem + DS::kRd;
    const int warp = threadIdx.x >> 5;
    unsigned pairs_done = 0u;
    int ps = 0;
    auto stamp = [&]() {
        if (prof != nullptr) {
            if (threadIdx.x == 0) prof[ps] = clock64();
            if (threadIdx.x == 32) prof[16 + ps] = clock64();
            ++ps;
        }
    };
    for (int kb = 0; kb < DS::NP; ++kb) {
        const int c0 = 32 * kb;
        stamp();
        if (warp == 0) {
            factor32_warp(S, DS::SP, c0, col, rd + c0, d_info, global_col0);
            invert32_warp<true>(S, DS::SP, c0, rd + c0, T + kb * 32 * DS::TP);
        } else if (kb > 0) {
            // rest of the trailing update of panel kb-1: macro-blocks (i, j), i >= 2, of the rows below it
            const int pc0 = c0 - 32, nmb = (BLK - c0) / 16, total = nmb * (nmb + 1) / 2;
            for (int u = 3 + warp - 1; u < total; u += kConsumerWarps - 1) {
                int i = (int)((sqrtf(8.0f * (float)u + 1.0f) - 1.0f) * 0.5f);
                while ((i + 1) * (i + 2) / 2 <= u) ++i;
                while (i * (i + 1) / 2 > u) --i;
                update_unit<BLK>(S, pc0, i, u - i * (i + 1) / 2);
            }
            // the columns of panel kb-1 are final (nobody writes them any more): off to global memory
            store_L_panel<BLK>(S, G, ldg, pc0, 32, kConsumerThreads - 32);
            if (DS::NP == 4 && kb == 3) {
                // look-ahead of the inverse: piece (1,0) needs T_0, T_1 and L_10, all final, L_10 stored two phases ago
                if (warp <= 4) inv_pair_first<BLK>(smem, 0, warp - 1);
                named_bar_sync<2, kConsumerThreads - 32>();
                if (warp <= 4) inv_pair_second<BLK>(smem, 0, warp - 1);
                pairs_done = 1u;
            }
        }
        stamp();
        cbar();
        if (kb + 1 < DS::NP) {
            stamp();
            const int units = (BLK - c0 - 32) / 16;
            for (int u = warp; u < units; u += kConsumerWarps) panel_unit<BLK>(S, T + kb * 32 * DS::TP, c0, u);
            cbar();
            stamp();
            if (warp < 3) update_unit<BLK>(S, c0, warp == 0 ? 0 : 1, warp == 2 ? 1 : 0);     // (0,0), (1,0), (1,1): piece kb+1
            cbar();
        }
    }
    stamp();
    // the last panel's columns (just the last diagonal piece)
    store_L_panel<BLK>(S, G, ldg, BLK - 32, 0, kConsumerThreads);
    return DS::NP == 4 ? 1u : pairs_done;    // (uniform: warp 0 did not go through the branch that sets it)
}

template <int BLK>
__device__ void load_lower_to_smem(double* S, const double* __restrict__ G, int ld) {
    constexpr int SP = DiagSmem<BLK>::SP;
    constexpr int PER = BLK * BLK / 2 / kConsumerThreads;   // double2 per thread (2, 8 or 32)
    constexpr int BATCH = PER < 16 ? PER : 16;               // 16-byte loads in flight per thread
    for (int b0 = 0; b0 < PER; b0 += BATCH) {
        double2 v[BATCH];
#pragma unroll
        for (int u = 0; u < BATCH; ++u) {
            const int idx = (b0 + u) * kConsumerThreads + threadIdx.x;
            const int r = idx / (BLK / 2), c = 2 * (idx % (BLK / 2));
            v[u] = (c <= r) ? __ldcg(reinterpret_cast<const double2*>(G + (size_t)r * ld + c)) : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int u = 0; u < BATCH; ++u) {
            const int idx = (b0 + u) * kConsumerThreads + threadIdx.x;
            const int r = idx / (BLK / 2), c = 2 * (idx % (BLK / 2));
            if (c == r) v[u].y = 0.0;                        // the element just above the diagonal
            *reinterpret_cast<double2*>(S + r * SP + c) = v[u];
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
    for (int idx = threadIdx.x; idx < BLK * BLK / 2; idx += kConsumerThreads) {
        const int r = idx / (BLK / 2), c = 2 * (idx % (BLK / 2));
        double2 v = make_double2(0.0, 0.0);
        if ((r >> 5) == (c >> 5)) v = *reinterpret_cast<const double2*>(T + (r >> 5) * 32 * DS::TP + (r & 31) * DS::TP + (c & 31));
        else if (c < r) v = *reinterpret_cast<const double2*>(S + r * DS::SP + c);
        __stcg(reinterpret_cast<double2*>(inv + (size_t)r * BLK + c), v);
    }
}

// POTRF job, all consumer threads: G = diagonal block (q,q) of L in global memory (leading
// dimension t), inv = invD(q).  smem is the (idle) operand ring.
template <int BLK>
__device__ void potrf_block(double* smem, double* __restrict__ G, int t, double* __restrict__ inv, int* d_info, int col0) {
    load_lower_to_smem<BLK>(smem, G, t);
    const unsigned pairs_done = chol_blocked<BLK>(smem, G, t, d_info, col0);
    cbar();                                  // every column of L has been read out of S before the inverse overwrites it
    inv_blocked<BLK>(smem, pairs_done);
    store_inverse<BLK>(smem, inv);
}

// inverse only (L given): the diagonal 32 x 32 inverses by one warp each, then the block assembly
template <int BLK>
__device__ void trtri_block(double* smem, const double* __restrict__ G, int t, double* __restrict__ inv) {
    using DS = DiagSmem<BLK>;
    load_lower_to_smem<BLK>(smem, G, t);
    const int warp = threadIdx.x >> 5;
    for (int kb = warp; kb < DS::NP; kb += kConsumerWarps)
        invert32_warp<false>(smem, DS::SP, 32 * kb, smem + DS::kRd + 32 * kb, smem + DS::kT + kb * 32 * DS::TP);
    cbar();
    inv_blocked<BLK>(smem);
    store_inverse<BLK>(smem, inv);
}

}  // namespace gpb
