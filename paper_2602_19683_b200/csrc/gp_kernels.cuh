// gp_kernels.cuh -- the HBM/ALU-bound kernels of the pipeline: fused covariance assembly
// (a1, a9), tile unpacking, the two triangular solves for alpha (a7, a8) and the fused
// cross-covariance + mean (a9, a10).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gp_tma.cuh"

namespace gpb {

struct HyperDev {
    double neg_inv_den;   // -1/den, den = 2*ell (Eq. 1 as printed) or 2*ell^2 (reading A1); formed once on the host:
                          // an FP64 division per matrix entry (~25 instructions, more than the exp) made the
                          // assembly issue-bound; exact for den a power of two (ell = 1, 2), else <= 1 ulp in the exponent
    double vertical;  // v
    double noise;     // sigma^2
};

// exp(x) for x <= 0, the only range Eq. 1 needs (x = -r^2/den).  The library exp() carries
// special-case branches and selects that made the assembly ISSUE-bound (ncu: issue slots 77 % busy,
// FP64 pipe 54 %); this is the same algorithm without them: k = round(x log2 e) by the 1.5*2^52 trick,
// f = x - k ln2 in two FMAs (|f| <= 0.347), degree-13 Taylor polynomial in Horner form (truncation
// 4e-18 relative), 2^k added into the exponent field.  Error ~1 ulp, like the library's.  Results
// below 2^-1021 (x < -708) are flushed to 0: an absolute error of 3e-308.
__device__ __forceinline__ double exp_nonpos(double x) {
    const double kMagic = 6755399441055744.0;                  // 1.5 * 2^52
    const double t = fma(x, 1.4426950408889634, kMagic);
    const int k = __double2loint(t);                           // round(x * log2 e), two's complement in the low word
    const double kd = t - kMagic;
    double f = fma(kd, -6.93147180369123816490e-01, x);        // ln2 high part (21 trailing zero bits)
    f = fma(kd, -1.90821492927058770002e-10, f);               // ln2 low part
    double p = 1.6059043836821613e-10;                         // 1/13!
    p = fma(p, f, 2.08767569878681e-09);                       // 1/12!
    p = fma(p, f, 2.505210838544172e-08);                      // 1/11!
    p = fma(p, f, 2.755731922398589e-07);                      // 1/10!
    p = fma(p, f, 2.7557319223985893e-06);                     // 1/9!
    p = fma(p, f, 2.48015873015873e-05);                       // 1/8!
    p = fma(p, f, 1.984126984126984e-04);                      // 1/7!
    p = fma(p, f, 1.388888888888889e-03);                      // 1/6!
    p = fma(p, f, 8.333333333333333e-03);                      // 1/5!
    p = fma(p, f, 4.1666666666666664e-02);                     // 1/4!
    p = fma(p, f, 1.6666666666666666e-01);                     // 1/3!
    p = fma(p, f, 0.5);
    p = fma(p, f, 1.0);
    p = fma(p, f, 1.0);
    const double r = __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
    return (x < -708.0) ? 0.0 : r;
}

// k(a,b) without the noise term -- PAPER.md:63, Eq. 1.  r2 accumulated in index order with FMA.
__device__ __forceinline__ double se_kernel(double r2, const HyperDev& h) { return h.vertical * exp_nonpos(r2 * h.neg_inv_den); }

// ---------------------------------------------------------------------------------------------
// Fused assembly: distance, exp, noise in one pass, one 64x64 output sub-block per CTA.
// Each thread produces a 4x4 patch (rows ty+16i, columns 4tx..4tx+3): 32 B contiguous per row
// per thread, a warp writes two full 512 B row segments per store pair -> fully coalesced.
// 1-D grid: blockIdx.x = tile index * sub-blocks per tile + sub-block.
// sym_lower: tile list is the lower-packed (I,J), J<=I; noise is added where global i == j.
// ---------------------------------------------------------------------------------------------
constexpr int kAsmBlk = 64;
constexpr int kAsmMaxD = 32;   // features staged in shared memory per pass; larger D is processed in chunks

__global__ void __launch_bounds__(256) assemble_tiles_kernel(const double* __restrict__ A, const double* __restrict__ B,
                                                             int D, HyperDev h, int tile, int tiles_b /* tiles per row (general) */,
                                                             int sym_lower, double* __restrict__ out) {
    extern __shared__ __align__(16) double sm[];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    // tile coordinates
    int I, J;
    const int sb = (tile + kAsmBlk - 1) / kAsmBlk;
    const int tidx = blockIdx.x / (sb * sb), sub = blockIdx.x % (sb * sb);
    if (sym_lower) {
        // invert tidx = I(I+1)/2 + J
        I = (int)((sqrt(8.0 * (double)tidx + 1.0) - 1.0) * 0.5);
        while ((int64_t)(I + 1) * (I + 2) / 2 <= tidx) ++I;
        while ((int64_t)I * (I + 1) / 2 > tidx) --I;
        J = tidx - (int)((int64_t)I * (I + 1) / 2);
    } else {
        I = tidx / tiles_b;
        J = tidx % tiles_b;
    }
    const int r0 = (sub / sb) * kAsmBlk, c0 = (sub % sb) * kAsmBlk;   // inside the tile
    const int64_t gi0 = (int64_t)I * tile + r0, gj0 = (int64_t)J * tile + c0;
    const int nrow = min(kAsmBlk, tile - r0), ncol = min(kAsmBlk, tile - c0);

    double acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;

    double* sA = sm;                       // [dchunk][64]  (d-major so that rows are bank-spread)
    double* sB = sm + kAsmMaxD * kAsmBlk;  // [dchunk][64]
    for (int d0 = 0; d0 < D; d0 += kAsmMaxD) {
        const int dc = min(kAsmMaxD, D - d0);
        __syncthreads();
        for (int idx = tid; idx < kAsmBlk * dc; idx += 256) {
            const int r = idx / dc, d = idx % dc;
            sA[d * kAsmBlk + r] = (r < nrow) ? A[(gi0 + r) * D + d0 + d] : 0.0;
            sB[d * kAsmBlk + r] = (r < ncol) ? B[(gj0 + r) * D + d0 + d] : 0.0;
        }
        __syncthreads();
        for (int d = 0; d < dc; ++d) {
            double a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = sA[d * kAsmBlk + ty + 16 * i];
            const double2 b01 = *reinterpret_cast<const double2*>(sB + d * kAsmBlk + 4 * tx);
            const double2 b23 = *reinterpret_cast<const double2*>(sB + d * kAsmBlk + 4 * tx + 2);
            b[0] = b01.x; b[1] = b01.y; b[2] = b23.x; b[3] = b23.y;
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const double diff = a[i] - b[j];
                    acc[i][j] = fma(diff, diff, acc[i][j]);
                }
        }
    }
    double* tbase = out + (size_t)tidx * tile * tile;
    const bool on_diagonal = sym_lower && gi0 == gj0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int r = ty + 16 * i;
        if (r >= nrow || 4 * tx >= ncol) continue;
        double k[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) k[j] = se_kernel(acc[i][j], h);
        if (on_diagonal) {      // CTA-uniform: only sub-blocks that straddle the global diagonal carry noise
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (r == 4 * tx + j) k[j] += h.noise;
        }
        double* dst = tbase + (size_t)(r0 + r) * tile + c0 + 4 * tx;
        __stcs(reinterpret_cast<double2*>(dst), make_double2(k[0], k[1]));
        __stcs(reinterpret_cast<double2*>(dst) + 1, make_double2(k[2], k[3]));
    }
}

// Dense rectangular variant: out [na x nb] row-major with leading dimension ld, out(i, j) = k(A_i, B_j), never any noise
// (the prior K_{X^_r, X^} of a block of test points against all of them, for the sharded covariance rows).
__global__ void __launch_bounds__(256) assemble_dense_kernel(const double* __restrict__ A, int64_t na, const double* __restrict__ B,
                                                             int64_t nb, int D, HyperDev h, double* __restrict__ out, int64_t ld) {
    extern __shared__ __align__(16) double sm[];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int64_t cb = (nb + kAsmBlk - 1) / kAsmBlk;
    const int64_t gi0 = (int64_t)(blockIdx.x / cb) * kAsmBlk, gj0 = (int64_t)(blockIdx.x % cb) * kAsmBlk;
    const int nrow = (int)min((int64_t)kAsmBlk, na - gi0), ncol = (int)min((int64_t)kAsmBlk, nb - gj0);
    double acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
    double* sA = sm;
    double* sB = sm + kAsmMaxD * kAsmBlk;
    for (int d0 = 0; d0 < D; d0 += kAsmMaxD) {
        const int dc = min(kAsmMaxD, D - d0);
        __syncthreads();
        for (int idx = tid; idx < kAsmBlk * dc; idx += 256) {
            const int r = idx / dc, d = idx % dc;
            sA[d * kAsmBlk + r] = (r < nrow) ? A[(gi0 + r) * D + d0 + d] : 0.0;
            sB[d * kAsmBlk + r] = (r < ncol) ? B[(gj0 + r) * D + d0 + d] : 0.0;
        }
        __syncthreads();
        for (int d = 0; d < dc; ++d) {
            double a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = sA[d * kAsmBlk + ty + 16 * i];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = sB[d * kAsmBlk + 4 * tx + j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const double diff = a[i] - b[j];
                    acc[i][j] = fma(diff, diff, acc[i][j]);
                }
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int r = ty + 16 * i;
        if (r >= nrow) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (4 * tx + j < ncol) out[(gi0 + r) * ld + gj0 + 4 * tx + j] = se_kernel(acc[i][j], h);
    }
}

// work items of the sharded covariance rows: block row gr0 + i of V^T against every block row gc, the whole contraction
// range in one item (no item depends on another)
__global__ void cov_row_items_kernel(uint4* __restrict__ items, int rows, int gr0, int NBm, int NB, unsigned op) {
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < rows * NBm; idx += gridDim.x * blockDim.x)
        items[idx] = make_uint4(op, (unsigned)(gr0 + idx / NBm), (unsigned)(idx % NBm), (unsigned)NB << 16);
}

// ROW_V items of one tile column: item i = (op, gr = i, gc = first block column of the tile column, 0)
__global__ void row_items_set_column_kernel(uint4* __restrict__ items, int rows, unsigned gc) {
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < rows; idx += gridDim.x * blockDim.x) {
        uint4 it = items[idx];
        it.y = (unsigned)idx;
        it.z = gc;
        it.w = 0u;
        items[idx] = it;
    }
}

// tiles -> dense (inspection helper)
__global__ void tiles_to_dense_kernel(const double* __restrict__ tiles, int64_t n, int64_t nb, int tile, int lower_packed,
                                      double* __restrict__ dense) {
    const int64_t total = n * nb;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = idx / nb, j = idx % nb;
        const int64_t I = i / tile, J = j / tile;
        double v = 0.0;
        if (lower_packed) {
            if (j <= i) v = tiles[((size_t)I * (I + 1) / 2 + J) * tile * tile + (i % tile) * tile + (j % tile)];
        } else {
            v = tiles[((size_t)I * (nb / tile) + J) * tile * tile + (i % tile) * tile + (j % tile)];
        }
        dense[idx] = v;
    }
}

// Sigma: copy the lower triangle onto the upper one so both are bit-identical (reading A12).
__global__ void mirror_lower_kernel(double* __restrict__ S, int64_t m) {
    __shared__ double tile[32][33];
    const int bi = blockIdx.y, bj = blockIdx.x;
    if (bj > bi) return;
    const int tx = threadIdx.x, ty = threadIdx.y;   // 32 x 8
    for (int r = ty; r < 32; r += 8) tile[r][tx] = S[((int64_t)bi * 32 + r) * m + (int64_t)bj * 32 + tx];
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        // element (bj*32 + r, bi*32 + tx) <- (bi*32 + tx, bj*32 + r)
        const int64_t row = (int64_t)bj * 32 + r, col = (int64_t)bi * 32 + tx;
        if (col > row) S[row * m + col] = tile[tx][r];
    }
}

// Predictive variances: var_a = prior - sum_i V^T[a][i]^2 over the
// general tiles of V^T (m x n).  One warp per test point, lanes stride the row, fixed reduction order.
__global__ void __launch_bounds__(256) posterior_var_kernel(const double* __restrict__ Vt, int64_t m, int64_t n, int tile,
                                                            double prior, double* __restrict__ var) {
    const int lane = threadIdx.x & 31;
    const int64_t a = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (a >= m) return;
    const int64_t Mt = n / tile;
    const double* rowbase = Vt + (a / tile) * Mt * (size_t)tile * tile + (a % tile) * (size_t)tile;
    double s = 0.0;
    for (int64_t J = 0; J < Mt; ++J) {
        const double2* row = reinterpret_cast<const double2*>(rowbase + J * (size_t)tile * tile);
        for (int c = lane; c < tile / 2; c += 32) {
            const double2 v = __ldcs(row + c);
            s = fma(v.x, v.x, s);
            s = fma(v.y, v.y, s);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) var[a] = prior - s;
}

// log p(y) = -1/2 y^T alpha - sum_i log L_ii - n/2 log(2 pi).  One CTA, fixed order.
__global__ void __launch_bounds__(1024) log_marginal_likelihood_kernel(const double* __restrict__ L, int64_t n, int tile,
                                                                        const double* __restrict__ y, const double* __restrict__ alpha,
                                                                        double* __restrict__ out) {
    __shared__ double s_q[32], s_l[32];
    double q = 0.0, ld = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += 1024) {
        q = fma(y[i], alpha[i], q);
        const int64_t I = i / tile, r = i % tile;
        ld += log(L[((size_t)I * (I + 1) / 2 + I) * (size_t)tile * tile + r * (size_t)tile + r]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { q += __shfl_xor_sync(0xffffffffu, q, o); ld += __shfl_xor_sync(0xffffffffu, ld, o); }
    if ((threadIdx.x & 31) == 0) { s_q[threadIdx.x >> 5] = q; s_l[threadIdx.x >> 5] = ld; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tq = 0.0, tl = 0.0;
        for (int k = 0; k < 32; ++k) { tq += s_q[k]; tl += s_l[k]; }
        out[0] = -0.5 * tq - tl - 0.5 * (double)n * 1.8378770664093454835606594728112;   // log(2 pi)
    }
}

// ---------------------------------------------------------------------------------------------
// Triangular solves for alpha.  Block rows/columns of SB (= the executor's block
// edge).  One CTA per block row; rows are handed out by a ticket so that a CTA only ever waits for
// rows claimed before it.  The off-diagonal part is a streaming GEMV that consumes x_p as soon as
// block p publishes it; the diagonal block is applied as a GEMV with its inverse.
//
// The n/SB diagonal steps form a latency chain (x_i needs x_{i-1}); everything else is bandwidth.
// To keep the chain short, a CTA (a) copies its inverted diagonal block into shared memory with
// cp.async before it starts streaming, (b) loads every block of L into registers BEFORE it waits
// for the matching piece of x, so that on the critical last block only the flag, 4 doubles of x,
// two shuffle reductions and the publish remain, and (c) lets every warp poll the flag itself
// instead of going through a CTA barrier.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int ld_acquire_i(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// relaxed gpu-scope accesses to the published solution: they go to L2, where every SM sees them
__device__ __forceinline__ double2 solve_ld2(const double* p) {
    double2 v;
    asm volatile("ld.relaxed.gpu.global.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ double solve_ld1(const double* p) {
    double v;
    asm volatile("ld.relaxed.gpu.global.f64 %0, [%1];\n" : "=d"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void solve_st1(double* p, double v) { asm volatile("st.relaxed.gpu.global.f64 [%0], %1;\n" ::"l"(p), "d"(v) : "memory"); }
__device__ __forceinline__ bool solve_pending(double v) { return __double_as_longlong(v) == kSolvePending; }
__device__ __forceinline__ void cp_async16_solve(void* smem_dst, const void* gmem_src) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all_solve() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

__device__ __forceinline__ const double* tile_block_ptr(const double* L, int t, int sbt, int gr, int gc, int sb) {
    const int I = gr / sbt, J = gc / sbt;
    return L + ((size_t)I * (I + 1) / 2 + J) * (size_t)t * t + (size_t)(gr % sbt) * sb * t + (size_t)(gc % sbt) * sb;
}

template <int SB>
struct SolveCfg {
    static constexpr int TX = SB / 4;             // threads across a row (4 columns each); divides 32
    static constexpr int TY = 256 / TX;           // row groups
    static constexpr int RPT = SB / TY;           // rows per thread
    // blocks of L in flight per CTA (register buffers of RPT x 4 doubles each).  More than one was measured for the 64- and
    // 32-row kernels (4 in flight): c2 0.396 -> 0.381 ms, c1 0.065 -> 0.069 ms, c3 with 64-row blocks 2.31 -> 2.66 ms: the
    // solves are not bound by the latency of a CTA's own stream (at c3 they move 4 TB/s, 62 % of the measured HBM rate,
    // at the smaller sizes the chain of diagonal steps is the bound), so one block in flight it stays.
    static constexpr int PD = 1;
    static constexpr int kSmemBytes = SB * SB * 8 + SB * 8 + TY * SB * 8;   // invD, rhs, cross-warp partials
};

// sum over the TX lanes that share a row group (TX is a power of two <= 32, groups are lane-aligned)
template <int TX>
__device__ __forceinline__ double group_sum(double v) {
#pragma unroll
    for (int o = TX / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Forward: x_i = invD_i (y_i - sum_{p<i} L(i,p) x_p).
template <int SB>
__global__ void __launch_bounds__(256, 1) forward_solve_kernel(const double* __restrict__ L, int t, int NB,
                                                               const double* __restrict__ invD, const double* __restrict__ y,
                                                               double* x, double* next_x, unsigned int* ticket) {
    using Cfg = SolveCfg<SB>;
    constexpr int TX = Cfg::TX, TY = Cfg::TY, RPT = Cfg::RPT;
    extern __shared__ __align__(16) double sm[];
    double* s_inv = sm;                 // SB x SB, row-major
    double* s_rhs = sm + SB * SB;       // SB
    __shared__ unsigned int s_row;
    __shared__ __align__(16) double s_x[2][SB];
    const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
    const int sbt = t / SB;
    if (tid == 0) s_row = atomicAdd(ticket, 1u);
    __syncthreads();
    const int i = (int)s_row;
    if (i >= NB) return;
    {   // (a) the inverted diagonal block, in the background
        const double* inv = invD + (size_t)i * SB * SB;
        for (int idx = tid; idx < SB * SB / 2; idx += 256) cp_async16_solve(s_inv + 2 * idx, inv + 2 * idx);
    }
    double acc[RPT];
#pragma unroll
    for (int r = 0; r < RPT; ++r) acc[r] = 0.0;
    constexpr int PD = Cfg::PD;
    double2 l[PD][RPT][2];
    auto load_block = [&](int slot, int pb) {      // (b) the blocks of L first ...
        const double* blk = tile_block_ptr(L, t, sbt, i, pb, SB);
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            const double2* row = reinterpret_cast<const double2*>(blk + (size_t)(ty + TY * r) * t + 4 * tx);
            l[slot][r][0] = __ldcs(row);
            l[slot][r][1] = __ldcs(row + 1);
        }
    };
#pragma unroll
    for (int sl = 0; sl < PD; ++sl)
        if (sl < i) load_block(sl, sl);
    for (int pb0 = 0; pb0 < i; pb0 += PD) {
#pragma unroll
        for (int sl = 0; sl < PD; ++sl) {
            const int pb = pb0 + sl;
            if (pb >= i) break;
            // (c) ... then the wait for x_p.  ONE warp polls the values (its lanes cover the whole piece) and hands them to
            // the others through shared memory: with every warp of every CTA polling, the L2 slice that holds x_p was
            // crowded (c3: 2.8 ms instead of 2.3), and a back-off costs more than it saves (__nanosleep is coarse: 4.9 ms).
            double* sx = s_x[pb & 1];
            if (tid < SB / 4) {
                double2 p01, p23;
                do {
                    p01 = solve_ld2(x + (size_t)pb * SB + 4 * tid);
                    p23 = solve_ld2(x + (size_t)pb * SB + 4 * tid + 2);
                } while (solve_pending(p01.x) || solve_pending(p01.y) || solve_pending(p23.x) || solve_pending(p23.y));
                *reinterpret_cast<double2*>(sx + 4 * tid) = p01;
                *reinterpret_cast<double2*>(sx + 4 * tid + 2) = p23;
            }
            __syncthreads();     // one barrier per block: the buffer written two blocks later is read before the next barrier
            const double2 x01 = *reinterpret_cast<const double2*>(sx + 4 * tx), x23 = *reinterpret_cast<const double2*>(sx + 4 * tx + 2);
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                acc[r] = fma(l[sl][r][0].x, x01.x, acc[r]);
                acc[r] = fma(l[sl][r][0].y, x01.y, acc[r]);
                acc[r] = fma(l[sl][r][1].x, x23.x, acc[r]);
                acc[r] = fma(l[sl][r][1].y, x23.y, acc[r]);
            }
            if (pb + PD < i) load_block(sl, pb + PD);
        }
    }
#pragma unroll
    for (int r = 0; r < RPT; ++r) acc[r] = group_sum<TX>(acc[r]);
    if (tx == 0) {
#pragma unroll
        for (int r = 0; r < RPT; ++r) s_rhs[ty + TY * r] = y[(size_t)i * SB + ty + TY * r] - acc[r];
    }
    cp_async_wait_all_solve();
    __syncthreads();
    // x_i = invD_i * rhs  (lower triangular inverse; its strict upper part is stored as zeros)
    double part[RPT];
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
        const double* row = s_inv + (size_t)(ty + TY * r) * SB + 4 * tx;
        part[r] = row[0] * s_rhs[4 * tx] + row[1] * s_rhs[4 * tx + 1] + row[2] * s_rhs[4 * tx + 2] + row[3] * s_rhs[4 * tx + 3];
    }
#pragma unroll
    for (int r = 0; r < RPT; ++r) part[r] = group_sum<TX>(part[r]);
    if (tx == 0) {
#pragma unroll
        for (int r = 0; r < RPT; ++r) solve_st1(x + (size_t)i * SB + ty + TY * r, part[r]);   // published by value: no flag, no fence
    }
    // y_i has been consumed (only this CTA reads it): mark block i of the backward solve's output "not yet computed"
    // (next_x may alias y)
    if (next_x != nullptr && tid < SB) next_x[(size_t)i * SB + tid] = __longlong_as_double(kSolvePending);
}

// Backward: x_j = invD_j^T (b_j - sum_{i>j} L(i,j)^T x_i); block columns handed out from the last.
template <int SB>
__global__ void __launch_bounds__(256, 1) backward_solve_kernel(const double* __restrict__ L, int t, int NB,
                                                                const double* __restrict__ invD, const double* __restrict__ b,
                                                                double* x, unsigned int* ticket) {
    using Cfg = SolveCfg<SB>;
    constexpr int TX = Cfg::TX, TY = Cfg::TY, RPT = Cfg::RPT;
    extern __shared__ __align__(16) double sm[];
    double* s_inv = sm;                          // SB x SB, row-major
    double* s_rhs = sm + SB * SB;                // SB
    double* s_part = sm + SB * SB + SB;          // TY x SB partial column sums
    __shared__ unsigned int s_col;
    __shared__ __align__(16) double s_x[2][SB];
    const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
    const int sbt = t / SB;
    if (tid == 0) s_col = atomicAdd(ticket, 1u);
    __syncthreads();
    if ((int)s_col >= NB) return;
    const int j = NB - 1 - (int)s_col;
    {
        const double* inv = invD + (size_t)j * SB * SB;
        for (int idx = tid; idx < SB * SB / 2; idx += 256) cp_async16_solve(s_inv + 2 * idx, inv + 2 * idx);
    }
    double acc[4] = {0.0, 0.0, 0.0, 0.0};        // columns 4tx..4tx+3, partial over this thread's rows
    constexpr int PD = Cfg::PD;
    double2 l[PD][RPT][2];
    auto load_block = [&](int slot, int ib) {
        const double* blk = tile_block_ptr(L, t, sbt, ib, j, SB);
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            const double2* row = reinterpret_cast<const double2*>(blk + (size_t)(ty + TY * r) * t + 4 * tx);
            l[slot][r][0] = __ldcs(row);
            l[slot][r][1] = __ldcs(row + 1);
        }
    };
#pragma unroll
    for (int sl = 0; sl < PD; ++sl)
        if (NB - 1 - sl > j) load_block(sl, NB - 1 - sl);
    for (int ib0 = NB - 1; ib0 > j; ib0 -= PD) {
#pragma unroll
        for (int sl = 0; sl < PD; ++sl) {
            const int ib = ib0 - sl;
            if (ib <= j) break;
            double* sx = s_x[ib & 1];            // x_ib: polled by value by one warp, handed over through shared memory
            if (tid < SB / 4) {
                double2 p01, p23;
                do {
                    p01 = solve_ld2(x + (size_t)ib * SB + 4 * tid);
                    p23 = solve_ld2(x + (size_t)ib * SB + 4 * tid + 2);
                } while (solve_pending(p01.x) || solve_pending(p01.y) || solve_pending(p23.x) || solve_pending(p23.y));
                *reinterpret_cast<double2*>(sx + 4 * tid) = p01;
                *reinterpret_cast<double2*>(sx + 4 * tid + 2) = p23;
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const double xv = sx[ty + TY * r];
                acc[0] = fma(l[sl][r][0].x, xv, acc[0]);
                acc[1] = fma(l[sl][r][0].y, xv, acc[1]);
                acc[2] = fma(l[sl][r][1].x, xv, acc[2]);
                acc[3] = fma(l[sl][r][1].y, xv, acc[3]);
            }
            if (ib - PD > j) load_block(sl, ib - PD);
        }
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) s_part[ty * SB + 4 * tx + c] = acc[c];
    cp_async_wait_all_solve();
    __syncthreads();
    if (tid < SB) {
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < TY; ++k) s += s_part[k * SB + tid];
        s_rhs[tid] = b[(size_t)j * SB + tid] - s;
    }
    __syncthreads();
    // x_j = invD_j^T rhs:  x[c] = sum_r inv[r][c] rhs[r]
    double part[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
        const int rr = ty + TY * r;
        const double rv = s_rhs[rr];
        const double* row = s_inv + (size_t)rr * SB + 4 * tx;
        part[0] = fma(row[0], rv, part[0]);
        part[1] = fma(row[1], rv, part[1]);
        part[2] = fma(row[2], rv, part[2]);
        part[3] = fma(row[3], rv, part[3]);
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) s_part[ty * SB + 4 * tx + c] = part[c];
    __syncthreads();
    if (tid < SB) {
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < TY; ++k) s += s_part[k * SB + tid];
        solve_st1(x + (size_t)j * SB + tid, s);
    }
}

// ---------------------------------------------------------------------------------------------
// Predictive mean, fused with the cross-covariance: mean[a] = sum_i k(xs_a, x_i) alpha_i.
// One CTA per kMeanTM test points; each thread strides over training points.  D <= kMeanMaxD staged
// in registers per training point; the test points live in shared memory.
// ---------------------------------------------------------------------------------------------
constexpr int kMeanTM = 8;

__global__ void __launch_bounds__(256) predict_mean_kernel(const double* __restrict__ X, int64_t n, int D,
                                                           const double* __restrict__ alpha, const double* __restrict__ Xs,
                                                           int64_t m, HyperDev h, double* __restrict__ mean) {
    extern __shared__ __align__(16) double sm[];   // [kMeanTM][D] test points, then [kMeanTM][256] reduction
    double* sXs = sm;
    double* sRed = sm + kMeanTM * D;
    const int tid = threadIdx.x;
    const int64_t a0 = (int64_t)blockIdx.x * kMeanTM;
    const int na = (int)min((int64_t)kMeanTM, m - a0);
    for (int idx = tid; idx < kMeanTM * D; idx += 256) {
        const int a = idx / D, d = idx % D;
        sXs[idx] = (a < na) ? Xs[(a0 + a) * D + d] : 0.0;
    }
    __syncthreads();
    double acc[kMeanTM];
#pragma unroll
    for (int a = 0; a < kMeanTM; ++a) acc[a] = 0.0;
    for (int64_t i = tid; i < n; i += 256) {
        double r2[kMeanTM];
#pragma unroll
        for (int a = 0; a < kMeanTM; ++a) r2[a] = 0.0;
        const double* xi = X + i * D;
        for (int d = 0; d < D; ++d) {
            const double xv = xi[d];
#pragma unroll
            for (int a = 0; a < kMeanTM; ++a) {
                const double diff = sXs[a * D + d] - xv;
                r2[a] = fma(diff, diff, r2[a]);
            }
        }
        const double al = alpha[i];
#pragma unroll
        for (int a = 0; a < kMeanTM; ++a) acc[a] = fma(se_kernel(r2[a], h), al, acc[a]);
    }
#pragma unroll
    for (int a = 0; a < kMeanTM; ++a) sRed[a * 256 + tid] = acc[a];
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (tid < s) {
#pragma unroll
            for (int a = 0; a < kMeanTM; ++a) sRed[a * 256 + tid] += sRed[a * 256 + tid + s];
        }
        __syncthreads();
    }
    if (tid < na) mean[a0 + tid] = sRed[tid * 256];
}

}  // namespace gpb
