// gp_gemm.cuh -- the one FP64 contraction of the pipeline:  C (-)= A * B^T
//
// A is [BM x K] row-major (leading dimension lda), B is [BN x K] row-major (ldb): the
// contraction index is contiguous in BOTH operands, which is exactly the form of every
// dense update in the tiled right-looking Cholesky and the predictor when tiles are stored
// row-major:
//   SYRK  K_II -= L_IJ L_IJ^T        (reading A3)
//   GEMM  K_IK -= L_IJ L_KJ^T        (reading A3)
//   TRSM  L_IJ  = K_IJ L_JJ^-T as products with inverted diagonal blocks
//   V solve / W = V^T V on the transposed factor V^T
//
// sm_100a has no FP64 kind of tcgen05.mma; the FP64 tensor path is the warp-level
// mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4), measured on this B200 at 37.19 TFLOP/s
// (= 148 SMs x 64 FMA/clk x 1.963 GHz, profiles/r01_fp64_peak.md), i.e. the full FP64 rate at
// 1/16 of the issue slots a DFMA loop needs.  One CTA computes a BM x BN block with 8 warps;
// operands are staged through a 4-deep cp.async (LDGSTS) ring in shared memory with a padded
// row stride (20 doubles) that makes every fragment LDS.64 bank-conflict-free.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gpb {

constexpr int kThreads = 256;       // 8 warps per CTA
constexpr int kBK = 16;             // contraction depth per pipeline stage (doubles)
constexpr int kStages = 4;
constexpr int kSmemStride = 20;     // doubles per staged row: 160 B, 160 mod 128 = 32 -> conflict-free

template <int BLK>
struct GemmCfg {
    // 8 warps as 2 (rows) x 4 (cols); each warp owns (BLK/2) x (BLK/4)
    static constexpr int WM = BLK / 2;
    static constexpr int WN = BLK / 4;
    static constexpr int MI = WM / 8;   // 8x8 accumulator blocks per warp along M
    static constexpr int NJ = WN / 8;   // and along N
    static constexpr int kStageDoubles = 2 * BLK * kSmemStride;
    static constexpr int kSmemBytes = kStages * kStageDoubles * 8;
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

enum GemmMode : int {
    kSub = 0,   // C <- C - A B^T
    kSet = 1,   // C <- A B^T            (C may alias A: all of A is read before C is written)
};

// Stage loader: rows [0,BLK) of A and of B, columns [k0, k0+kBK), into one ring slot.
template <int BLK>
__device__ __forceinline__ void gemm_load_stage(double* slot, const double* __restrict__ A, int lda,
                                                const double* __restrict__ B, int ldb, int k0, int tid) {
    constexpr int kChunksPerRow = kBK / 2;                 // 16-byte chunks
    constexpr int kChunks = BLK * kChunksPerRow;           // per operand
    double* sA = slot;
    double* sB = slot + BLK * kSmemStride;
#pragma unroll
    for (int c = tid; c < kChunks; c += kThreads) {
        const int row = c / kChunksPerRow, kc = c % kChunksPerRow;
        cp_async16(sA + row * kSmemStride + kc * 2, A + (size_t)row * lda + k0 + kc * 2);
    }
#pragma unroll
    for (int c = tid; c < kChunks; c += kThreads) {
        const int row = c / kChunksPerRow, kc = c % kChunksPerRow;
        cp_async16(sB + row * kSmemStride + kc * 2, B + (size_t)row * ldb + k0 + kc * 2);
    }
}

// One CTA: C[BLK x BLK] (ldc) (-)= A[BLK x K] * B[BLK x K]^T.   K % kBK == 0, K >= kBK.
// lower_only: skip the store of 8x8 accumulator blocks strictly above the diagonal of the
// block (used for diagonal blocks of the symmetric matrix; their upper part is never read).
// All 256 threads must call this; `smem` is the dynamic shared memory ring.
template <int BLK>
__device__ __forceinline__ void gemm_nt_block(double* __restrict__ C, int ldc, const double* __restrict__ A,
                                              int lda, const double* __restrict__ B, int ldb, int K,
                                              int mode, double* smem) {
    using Cfg = GemmCfg<BLK>;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = lane >> 2, t = lane & 3;
    const int wm = (warp >> 2) * Cfg::WM, wn = (warp & 3) * Cfg::WN;

    double acc[Cfg::MI][Cfg::NJ][2];
    const int KT = K / kBK;

    // prologue: first kStages-1 stages in flight before anything else
#pragma unroll
    for (int s = 0; s < kStages - 1; ++s) {
        if (s < KT) gemm_load_stage<BLK>(smem + s * Cfg::kStageDoubles, A, lda, B, ldb, s * kBK, tid);
        cp_async_commit();
    }
    // accumulators start at -C (kSub) so that the final store is -(acc) = C - A B^T
    if (mode == kSub) {
#pragma unroll
        for (int i = 0; i < Cfg::MI; ++i)
#pragma unroll
            for (int j = 0; j < Cfg::NJ; ++j) {
                const double2 c = __ldcg(reinterpret_cast<const double2*>(
                    C + (size_t)(wm + 8 * i + g) * ldc + wn + 8 * j + 2 * t));
                acc[i][j][0] = -c.x;
                acc[i][j][1] = -c.y;
            }
    } else {
#pragma unroll
        for (int i = 0; i < Cfg::MI; ++i)
#pragma unroll
            for (int j = 0; j < Cfg::NJ; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    }

    for (int kt = 0; kt < KT; ++kt) {
        cp_async_wait<kStages - 2>();
        __syncthreads();
        {
            const int nk = kt + kStages - 1;
            if (nk < KT) gemm_load_stage<BLK>(smem + (nk % kStages) * Cfg::kStageDoubles, A, lda, B, ldb, nk * kBK, tid);
            cp_async_commit();
        }
        const double* sA = smem + (kt % kStages) * Cfg::kStageDoubles + (wm + g) * kSmemStride + t;
        const double* sB = smem + (kt % kStages) * Cfg::kStageDoubles + BLK * kSmemStride + (wn + g) * kSmemStride + t;
#pragma unroll
        for (int ks = 0; ks < kBK / 4; ++ks) {
            double a[Cfg::MI], b[Cfg::NJ];
#pragma unroll
            for (int i = 0; i < Cfg::MI; ++i) a[i] = sA[i * 8 * kSmemStride + ks * 4];
#pragma unroll
            for (int j = 0; j < Cfg::NJ; ++j) b[j] = sB[j * 8 * kSmemStride + ks * 4];
#pragma unroll
            for (int i = 0; i < Cfg::MI; ++i)
#pragma unroll
                for (int j = 0; j < Cfg::NJ; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_async_wait<0>();
    __syncthreads();   // every read of A/B (and of the ring) is complete: C may alias A, ring may be reused

    const double sgn = (mode == kSub) ? -1.0 : 1.0;
#pragma unroll
    for (int i = 0; i < Cfg::MI; ++i)
#pragma unroll
        for (int j = 0; j < Cfg::NJ; ++j) {
            double2 c;
            c.x = sgn * acc[i][j][0];
            c.y = sgn * acc[i][j][1];
            __stcg(reinterpret_cast<double2*>(C + (size_t)(wm + 8 * i + g) * ldc + wn + 8 * j + 2 * t), c);
        }
}

}  // namespace gpb
