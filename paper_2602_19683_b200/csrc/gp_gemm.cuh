// gp_gemm.cuh -- the one FP64 contraction of the pipeline:  C (-)= A * B^T   (consumer side)
//
// A is [BLK x K] row-major, B is [BLK x K] row-major: the contraction index is contiguous in BOTH
// operands, which is exactly the form of every dense update in the tiled right-looking Cholesky
// and the predictor when tiles are stored row-major:
//   SYRK  K_II -= L_IJ L_IJ^T        (reading A3)
//   GEMM  K_IK -= L_IJ L_KJ^T        (reading A3)
//   TRSM  L_IJ  = K_IJ L_JJ^-T as products with inverted diagonal blocks
//   V solve / W = V^T V on the transposed factor V^T
//
// sm_100a has no FP64 kind of tcgen05.mma; the FP64 tensor path is the warp-level
// mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4), measured on this B200 at 37.1 TFLOP/s
// (= 148 SMs x 64 FMA/clk x 1.965 GHz), i.e. the full FP64 rate at 1/16 of the issue slots a DFMA
// loop needs.  An LDS.64 + DMMA loop over operands that are already in shared memory reaches that
// rate with 8 warps of 64x32 (measured 37.0 TFLOP/s); what kept the first version of this kernel
// at 75 % was the all-thread cp.async issue and the CTA-wide barrier per k-stage.  So the operands
// now arrive by TMA (one elected producer lane, gp_exec.cuh) into a ring of 128-byte-swizzled
// stages guarded by full/empty mbarriers, and the 8 consumer warps here never meet a CTA barrier.
//
// Stage layout (per operand): BLK rows x 16 doubles = BLK x 128 B, written by TMA with
// CU_TENSOR_MAP_SWIZZLE_128B: the 16-byte chunk c of row r sits at chunk (c ^ (r & 7)).
// Fragment mapping: DMMA lane (g = lane/4, t = lane%4) supplies A[row g][k t].  Accumulator
// block i of a warp uses the rows  16*(i/2) + 2*g + (i%2)  of the warp's slab, so the four rows a
// half-warp touches differ in bits 1-2 of (r & 7) and its 16 LDS.64 fall into 16 distinct 8-byte
// bank pairs: conflict-free under the TMA swizzle, no padding.  Columns (B rows) likewise.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gp_tma.cuh"

namespace gpb {

constexpr int kConsumerWarps = 8;
constexpr int kConsumerThreads = kConsumerWarps * 32;
constexpr int kThreads = kConsumerThreads + 128;  // + the producer warpgroup (one working warp; registers are
                                                  //   re-balanced per warpgroup with setmaxnreg, which is why it is a whole one)
constexpr int kConsumerRegs = 224;                // the CTA is launched with 384 x 168 registers; 256 x 224 + 128 x 56 is the same pool
constexpr int kProducerRegs = 56;
constexpr int kBK = 16;                           // contraction depth per stage = one 128-byte swizzle row
constexpr int kStages = 7;                       // 7 x 32 KB (b = 128) + barriers fits the 227 KB of an SM; one stage is always held back (deferred release)
constexpr int kJobSlots = 4;

template <int BLK>
struct GemmCfg {
    // 8 warps as 2 (rows) x 4 (cols); each warp owns (BLK/2) x (BLK/4)
    static constexpr int WM = BLK / 2;
    static constexpr int WN = BLK / 4;
    static constexpr int MI = WM / 8;   // 8x8 accumulator blocks per warp along M (2, 4 or 8: even)
    static constexpr int NJ = WN / 8;   // and along N (1, 2 or 4)
    // A stage holds kSub sub-tiles of kBK columns per operand (each BLK rows x 128 B, written by its own TMA box).  64-blocks
    // take two: a 16-deep stage is only 32 DMMAs per warp, and the full/empty barrier round of every stage cost ~10 % of
    // the 64-block contraction (2.6 us per 64^3 product against 2.1 at the pipe's rate).
    static constexpr int kSub = BLK == 64 ? 2 : 1;
    static constexpr int kStageDepth = kBK * kSub;
    static constexpr int kSubBytes = BLK * kBK * 8;
    static constexpr int kOperandBytes = kSubBytes * kSub;
    static constexpr int kStageBytes = 2 * kOperandBytes;
    static constexpr int kRingBytes = kStages * kStageBytes;
    static_assert(MI % 2 == 0, "row interleave needs an even number of accumulator blocks");
};

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

enum GemmMode : int {
    kSub = 0,   // C <- C - A B^T
    kSet = 1,   // C <- A B^T            (C may alias A: A is in shared memory before C is written)
};

// Per-lane geometry of one consumer warp.
template <int BLK>
struct WarpTile {
    using Cfg = GemmCfg<BLK>;
    int wm, wn, g, t;
    uint32_t a_off[2];                       // byte offset inside the A operand of a stage, accumulator blocks i even / odd
    uint32_t b_off[2];                       // same for B (only [0] when NJ == 1)

    __device__ __forceinline__ static uint32_t swz(int row, int t) {
        return (uint32_t)(row * 128 + ((((row & 7) ^ (t >> 1))) << 4) + (t & 1) * 8);
    }
    __device__ __forceinline__ int row_of(int i) const { return wm + 16 * (i >> 1) + 2 * g + (i & 1); }
    // column of B-row index nn (0..7) of accumulator block j
    __device__ __forceinline__ int col_of(int j, int nn) const {
        return (Cfg::NJ % 2 == 0) ? wn + 16 * (j >> 1) + 2 * nn + (j & 1) : wn + 8 * j + nn;
    }
    __device__ __forceinline__ void init(int warp, int lane) {
        g = lane >> 2;
        t = lane & 3;
        wm = (warp >> 2) * Cfg::WM;
        wn = (warp & 3) * Cfg::WN;
        a_off[0] = swz(wm + 2 * g, t);
        a_off[1] = swz(wm + 2 * g + 1, t);
        if (Cfg::NJ % 2 == 0) {
            b_off[0] = swz(wn + 2 * g, t);
            b_off[1] = swz(wn + 2 * g + 1, t);
        } else {
            b_off[0] = b_off[1] = swz(wn + g, t);
        }
    }
};

// One k-stage (kSub sub-tiles of 16) of the warp's (MI*8) x (NJ*8) product out of a filled ring slot.
template <int BLK>
__device__ __forceinline__ void consume_stage(const char* stage, const WarpTile<BLK>& w,
                                              double (&acc)[GemmCfg<BLK>::MI][GemmCfg<BLK>::NJ][2]) {
    using Cfg = GemmCfg<BLK>;
#pragma unroll
    for (int sub = 0; sub < Cfg::kSub; ++sub) {
    const char* sA = stage + sub * Cfg::kSubBytes;
    const char* sB = stage + Cfg::kOperandBytes + sub * Cfg::kSubBytes;
#pragma unroll
    for (int ks = 0; ks < kBK / 4; ++ks) {
        double a[Cfg::MI], b[Cfg::NJ];
        // k = 4*ks + t lives in chunk (2*ks + t/2) ^ (row & 7): the ks part is an XOR of bits 5-6
        const uint32_t a0 = w.a_off[0] ^ (uint32_t)(ks << 5), a1 = w.a_off[1] ^ (uint32_t)(ks << 5);
        const uint32_t b0 = w.b_off[0] ^ (uint32_t)(ks << 5), b1 = w.b_off[1] ^ (uint32_t)(ks << 5);
#pragma unroll
        for (int i = 0; i < Cfg::MI; ++i)
            a[i] = *reinterpret_cast<const double*>(sA + ((i & 1) ? a1 : a0) + (i >> 1) * 16 * 128);
#pragma unroll
        for (int j = 0; j < Cfg::NJ; ++j) {
            if (Cfg::NJ % 2 == 0) b[j] = *reinterpret_cast<const double*>(sB + ((j & 1) ? b1 : b0) + (j >> 1) * 16 * 128);
            else b[j] = *reinterpret_cast<const double*>(sB + b0 + j * 8 * 128);
        }
#pragma unroll
        for (int i = 0; i < Cfg::MI; ++i)
#pragma unroll
            for (int j = 0; j < Cfg::NJ; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
    }
}

// Epilogue of one warp: C <- C - acc (kSub) or C <- acc (kSet).  Lane (g,t) of accumulator block
// (i,j) holds rows row_of(i), columns col_of(j, 2t) and col_of(j, 2t+1); with NJ even a lane owns
// four consecutive columns per (i, j/2).
template <int BLK>
__device__ __forceinline__ void store_tile(double* __restrict__ C, int ldc, int mode, const WarpTile<BLK>& w,
                                           double (&acc)[GemmCfg<BLK>::MI][GemmCfg<BLK>::NJ][2]) {
    using Cfg = GemmCfg<BLK>;
    constexpr int GI = 2;                    // rows in flight per batch of loads (MI is even)
    constexpr int NV = Cfg::NJ;              // double2 vectors per row per lane
    // vector v of a row: NJ even: columns wn + 16*(v/2) + 4t + 2*(v%2) .. +1;  NJ odd: wn + 8v + 2t .. +1
    const int cbase = (Cfg::NJ % 2 == 0) ? w.wn + 4 * w.t : w.wn + 2 * w.t;
#pragma unroll
    for (int i0 = 0; i0 < Cfg::MI; i0 += GI) {
        double2 old[GI][NV];
        double* crow[GI];
#pragma unroll
        for (int ii = 0; ii < GI; ++ii) {
            crow[ii] = C + (size_t)w.row_of(i0 + ii) * ldc + cbase;
            if (mode == kSub) {
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    const int coff = (Cfg::NJ % 2 == 0) ? 16 * (v >> 1) + 2 * (v & 1) : 8 * v;
                    old[ii][v] = __ldcg(reinterpret_cast<const double2*>(crow[ii] + coff));
                }
            }
        }
#pragma unroll
        for (int ii = 0; ii < GI; ++ii) {
            const int i = i0 + ii;
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const int coff = (Cfg::NJ % 2 == 0) ? 16 * (v >> 1) + 2 * (v & 1) : 8 * v;
                double2 r;
                if (Cfg::NJ % 2 == 0) r = make_double2(acc[i][2 * (v >> 1)][v & 1], acc[i][2 * (v >> 1) + 1][v & 1]);
                else r = make_double2(acc[i][v][0], acc[i][v][1]);
                if (mode == kSub) { r.x = old[ii][v].x - r.x; r.y = old[ii][v].y - r.y; }
                __stcg(reinterpret_cast<double2*>(crow[ii] + coff), r);
            }
        }
    }
}

}  // namespace gpb
