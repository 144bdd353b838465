// gp_ozaki.cuh -- SURVEY.md 8(f) row 3 ("mixed-precision calculations to take advantage of
// modern hardware capabilities"): the building block of a tensor-core route past the FP64 pipe.
//
// sm_100a has no FP64 kind of tcgen05.mma, and the FP64 DMMA path of gp_gemm.cuh already runs at 93 % of the
// chip's FP64 rate.  The only way to a materially faster  C -= A B^T  in FP64 accuracy is to EMULATE it on the
// integer tensor cores (the Ozaki scheme): write every operand entry in fixed point with one global scale,
//     x / scale = sum_{p=0}^{S-1} d_p 2^{-b (p+1)},      d_p in [-2^(b-1), 2^(b-1) - 1]   (balanced digits, int8),
// so that
//     A B^T = scaleA scaleB sum_{lvl} 2^{-b (lvl + 2)} sum_{p+q = lvl} D_p(A) D_q(B)^T .
// Every digit-plane product is an int8 GEMM whose int32 accumulation is EXACT, products of equal weight share one
// accumulator, and only the final recombination of the S level sums rounds (in FP64).  Pairs with p + q >= S are
// dropped: that is 2^-(b (S + 1)) relative to scaleA scaleB per term, below the FP64 rounding of the result.
// S = 7 planes of b = 8 bits (56 bits of fixed point, S (S + 1) / 2 = 28 int8 GEMMs per FP64 GEMM).  Round 2 began with
// 8 planes of 7 bits (36 GEMMs; a CPU study of the tiled Cholesky with emulated updates at cond(K) = 4e4 gave
// |L - L_fp64| / |L| = 1.7e-9 / 1.4e-11 / 1.2e-13 for 42 / 49 / 56 bits, so 56 bits is what north_star's 1e-10 needs
// with margin); the 8-bit digits keep the 56 bits with 22 % fewer MMAs, which counts double because the kernel
// runs into the board's POWER limit on real operands (profiles/r02_ozaki_bounds.md).  The price is the depth one
// accumulator can take: 7 * 2^14 * k < 2^31 means k <= 16384 (kMaxK), longer contractions run in segments.
// The digits are balanced (round to nearest), not the bytes of the two's complement: unsigned low digits would
// turn the dropped terms into a bias instead of zero-mean noise.
//
// Kernels (Blackwell-native: tcgen05.mma kind::i8, accumulators in TMEM, operands by TMA):
//   * ozaki_contract_kernel3 (the default): 128 x 128 output tile, levels in two passes -- see its own comment;
//   * ozaki_contract_kernel: 128 x 64 output tile for shapes that are not multiples of 128; all S level accumulators
//     in tensor memory at once (7 x 64 columns); a stage holds one 32-deep k-chunk of ALL planes of both operands
//     (two 3-D TMA loads with the 32-byte swizzle), ring of 4 stages; warp 0 = TMA producer, warp 1 = MMA issuer,
//     warps 2-5 = epilogue (tcgen05.ld the level sums of a row segment, recombine smallest weight first, C -= result).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "gp_tma.cuh"

namespace gpb {
namespace oz {

constexpr int kPlanes = 7;           // S
constexpr int kDigitBits = 8;        // balanced base-256 digits in [-128, 127]: S * bits = 56 bits of fixed point
constexpr int kFixedBits = kPlanes * kDigitBits;
constexpr long long kDigitHalf = 1ll << (kDigitBits - 1), kDigitMask = (1ll << kDigitBits) - 1;
// int32 accumulators: a level sums at most S products of two digits per k-step, S * 2^(2 (bits - 1)) * k < 2^31
constexpr int kMaxK = 16384;         // 7 * 2^14 * 16384 = 1.88e9 < 2^31; longer contractions are run in segments
constexpr int kTileM = 128, kTileN = 64, kChunk = 32;
constexpr int kStagesOz = 4;
constexpr int kABytes = kPlanes * kTileM * kChunk;       // 32 KB
constexpr int kBBytes = kPlanes * kTileN * kChunk;       // 16 KB
constexpr int kStageBytesOz = kABytes + kBBytes;
constexpr int kThreadsOz = 192;
constexpr int kSmemOz = kStagesOz * kStageBytesOz + 1024 + 256;
constexpr int kTmemCols = 512;

// ---- slicing: FP64 -> S planes of balanced base-128 digits ------------------------------------------------------
// planes[p][r][k] (int8, row-major rows x k per plane).  |x| <= 0.498 scale is required (the top digit must stay <= 127).
__global__ void __launch_bounds__(256) slice_kernel(const double* __restrict__ X, int64_t rows, int64_t k, int64_t ld, double inv_scale,
                                                    int8_t* __restrict__ planes, int* __restrict__ overflow) {
    const int64_t total = rows * (k / 4);
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = idx / (k / 4), c = 4 * (idx % (k / 4));
        uint32_t packed[kPlanes];
#pragma unroll
        for (int p = 0; p < kPlanes; ++p) packed[p] = 0u;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const double x = X[r * ld + c + e] * inv_scale;                       // |x| <= 1/2
            long long I = __double2ll_rn(x * (double)(1ull << kFixedBits));
#pragma unroll
            for (int p = kPlanes - 1; p >= 0; --p) {
                const long long d = ((I + kDigitHalf) & kDigitMask) - kDigitHalf;
                I = (I - d) >> kDigitBits;
                packed[p] |= (uint32_t)((int)d & 0xff) << (8 * e);
            }
            if (I != 0) atomicExch(overflow, 1);
        }
#pragma unroll
        for (int p = 0; p < kPlanes; ++p) *reinterpret_cast<uint32_t*>(planes + ((size_t)p * rows + r) * k + c) = packed[p];
    }
}

// The same for tile column J of a lower-packed tiled matrix (tiles (I, J), I > J) into DENSE planes [p][n][n] of the
// whole matrix (row = global row, column = global column), with the scale read from device memory.
__global__ void __launch_bounds__(256) slice_tile_column_kernel(const double* __restrict__ tiles, int64_t n, int t, int J,
                                                                const double* __restrict__ scale, int8_t* __restrict__ planes) {
    const double inv_scale = 1.0 / *scale;
    const int64_t rows = n - (int64_t)(J + 1) * t;          // rows below the diagonal tile
    const int64_t total = rows * (t / 4);
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t rr = idx / (t / 4);
        const int c = 4 * (int)(idx % (t / 4));
        const int64_t gi = (int64_t)(J + 1) * t + rr;
        const int64_t I = gi / t, r = gi % t;
        const double* src = tiles + ((size_t)I * (I + 1) / 2 + J) * (size_t)t * t + (size_t)r * t + c;
        const double2 v01 = *reinterpret_cast<const double2*>(src), v23 = *reinterpret_cast<const double2*>(src + 2);
        const double xs[4] = {v01.x, v01.y, v23.x, v23.y};
        uint32_t packed[kPlanes];
#pragma unroll
        for (int p = 0; p < kPlanes; ++p) packed[p] = 0u;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            long long I56 = __double2ll_rn(xs[e] * inv_scale * (double)(1ull << kFixedBits));
#pragma unroll
            for (int p = kPlanes - 1; p >= 0; --p) {
                const long long d = ((I56 + kDigitHalf) & kDigitMask) - kDigitHalf;
                I56 = (I56 - d) >> kDigitBits;
                packed[p] |= (uint32_t)((int)d & 0xff) << (8 * e);
            }
        }
#pragma unroll
        for (int p = 0; p < kPlanes; ++p)
            *reinterpret_cast<uint32_t*>(planes + ((size_t)p * n + gi) * n + (size_t)J * t + c) = packed[p];
    }
}

// scale <- 2 * 2^ceil(log2(sqrt(max_i K_ii))): every entry of the Cholesky factor obeys |L_ij| <= sqrt(K_ii), so
// |L| <= scale / 2 and one global fixed-point scale serves the whole factor.  One CTA.
__global__ void __launch_bounds__(1024) factor_scale_kernel(const double* __restrict__ tiles, int64_t n, int t, double* __restrict__ scale) {
    __shared__ double s_max[32];
    double m = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += 1024) {
        const int64_t I = i / t, r = i % t;
        m = fmax(m, tiles[((size_t)I * (I + 1) / 2 + I) * (size_t)t * t + r * (size_t)t + r]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 0; k < 32; ++k) m = fmax(m, s_max[k]);
        int e;
        const double f = frexp(sqrt(m > 0.0 ? m : 1.0), &e);      // sqrt(m) = f 2^e, f in [0.5, 1)
        const double sc = ldexp(1.0, e + 1 + (f > 0.98 ? 1 : 0)); // >= 2 sqrt(m) / 0.98: the top digit of a balanced expansion stays below 2^(b-1)
        scale[0] = sc;
        scale[1] = sc * sc;                                          // the weight factor of a product of two such operands
    }
}

// The same from a FINISHED factor: scale[0] <- power of two >= 2 max |L_ij| (lower tiles), scale[1] <- sv (given),
// scale[2] <- scale[0] * sv, scale[3] <- sv * sv.  Two launches: a grid-wide maximum (positive doubles order like their
// bit patterns), then the finish.
__global__ void __launch_bounds__(256) absmax_lower_tiles_kernel(const double* __restrict__ tiles, int64_t count, unsigned long long* __restrict__ bits) {
    double m = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (int64_t)gridDim.x * blockDim.x) m = fmax(m, fabs(tiles[i]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m == m) atomicMax(bits, (unsigned long long)__double_as_longlong(m));
}
__global__ void finish_scales_kernel(const unsigned long long* __restrict__ bits, double sv, double* __restrict__ scale) {
    const double m = __longlong_as_double((long long)*bits);
    int e;
    const double f = frexp(m > 0.0 ? m : 1.0, &e);
    const double sl = ldexp(1.0, e + 1 + (f > 0.98 ? 1 : 0));
    scale[0] = sl;
    scale[1] = sv;
    scale[2] = sl * sv;
    scale[3] = sv * sv;
}

// tile column J of a GP_GENERAL tiled m x n matrix (all tile rows) -> dense planes [p][m][n]
__global__ void __launch_bounds__(256) slice_general_column_kernel(const double* __restrict__ tiles, int64_t m, int64_t n, int t, int J,
                                                                   const double* __restrict__ scale, int8_t* __restrict__ planes) {
    const double inv_scale = 1.0 / *scale;
    const int64_t total = m * (t / 4);
    const int64_t Mt = n / t;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t gi = idx / (t / 4);
        const int c = 4 * (int)(idx % (t / 4));
        const int64_t a = gi / t, r = gi % t;
        const double* src = tiles + ((size_t)a * Mt + J) * (size_t)t * t + (size_t)r * t + c;
        const double2 v01 = *reinterpret_cast<const double2*>(src), v23 = *reinterpret_cast<const double2*>(src + 2);
        const double xs[4] = {v01.x, v01.y, v23.x, v23.y};
        uint32_t packed[kPlanes];
#pragma unroll
        for (int p = 0; p < kPlanes; ++p) packed[p] = 0u;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            long long I56 = __double2ll_rn(xs[e] * inv_scale * (double)(1ull << kFixedBits));
#pragma unroll
            for (int p = kPlanes - 1; p >= 0; --p) {
                const long long d = ((I56 + kDigitHalf) & kDigitMask) - kDigitHalf;
                I56 = (I56 - d) >> kDigitBits;
                packed[p] |= (uint32_t)((int)d & 0xff) << (8 * e);
            }
        }
#pragma unroll
        for (int p = 0; p < kPlanes; ++p)
            *reinterpret_cast<uint32_t*>(planes + ((size_t)p * m + gi) * n + (size_t)J * t + c) = packed[p];
    }
}

// version counters of the blocks of tile column J of V^T <- "J updates applied"
__global__ void set_general_column_versions_kernel(int* __restrict__ ver, int NBm, int NB, int nbt, int J, int per_version) {
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < NBm * nbt; idx += gridDim.x * blockDim.x)
        ver[(size_t)(idx / nbt) * NB + J * nbt + idx % nbt] = J * per_version;
}

// version counters of the blocks of tile column J <- "J trailing updates applied" (they were applied by the emulated
// contraction, which does not go through the executor's counters)
__global__ void set_column_versions_kernel(int* __restrict__ ver, int NB, int nbt, int J, int per_version) {
    const int c0 = J * nbt;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < (NB - c0) * nbt; idx += gridDim.x * blockDim.x) {
        const int gr = c0 + idx / nbt, gc = c0 + idx % nbt;
        if (gc <= gr) ver[(size_t)gr * NB + gc] = J * per_version;
    }
}

// ---- tcgen05 / TMEM wrappers ----------------------------------------------------------------------------------------
__device__ __forceinline__ void tmem_alloc(uint32_t* slot_in_smem, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(slot_in_smem)), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(taddr), "r"(cols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); }
// all MMAs issued so far by this thread arrive on `bar` when they have completed (implies fence::before_thread_sync)
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
// D[tmem] (+)= A[smem] B[smem]^T, int8 x int8 -> int32, M = 128, N = 64, K = 32
__device__ __forceinline__ void mma_i8(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        " .reg .pred p;\n"
        " setp.ne.b32 p, %4, 0;\n"
        " tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n"
        "}\n" ::"r"(tmem_d),
        "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate), "r"(0u)
        : "memory");
}
// 16 consecutive 32-bit columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, int32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]), "=r"(v[10]),
          "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
}
// one lane of a converged warp; the loops of the wide kernel are run by WHOLE warps with the side effects under this
// predicate: code under `if (lane == 0)` makes ptxas treat every operand as divergent and wrap each tcgen05.mma in an
// R2UR + ELECT + BRA.U.ANY loop, code that is uniform across the warp keeps descriptors in uniform registers
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n .reg .pred P;\n elect.sync _|P, 0xffffffff;\n selp.u32 %0, 1, 0, P;\n}\n" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory"); }

__device__ __forceinline__ void tma_load_3d(void* smem_dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cta.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];\n" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
                 : "memory");
}

// shared-memory matrix descriptor: K-major operand, rows of 32 bytes written by TMA with the 32-byte swizzle
// (8-row atoms of 256 B): start address >> 4 | LBO (unused for swizzled K-major) | SBO = 256 B | version 1 | SWIZZLE_32B
__device__ __forceinline__ uint64_t smem_desc_sw32(uint32_t saddr) {
    return (uint64_t)((saddr >> 4) & 0x3fffu) | ((uint64_t)1 << 16) | ((uint64_t)(256 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)6 << 61);
}
// instruction descriptor: D = S32, A = B = signed int8, both K-major, N = 64, M = 128, dense, no saturation
constexpr uint32_t kIdescI8 = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(kTileN >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);

struct OzParams {
    double* C;            // dense: C [tiles_m * 128, ldc];  tiled: the lower-packed tiles of the factorisation
    int64_t ldc;
    int tiles_m, tiles_n, kchunks;
    double w_last;        // scaleA * scaleB * 2^(-7 (S + 1)): weight of level S - 1; level l weighs scaleA scaleB 2^(-7 (l + 2))
    const double* scale;  // optional device scalar: the weights are multiplied by it (= scaleA * scaleB of operands that were
                          // sliced with scales found on the device)
    // output modes:  0 dense C (ldc);  1 tile column J of a LOWER-PACKED matrix of t x t tiles, rows from tile row J down
    // (gp_cholesky_tiled_mixed);  2 tile column J of a GP_GENERAL matrix with Mt tile columns, all tile rows (the V^T solve);
    // 3 dense C, only the 128 x TN pieces that touch the lower triangle (Sigma)
    int tiled, t, J, Mt;
    int row0a, row0b;     // first operand row of A and of B in their digit planes
    int kc0;              // first k-chunk (the contraction covers the chunks [kc0, kc0 + kchunks))
};

// tile (tm, tn) -> is it wanted, and where does row `r` (0..127) of it live
struct OzTile {
    bool wanted;
    double* c;            // address of element (row 0 of the tile, column 0 of the tile)
    int64_t ld;
    // the same place in the 2-D view [rows][ld] of the output array (dense: the matrix itself; tiled: tile after tile, each
    // t rows of t entries) that the wide kernel's tensor map for C describes
    int row0, col0;
};
// Order in which the wide kernel's CTAs walk the output tiles: bands of kBand3 tile rows, column by column inside a
// band, so that the ~148 tiles in flight form a 12 x 12 square and share 24 operand row blocks instead of the 3 + 64 of
// a row-major walk over a wide matrix (8192 x 8192 x 4096: 15.0 -> 4.0 GB of DRAM reads per launch, ncu; 111 -> 122 TFLOP/s-equivalent under the power cap).
constexpr int kBand3 = 12;
__device__ __forceinline__ void oz3_tile_coords(const OzParams& p, int tile, int& tm, int& tn) {
    if (p.tiles_n <= kBand3) {          // a narrow output (the tile columns of the factorisation): row-major is already compact
        tm = tile / p.tiles_n;
        tn = tile - tm * p.tiles_n;
        return;
    }
    const int per_band = kBand3 * p.tiles_n;
    const int band = tile / per_band, r = tile - band * per_band;
    const int rows = min(kBand3, p.tiles_m - band * kBand3);
    tn = r / rows;
    tm = band * kBand3 + (r - tn * rows);
}

template <int TN = kTileN>
__device__ __forceinline__ OzTile oz_tile(const OzParams& p, int tm, int tn) {
    OzTile o;
    if (p.tiled == 0 || p.tiled == 3) {
        o.wanted = p.tiled == 0 || tn * TN < (tm + 1) * kTileM;
        o.ld = p.ldc;
        o.row0 = tm * kTileM;
        o.col0 = tn * TN;
        o.c = p.C + (size_t)o.row0 * p.ldc + (size_t)o.col0;
        return o;
    }
    const int bpt = p.t / kTileM;                       // 128-row blocks per tile edge
    if (p.tiled == 2) {
        const int a = tm / bpt, rblk = tm % bpt;
        o.wanted = true;
        o.ld = p.t;
        o.row0 = (a * p.Mt + p.J) * p.t + rblk * kTileM;
        o.col0 = tn * TN;
        o.c = p.C + (size_t)o.row0 * p.t + (size_t)o.col0;
        return o;
    }
    const int I = p.J + tm / bpt, rblk = tm % bpt;
    // on the diagonal tile only the lower part is data: skip 128 x TN pieces that lie wholly above the diagonal
    o.wanted = !(I == p.J && tn * TN >= (rblk + 1) * kTileM);
    o.ld = p.t;
    o.row0 = (I * (I + 1) / 2 + p.J) * p.t + rblk * kTileM;
    o.col0 = tn * TN;
    o.c = p.C + (size_t)o.row0 * p.t + (size_t)o.col0;
    return o;
}

__global__ void __launch_bounds__(kThreadsOz, 1)
ozaki_contract_kernel(const __grid_constant__ OzParams p, const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB) {
    extern __shared__ char smem_raw[];
    char* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* full = reinterpret_cast<uint64_t*>(base + kStagesOz * kStageBytesOz);
    uint64_t* empty = full + kStagesOz;
    uint64_t* tmem_full = empty + kStagesOz;
    uint64_t* tmem_empty = tmem_full + 1;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tmem_empty + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStagesOz; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        mbar_init(tmem_full, 1);
        mbar_init(tmem_empty, 4);
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc(tmem_slot, kTmemCols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const int ntiles = p.tiles_m * p.tiles_n;

    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            tma_prefetch_desc(&mapA);
            tma_prefetch_desc(&mapB);
            int stage = 0, phase = 0;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                const int tm = tile / p.tiles_n, tn = tile % p.tiles_n;
                if (!oz_tile(p, tm, tn).wanted) continue;
                for (int kc = 0; kc < p.kchunks; ++kc) {
                    mbar_wait(&empty[stage], (uint32_t)(phase ^ 1));
                    char* dst = base + (size_t)stage * kStageBytesOz;
                    mbar_arrive_expect_tx(&full[stage], (uint32_t)kStageBytesOz);
                    tma_load_3d(dst, &mapA, (p.kc0 + kc) * kChunk, p.row0a + tm * kTileM, 0, &full[stage]);
                    tma_load_3d(dst + kABytes, &mapB, (p.kc0 + kc) * kChunk, p.row0b + tn * kTileN, 0, &full[stage]);
                    if (++stage == kStagesOz) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer =====
        if (lane == 0) {
            int stage = 0, phase = 0, tphase = 0;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                if (!oz_tile(p, tile / p.tiles_n, tile % p.tiles_n).wanted) continue;
                mbar_wait(tmem_empty, (uint32_t)(tphase ^ 1));          // the epilogue has drained the previous tile
                tc_fence_after();
                for (int kc = 0; kc < p.kchunks; ++kc) {
                    mbar_wait(&full[stage], (uint32_t)phase);
                    tc_fence_after();
                    const uint32_t sa = smem_u32(base + (size_t)stage * kStageBytesOz), sb = sa + kABytes;
#pragma unroll
                    for (int pa = 0; pa < kPlanes; ++pa) {
                        const uint64_t da = smem_desc_sw32(sa + pa * (kTileM * kChunk));
#pragma unroll
                        for (int pb = 0; pb + pa < kPlanes; ++pb) {
                            const uint64_t db = smem_desc_sw32(sb + pb * (kTileN * kChunk));
                            // level pa + pb: its first product of the tile is (kc = 0, pa = 0)
                            mma_i8(tmem_base + (uint32_t)((pa + pb) * kTileN), da, db, kIdescI8, (kc > 0 || pa > 0) ? 1u : 0u);
                        }
                    }
                    tc_commit(&empty[stage]);                          // the stage is free once these MMAs have read it
                    if (++stage == kStagesOz) { stage = 0; phase ^= 1; }
                }
                tc_commit(tmem_full);                                   // the tile's eight level sums are complete
                tphase ^= 1;
            }
        }
    } else {
        // ===== epilogue: 4 warps, warp w owns the TMEM lanes 32 (w % 4) .. +31 = rows of the tile =====
        const int quad = warp & 3;
        int tphase = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const OzTile ot = oz_tile(p, tile / p.tiles_n, tile % p.tiles_n);
            if (!ot.wanted) continue;
            mbar_wait(tmem_full, (uint32_t)tphase);
            tc_fence_after();
            double* crow = ot.c + (size_t)(32 * quad + lane) * ot.ld;
            const double wl = p.scale ? p.w_last * (*p.scale) : p.w_last;
#pragma unroll 1
            for (int c0 = 0; c0 < kTileN; c0 += 16) {
                double acc[16];
#pragma unroll
                for (int j = 0; j < 16; ++j) acc[j] = 0.0;
                double w = wl;
#pragma unroll
                for (int lvl = kPlanes - 1; lvl >= 0; --lvl) {           // smallest weight first
                    int32_t v[16];
                    tmem_ld16(tmem_base + ((uint32_t)(32 * quad) << 16) + (uint32_t)(lvl * kTileN + c0), v);
                    tmem_ld_wait();
#pragma unroll
                    for (int j = 0; j < 16; ++j) acc[j] = fma((double)v[j], w, acc[j]);
                    w *= (double)(1 << kDigitBits);
                }
#pragma unroll
                for (int j = 0; j < 16; j += 2) {
                    double2 c = *reinterpret_cast<double2*>(crow + c0 + j);
                    c.x -= acc[j];
                    c.y -= acc[j + 1];
                    *reinterpret_cast<double2*>(crow + c0 + j) = c;
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tmem_empty);
            tphase ^= 1;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
}


// ---- the wide shape: 128 x 128 output tile, 128-byte k-chunks, the levels in TWO passes --------------------------------
// What bounds the 128 x 64 kernel above was measured with probes (profiles/r02_ozaki_bounds.md): with the TMA loads
// removed it runs at the SAME rate, so it is not the operand stream from L2; a bare issue loop shows that a
// tcgen05.mma kind::i8 of 128 x 64 x 32 takes 48 cycles, not 32 -- every MMA re-reads its 4 KB A operand and 2 KB B
// operand from shared memory, 192 B/clk against a port of 128 B/clk -- while 128 x 128 x 32 takes 64 cycles = the
// full 8192 MAC/clk/SM.  So N must be 128, and then tensor memory (512 columns) holds four level sums, not eight:
// the levels are done in two passes over k (pass 0: the high levels, which need the leading planes only; pass 1:
// the rest).  The first two-pass kernel (round 2, removed) kept a whole 32-byte k-chunk of ALL planes per stage and
// was bound by the L2 -> shared-memory stream instead: TMA boxes with 32-byte rows move 9 TB/s over the chip,
// boxes with 128-byte rows 20-29 TB/s (same probe file).  This kernel therefore streams ONE plane of ONE operand
// per slot (128 rows x 128 bytes of k, 128-byte swizzle, 16 KB) through two rings:
//   * step pa of a k-chunk multiplies plane pa of A with the planes pb of B whose level pa + pb lies in the pass's
//     range [LO, HI]: a window of at most four B planes that slides down by one plane per step.  A planes live for
//     one step, B planes are loaded in the order HI, HI-1, ... 0 and retire in the same order: both rings are FIFOs
//     (5 A slots, 8 B slots), each with its own producer warp, so the operands of a step are requested at least
//     2500 cycles before the step is issued;
//   * per step up to 4 x 4 MMAs (128 x 128 x 32 each, the k-steps of a chunk address 32-byte columns of the
//     swizzled rows); tcgen05.commit retires the A slot and the B plane that leaves the window;
//   * epilogue by eight warps (two per TMEM lane quarter, 64 columns each): the pass's level sums -> FP64, smallest
//     weight first, C -= result.  Pass 0 and pass 1 both update C in place.
constexpr int kTileN3 = 128;
constexpr int kChunk3 = 128;                                   // bytes of k per slot
constexpr int kKSteps3 = kChunk3 / kChunk;                      // MMAs (K = 32) per plane pair and chunk
constexpr int kSlotBytes3 = kTileM * kChunk3;                   // 16 KB
constexpr int kNA3 = 5, kNB3 = 8;
constexpr int kThreads3 = 352;                                  // warp 0 A producer, 1 MMA issuer, 2-9 epilogue, 10 B producer
constexpr int kSmemOz3 = (kNA3 + kNB3) * kSlotBytes3 + 16384 + 1024 + 512;   // slots, epilogue staging, alignment slack, barriers
constexpr uint32_t kIdescI8N128 = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(kTileN3 >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);

// the level range of a pass
__host__ __device__ constexpr int oz3_lo(int pass) { return pass == 0 ? 0 : kPlanes / 2; }
__host__ __device__ constexpr int oz3_hi(int pass) { return pass == 0 ? kPlanes / 2 - 1 : kPlanes - 1; }

// K-major operand whose rows are 128 bytes written by TMA with the 128-byte swizzle (8-row atoms of 1024 B)
__device__ __forceinline__ uint64_t smem_desc_sw128(uint32_t saddr) {
    return (uint64_t)((saddr >> 4) & 0x3fffu) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__device__ __forceinline__ void mma_i8_n128(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t accumulate) {
    mma_i8(tmem_d, desc_a, desc_b, kIdescI8N128, accumulate);
}

__device__ long long g_oz3_probe[8];       // PROBE > 0 only: clock64 stamps of the second tile of CTA 0

struct Oz3Smem {
    char* slotA;
    char* slotB;
    uint64_t *fullA, *emptyA, *fullB, *emptyB, *tmem_full, *tmem_empty;
};

// the same instructions under a predicate instead of a C++ branch: a branch around every MMA splits the issue loop into
// basic blocks and ptxas then rebuilds the descriptors (R2UR and a dozen uniform ops) between the waits and the first MMA
// of each step, which is exactly where the tensor core's two-deep queue runs dry
__device__ __forceinline__ void mma_i8_n128_if(uint32_t leader, uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t accumulate) {
    asm volatile(
        "{\n"
        " .reg .pred p, q;\n"
        " setp.ne.b32 p, %4, 0;\n"
        " setp.ne.b32 q, %6, 0;\n"
        " @q tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n"
        "}\n" ::"r"(tmem_d),
        "l"(desc_a), "l"(desc_b), "r"(kIdescI8N128), "r"(accumulate), "r"(0u), "r"(leader)
        : "memory");
}
__device__ __forceinline__ void tc_commit_if(uint32_t leader, uint64_t* bar) {
    asm volatile("{\n .reg .pred q;\n setp.ne.b32 q, %1, 0;\n @q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n}\n" ::"r"(smem_u32(bar)),
                 "r"(leader)
                 : "memory");
}

// issuer: one pass over the k range for one tile.  The tensor core's instruction queue is about two MMAs deep (a pause
// of more than ~100 cycles in the issuing thread is a bubble in the pipe: profiles/r02_ozaki_bounds.md), so the
// mbarrier waits of the NEXT step are interleaved with the last MMAs of the current one, ring positions advance
// without divisions, and a step's descriptors are one add away from words computed a step ahead.
template <int LO, int HI, int PROBE>
__device__ __forceinline__ void oz3_issue_pass(const Oz3Smem& sm, uint32_t tmem_base, int nchunks, uint32_t& cntA, uint32_t& cntB, uint32_t leader) {
    constexpr int QMAX = HI < kPlanes - 1 ? HI : kPlanes - 1;       // B planes QMAX .. 0 and A planes 0 .. QMAX take part
    constexpr uint64_t kDescHi = ((uint64_t)(1024 >> 4) | ((uint64_t)1 << 14) | ((uint64_t)2 << 29)) << 32;   // SBO, version, SWIZZLE_128B
    constexpr uint32_t kSlotLo = (uint32_t)(kSlotBytes3 >> 4);
    static_assert((kNB3 & (kNB3 - 1)) == 0, "the B ring is indexed with a mask");
    const uint32_t a_lo0 = ((smem_u32(sm.slotA) >> 4) & 0x3fffu) | (1u << 16);
    const uint32_t b_lo0 = ((smem_u32(sm.slotB) >> 4) & 0x3fffu) | (1u << 16);
    auto wait_b = [&](uint32_t cb, int q) { const uint32_t c = cb + (uint32_t)(QMAX - q); mbar_wait(&sm.fullB[c & (kNB3 - 1)], (c / kNB3) & 1u); };
    // ring position of the A plane of the current step, and of the next one
    uint32_t sa = cntA % kNA3, pha = (cntA / kNA3) & 1u;
    // prologue: the operands of step 0 of chunk 0
#pragma unroll
    for (int q = QMAX; q >= 0; --q)
        if (LO - q <= 0) wait_b(cntB, q);
    mbar_wait(&sm.fullA[sa], pha);
    for (int kc = 0; kc < nchunks; ++kc) {
        const bool more = kc + 1 < nchunks;
#pragma unroll
        for (int pa = 0; pa <= QMAX; ++pa) {
            const uint32_t san = sa + 1 == kNA3 ? 0u : sa + 1, phan = sa + 1 == kNA3 ? pha ^ 1u : pha;
            const uint32_t a_lo = a_lo0 + sa * kSlotLo;
            tc_fence_after();
            // this step's MMAs: pb in [max(0, LO - pa), min(S - 1, HI - pa)], 4 k-steps each
            const int pb_lo = LO - pa > 0 ? LO - pa : 0, pb_hi = HI - pa < kPlanes - 1 ? HI - pa : kPlanes - 1;
            const int n_mma = (pb_hi - pb_lo + 1) * kKSteps3;
            // waits owed to the NEXT step: (pa + 1 of this chunk) or (step 0 of the next chunk)
            const bool wrap = pa == QMAX;
            const int n_wait = wrap ? (QMAX - (LO > 0 ? LO : 0) + 1) + 1 : ((LO - (pa + 1) >= 0) ? 2 : 1);
            auto next_wait = [&](int j) {            // j-th wait owed to the next step; the A plane comes last
                if (!wrap) {
                    if (LO - (pa + 1) >= 0 && j == 0) wait_b(cntB, LO - (pa + 1));
                    else mbar_wait(&sm.fullA[san], phan);
                } else if (more) {
                    if (j < n_wait - 1) wait_b(cntB + QMAX + 1, QMAX - j);
                    else mbar_wait(&sm.fullA[san], phan);
                }
            };
            // the last wait is followed by kTail more MMAs of this step, so that the queue is full across the step boundary
            constexpr int kTail = 2;
            const int first_after = n_mma - kTail - n_wait;                  // wait j follows MMA first_after + j
#pragma unroll
            for (int j = 0; j < n_wait; ++j)
                if (first_after + j < 0) next_wait(j);                        // more waits than MMAs: the surplus first
#pragma unroll
            for (int w = 0; w < 4; ++w) {                                    // the window holds at most four B planes
                const int pb = pb_lo + w;
                if (pb > pb_hi) continue;
                const uint32_t b_lo = b_lo0 + ((cntB + (uint32_t)(QMAX - pb)) & (kNB3 - 1)) * kSlotLo;
#pragma unroll
                for (int ks = 0; ks < kKSteps3; ++ks) {
                    const int m = w * kKSteps3 + ks;
                    if (PROBE != 2)
                        mma_i8_n128_if(leader, tmem_base + (uint32_t)((pa + pb - LO) * kTileN3), kDescHi | (a_lo + ks * (kChunk >> 4)),
                                       kDescHi | (b_lo + ks * (kChunk >> 4)), (kc > 0 || pa > 0 || ks > 0) ? 1u : 0u);
                    if (m == n_mma - 1) {
                        // the step is issued: retire its A slot and the B plane that leaves the window
                        tc_commit_if(leader, &sm.emptyA[sa]);
#pragma unroll
                        for (int q = QMAX; q >= 0; --q) {
                            const int last = HI - q < kPlanes - 1 ? HI - q : kPlanes - 1;
                            if (last == pa) tc_commit_if(leader, &sm.emptyB[(cntB + (uint32_t)(QMAX - q)) & (kNB3 - 1)]);
                        }
                    }
                    const int jw = m - first_after;
                    if (jw >= 0 && jw < n_wait) next_wait(jw);
                }
            }
            sa = san;
            pha = phan;
            ++cntA;
        }
        cntB += QMAX + 1;
    }
}

// int32 -> double without the (slow) I2F.F64: the bits 0x43300000'(v + 2^31) are the double 2^52 + 2^31 + v
__device__ __forceinline__ double i32_to_f64(int32_t v) {
    return __hiloint2double(0x43300000, (int)((uint32_t)v ^ 0x80000000u)) - 4503601774854144.0;
}

// C -= tile without reading C in the SM: the negated update goes to shared memory and from there to global memory as a
// bulk FP64 reduction (TMA, executed in L2), one 2-D box of 32 rows x 8 columns per warp and step.  The first epilogue
// read-modify-wrote C with LDG/STG: 20 000 cycles per pass and tile (row-strided 16-byte accesses at HBM latency) in
// which the tensor core has nothing to do, because the next pass needs the same tensor memory.  One 64-byte 1-D bulk
// reduction per lane was no better (2048 small operations per pass: the TMA unit's issue rate); the boxed form is 64
// operations per pass (profiles/r02_ozaki_bounds.md).
__device__ __forceinline__ void tensor_reduce_add_2d(const CUtensorMap* map, int c0, int c1, const void* ssrc) {
    asm volatile("cp.reduce.async.bulk.tensor.2d.global.shared::cta.add.tile.bulk_group [%0, {%1, %2}], [%3];\n" ::"l"(reinterpret_cast<uint64_t>(map)), "r"(c0),
                 "r"(c1), "r"(smem_u32(ssrc))
                 : "memory");
}
__device__ __forceinline__ void bulk_commit_group() { asm volatile("cp.async.bulk.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_group_read0() { asm volatile("cp.async.bulk.wait_group.read 0;\n" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_group0() { asm volatile("cp.async.bulk.wait_group 0;\n" ::: "memory"); }

constexpr int kStageCols3 = 8;                                   // columns per box (64 bytes per row)
constexpr int kStageWarpBytes3 = 32 * kStageCols3 * 8;           // one box: 32 rows x 64 B
constexpr int kStageBytes3 = 8 * kStageWarpBytes3;               // eight epilogue warps

// epilogue of one pass: this warp's 32 rows x 64 columns.  `stage` = this warp's box, (row0, col0) = its first row and
// the tile's first column in the 2-D view of C.
template <int LO, int HI, int PROBE = 0>
__device__ __forceinline__ void oz3_epilogue_pass(uint32_t tmem_base, int quad, int half, int lane, const CUtensorMap* mapC, int row0, int col0, double w_hi,
                                                  double* stage) {
    constexpr int NACC = HI - LO + 1;
#pragma unroll 1
    for (int c0 = 64 * half; c0 < 64 * half + 64; c0 += 16) {
        int32_t v[NACC][16];
#pragma unroll
        for (int a = 0; a < NACC; ++a) tmem_ld16(tmem_base + ((uint32_t)(32 * quad) << 16) + (uint32_t)(a * kTileN3 + c0), v[a]);
        tmem_ld_wait();
        double acc[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) acc[j] = 0.0;
        double w = -w_hi;                                               // the NEGATED update is added to C
#pragma unroll
        for (int a = NACC - 1; a >= 0; --a) {                          // smallest weight first
#pragma unroll
            for (int j = 0; j < 16; ++j) acc[j] = fma(i32_to_f64(v[a][j]), w, acc[j]);
            w *= (double)(1 << kDigitBits);
        }
#pragma unroll
        for (int h = 0; h < 16 / kStageCols3; ++h) {
            if (lane == 0) bulk_wait_group_read0();                     // the previous reduction has read the box
            __syncwarp();
#pragma unroll
            for (int j = 0; j < kStageCols3; j += 2)
                *reinterpret_cast<double2*>(stage + lane * kStageCols3 + j) = make_double2(acc[h * kStageCols3 + j], acc[h * kStageCols3 + j + 1]);
            fence_proxy_async_shared();
            __syncwarp();
            if (lane == 0) {
                if (PROBE != 4) tensor_reduce_add_2d(mapC, col0 + c0 + h * kStageCols3, row0, stage);
                bulk_commit_group();
            }
        }
    }
}

// mapA / mapB: boxes of {128 bytes of k, 128 rows, 1 plane}, 128-byte swizzle; mapC: FP64, the 2-D view of the output
// array (see OzTile), boxes of {8 columns, 32 rows}, no swizzle.  p.kc0 / p.kchunks count 32-byte chunks and
// must be multiples of 4; p.tiles_n counts 128-column tiles.  PROBE (measurement only, 0 in the product): 1 = the producers
// skip their TMA loads (the MMAs run on whatever the slots hold), 2 = the issuer skips its MMAs (loads only), 4 = the
// epilogue skips its reductions into C; every PROBE > 0 leaves time stamps of the second tile of CTA 0 in g_oz3_probe
// (pass 0: issue start, issue end; pass 1: issue start, issue end; then epilogue start / end of pass 0 and of pass 1).
template <int PROBE = 0>
__global__ void __launch_bounds__(kThreads3, 1)
ozaki_contract_kernel3(const __grid_constant__ OzParams p, const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
                       const __grid_constant__ CUtensorMap mapC) {
    extern __shared__ char smem_raw[];
    char* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    Oz3Smem sm;
    sm.slotA = base;
    sm.slotB = base + kNA3 * kSlotBytes3;
    char* staging = base + (kNA3 + kNB3) * kSlotBytes3;
    sm.fullA = reinterpret_cast<uint64_t*>(staging + kStageBytes3);
    sm.emptyA = sm.fullA + kNA3;
    sm.fullB = sm.emptyA + kNA3;
    sm.emptyB = sm.fullB + kNB3;
    sm.tmem_full = sm.emptyB + kNB3;
    sm.tmem_empty = sm.tmem_full + 1;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sm.tmem_empty + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kNA3; ++s) { mbar_init(&sm.fullA[s], 1); mbar_init(&sm.emptyA[s], 1); }
        for (int s = 0; s < kNB3; ++s) { mbar_init(&sm.fullB[s], 1); mbar_init(&sm.emptyB[s], 1); }
        mbar_init(sm.tmem_full, 1);
        mbar_init(sm.tmem_empty, 8);
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc(tmem_slot, kTmemCols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const int ntiles = p.tiles_m * p.tiles_n;
    const int nchunks = p.kchunks / kKSteps3;
    const int kbyte0 = p.kc0 * kChunk;

    if (warp == 0 || warp == 10) {
        // ===== producers (whole warps, side effects by one elected lane): warp 0 streams the A planes 0 .. HI of every
        // (pass, chunk), warp 10 the B planes HI .. 0 =====
        const bool leader = elect_one();
        const bool isA = warp == 0;
        const CUtensorMap* map = isA ? &mapA : &mapB;
        if (leader) tma_prefetch_desc(map);
        uint64_t* full = isA ? sm.fullA : sm.fullB;
        uint64_t* empty = isA ? sm.emptyA : sm.emptyB;
        char* slots = isA ? sm.slotA : sm.slotB;
        const uint32_t nslots = isA ? kNA3 : kNB3;
        uint32_t cnt = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            int tm, tn;
            oz3_tile_coords(p, tile, tm, tn);
            const OzTile ot = oz_tile<kTileN3>(p, tm, tn);
            if (!ot.wanted) continue;
            const int row = isA ? p.row0a + tm * kTileM : p.row0b + tn * kTileN3;
            for (int pass = 0; pass < 2; ++pass) {
                const int qmax = oz3_hi(pass);
                for (int kc = 0; kc < nchunks; ++kc) {
                    for (int i = 0; i <= qmax; ++i) {
                        const uint32_t slot = cnt % nslots;
                        mbar_wait(&empty[slot], ((cnt / nslots) & 1u) ^ 1u);
                        if (leader) {
                            if (PROBE == 1) {
                                mbar_arrive(&full[slot]);
                            } else {
                                mbar_arrive_expect_tx(&full[slot], (uint32_t)kSlotBytes3);
                                tma_load_3d(slots + (size_t)slot * kSlotBytes3, map, kbyte0 + kc * kChunk3, row, isA ? i : qmax - i, &full[slot]);
                            }
                        }
                        ++cnt;
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (whole warp; the MMAs and commits by one elected lane) =====
        const uint32_t leader = elect_one() ? 1u : 0u;
        uint32_t cntA = 0, cntB = 0, tphase = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            int tm, tn;
            oz3_tile_coords(p, tile, tm, tn);
            if (!oz_tile<kTileN3>(p, tm, tn).wanted) continue;
            const bool stamp = PROBE >= 1 && blockIdx.x == 0 && tile == (int)(blockIdx.x + gridDim.x) && leader != 0u;
            mbar_wait(sm.tmem_empty, tphase ^ 1u);                 // the epilogue has drained the previous level sums
            tc_fence_after();
            if (stamp) g_oz3_probe[0] = clock64();
            oz3_issue_pass<oz3_lo(0), oz3_hi(0), PROBE>(sm, tmem_base, nchunks, cntA, cntB, leader);
            if (stamp) g_oz3_probe[1] = clock64();
            tc_commit_if(leader, sm.tmem_full);
            tphase ^= 1u;
            mbar_wait(sm.tmem_empty, tphase ^ 1u);
            tc_fence_after();
            if (stamp) g_oz3_probe[2] = clock64();
            oz3_issue_pass<oz3_lo(1), oz3_hi(1), PROBE>(sm, tmem_base, nchunks, cntA, cntB, leader);
            if (stamp) g_oz3_probe[3] = clock64();
            tc_commit_if(leader, sm.tmem_full);
            tphase ^= 1u;
        }
    } else {
        // ===== epilogue: warps 2-9; warp w owns the TMEM lanes 32 (w % 4) .. +31 (rows) and 64 of the 128 columns =====
        const int quad = warp & 3, half = (warp - 2) >> 2;
        uint32_t tphase = 0;
        const double s2 = p.scale ? (*p.scale) : 1.0;
        double* stage = reinterpret_cast<double*>(staging + (warp - 2) * kStageWarpBytes3);
        if (lane == 0) tma_prefetch_desc(&mapC);
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            int tm, tn;
            oz3_tile_coords(p, tile, tm, tn);
            const OzTile ot = oz_tile<kTileN3>(p, tm, tn);
            if (!ot.wanted) continue;
#pragma unroll
            for (int pass = 0; pass < 2; ++pass) {
                mbar_wait(sm.tmem_full, tphase);
                tc_fence_after();
                bulk_wait_group0();                                    // this lane's earlier reductions (pass 0 of this tile) are complete
                const bool stamp = PROBE >= 1 && blockIdx.x == 0 && tile == (int)(blockIdx.x + gridDim.x) && warp == 2 && lane == 0;
                if (stamp) g_oz3_probe[4 + 2 * pass] = clock64();
                // weight of the last level of the pass: w_last is that of level S - 1, a level up weighs 2^bits more
                if (pass == 0)
                    oz3_epilogue_pass<oz3_lo(0), oz3_hi(0), PROBE>(tmem_base, quad, half, lane, &mapC, ot.row0 + 32 * quad, ot.col0,
                                                                  p.w_last * s2 * (double)(1ull << (kDigitBits * (kPlanes - 1 - oz3_hi(0)))), stage);
                else
                    oz3_epilogue_pass<oz3_lo(1), oz3_hi(1), PROBE>(tmem_base, quad, half, lane, &mapC, ot.row0 + 32 * quad, ot.col0, p.w_last * s2, stage);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(sm.tmem_empty);
                if (stamp) g_oz3_probe[5 + 2 * pass] = clock64();
                tphase ^= 1u;
            }
        }
        bulk_wait_group0();                                            // every reduction into C has completed before the kernel ends
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
}

// ---- the tensor core's int8 rate by a bare issue loop (measurement support) ---------------------------------------------
// One thread per SM issues tcgen05.mma kind::i8 of 128 x N x 32 on whatever shared memory holds, 16 per iteration into
// rotating accumulators; cycles[0] <- clock64 ticks of CTA 0's loop (issue to completion).  Measured on B200 at 1965 MHz:
// N = 64: 48 cycles per MMA (the 6 KB of operands an MMA reads from shared memory at 128 B/clk), N = 128: 64, N = 256: 128
// (= 8192 int8 MAC per cycle and SM, 4.56 POPS over the chip).  A pause of the issuing thread of up to ~100 cycles per
// 16 MMAs is absorbed, 200 cycles cost 110: the instruction queue is about two MMAs deep.
template <int N>
__global__ void __launch_bounds__(128, 1) int8_mma_peak_kernel(int iters, long long* __restrict__ cycles) {
    extern __shared__ char smem_raw[];
    char* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    __shared__ uint64_t bar;
    __shared__ uint32_t slot;
    const int warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) { mbar_init(&bar, 1); fence_mbar_init(); }
    if (warp == 0) tmem_alloc(&slot, kTmemCols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = slot;
    constexpr uint32_t idesc = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
    constexpr int NACC = kTmemCols / N;
    if (threadIdx.x == 0) {
        const uint32_t sa = smem_u32(base), sb = sa + 4 * kSlotBytes3;
        const long long t0 = clock64();
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int j = 0; j < 16; ++j)
                mma_i8(tmem + (uint32_t)((j % NACC) * N), smem_desc_sw128(sa + (j & 3) * kSlotBytes3 + (j >> 2) * kChunk),
                       smem_desc_sw128(sb + ((j * 3) & 3) * (N * kChunk3) + (j >> 2) * kChunk), idesc, 1u);
        }
        tc_commit(&bar);
        mbar_wait(&bar, 0);
        if (blockIdx.x == 0 && cycles) cycles[0] = clock64() - t0;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, kTmemCols);
}
constexpr int kSmemInt8Peak = 4 * kSlotBytes3 + 4 * 256 * kChunk3 + 2048;

}  // namespace oz
}  // namespace gpb
