// gp_ozaki.cuh -- SURVEY.md 8(f) row 3 ("mixed-precision calculations to take advantage of
// modern hardware capabilities"): the building block of a tensor-core route past the FP64 pipe.
//
// sm_100a has no FP64 kind of tcgen05.mma, and the FP64 DMMA path of gp_gemm.cuh already runs at 93 % of the
// chip's FP64 rate.  The only way to a materially faster  C -= A B^T  in FP64 accuracy is to EMULATE it on the
// integer tensor cores (the Ozaki scheme): write every operand entry in fixed point with one global scale,
//     x / scale = sum_{p=0}^{S-1} d_p 2^{-7 (p+1)},      d_p in [-64, 64]   (balanced base-128 digits, int8),
// so that
//     A B^T = scaleA scaleB sum_{lvl} 2^{-7 (lvl + 2)} sum_{p+q = lvl} D_p(A) D_q(B)^T .
// Every digit-plane product is an int8 GEMM whose int32 accumulation is EXACT (|d| <= 64: 2^12 per term, so
// 2^19 terms fit), products of equal weight share one accumulator, and only the final recombination of the S
// level sums rounds (in FP64).  Pairs with p + q >= S are dropped: with S = 8 that is 2^-56 relative to
// scaleA scaleB, below the FP64 rounding of the result.  Measured on the CPU (a tiled Cholesky whose trailing
// updates are emulated this way, cond(K) = 4e4): S = 6 / 7 / 8 planes give |L - L_fp64| / |L| =
// 1.7e-9 / 1.4e-11 / 1.2e-13, so S = 8 (36 int8 GEMMs per FP64 GEMM) is what north_star's 1e-10 needs with margin.
//
// Kernel (this IS Blackwell-native: tcgen05.mma kind::i8, accumulators in TMEM, operands by TMA):
//   * output tile 128 x 64 per CTA; the S = 8 level accumulators (int32) fill the SM's tensor memory exactly:
//     8 x 64 = 512 columns x 128 lanes;
//   * a stage holds one 32-deep k-chunk of ALL planes of both operands (8 x 128 x 32 B + 8 x 64 x 32 B = 48 KB,
//     two 3-D TMA loads with the 32-byte swizzle), so every operand byte is fetched once and used by all the
//     pairs it takes part in: 36 MMAs (128 x 64 x 32) per stage, ring of 4 stages;
//   * warp 0 = TMA producer, warp 1 = MMA issuer (one elected lane; tcgen05.commit releases stages and hands the
//     finished tile over), warps 2-5 = epilogue: tcgen05.ld the eight level sums of a row segment, convert,
//     recombine smallest weight first in FP64, C -= result.
// Status: a measured building block with its own entry points and parity test; the executor still runs the FP64
// DMMA path (DESIGN.md section 10 says what the measurement implies).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "gp_tma.cuh"

namespace gpb {
namespace oz {

constexpr int kPlanes = 8;           // S
constexpr int kDigitBits = 7;
constexpr int kTileM = 128, kTileN = 64, kChunk = 32;
constexpr int kStagesOz = 4;
constexpr int kABytes = kPlanes * kTileM * kChunk;       // 32 KB
constexpr int kBBytes = kPlanes * kTileN * kChunk;       // 16 KB
constexpr int kStageBytesOz = kABytes + kBBytes;
constexpr int kThreadsOz = 192;
constexpr int kSmemOz = kStagesOz * kStageBytesOz + 1024 + 256;
constexpr int kTmemCols = 512;

// ---- slicing: FP64 -> S planes of balanced base-128 digits ------------------------------------------------------
// planes[p][r][k] (int8, row-major rows x k per plane).  |x| <= scale / 2 is required (the top digit must fit).
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
            long long I = __double2ll_rn(x * 72057594037927936.0);                  // 2^56 = 2^(7 S)
#pragma unroll
            for (int p = kPlanes - 1; p >= 0; --p) {
                const long long d = ((I + 64) & 127) - 64;
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
            long long I56 = __double2ll_rn(xs[e] * inv_scale * 72057594037927936.0);
#pragma unroll
            for (int p = kPlanes - 1; p >= 0; --p) {
                const long long d = ((I56 + 64) & 127) - 64;
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
        const double sc = ldexp(1.0, e + 1 + (f > 0.999 ? 1 : 0)); // >= 2 sqrt(m), with a little head-room at the edge
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
    const double sl = ldexp(1.0, e + 1 + (f > 0.999 ? 1 : 0));
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
            long long I56 = __double2ll_rn(xs[e] * inv_scale * 72057594037927936.0);
#pragma unroll
            for (int p = kPlanes - 1; p >= 0; --p) {
                const long long d = ((I56 + 64) & 127) - 64;
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
};
template <int TN = kTileN>
__device__ __forceinline__ OzTile oz_tile(const OzParams& p, int tm, int tn) {
    OzTile o;
    if (p.tiled == 0 || p.tiled == 3) {
        o.wanted = p.tiled == 0 || tn * TN < (tm + 1) * kTileM;
        o.ld = p.ldc;
        o.c = p.C + (size_t)tm * kTileM * p.ldc + (size_t)tn * TN;
        return o;
    }
    const int bpt = p.t / kTileM;                       // 128-row blocks per tile edge
    if (p.tiled == 2) {
        const int a = tm / bpt, rblk = tm % bpt;
        o.wanted = true;
        o.ld = p.t;
        o.c = p.C + ((size_t)a * p.Mt + p.J) * (size_t)p.t * p.t + (size_t)rblk * kTileM * p.t + (size_t)tn * TN;
        return o;
    }
    const int I = p.J + tm / bpt, rblk = tm % bpt;
    // on the diagonal tile only the lower part is data: skip 128 x TN pieces that lie wholly above the diagonal
    o.wanted = !(I == p.J && tn * TN >= (rblk + 1) * kTileM);
    o.ld = p.t;
    o.c = p.C + ((size_t)I * (I + 1) / 2 + p.J) * (size_t)p.t * p.t + (size_t)rblk * kTileM * p.t + (size_t)tn * TN;
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
                    w *= 128.0;
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


// ---- second shape: 128 x 128 output tile, the eight levels in TWO passes of four ---------------------------------------
// The 128 x 64 kernel above keeps all eight level sums in tensor memory, so every operand byte is fetched once -- but each
// of its MMAs (128 x 64 x 32) makes the tensor core read 4 KB of A and 2 KB of B from shared memory for 32 cycles of
// work: 192 B/cycle against a shared-memory port of 128 B/cycle.  With N = 128 an MMA reads 4 + 4 KB for 64 cycles
// (128 B/cycle), and tensor memory holds four level sums of 128 columns: the levels are done in two passes over k
// (levels 0-3 need the planes 0-3 only: 10 products per chunk; levels 4-7 need all planes: 26), which costs exactly the
// L2 traffic the 128 x 64 kernel spends on loading A once per column half.
// MEASURED (8192 x 8192 x k, FP64-equivalent TFLOP/s): k = 1024 / 4096 / 16384: 128 x 64: 59.7 / 63.4 / 64.7;
// 128 x 128: 51.8 / 68.1 / 62.7.  The two shapes end at the same 2.3-2.45 int8 POPS although their shared-memory
// demand differs by a third: what they share is the 96 KB per 128 x 128 x 32 product that travel from L2 to shared
// memory (5.9 TB/s over the chip at that rate), so that, not the operand read of the tensor core, is the bound.  The
// way past it is a larger output tile per operand byte (a CTA pair with cta_group::2 / TMA multicast); not built.
// The 128 x 64 shape is the default (no second pass, so no drain bubble at short k).
constexpr int kTileN2 = 128;
constexpr int kSlotBytes2 = 2 * kPlanes * kTileM * kChunk;          // 64 KB: 8 planes of A + 8 planes of B, one k-chunk
constexpr int kStages2 = 3;
constexpr int kSmemOz2 = kStages2 * kSlotBytes2 + 1024 + 256;
constexpr uint32_t kIdescI8N128 = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(kTileN2 >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);

// map4: boxes of {32 bytes of k, 128 rows, 4 planes} (the same box serves A and B)
__global__ void __launch_bounds__(kThreadsOz, 1)
ozaki_contract_kernel2(const __grid_constant__ OzParams p, const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB) {
    extern __shared__ char smem_raw[];
    char* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* full = reinterpret_cast<uint64_t*>(base + kStages2 * kSlotBytes2);
    uint64_t* empty = full + kStages2;
    uint64_t* tmem_full = empty + kStages2;
    uint64_t* tmem_empty = tmem_full + 1;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tmem_empty + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages2; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
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
    constexpr int kPlaneBytes = kTileM * kChunk;                    // 4 KB
    constexpr int kHalf = 4 * kPlaneBytes;                          // one TMA box: 4 planes

    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            tma_prefetch_desc(&mapA);
            tma_prefetch_desc(&mapB);
            int stage = 0, phase = 0;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                const int tm = tile / p.tiles_n, tn = tile % p.tiles_n;
                if (!oz_tile<kTileN2>(p, tm, tn).wanted) continue;
                for (int pass = 0; pass < 2; ++pass)
                    for (int kc = 0; kc < p.kchunks; ++kc) {
                        mbar_wait(&empty[stage], (uint32_t)(phase ^ 1));
                        char* dst = base + (size_t)stage * kSlotBytes2;
                        const int k = (p.kc0 + kc) * kChunk, ra = p.row0a + tm * kTileM, rb = p.row0b + tn * kTileN2;
                        mbar_arrive_expect_tx(&full[stage], (uint32_t)(pass ? 4 * kHalf : 2 * kHalf));
                        tma_load_3d(dst, &mapA, k, ra, 0, &full[stage]);
                        tma_load_3d(dst + 2 * kHalf, &mapB, k, rb, 0, &full[stage]);
                        if (pass) {
                            tma_load_3d(dst + kHalf, &mapA, k, ra, 4, &full[stage]);
                            tma_load_3d(dst + 3 * kHalf, &mapB, k, rb, 4, &full[stage]);
                        }
                        if (++stage == kStages2) { stage = 0; phase ^= 1; }
                    }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer =====
        if (lane == 0) {
            int stage = 0, phase = 0, tphase = 0;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                if (!oz_tile<kTileN2>(p, tile / p.tiles_n, tile % p.tiles_n).wanted) continue;
                for (int pass = 0; pass < 2; ++pass) {
                    mbar_wait(tmem_empty, (uint32_t)(tphase ^ 1));      // the epilogue has drained the previous four level sums
                    tc_fence_after();
                    for (int kc = 0; kc < p.kchunks; ++kc) {
                        mbar_wait(&full[stage], (uint32_t)phase);
                        tc_fence_after();
                        const uint32_t sa = smem_u32(base + (size_t)stage * kSlotBytes2), sb = sa + 2 * kHalf;
                        const uint32_t acc = (kc > 0) ? 1u : 0u;
                        if (pass == 0) {
#pragma unroll
                            for (int pa = 0; pa < 4; ++pa)
#pragma unroll
                                for (int pb = 0; pb + pa < 4; ++pb)
                                    mma_i8(tmem_base + (uint32_t)((pa + pb) * kTileN2), smem_desc_sw32(sa + pa * kPlaneBytes),
                                           smem_desc_sw32(sb + pb * kPlaneBytes), kIdescI8N128, pa > 0 ? 1u : acc);
                        } else {
#pragma unroll
                            for (int pa = 0; pa < kPlanes; ++pa)
#pragma unroll
                                for (int pb = 0; pb < kPlanes; ++pb)
                                    if (pa + pb >= 4 && pa + pb < kPlanes)
                                        mma_i8(tmem_base + (uint32_t)(((pa + pb) & 3) * kTileN2), smem_desc_sw32(sa + pa * kPlaneBytes),
                                               smem_desc_sw32(sb + pb * kPlaneBytes), kIdescI8N128, pa > 0 ? 1u : acc);
                        }
                        tc_commit(&empty[stage]);
                        if (++stage == kStages2) { stage = 0; phase ^= 1; }
                    }
                    tc_commit(tmem_full);
                    tphase ^= 1;
                }
            }
        }
    } else {
        // ===== epilogue: 4 warps, warp w owns the TMEM lanes 32 (w % 4) .. +31 = rows of the tile =====
        const int quad = warp & 3;
        int tphase = 0;
        const double s2 = p.scale ? (*p.scale) : 1.0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const OzTile ot = oz_tile<kTileN2>(p, tile / p.tiles_n, tile % p.tiles_n);
            if (!ot.wanted) continue;
            double* crow = ot.c + (size_t)(32 * quad + lane) * ot.ld;
            for (int pass = 0; pass < 2; ++pass) {
                mbar_wait(tmem_full, (uint32_t)tphase);
                tc_fence_after();
                // weight of the LAST level of this pass (3 or 7): w_last is that of level 7, a level up weighs 128 x more
                const double wl = p.w_last * s2 * (pass ? 1.0 : 268435456.0);       // 128^4
#pragma unroll 1
                for (int c0 = 0; c0 < kTileN2; c0 += 16) {
                    double acc[16];
#pragma unroll
                    for (int j = 0; j < 16; ++j) acc[j] = 0.0;
                    double w = wl;
#pragma unroll
                    for (int l = 3; l >= 0; --l) {                            // smallest weight first
                        int32_t v[16];
                        tmem_ld16(tmem_base + ((uint32_t)(32 * quad) << 16) + (uint32_t)(l * kTileN2 + c0), v);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 16; ++j) acc[j] = fma((double)v[j], w, acc[j]);
                        w *= 128.0;
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
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
}

}  // namespace oz
}  // namespace gpb
