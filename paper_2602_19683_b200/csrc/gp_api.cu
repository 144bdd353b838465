// gp_api.cu -- C ABI of libgp_b200.so (include/gp_b200.h): argument validation, workspace
// carving, host-side construction of the static tile-task schedule, kernel launches.
// No library linear algebra (cuBLAS / cuSOLVER) is linked or called anywhere in this library.
#include "../../include/gp_b200.h"

#include <atomic>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <algorithm>
#include <cstring>
#include <map>
#include <mutex>
#include <tuple>
#include <vector>

#include "gp_exec.cuh"
#include "gp_kernels.cuh"
#include "gp_ozaki.cuh"
#include "gp_peak.cuh"
#include "gp_schedule.h"

using namespace gpb;

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// workspace common header: [0, 256) ticket counters, [256, kHdrBytes) per-worker executor statistics
constexpr size_t kStatsOff = 256;
constexpr size_t kHdrBytes = 16384;
constexpr size_t kStatsBytes = 64;   // 8 uint64 per worker, see gp_exec_stats
constexpr int kMaxWorkers = (int)((kHdrBytes - kStatsOff) / kStatsBytes);

// Block edge b: the unit of work and of dependency tracking inside a storage tile (any b in {128, 64, 32} that
// divides the tile works; the tile only fixes the addressing).  128-blocks give the contraction its full rate
// (93 % of the FP64 peak at n = 32768) but every step of the serial spine -- POTRF of a diagonal block, TRSM of
// the block below, update of the next diagonal block -- is then 38 + 24 + 24 us; with 64-blocks it is
// 15 + 7 + 7 us per 64 columns.  Measured Cholesky, b = 64 vs 128: n = 1024: 0.47 / 0.70 ms, 4096: 1.88 / 2.94,
// 6144: 3.96 / 4.58, 8192: 7.17 / 7.43, 16384: the 128-block wins.  So: 64 up to n = 8192, else 128.
std::atomic<int> g_block_edge{0};        // 0 = auto; set by gp_set_block_edge (measurement support)

int pick_block(int tile, int64_t n) {
    int cap = g_block_edge.load(std::memory_order_relaxed);
    if (cap <= 0) cap = n <= 8192 ? 64 : 128;
    if (cap >= 128 && tile % 128 == 0) return 128;
    if (cap >= 64 && tile % 64 == 0) return 64;
    return 32;
}

bool hyper_ok(const gp_hyper& h) {
    return std::isfinite(h.lengthscale) && std::isfinite(h.vertical) && std::isfinite(h.noise) && h.lengthscale > 0.0 &&
           h.vertical > 0.0 && h.noise >= 0.0;
}

HyperDev to_dev(const gp_hyper& h) {
    HyperDev d;
    const double den = h.ell_squared ? 2.0 * h.lengthscale * h.lengthscale : 2.0 * h.lengthscale;
    d.neg_inv_den = -1.0 / den;
    d.vertical = h.vertical;
    d.noise = h.noise;
    return d;
}

// ---- scheduling granularity ---------------------------------------------------------------------
// The tile tasks of PAPER.md Fig. 1 are formed over SCHEDULING tiles of g x g blocks; g is the library's
// choice and independent of the storage tile of the API.  Small g = short serial chains (the TRSM tile task
// of a block row is a chain of g dependent block solves): best while the critical path bounds the run
// (measured at n = 8192: g = 1 / 2 / 4 / 8 -> 7.45 / 8.15 / 8.61 / 10.2 ms).  Large g = fewer, longer work
// items whose operand panels are shared in L2: best once the trailing updates dominate (n = 32768, g = 8:
// 93 % of the FP64 peak).  Auto: g = 1 up to 96 block columns, else the largest divisor of the block counts
// that keeps about 32 scheduling tiles per dimension.
std::atomic<int> g_sched_blocks{0};      // 0 = auto; set by gp_set_schedule_granularity (measurement support)

int gcd_int(int a, int b) { while (b) { const int t = a % b; a = b; b = t; } return a; }

int pick_sched_blocks(int NB, int NBm) {
    const int common = NBm > 0 ? gcd_int(NB, NBm) : NB;
    int want = g_sched_blocks.load(std::memory_order_relaxed);
    if (want <= 0) want = NB <= 96 ? 1 : NB / 32;
    int g = 1;
    for (int d = 1; d <= want && d <= common; ++d)
        if (common % d == 0) g = d;
    return g;
}

int tile_ok(int64_t n, int tile) {
    if (tile <= 0 || tile % 32 != 0) return GP_ERR_TILE;
    if (n % tile != 0) return GP_ERR_TILE;
    return GP_OK;
}

// Per-device state (the schedule cache is keyed by device, so several devices in one process are
// supported): SM count and which kernels already had their dynamic shared-memory limit raised.
constexpr int kMaxDevices = 64;
std::atomic<int> g_sms[kMaxDevices];
std::atomic<uint32_t> g_configured[kMaxDevices];

int current_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) return 0;
    return dev;
}

int sm_count() {
    const int dev = current_device();
    const int slot = dev < kMaxDevices ? dev : kMaxDevices - 1;
    int sms = g_sms[slot].load(std::memory_order_relaxed);
    if (sms == 0 || dev >= kMaxDevices) {
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) sms = 148;
        if (dev < kMaxDevices) g_sms[slot].store(sms, std::memory_order_relaxed);
    }
    return sms;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize applies per device: set it once per (device, kernel).
enum KernelBit : uint32_t { KB_EXEC128 = 1, KB_EXEC64 = 2, KB_EXEC32 = 4, KB_TRTRI128 = 8, KB_TRTRI64 = 16, KB_TRTRI32 = 32,
                            KB_SOLVE128 = 64, KB_SOLVE64 = 128, KB_SOLVE32 = 256 };
template <class F>
int configure_once(uint32_t bit, F&& set) {
    const int dev = current_device();
    if (dev < kMaxDevices && (g_configured[dev].load(std::memory_order_acquire) & bit)) return GP_OK;
    if (!set()) return GP_ERR_CUDA;
    if (dev < kMaxDevices) g_configured[dev].fetch_or(bit, std::memory_order_release);
    return GP_OK;
}

// ---- device-resident schedule cache ---------------------------------------------------------
struct CachedSchedule {
    Item* d_items = nullptr;
    int nitems = 0;
};
std::mutex g_mu;
std::map<std::tuple<int, int, int, int, int, int>, CachedSchedule> g_cache;   // (device, kind, M, Mm, nbt, blk)

// kind 0: Cholesky, 1: predictor with Sigma, 2: predictor without (variances only).
// The first request for a key builds the schedule on the host (list-scheduling simulation: 0.2 s for the
// n = 32768 / tile 1024 factorisation, 1.3 s for n = 65536 / tile 2048) and uploads it with a synchronous
// copy; gp_prepare() does this ahead of time so that the compute calls never block (include/gp_b200.h).
int get_schedule(int kind, int M, int Mm, int nbt, int blk, int workers, CachedSchedule* out) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return GP_ERR_CUDA;
    std::lock_guard<std::mutex> lk(g_mu);
    auto key = std::make_tuple(dev, kind, M, Mm, nbt, blk);
    auto it = g_cache.find(key);
    if (it != g_cache.end()) { *out = it->second; return GP_OK; }
    std::vector<SchedItem> items;
    if (kind == 0) build_cholesky_schedule(M, nbt, workers, items, blk);
    else build_predict_schedule(M, Mm, nbt, workers, items, blk, nullptr, true, /*with_sigma=*/kind == 1);
    static_assert(sizeof(SchedItem) == sizeof(Item), "schedule item layout");
    CachedSchedule cs;
    cs.nitems = (int)items.size();
    if (cudaMalloc(&cs.d_items, items.size() * sizeof(Item) + 16) != cudaSuccess) return GP_ERR_CUDA;
    if (cudaMemcpy(cs.d_items, items.data(), items.size() * sizeof(Item), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaFree(cs.d_items);
        return GP_ERR_CUDA;
    }
    g_cache[key] = cs;
    *out = cs;
    return GP_OK;
}

// ---- TMA tensor maps ---------------------------------------------------------------------------
// cuTensorMapEncodeTiled is fetched from the driver at run time (no link-time libcuda dependency).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)ptr;
    }
    return fn;
}

// Row-major FP64 matrix [rows x cols] (contiguous rows) viewed through boxes of b rows x 16 doubles
// (one 128-byte swizzle row per matrix row): the operand panels of the contraction kernel.
int make_map(CUtensorMap* map, const double* base, uint64_t rows, uint64_t cols, int b) {
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return GP_ERR_CUDA;
    const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)cols * sizeof(double)};
    const cuuint32_t box[2] = {(cuuint32_t)kBK, (cuuint32_t)b};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? GP_OK : GP_ERR_CUDA;
}

struct ExecMaps { CUtensorMap L, V, D; };

// maps for the executor: L (lower-packed tiles as a [tiles*t, t] matrix), V^T (general tiles, same view;
// the L map again when there is no V^T) and the inverted diagonal blocks ([NB*b, b]).
int make_exec_maps(ExecMaps* mp, const ExecParams& p, int b, int64_t m) {
    const uint64_t M = (uint64_t)p.Mt, t = (uint64_t)p.t;
    int rc = make_map(&mp->L, p.L, M * (M + 1) / 2 * t, t, b);
    if (rc != GP_OK) return rc;
    if (p.Vt) rc = make_map(&mp->V, p.Vt, (uint64_t)(m / p.t) * M * t, t, b);
    else mp->V = mp->L;
    if (rc != GP_OK) return rc;
    return make_map(&mp->D, p.invD, (uint64_t)p.NB * b, (uint64_t)b, b);
}

template <int BLK>
int launch_exec(const ExecParams& p, const ExecMaps& mp, int workers, cudaStream_t st) {
    constexpr int smem = exec_smem_bytes<BLK>();
    const int rc = configure_once(BLK == 128 ? KB_EXEC128 : (BLK == 64 ? KB_EXEC64 : KB_EXEC32), [] {
        return cudaFuncSetAttribute(exec_kernel<BLK>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) == cudaSuccess;
    });
    if (rc != GP_OK) return rc;
    exec_kernel<BLK><<<workers, kThreads, smem, st>>>(p, mp.L, mp.V, mp.D);
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

int launch_exec_any(int b, const ExecParams& p, int64_t m, int workers, cudaStream_t st) {
    ExecMaps mp;
    const int rc = make_exec_maps(&mp, p, b, m);
    if (rc != GP_OK) return rc;
    switch (b) {
        case 128: return launch_exec<128>(p, mp, workers, st);
        case 64: return launch_exec<64>(p, mp, workers, st);
        default: return launch_exec<32>(p, mp, workers, st);
    }
}

template <int BLK>
int launch_trtri(const double* L, int t, int nbt, int NB, double* invD, cudaStream_t st, double* fill = nullptr) {
    constexpr int smem = DiagSmem<BLK>::kBytes;
    const int rc = configure_once(BLK == 128 ? KB_TRTRI128 : (BLK == 64 ? KB_TRTRI64 : KB_TRTRI32), [] {
        return cudaFuncSetAttribute(trtri_diag_kernel<BLK>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) == cudaSuccess;
    });
    if (rc != GP_OK) return rc;
    trtri_diag_kernel<BLK><<<NB, kConsumerThreads, smem, st>>>(L, t, nbt, invD, fill);
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

int launch_trtri_any(int b, const double* L, int t, int NB, double* invD, cudaStream_t st, double* fill = nullptr) {
    switch (b) {
        case 128: return launch_trtri<128>(L, t, t / 128, NB, invD, st, fill);
        case 64: return launch_trtri<64>(L, t, t / 64, NB, invD, st, fill);
        default: return launch_trtri<32>(L, t, t / 32, NB, invD, st, fill);
    }
}

template <int SB>
int launch_solves(const double* dL, int tile, int NB, const double* invD, const double* dY, double* beta, double* dAlpha,
                  unsigned int* ticket, cudaStream_t st) {
    constexpr int smem = SolveCfg<SB>::kSmemBytes;
    const int rc = configure_once(SB == 128 ? KB_SOLVE128 : (SB == 64 ? KB_SOLVE64 : KB_SOLVE32), [] {
        return cudaFuncSetAttribute(forward_solve_kernel<SB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) == cudaSuccess &&
               cudaFuncSetAttribute(backward_solve_kernel<SB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) == cudaSuccess;
    });
    if (rc != GP_OK) return rc;
    forward_solve_kernel<SB><<<NB, 256, smem, st>>>(dL, tile, NB, invD, dY, beta, dAlpha, ticket);
    backward_solve_kernel<SB><<<NB, 256, smem, st>>>(dL, tile, NB, invD, beta, dAlpha, ticket + 1);
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

int workers_for(int sched_width) {
    const int sms = sm_count();
    if (sched_width <= 0) return sms < kMaxWorkers ? sms : kMaxWorkers;
    const int w = sched_width < sms ? sched_width : sms;   // one resident CTA per SM: more cannot be co-resident
    return w < kMaxWorkers ? w : kMaxWorkers;
}

int launch_assemble(const double* dA, int64_t na, const double* dB, int64_t nb, int D, const HyperDev& h, int tile, int sym_lower,
                    double* out, cudaStream_t st) {
    const int64_t Ma = na / tile, Mb = nb / tile;
    const int64_t ntiles = sym_lower ? Ma * (Ma + 1) / 2 : Ma * Mb;
    const int sb = (tile + kAsmBlk - 1) / kAsmBlk;
    if (ntiles * sb * sb > 2147483647LL) return GP_ERR_SIZE;
    dim3 grid((unsigned)(ntiles * sb * sb));
    const size_t smem = 2 * (size_t)kAsmMaxD * kAsmBlk * sizeof(double);
    assemble_tiles_kernel<<<grid, 256, smem, st>>>(dA, dB, D, h, tile, (int)Mb, sym_lower, out);
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

// workspace layouts ---------------------------------------------------------------------------
struct CholWs { size_t ticket, verL, invD, total; };
CholWs chol_ws(int64_t n, int b) {
    const size_t NB = (size_t)(n / b);
    CholWs w;
    w.ticket = 0;
    w.verL = kHdrBytes;
    w.invD = align_up(w.verL + NB * NB * sizeof(int), 256);
    w.total = w.invD + NB * (size_t)b * b * sizeof(double);
    return w;
}
struct SolveWs { size_t ticket, flags, beta, invD, total; };
SolveWs solve_ws(int64_t n, int b) {
    const size_t NB = (size_t)(n / b);
    SolveWs w;
    w.ticket = 0;
    w.flags = kHdrBytes;
    w.beta = align_up(w.flags + 2 * NB * sizeof(int), 256);
    w.invD = align_up(w.beta + (size_t)n * sizeof(double), 256);
    w.total = w.invD + NB * (size_t)b * b * sizeof(double);
    return w;
}
struct CovWs { size_t ticket, verV, verS, invD, Vt, total; };
CovWs cov_ws(int64_t n, int64_t m, int b) {
    const size_t NB = (size_t)(n / b), NBm = (size_t)(m / b);
    CovWs w;
    w.ticket = 0;
    w.verV = kHdrBytes;
    w.verS = align_up(w.verV + NBm * NB * sizeof(int), 256);
    w.invD = align_up(w.verS + NBm * NBm * sizeof(int), 256);
    w.Vt = align_up(w.invD + NB * (size_t)b * b * sizeof(double), 256);
    w.total = w.Vt + (size_t)m * (size_t)n * sizeof(double);
    return w;
}

}  // namespace

extern "C" {

int gp_block_size(int tile) {
    if (tile <= 0 || tile % 32 != 0) return GP_ERR_TILE;
    return tile % 128 == 0 ? 128 : (tile % 64 == 0 ? 64 : 32);
}

int gp_block_size_for(int64_t n, int tile) {
    if (n <= 0) return GP_ERR_SIZE;
    const int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    return pick_block(tile, n);
}

int gp_set_block_edge(int b) {
    if (b != 0 && b != 32 && b != 64 && b != 128) return GP_ERR_SIZE;
    g_block_edge.store(b, std::memory_order_relaxed);
    return GP_OK;
}

const char* gp_strerror(int code) {
    switch (code) {
        case GP_OK: return "ok";
        case GP_ERR_NULL: return "required pointer is NULL";
        case GP_ERR_SIZE: return "invalid size (n, m, na, nb or D)";
        case GP_ERR_TILE: return "invalid tile size (must be a positive multiple of 32 dividing n and m)";
        case GP_ERR_HYPER: return "invalid hyperparameters";
        case GP_ERR_WORKSPACE: return "workspace too small";
        case GP_ERR_CUDA: return "CUDA runtime error";
        case GP_ERR_MODE: return "unknown layout mode";
        case GP_ERR_LIMIT: return "problem exceeds the fixed scratch of the no-allocation entry point (gp_solve_noalloc: n <= 8192)";
        default: return "unknown error code";
    }
}

int gp_workspace_bytes(int64_t n, int64_t m, int D, int tile, size_t* chol, size_t* solve, size_t* full_cov) {
    if (n <= 0 || m < 0 || D <= 0) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    if (m > 0 && m % tile != 0) return GP_ERR_TILE;
    const int b = pick_block(tile, n);
    if (chol) *chol = chol_ws(n, b).total;
    if (solve) *solve = solve_ws(n, b).total;
    if (full_cov) *full_cov = m > 0 ? cov_ws(n, m, b).total : 0;
    return GP_OK;
}

int gp_assemble_tiles(const double* dA, int64_t na, const double* dB, int64_t nb, int D, gp_hyper h, int tile, int mode,
                      double* dTiles, void* stream) {
    if (!dA || !dB || !dTiles) return GP_ERR_NULL;
    if (na <= 0 || nb <= 0 || D <= 0) return GP_ERR_SIZE;
    if (mode != GP_SYM_LOWER && mode != GP_GENERAL) return GP_ERR_MODE;
    int rc = tile_ok(na, tile);
    if (rc != GP_OK) return rc;
    rc = tile_ok(nb, tile);
    if (rc != GP_OK) return rc;
    if (!hyper_ok(h)) return GP_ERR_HYPER;
    if (mode == GP_SYM_LOWER && (dA != dB || na != nb)) return GP_ERR_SIZE;
    return launch_assemble(dA, na, dB, nb, D, to_dev(h), tile, mode == GP_SYM_LOWER ? 1 : 0, dTiles, (cudaStream_t)stream);
}

int gp_tiles_to_dense(const double* dTiles, int64_t n, int64_t nb, int tile, int lower_packed, double* dDense, void* stream) {
    if (!dTiles || !dDense) return GP_ERR_NULL;
    if (n <= 0) return GP_ERR_SIZE;
    if (lower_packed) nb = n;
    if (nb <= 0) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    rc = tile_ok(nb, tile);
    if (rc != GP_OK) return rc;
    tiles_to_dense_kernel<<<sm_count() * 8, 256, 0, (cudaStream_t)stream>>>(dTiles, n, nb, tile, lower_packed, dDense);
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

int gp_cholesky_task_counts(int64_t n, int tile, int64_t* tile_tasks, int64_t* work_items) {
    if (n <= 0) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    const int64_t M = n / tile;
    if (tile_tasks) *tile_tasks = M + M * (M - 1) / 2 + M * (M - 1) / 2 + M * (M - 1) * (M - 2) / 6;
    if (work_items) {
        std::vector<SchedItem> items;
        const int b = pick_block(tile, n), NB = (int)(n / b), g = pick_sched_blocks(NB, 0);
        build_cholesky_schedule(NB / g, g, 148, items, b, nullptr, false);
        *work_items = (int64_t)items.size();
    }
    return GP_OK;
}

int gp_cholesky_tiled(double* dKL, int64_t n, int tile, int sched_width, int* d_info, void* dWork, size_t work_bytes, void* stream) {
    if (!dKL || !d_info || !dWork) return GP_ERR_NULL;
    if (n <= 0 || n > (int64_t)1 << 22) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    const int b = pick_block(tile, n);
    if (n / b > 65535) return GP_ERR_SIZE;            // block indices travel in 16 bits of a work item
    const CholWs w = chol_ws(n, b);
    if (work_bytes < w.total) return GP_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const int M = (int)(n / tile), nbt = tile / b, NB = (int)(n / b);
    const int workers = workers_for(sched_width);
    const int g = pick_sched_blocks(NB, 0);
    CachedSchedule cs;
    rc = get_schedule(0, NB / g, 0, g, b, sm_count(), &cs);
    if (rc != GP_OK) return rc;
    char* ws = (char*)dWork;
    if (cudaMemsetAsync(ws, 0, w.invD, st) != cudaSuccess) return GP_ERR_CUDA;        // ticket + version counters
    if (cudaMemsetAsync(d_info, 0, sizeof(int), st) != cudaSuccess) return GP_ERR_CUDA;
    ExecParams p;
    memset(&p, 0, sizeof(p));
    p.L = dKL;
    p.invD = (double*)(ws + w.invD);
    p.verL = (int*)(ws + w.verL);
    p.items = cs.d_items;
    p.nitems = cs.nitems;
    p.ticket = (unsigned int*)(ws + w.ticket);
    p.stats = (unsigned long long*)(ws + kStatsOff);
    p.d_info = d_info;
    p.t = tile;
    p.nbt = nbt;
    p.snbt = g;
    p.NB = NB;
    p.Mt = M;
    return launch_exec_any(b, p, 0, workers, st);
}

int gp_solve(const double* dL, int64_t n, int tile, const double* dY, double* dAlpha, double* dBeta, void* dWork, size_t work_bytes,
             void* stream) {
    if (!dL || !dY || !dAlpha || !dWork) return GP_ERR_NULL;
    if (n <= 0) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    const int b = pick_block(tile, n);
    const SolveWs w = solve_ws(n, b);
    if (work_bytes < w.total) return GP_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const int NB = (int)(n / b);
    char* ws = (char*)dWork;
    if (cudaMemsetAsync(ws, 0, w.beta, st) != cudaSuccess) return GP_ERR_CUDA;
    double* invD = (double*)(ws + w.invD);
    double* beta = dBeta ? dBeta : (double*)(ws + w.beta);
    unsigned int* ticket = (unsigned int*)(ws + w.ticket);
    // the kernel that inverts the diagonal blocks also marks beta "not yet computed" (the forward solve marks alpha)
    rc = launch_trtri_any(b, dL, tile, NB, invD, st, beta);
    if (rc != GP_OK) return rc;
    switch (b) {
        case 128: rc = launch_solves<128>(dL, tile, NB, invD, dY, beta, dAlpha, ticket, st); break;
        case 64: rc = launch_solves<64>(dL, tile, NB, invD, dY, beta, dAlpha, ticket, st); break;
        default: rc = launch_solves<32>(dL, tile, NB, invD, dY, beta, dAlpha, ticket, st); break;
    }
    if (rc != GP_OK) return rc;
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

// ---- gp_solve without any allocation: the scratch is a static device array of the library ----------------------------------
}  // extern "C"
namespace {
// In HOST code this name is only a stand-in for the symbol, not a device address: the address is taken per device with
// cudaGetSymbolAddress (below) and that pointer is what the kernels receive.
static __device__ __align__(256) unsigned char g_solve_noalloc_scratch[GP_SOLVE_NOALLOC_BYTES];
void* g_solve_noalloc_ptr[kMaxDevices];          // per device, guarded by g_mu

int solve_noalloc_scratch(void** out) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return GP_ERR_CUDA;
    if (dev < 0 || dev >= kMaxDevices) return GP_ERR_SIZE;
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_solve_noalloc_ptr[dev]) {
        void* ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, g_solve_noalloc_scratch) != cudaSuccess || !ptr) return GP_ERR_CUDA;   // with `dev` current
        g_solve_noalloc_ptr[dev] = ptr;
    }
    *out = g_solve_noalloc_ptr[dev];
    return GP_OK;
}
}  // namespace
extern "C" {

int gp_solve_noalloc(const double* dL, int64_t n, int tile, const double* dY, double* dAlpha, double* dBeta, void* stream) {
    if (!dL || !dY || !dAlpha) return GP_ERR_NULL;
    if (n <= 0) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    if (n > GP_SOLVE_NOALLOC_MAX_N || solve_ws(n, pick_block(tile, n)).total > (size_t)GP_SOLVE_NOALLOC_BYTES) return GP_ERR_LIMIT;
    void* scratch = nullptr;
    if ((rc = solve_noalloc_scratch(&scratch)) != GP_OK) return rc;
    // the existing path, unchanged, on the static scratch: it clears its counters and marks beta / alpha "not yet computed"
    // itself, so the previous call's contents do not matter
    return gp_solve(dL, n, tile, dY, dAlpha, dBeta, scratch, (size_t)GP_SOLVE_NOALLOC_BYTES, stream);
}

int gp_predict_mean(const double* dX, int64_t n, int D, const double* dAlpha, const double* dXs, int64_t m, gp_hyper h, double* dMean,
                    void* stream) {
    if (!dX || !dAlpha || !dXs || !dMean) return GP_ERR_NULL;
    if (n <= 0 || m <= 0 || D <= 0 || D > 512) return GP_ERR_SIZE;
    if (!hyper_ok(h)) return GP_ERR_HYPER;
    const unsigned grid = (unsigned)((m + kMeanTM - 1) / kMeanTM);
    const size_t smem = ((size_t)kMeanTM * D + (size_t)kMeanTM * 256) * sizeof(double);
    predict_mean_kernel<<<grid, 256, smem, (cudaStream_t)stream>>>(dX, n, D, dAlpha, dXs, m, to_dev(h), dMean);
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

// a9, a11, a12 (dSigma != NULL) or the variance-only variant (dSigma == NULL, dVar != NULL)
static int run_predictor(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m, gp_hyper h, int tile,
                         int sched_width, double* dSigma, double* dVar, void* dWork, size_t work_bytes, void* stream,
                         double* dVtExt = nullptr) {
    if (!dL || !dX || !dXs || (!dSigma && !dVar && !dVtExt) || !dWork) return GP_ERR_NULL;
    if (n <= 0 || m <= 0 || D <= 0 || n > (int64_t)1 << 22 || m > (int64_t)1 << 22) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    rc = tile_ok(m, tile);
    if (rc != GP_OK) return rc;
    if (!hyper_ok(h)) return GP_ERR_HYPER;
    const int b = pick_block(tile, n);
    if (n / b > 65535 || m / b > 65535) return GP_ERR_SIZE;   // block indices travel in 16 bits of a work item
    const CovWs w = cov_ws(n, m, b);
    if (work_bytes < w.total) return GP_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const int M = (int)(n / tile), nbt = tile / b, NB = (int)(n / b), NBm = (int)(m / b);
    const int workers = workers_for(sched_width);
    const int g = pick_sched_blocks(NB, NBm);
    CachedSchedule cs;
    rc = get_schedule(dSigma ? 1 : 2, NB / g, NBm / g, g, b, sm_count(), &cs);
    if (rc != GP_OK) return rc;
    char* ws = (char*)dWork;
    const HyperDev hd = to_dev(h);
    double* Vt = dVtExt ? dVtExt : (double*)(ws + w.Vt);
    double* invD = (double*)(ws + w.invD);
    if (cudaMemsetAsync(ws, 0, w.invD, st) != cudaSuccess) return GP_ERR_CUDA;
    // a9: K_{X^,X} (m x n, noise-free) straight into the V^T buffer; prior K_{X^,X^} straight into Sigma
    rc = launch_assemble(dXs, m, dX, n, D, hd, tile, 0, Vt, st);
    if (rc != GP_OK) return rc;
    if (dSigma) {
        // dense m x m = one "tile" of edge m
        const int sb = (int)((m + kAsmBlk - 1) / kAsmBlk);
        if ((int64_t)sb * sb > 2147483647LL) return GP_ERR_SIZE;
        dim3 grid((unsigned)(sb * sb));
        const size_t smem = 2 * (size_t)kAsmMaxD * kAsmBlk * sizeof(double);
        assemble_tiles_kernel<<<grid, 256, smem, st>>>(dXs, dXs, D, hd, (int)m, 1, 0, dSigma);
        if (cudaGetLastError() != cudaSuccess) return GP_ERR_CUDA;
    }
    rc = launch_trtri_any(b, dL, tile, NB, invD, st);
    if (rc != GP_OK) return rc;
    ExecParams p;
    memset(&p, 0, sizeof(p));
    p.L = const_cast<double*>(dL);
    p.Vt = Vt;
    p.S = dSigma;
    p.invD = invD;
    p.verV = (int*)(ws + w.verV);
    p.verS = (int*)(ws + w.verS);
    p.items = cs.d_items;
    p.nitems = cs.nitems;
    p.ticket = (unsigned int*)(ws + w.ticket);
    p.stats = (unsigned long long*)(ws + kStatsOff);
    p.t = tile;
    p.nbt = nbt;
    p.snbt = g;
    p.NB = NB;
    p.NBm = NBm;
    p.Mt = M;
    p.m = m;
    p.L_final = 1;
    rc = launch_exec_any(b, p, m, workers, st);
    if (rc != GP_OK) return rc;
    if (dSigma) {
        dim3 mg((unsigned)(m / 32), (unsigned)(m / 32));
        mirror_lower_kernel<<<mg, dim3(32, 8), 0, st>>>(dSigma, m);
    } else if (dVar) {
        // var_a = k(x^_a, x^_a) - sum_i V_ia^2 with k(x,x) = v (noise-free prior, reading A2): one warp per test point
        posterior_var_kernel<<<(unsigned)((m + 7) / 8), 256, 0, st>>>(Vt, m, n, tile, hd.vertical, dVar);
    }
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

int gp_predict_full_cov(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m, gp_hyper h, int tile,
                        int sched_width, double* dSigma, void* dWork, size_t work_bytes, void* stream) {
    if (!dSigma) return GP_ERR_NULL;
    return run_predictor(dL, dX, n, D, dXs, m, h, tile, sched_width, dSigma, nullptr, dWork, work_bytes, stream);
}

int gp_predict_variance(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m, gp_hyper h, int tile,
                        int sched_width, double* dVar, void* dWork, size_t work_bytes, void* stream) {
    if (!dVar) return GP_ERR_NULL;
    return run_predictor(dL, dX, n, D, dXs, m, h, tile, sched_width, nullptr, dVar, dWork, work_bytes, stream);
}

int gp_predict_vt(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m, gp_hyper h, int tile, int sched_width,
                  double* dVt, void* dWork, size_t work_bytes, void* stream) {
    if (!dVt) return GP_ERR_NULL;
    return run_predictor(dL, dX, n, D, dXs, m, h, tile, sched_width, nullptr, nullptr, dWork, work_bytes, stream, dVt);
}

int gp_cov_rows_workspace_bytes(int64_t n, int64_t m, int64_t rows, int tile, size_t* bytes) {
    if (!bytes) return GP_ERR_NULL;
    if (n <= 0 || m <= 0 || rows <= 0) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc == GP_OK) rc = tile_ok(m, tile);
    if (rc == GP_OK) rc = tile_ok(rows, tile);
    if (rc != GP_OK) return rc;
    const int b = pick_block(tile, n);
    const size_t NBm = (size_t)(m / b);
    *bytes = kHdrBytes + align_up(NBm * NBm * sizeof(int), 256) + align_up((size_t)(rows / b) * NBm * sizeof(Item), 256) + 256;
    return GP_OK;
}

int gp_predict_cov_rows(const double* dVtAll, const double* dXsAll, int64_t n, int64_t m, int D, int64_t row0, int64_t rows, gp_hyper h,
                        int tile, int sched_width, double* dSigmaRows, void* dWork, size_t work_bytes, void* stream) {
    if (!dVtAll || !dXsAll || !dSigmaRows || !dWork) return GP_ERR_NULL;
    if (n <= 0 || m <= 0 || D <= 0 || rows <= 0 || row0 < 0 || row0 + rows > m || n > (int64_t)1 << 22 || m > (int64_t)1 << 22) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc == GP_OK) rc = tile_ok(m, tile);
    if (rc == GP_OK) rc = tile_ok(rows, tile);
    if (rc != GP_OK) return rc;
    if (row0 % tile != 0) return GP_ERR_TILE;
    if (!hyper_ok(h)) return GP_ERR_HYPER;
    const int b = pick_block(tile, n);
    if (n / b > 65535 || m / b > 65535) return GP_ERR_SIZE;
    size_t need = 0;
    gp_cov_rows_workspace_bytes(n, m, rows, tile, &need);
    if (work_bytes < need) return GP_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const int NB = (int)(n / b), NBm = (int)(m / b), nrows = (int)(rows / b), gr0 = (int)(row0 / b);
    char* ws = (char*)dWork;
    const size_t off_ver = kHdrBytes, off_items = off_ver + align_up((size_t)NBm * NBm * sizeof(int), 256);
    if (cudaMemsetAsync(ws, 0, off_items, st) != cudaSuccess) return GP_ERR_CUDA;
    const HyperDev hd = to_dev(h);
    {   // the prior K_{X^_r, X^} straight into the output rows
        const int64_t rb = (rows + kAsmBlk - 1) / kAsmBlk, cb = (m + kAsmBlk - 1) / kAsmBlk;
        if (rb * cb > 2147483647LL) return GP_ERR_SIZE;
        const size_t smem = 2 * (size_t)kAsmMaxD * kAsmBlk * sizeof(double);
        assemble_dense_kernel<<<(unsigned)(rb * cb), 256, smem, st>>>(dXsAll + row0 * D, rows, dXsAll, m, D, hd, dSigmaRows, m);
        if (cudaGetLastError() != cudaSuccess) return GP_ERR_CUDA;
    }
    Item* items = (Item*)(ws + off_items);
    cov_row_items_kernel<<<(nrows * NBm + 255) / 256, 256, 0, st>>>((uint4*)items, nrows, gr0, NBm, NB, (unsigned)OP_UPD_S);
    ExecParams p;
    memset(&p, 0, sizeof(p));
    p.L = const_cast<double*>(dVtAll);        // no item touches L: the pointer only has to be mappable
    p.Vt = const_cast<double*>(dVtAll);
    p.S = dSigmaRows;
    p.invD = (double*)ws;
    p.verV = (int*)(ws + off_ver);
    p.verS = (int*)(ws + off_ver);
    p.items = items;
    p.nitems = nrows * NBm;
    p.ticket = (unsigned int*)ws;
    p.stats = (unsigned long long*)(ws + kStatsOff);
    p.t = tile;
    p.nbt = tile / b;
    p.snbt = NB;                               // one version per item: the whole contraction range is one "column"
    p.NB = NB;
    p.NBm = NBm;
    p.Mt = (int)(n / tile);
    p.m = m;
    p.s_row0 = gr0;
    p.L_final = 1;
    p.no_deps = 1;
    // the L map is built over [Mt (Mt + 1) / 2 * t, t]: keep it inside the V^T buffer, which has m / t * Mt * t rows
    {
        ExecMaps mp;
        int rc2 = make_map(&mp.V, dVtAll, (uint64_t)(m / tile) * (uint64_t)p.Mt * (uint64_t)tile, (uint64_t)tile, b);
        if (rc2 != GP_OK) return rc2;
        mp.L = mp.V;
        mp.D = mp.V;
        switch (b) {
            case 128: rc = launch_exec<128>(p, mp, workers_for(sched_width), st); break;
            case 64: rc = launch_exec<64>(p, mp, workers_for(sched_width), st); break;
            default: rc = launch_exec<32>(p, mp, workers_for(sched_width), st); break;
        }
    }
    return rc;
}

int gp_log_marginal_likelihood(const double* dL, int64_t n, int tile, const double* dY, const double* dAlpha, double* d_out,
                               void* stream) {
    if (!dL || !dY || !dAlpha || !d_out) return GP_ERR_NULL;
    if (n <= 0) return GP_ERR_SIZE;
    const int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    log_marginal_likelihood_kernel<<<1, 1024, 0, (cudaStream_t)stream>>>(dL, n, tile, dY, dAlpha, d_out);
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

int gp_prepare(int64_t n, int64_t m, int tile, int what, double* build_ms) {
    if (n <= 0 || m < 0 || n > (int64_t)1 << 22 || m > (int64_t)1 << 22) return GP_ERR_SIZE;
    if ((what & ~(GP_PREPARE_CHOLESKY | GP_PREPARE_FULL_COV | GP_PREPARE_VARIANCE)) != 0 || what == 0) return GP_ERR_MODE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    const bool pred = (what & (GP_PREPARE_FULL_COV | GP_PREPARE_VARIANCE)) != 0;
    if (pred && m <= 0) return GP_ERR_SIZE;
    if (pred && (rc = tile_ok(m, tile)) != GP_OK) return rc;
    const int b = pick_block(tile, n);
    if (n / b > 65535 || m / b > 65535) return GP_ERR_SIZE;
    const int NB = (int)(n / b), NBm = (int)(m / b);
    const int gc = pick_sched_blocks(NB, 0), gp = pred ? pick_sched_blocks(NB, NBm) : 1;
    const auto t0 = std::chrono::steady_clock::now();
    CachedSchedule cs;
    if ((what & GP_PREPARE_CHOLESKY) && (rc = get_schedule(0, NB / gc, 0, gc, b, sm_count(), &cs)) != GP_OK) return rc;
    if ((what & GP_PREPARE_FULL_COV) && (rc = get_schedule(1, NB / gp, NBm / gp, gp, b, sm_count(), &cs)) != GP_OK) return rc;
    if ((what & GP_PREPARE_VARIANCE) && (rc = get_schedule(2, NB / gp, NBm / gp, gp, b, sm_count(), &cs)) != GP_OK) return rc;
    if (build_ms) *build_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    return GP_OK;
}

int gp_set_schedule_granularity(int blocks) {
    if (blocks < 0 || blocks > 4096) return GP_ERR_SIZE;
    g_sched_blocks.store(blocks, std::memory_order_relaxed);
    return GP_OK;
}

int gp_schedule_granularity(int64_t n, int64_t m, int tile) {
    if (n <= 0 || m < 0) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    if (m > 0 && (rc = tile_ok(m, tile)) != GP_OK) return rc;
    const int b = pick_block(tile, n);
    return pick_sched_blocks((int)(n / b), (int)(m / b));
}

void gp_release_cached_schedules(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    cudaDeviceSynchronize();
    for (auto& kv : g_cache) cudaFree(kv.second.d_items);
    g_cache.clear();
}

}  // extern "C"

// ---- whole pipeline on host buffers -----------------------------------------------------------
namespace {
struct PipeWs { size_t X, y, Xs, KL, alpha, beta, mean, Sigma, info, scratch, scratch_bytes, total; };
int pipe_ws(int64_t n, int64_t m, int D, int tile, PipeWs* w, bool mixed = false) {
    size_t c = 0, s = 0, f = 0;
    int rc = gp_workspace_bytes(n, m, D, tile, &c, &s, &f);
    if (rc != GP_OK) return rc;
    if (mixed) {        // the emulated path: its scratch (digit planes of L and V^T) replaces the executor's
        if ((rc = gp_mixed_workspace_bytes(n, tile, &c)) != GP_OK) return rc;
        if (m > 0 && (rc = gp_mixed_predict_workspace_bytes(n, m, tile, &f)) != GP_OK) return rc;
    }
    const size_t M = (size_t)(n / tile);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    w->X = take((size_t)n * D * 8);
    w->y = take((size_t)n * 8);
    w->Xs = take((size_t)(m > 0 ? m : 1) * D * 8);
    w->KL = take(M * (M + 1) / 2 * (size_t)tile * tile * 8);
    w->alpha = take((size_t)n * 8);
    w->beta = take((size_t)n * 8);
    w->mean = take((size_t)(m > 0 ? m : 1) * 8);
    w->Sigma = take((size_t)m * m * 8 + 8);
    w->info = take(sizeof(int));
    w->scratch_bytes = c > s ? (c > f ? c : f) : (s > f ? s : f);
    w->scratch = take(w->scratch_bytes);
    w->total = off;
    return GP_OK;
}
}  // namespace

extern "C" {

int gp_pipeline_workspace_bytes(int64_t n, int64_t m, int D, int tile, size_t* bytes) {
    if (!bytes) return GP_ERR_NULL;
    PipeWs w;
    int rc = pipe_ws(n, m, D, tile, &w);
    if (rc != GP_OK) return rc;
    *bytes = w.total;
    return GP_OK;
}

int gp_pipeline_mixed_workspace_bytes(int64_t n, int64_t m, int D, int tile, size_t* bytes) {
    if (!bytes) return GP_ERR_NULL;
    PipeWs w;
    int rc = pipe_ws(n, m, D, tile, &w, true);
    if (rc != GP_OK) return rc;
    *bytes = w.total;
    return GP_OK;
}

static int pipeline_host_impl(bool mixed, const double* hX, const double* hY, const double* hXs, int64_t n, int64_t m, int D, gp_hyper h, int tile,
                              int sched_width, double* hMean, double* hSigma, double* hAlpha, int* h_info, void* dWork, size_t work_bytes,
                              void* stream) {
    if (!hX || !hY || !hXs || !hMean || !h_info || !dWork) return GP_ERR_NULL;
    if (m <= 0) return GP_ERR_SIZE;
    if (!hyper_ok(h)) return GP_ERR_HYPER;
    PipeWs w;
    int rc = pipe_ws(n, m, D, tile, &w, mixed);
    if (rc != GP_OK) return rc;
    if (work_bytes < w.total) return GP_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    char* ws = (char*)dWork;
    double *dX = (double*)(ws + w.X), *dY = (double*)(ws + w.y), *dXs = (double*)(ws + w.Xs), *dKL = (double*)(ws + w.KL);
    double *dAlpha = (double*)(ws + w.alpha), *dBeta = (double*)(ws + w.beta), *dMean = (double*)(ws + w.mean);
    double* dSigma = (double*)(ws + w.Sigma);
    int* d_info = (int*)(ws + w.info);
    void* scratch = ws + w.scratch;
    if (cudaMemcpyAsync(dX, hX, (size_t)n * D * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return GP_ERR_CUDA;
    if (cudaMemcpyAsync(dY, hY, (size_t)n * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return GP_ERR_CUDA;
    if (cudaMemcpyAsync(dXs, hXs, (size_t)m * D * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return GP_ERR_CUDA;
    if ((rc = gp_assemble_tiles(dX, n, dX, n, D, h, tile, GP_SYM_LOWER, dKL, stream)) != GP_OK) return rc;
    rc = mixed ? gp_cholesky_tiled_mixed(dKL, n, tile, sched_width, d_info, scratch, w.scratch_bytes, stream)
               : gp_cholesky_tiled(dKL, n, tile, sched_width, d_info, scratch, w.scratch_bytes, stream);
    if (rc != GP_OK) return rc;
    if ((rc = gp_solve(dKL, n, tile, dY, dAlpha, dBeta, scratch, w.scratch_bytes, stream)) != GP_OK) return rc;
    if ((rc = gp_predict_mean(dX, n, D, dAlpha, dXs, m, h, dMean, stream)) != GP_OK) return rc;
    if (hSigma) {
        rc = mixed ? gp_predict_full_cov_mixed(dKL, dX, n, D, dXs, m, h, tile, sched_width, dSigma, scratch, w.scratch_bytes, stream)
                   : gp_predict_full_cov(dKL, dX, n, D, dXs, m, h, tile, sched_width, dSigma, scratch, w.scratch_bytes, stream);
        if (rc != GP_OK)
            return rc;
        if (cudaMemcpyAsync(hSigma, dSigma, (size_t)m * m * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return GP_ERR_CUDA;
    }
    if (cudaMemcpyAsync(hMean, dMean, (size_t)m * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return GP_ERR_CUDA;
    if (hAlpha && cudaMemcpyAsync(hAlpha, dAlpha, (size_t)n * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return GP_ERR_CUDA;
    if (cudaMemcpyAsync(h_info, d_info, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess) return GP_ERR_CUDA;
    return cudaStreamSynchronize(st) == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

int gp_pipeline_host(const double* hX, const double* hY, const double* hXs, int64_t n, int64_t m, int D, gp_hyper h, int tile,
                     int sched_width, double* hMean, double* hSigma, double* hAlpha, int* h_info, void* dWork, size_t work_bytes,
                     void* stream) {
    return pipeline_host_impl(false, hX, hY, hXs, n, m, D, h, tile, sched_width, hMean, hSigma, hAlpha, h_info, dWork, work_bytes, stream);
}

int gp_pipeline_host_mixed(const double* hX, const double* hY, const double* hXs, int64_t n, int64_t m, int D, gp_hyper h, int tile,
                           int sched_width, double* hMean, double* hSigma, double* hAlpha, int* h_info, void* dWork, size_t work_bytes,
                           void* stream) {
    return pipeline_host_impl(true, hX, hY, hXs, n, m, D, h, tile, sched_width, hMean, hSigma, hAlpha, h_info, dWork, work_bytes, stream);
}

int gp_fp64_peak_launch(int mode, int iters, double* d_sink, double* flops, void* stream) {
    if (!d_sink) return GP_ERR_NULL;
    if (iters <= 0) return GP_ERR_SIZE;
    if (mode != 0 && mode != 1) return GP_ERR_MODE;
    const int grid = sm_count() * kPeakCtasPerSm;
    if (mode == 0) {
        peak_dmma_kernel<<<grid, kPeakThreads, 0, (cudaStream_t)stream>>>(d_sink, iters, 1.0);
        if (flops) *flops = (double)grid * (kPeakThreads / 32) * (double)iters * kPeakChains * 512.0;   // 2*8*8*4 per DMMA
    } else {
        peak_dfma_kernel<<<grid, kPeakThreads, 0, (cudaStream_t)stream>>>(d_sink, iters, 1.0);
        if (flops) *flops = (double)grid * kPeakThreads * (double)iters * kPeakChains * 2.0;
    }
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

int gp_contraction_bench_launch(int K, int reps, void* d_buf, size_t buf_bytes, double* flops, size_t* need_bytes, void* stream) {
    constexpr int b = 128;
    if (K < b || K % b != 0 || K > 8192 || reps <= 0) return GP_ERR_SIZE;
    // a synthetic lower-packed matrix with tile edge K: tile column 0 supplies the A and B panels,
    // the tiles (I, J >= 1) supply the C blocks; every item is UPD_L(gr, gc, 0, K/b) without dependencies
    const int nbt = K / b;
    const int M = 1 + (12 / nbt > 1 ? 12 / nbt : 1);
    const int NB = M * nbt, ctas = sm_count();
    const size_t tiles_bytes = (size_t)M * (M + 1) / 2 * K * K * sizeof(double);
    const size_t ver_off = align_up(tiles_bytes, 256) + kHdrBytes;
    const size_t items_off = align_up(ver_off + (size_t)NB * NB * sizeof(int), 256);
    const size_t nitems = (size_t)ctas * reps;
    const size_t total = items_off + nitems * sizeof(Item);
    if (need_bytes) *need_bytes = total;
    if (!d_buf) return need_bytes ? GP_OK : GP_ERR_NULL;
    if (buf_bytes < total) return GP_ERR_WORKSPACE;
    std::vector<Item> cblocks;
    for (int gr = nbt; gr < NB; ++gr)
        for (int gc = nbt; gc < (gr / nbt + 1) * nbt; ++gc) {
            Item it;
            it.op = OP_UPD_L; it.gr = (uint32_t)gr; it.gc = (uint32_t)gc; it.q = (uint32_t)nbt << 16;
            cblocks.push_back(it);
        }
    std::vector<Item> items(nitems);
    for (size_t i = 0; i < nitems; ++i) items[i] = cblocks[i % cblocks.size()];
    char* ws = (char*)d_buf;
    cudaStream_t st = (cudaStream_t)stream;
    if (cudaMemcpy(ws + items_off, items.data(), nitems * sizeof(Item), cudaMemcpyHostToDevice) != cudaSuccess) return GP_ERR_CUDA;
    if (cudaMemsetAsync(ws + align_up(tiles_bytes, 256), 0, items_off - align_up(tiles_bytes, 256), st) != cudaSuccess) return GP_ERR_CUDA;
    ExecParams p;
    memset(&p, 0, sizeof(p));
    p.L = (double*)d_buf;
    p.invD = (double*)d_buf;
    p.verL = (int*)(ws + ver_off);
    p.items = (const Item*)(ws + items_off);
    p.nitems = (int)nitems;
    p.ticket = (unsigned int*)(ws + align_up(tiles_bytes, 256));
    p.stats = (unsigned long long*)(ws + align_up(tiles_bytes, 256) + kStatsOff);
    p.d_info = (int*)(ws + align_up(tiles_bytes, 256) + 128);
    p.t = K;
    p.nbt = nbt;
    p.snbt = nbt;
    p.NB = NB;
    p.Mt = M;
    p.no_deps = 1;
    if (flops) *flops = (double)nitems * 2.0 * b * b * K;
    return launch_exec_any(b, p, 0, ctas, st);
}

}  // extern "C"

// ---- split-operand (Ozaki) contraction on the int8 tensor cores -------------------------
namespace {
// planes [S][rows][k] (int8) viewed through boxes of {chunk bytes of k, box_rows rows, box_planes planes}; the swizzle is as
// wide as the box row (32 bytes: all planes of a k-chunk per box; 128 bytes: one plane per box)
int make_plane_map(CUtensorMap* map, const int8_t* planes, uint64_t rows, uint64_t k, uint32_t box_rows, uint32_t box_planes = oz::kPlanes,
                   uint32_t chunk = oz::kChunk) {
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return GP_ERR_CUDA;
    const cuuint64_t dims[3] = {(cuuint64_t)k, (cuuint64_t)rows, (cuuint64_t)oz::kPlanes};
    const cuuint64_t strides[2] = {(cuuint64_t)k, (cuuint64_t)(rows * k)};
    const cuuint32_t box[3] = {chunk, box_rows, box_planes};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<int8_t*>(planes), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, chunk == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_32B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? GP_OK : GP_ERR_CUDA;
}
}  // namespace

namespace {
// the 2-D view [rows][ld] of an FP64 output array, boxes of {8 columns, 32 rows}: the wide kernel's bulk reductions into C
int make_c_map(CUtensorMap* map, double* C, uint64_t ld, uint64_t rows) {
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return GP_ERR_CUDA;
    const cuuint64_t dims[2] = {(cuuint64_t)ld, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)(ld * sizeof(double))};
    const cuuint32_t box[2] = {(cuuint32_t)oz::kStageCols3, 32};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, C, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? GP_OK : GP_ERR_CUDA;
}

std::atomic<int> g_ozaki_tile_n{0};       // 0 = auto (128 when the shape allows), 64, 128: gp_set_ozaki_tile_n (measurement support)

// launches the emulated contraction described by q (kc0 / kchunks in 32-byte chunks) with the tile shape that fits:
// the 128 x 128 two-pass kernel when the column count and the k range are multiples of 128, else the 128 x 64 one.
// A contraction deeper than oz::kMaxK (the depth an int32 level accumulator can take) runs as several launches over
// consecutive k segments, each subtracting its part from C.
// c_rows: rows of the 2-D view [c_rows][ld] of the output array (dense: the rows of C, ld = ldc; tiled: tiles x t, ld = t)
int launch_ozaki(oz::OzParams q, const int8_t* planesA, uint64_t rowsA, const int8_t* planesB, uint64_t rowsB, uint64_t kdim, int64_t ncols,
                 uint64_t c_rows, cudaStream_t st) {
    const int want = g_ozaki_tile_n.load(std::memory_order_relaxed);
    const bool wide = want != 64 && ncols % oz::kTileN3 == 0 && q.kchunks % oz::kKSteps3 == 0 && q.kc0 % oz::kKSteps3 == 0 && kdim % oz::kChunk3 == 0;
    CUtensorMap mapA, mapB, mapC;
    int rc;
    if (wide) {
        if ((rc = make_plane_map(&mapA, planesA, rowsA, kdim, oz::kTileM, 1, oz::kChunk3)) != GP_OK) return rc;
        if ((rc = make_plane_map(&mapB, planesB, rowsB, kdim, oz::kTileN3, 1, oz::kChunk3)) != GP_OK) return rc;
        if ((rc = make_c_map(&mapC, q.C, (q.tiled == 1 || q.tiled == 2) ? (uint64_t)q.t : (uint64_t)q.ldc, c_rows)) != GP_OK) return rc;
        rc = configure_once(1024u, [] {
            return cudaFuncSetAttribute(oz::ozaki_contract_kernel3<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz::kSmemOz3) == cudaSuccess;
        });
        q.tiles_n = (int)(ncols / oz::kTileN3);
    } else {
        if ((rc = make_plane_map(&mapA, planesA, rowsA, kdim, oz::kTileM)) != GP_OK) return rc;
        if ((rc = make_plane_map(&mapB, planesB, rowsB, kdim, oz::kTileN)) != GP_OK) return rc;
        rc = configure_once(512u, [] {
            return cudaFuncSetAttribute(oz::ozaki_contract_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, oz::kSmemOz) == cudaSuccess;
        });
        q.tiles_n = (int)(ncols / oz::kTileN);
    }
    if (rc != GP_OK) return rc;
    const int grid = (int)std::min<int64_t>((int64_t)q.tiles_m * q.tiles_n, sm_count());
    const int seg_chunks = oz::kMaxK / oz::kChunk;                      // a multiple of 4
    const int first = q.kc0, total = q.kchunks;
    for (int done = 0; done < total; done += seg_chunks) {
        q.kc0 = first + done;
        q.kchunks = std::min(seg_chunks, total - done);
        if (wide)
            oz::ozaki_contract_kernel3<0><<<grid, oz::kThreads3, oz::kSmemOz3, st>>>(q, mapA, mapB, mapC);
        else
            oz::ozaki_contract_kernel<<<grid, oz::kThreadsOz, oz::kSmemOz, st>>>(q, mapA, mapB);
    }
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}
}  // namespace

extern "C" int gp_set_ozaki_tile_n(int n) {
    if (n != 0 && n != 64 && n != 128) return GP_ERR_SIZE;
    g_ozaki_tile_n.store(n, std::memory_order_relaxed);
    return GP_OK;
}

// ---- measurement support for the emulated contraction (bench.py --ozaki-probe; profiles/r02_ozaki_bounds.md) ----
extern "C" int gp_int8_mma_peak_launch(int n_cols, int iters, long long* d_cycles, double* ops, void* stream) {
    if (iters <= 0 || (n_cols != 64 && n_cols != 128 && n_cols != 256)) return GP_ERR_SIZE;
    cudaStream_t st = (cudaStream_t)stream;
    const int grid = sm_count();
    cudaError_t e;
    if (n_cols == 64) {
        e = cudaFuncSetAttribute(oz::int8_mma_peak_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz::kSmemInt8Peak);
        if (e == cudaSuccess) oz::int8_mma_peak_kernel<64><<<grid, 128, oz::kSmemInt8Peak, st>>>(iters, d_cycles);
    } else if (n_cols == 128) {
        e = cudaFuncSetAttribute(oz::int8_mma_peak_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz::kSmemInt8Peak);
        if (e == cudaSuccess) oz::int8_mma_peak_kernel<128><<<grid, 128, oz::kSmemInt8Peak, st>>>(iters, d_cycles);
    } else {
        e = cudaFuncSetAttribute(oz::int8_mma_peak_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz::kSmemInt8Peak);
        if (e == cudaSuccess) oz::int8_mma_peak_kernel<256><<<grid, 128, oz::kSmemInt8Peak, st>>>(iters, d_cycles);
    }
    if (e != cudaSuccess) return GP_ERR_CUDA;
    if (ops) *ops = 2.0 * oz::kTileM * (double)n_cols * oz::kChunk * 16.0 * (double)iters * (double)grid;
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

extern "C" int gp_ozaki_probe_launch(int probe, const int8_t* dAplanes, int64_t ma, const int8_t* dBplanes, int64_t nb, int64_t k, double* dC,
                                     int64_t ldc, void* stream) {
    if (!dAplanes || !dBplanes || !dC) return GP_ERR_NULL;
    if (probe != 0 && probe != 1 && probe != 2 && probe != 4) return GP_ERR_MODE;
    if (ma <= 0 || nb <= 0 || k <= 0 || ma % oz::kTileM != 0 || nb % oz::kTileN3 != 0 || k % oz::kChunk3 != 0 || k > oz::kMaxK || ldc < nb || ldc % 2 != 0)
        return GP_ERR_SIZE;
    oz::OzParams q;
    memset(&q, 0, sizeof(q));
    q.C = dC;
    q.ldc = ldc;
    q.tiles_m = (int)(ma / oz::kTileM);
    q.tiles_n = (int)(nb / oz::kTileN3);
    q.kchunks = (int)(k / oz::kChunk);
    q.w_last = std::ldexp(1.0, -oz::kDigitBits * (oz::kPlanes + 1));
    CUtensorMap mapA, mapB, mapC;
    int rc;
    if ((rc = make_plane_map(&mapA, dAplanes, (uint64_t)ma, (uint64_t)k, oz::kTileM, 1, oz::kChunk3)) != GP_OK) return rc;
    if ((rc = make_plane_map(&mapB, dBplanes, (uint64_t)nb, (uint64_t)k, oz::kTileN3, 1, oz::kChunk3)) != GP_OK) return rc;
    if ((rc = make_c_map(&mapC, dC, (uint64_t)ldc, (uint64_t)ma)) != GP_OK) return rc;
    const int grid = (int)std::min<int64_t>((int64_t)q.tiles_m * q.tiles_n, sm_count());
    cudaStream_t st = (cudaStream_t)stream;
#define GPB_PROBE_CASE(P)                                                                                                              \
    case P:                                                                                                                            \
        if (cudaFuncSetAttribute(oz::ozaki_contract_kernel3<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz::kSmemOz3) != cudaSuccess) \
            return GP_ERR_CUDA;                                                                                                        \
        oz::ozaki_contract_kernel3<P><<<grid, oz::kThreads3, oz::kSmemOz3, st>>>(q, mapA, mapB, mapC);                                 \
        break;
    switch (probe) {
        GPB_PROBE_CASE(0)
        GPB_PROBE_CASE(1)
        GPB_PROBE_CASE(2)
        GPB_PROBE_CASE(4)
    }
#undef GPB_PROBE_CASE
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

extern "C" int gp_ozaki_probe_stamps(long long* h_stamps8) {
    if (!h_stamps8) return GP_ERR_NULL;
    return cudaMemcpyFromSymbol(h_stamps8, oz::g_oz3_probe, 8 * sizeof(long long)) == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

extern "C" int gp_ozaki_planes(void) { return oz::kPlanes; }
extern "C" int gp_ozaki_digit_bits(void) { return oz::kDigitBits; }

extern "C" int gp_ozaki_plane_bytes(int64_t rows, int64_t k, size_t* bytes) {
    if (!bytes) return GP_ERR_NULL;
    if (rows <= 0 || k <= 0 || k % oz::kChunk != 0) return GP_ERR_SIZE;
    *bytes = (size_t)oz::kPlanes * (size_t)rows * (size_t)k;
    return GP_OK;
}

extern "C" int gp_ozaki_slice(const double* dX, int64_t rows, int64_t k, int64_t ld, double scale, int8_t* dPlanes, int* d_overflow,
                              void* stream) {
    if (!dX || !dPlanes || !d_overflow) return GP_ERR_NULL;
    if (rows <= 0 || k <= 0 || k % oz::kChunk != 0 || ld < k) return GP_ERR_SIZE;
    if (!(scale > 0.0) || !std::isfinite(scale)) return GP_ERR_HYPER;
    cudaStream_t st = (cudaStream_t)stream;
    if (cudaMemsetAsync(d_overflow, 0, sizeof(int), st) != cudaSuccess) return GP_ERR_CUDA;
    const int64_t total = rows * (k / 4);
    const unsigned grid = (unsigned)std::min<int64_t>((total + 255) / 256, (int64_t)sm_count() * 16);
    oz::slice_kernel<<<grid, 256, 0, st>>>(dX, rows, k, ld, 1.0 / scale, dPlanes, d_overflow);
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

extern "C" int gp_ozaki_contract(const int8_t* dAplanes, int64_t ma, const int8_t* dBplanes, int64_t nb, int64_t k, double scaleA,
                                 double scaleB, double* dC, int64_t ldc, void* stream) {
    if (!dAplanes || !dBplanes || !dC) return GP_ERR_NULL;
    if (ma <= 0 || nb <= 0 || k <= 0 || ma % oz::kTileM != 0 || nb % oz::kTileN != 0 || k % oz::kChunk != 0 || k > (1 << 22) || ldc < nb || ldc % 2 != 0)
        return GP_ERR_SIZE;
    if (!(scaleA > 0.0) || !(scaleB > 0.0) || !std::isfinite(scaleA * scaleB)) return GP_ERR_HYPER;
    oz::OzParams p;
    memset(&p, 0, sizeof(p));
    p.C = dC;
    p.ldc = ldc;
    p.tiles_m = (int)(ma / oz::kTileM);
    p.kchunks = (int)(k / oz::kChunk);
    p.w_last = scaleA * scaleB * std::ldexp(1.0, -oz::kDigitBits * (oz::kPlanes + 1));
    return launch_ozaki(p, dAplanes, (uint64_t)ma, dBplanes, (uint64_t)nb, (uint64_t)k, nb, (uint64_t)ma, (cudaStream_t)stream);
}

// ---- gp_cholesky_tiled_mixed: FP64 panels + emulated trailing updates ------------------------
namespace {
struct MixedWs { size_t ticket, verL, invD, scale, planes, total; };
MixedWs mixed_ws(int64_t n) {
    // panels run with 128-blocks or, when few block rows are left below the diagonal tile, with 64-blocks (mixed_panel_block):
    // version counters for the finer grid, inverted diagonal blocks for the coarser one (n x 128 doubles covers n x 64)
    const CholWs c = chol_ws(n, 64), c128 = chol_ws(n, 128);
    MixedWs w;
    w.ticket = c.ticket;
    w.verL = c.verL;
    w.invD = c.invD;
    w.scale = align_up(c.invD + (c128.total - c128.invD), 256);
    w.planes = align_up(w.scale + 256, 1024);
    w.total = w.planes + (size_t)oz::kPlanes * (size_t)n * (size_t)n;
    return w;
}
int mixed_ok(int64_t n, int tile) {
    if (n <= 0 || n > (int64_t)1 << 22) return GP_ERR_SIZE;
    const int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    if (tile % 128 != 0) return GP_ERR_TILE;
    if (n / tile > 60) return GP_ERR_SIZE;                 // one ticket counter per panel launch in the 256-byte header
    if (n > 65536 + 128) return GP_ERR_SIZE;               // 8.6 GB of digit planes per 32768^2 entries: the workspace is the limit
    return GP_OK;
}
}  // namespace

extern "C" int gp_mixed_workspace_bytes(int64_t n, int tile, size_t* bytes) {
    if (!bytes) return GP_ERR_NULL;
    const int rc = mixed_ok(n, tile);
    if (rc != GP_OK) return rc;
    *bytes = mixed_ws(n).total;
    return GP_OK;
}

// The four steps of the mixed factorisation.  gp_cholesky_tiled_mixed runs them in a loop; a multi-GPU driver
// (paper_2602_19683_b200/multi_gpu.py, block-cyclic tile columns) interleaves them with panel broadcasts.
namespace {
struct MixedCtx {
    MixedWs w;
    char* ws;
    int M, nbt, NB;
    cudaStream_t st;
};
int mixed_ctx(int64_t n, int tile, void* dWork, size_t work_bytes, void* stream, MixedCtx* c) {
    if (!dWork) return GP_ERR_NULL;
    const int rc = mixed_ok(n, tile);
    if (rc != GP_OK) return rc;
    c->w = mixed_ws(n);
    if (work_bytes < c->w.total) return GP_ERR_WORKSPACE;
    c->ws = (char*)dWork;
    c->M = (int)(n / tile);
    c->nbt = tile / 128;
    c->NB = (int)(n / 128);
    c->st = (cudaStream_t)stream;
    return GP_OK;
}
// Block edge of the FP64 panel step of column J.  A panel is the chain of the diagonal tile and, below it, one chain per block
// row (the solves of a block row depend on each other, a chain keeps one SM busy): with r block rows on W workers the step takes
// about ceil(r / W) chain times.  Measured at n = 32768, tile 1024 (ms, by 128-block rows left below the diagonal tile):
//   128-blocks: <= 144 rows 0.90, 152-248 rows 1.45-1.57;   64-blocks: <= 72 rows 0.60, 80-144 rows 0.94, 152-216 rows 1.23-1.33,
//   224-248 rows 1.65-1.73 -- i.e. T128 = 1 + 0.67 (waves128 - 1), T64 = 0.67 + 0.38 (waves64 - 1) in units of the 128-block chain.
// The cheaper one is taken (c3: J = 4-12 and J >= 22 with 64-blocks: panels 37.9 -> 32 ms).  Emitting the block rows RIGHT-looking
// (every solved block updates the blocks to its right at once, so that a row is spread over several SMs) was built and measured
// too: 37.5 ms with 128-blocks against 36.6 ms left-looking -- the depth-one items cost more than the waves they remove.
int mixed_panel_block(int M, int tile, int J) {
    const int cap = g_block_edge.load(std::memory_order_relaxed);      // gp_set_block_edge: measurement override
    if (cap == 64 || cap == 128) return cap;
    const int rows128 = (M - J - 1) * (tile / 128), W = sm_count();
    const int w128 = rows128 > 0 ? (rows128 + W - 1) / W : 1, w64 = rows128 > 0 ? (2 * rows128 + W - 1) / W : 1;
    const double t128 = 1.0 + 0.67 * (w128 - 1), t64 = 0.67 + 0.38 * (w64 - 1);
    return t64 < t128 ? 64 : 128;
}

int get_panel_schedule(int M, int nbt, int J, int b, CachedSchedule* out) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return GP_ERR_CUDA;
    std::lock_guard<std::mutex> lk(g_mu);
    auto key = std::make_tuple(dev, 16 + J, M, 0, nbt, b);
    auto it = g_cache.find(key);
    if (it != g_cache.end()) { *out = it->second; return GP_OK; }
    std::vector<SchedItem> items;
    build_panel_schedule(M, nbt, J, sm_count(), items, b);
    CachedSchedule cs;
    cs.nitems = (int)items.size();
    if (cudaMalloc(&cs.d_items, items.size() * sizeof(Item) + 16) != cudaSuccess) return GP_ERR_CUDA;
    if (cudaMemcpy(cs.d_items, items.data(), items.size() * sizeof(Item), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaFree(cs.d_items);
        return GP_ERR_CUDA;
    }
    g_cache[key] = cs;
    *out = cs;
    return GP_OK;
}
}  // namespace

extern "C" int gp_mixed_begin(const double* dKL, int64_t n, int tile, int* d_info, void* dWork, size_t work_bytes, void* stream) {
    if (!dKL || !d_info) return GP_ERR_NULL;
    MixedCtx c;
    const int rc = mixed_ctx(n, tile, dWork, work_bytes, stream, &c);
    if (rc != GP_OK) return rc;
    if (cudaMemsetAsync(c.ws, 0, c.w.invD, c.st) != cudaSuccess) return GP_ERR_CUDA;          // tickets, statistics, version counters
    if (cudaMemsetAsync(d_info, 0, sizeof(int), c.st) != cudaSuccess) return GP_ERR_CUDA;
    oz::factor_scale_kernel<<<1, 1024, 0, c.st>>>(dKL, n, tile, (double*)(c.ws + c.w.scale));
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

extern "C" int gp_mixed_update_column(double* dKL, int64_t n, int tile, int J, int k_tile0, int k_tile1, void* dWork, size_t work_bytes,
                                      void* stream) {
    if (!dKL) return GP_ERR_NULL;
    MixedCtx c;
    int rc = mixed_ctx(n, tile, dWork, work_bytes, stream, &c);
    if (rc != GP_OK) return rc;
    if (J < 0 || J >= c.M || k_tile0 < 0 || k_tile1 > J || k_tile0 > k_tile1) return GP_ERR_SIZE;
    if (k_tile0 == k_tile1) return GP_OK;
    int8_t* planes = (int8_t*)(c.ws + c.w.planes);
    oz::OzParams q;
    memset(&q, 0, sizeof(q));
    q.C = dKL;
    q.tiles_m = (c.M - J) * (tile / oz::kTileM);
    q.kchunks = (int)((int64_t)(k_tile1 - k_tile0) * tile / oz::kChunk);
    q.kc0 = (int)((int64_t)k_tile0 * tile / oz::kChunk);
    q.w_last = std::ldexp(1.0, -oz::kDigitBits * (oz::kPlanes + 1));
    q.scale = (const double*)(c.ws + c.w.scale) + 1;          // scale^2
    q.tiled = 1;
    q.t = tile;
    q.J = J;
    q.row0a = q.row0b = J * tile;
    // both operands come from the dense digit planes [S][n][n] of the whole matrix
    return launch_ozaki(q, planes, (uint64_t)n, planes, (uint64_t)n, (uint64_t)n, tile, (uint64_t)c.M * (c.M + 1) / 2 * (uint64_t)tile, c.st);
}

namespace {
int mixed_panel_impl(double* dKL, int64_t n, int tile, int J, int sched_width, int* d_info, void* dWork, size_t work_bytes, double* const* peers,
                     int npeers, void* stream) {
    if (!dKL || !d_info) return GP_ERR_NULL;
    if (npeers < 0 || npeers > kMaxPeers || (npeers > 0 && !peers)) return GP_ERR_SIZE;
    for (int k = 0; k < npeers; ++k)
        if (!peers[k] || peers[k] == dKL) return GP_ERR_NULL;
    MixedCtx c;
    int rc = mixed_ctx(n, tile, dWork, work_bytes, stream, &c);
    if (rc != GP_OK) return rc;
    if (J < 0 || J >= c.M) return GP_ERR_SIZE;
    const int b = mixed_panel_block(c.M, tile, J);
    const int nbt = tile / b, NB = (int)(n / b);
    CachedSchedule cs;
    if ((rc = get_panel_schedule(c.M, nbt, J, b, &cs)) != GP_OK) return rc;
    ExecParams p;
    memset(&p, 0, sizeof(p));
    p.L = dKL;
    p.invD = (double*)(c.ws + c.w.invD);
    p.verL = (int*)(c.ws + c.w.verL);
    p.stats = (unsigned long long*)(c.ws + kStatsOff);
    p.d_info = d_info;
    p.t = tile;
    p.nbt = nbt;
    p.snbt = nbt;
    p.NB = NB;
    p.Mt = c.M;
    p.items = cs.d_items;
    p.nitems = cs.nitems;
    p.ticket = (unsigned int*)(c.ws + c.w.ticket) + J;
    p.npeers = npeers;
    for (int k = 0; k < npeers; ++k) p.peerL[k] = peers[k];
    // the J trailing updates of this column were applied by the emulated contraction, outside the executor's counters
    if (cudaMemsetAsync(p.ticket, 0, sizeof(unsigned int), c.st) != cudaSuccess) return GP_ERR_CUDA;
    oz::set_column_versions_kernel<<<(NB * nbt + 255) / 256, 256, 0, c.st>>>(p.verL, NB, nbt, J, kConsumerWarps);
    return launch_exec_any(b, p, 0, workers_for(sched_width), c.st);
}
}  // namespace

extern "C" int gp_mixed_panel(double* dKL, int64_t n, int tile, int J, int sched_width, int* d_info, void* dWork, size_t work_bytes,
                              void* stream) {
    return mixed_panel_impl(dKL, n, tile, J, sched_width, d_info, dWork, work_bytes, nullptr, 0, stream);
}

extern "C" int gp_mixed_panel_bcast(double* dKL, int64_t n, int tile, int J, int sched_width, int* d_info, void* dWork, size_t work_bytes,
                                    double* const* peers, int npeers, void* stream) {
    return mixed_panel_impl(dKL, n, tile, J, sched_width, d_info, dWork, work_bytes, peers, npeers, stream);
}

extern "C" int gp_mixed_slice_column(const double* dKL, int64_t n, int tile, int J, void* dWork, size_t work_bytes, void* stream) {
    if (!dKL) return GP_ERR_NULL;
    MixedCtx c;
    const int rc = mixed_ctx(n, tile, dWork, work_bytes, stream, &c);
    if (rc != GP_OK) return rc;
    if (J < 0 || J >= c.M) return GP_ERR_SIZE;
    if (J + 1 == c.M) return GP_OK;                          // the last column has no tile below its diagonal tile
    const int64_t total = (n - (int64_t)(J + 1) * tile) * (tile / 4);
    const unsigned grid = (unsigned)std::min<int64_t>((total + 255) / 256, (int64_t)sm_count() * 16);
    oz::slice_tile_column_kernel<<<grid, 256, 0, c.st>>>(dKL, n, tile, J, (const double*)(c.ws + c.w.scale), (int8_t*)(c.ws + c.w.planes));
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}

extern "C" int gp_cholesky_tiled_mixed(double* dKL, int64_t n, int tile, int sched_width, int* d_info, void* dWork, size_t work_bytes,
                                       void* stream) {
    int rc = gp_mixed_begin(dKL, n, tile, d_info, dWork, work_bytes, stream);
    if (rc != GP_OK) return rc;
    const int M = (int)(n / tile);
    for (int J = 0; J < M; ++J) {
        // left-looking: tile column J -= L(J:, 0:J) L(J, 0:J)^T in one emulated contraction of depth J * tile, then its
        // FP64 panel step, then its digit planes
        if ((rc = gp_mixed_update_column(dKL, n, tile, J, 0, J, dWork, work_bytes, stream)) != GP_OK) return rc;
        if ((rc = gp_mixed_panel(dKL, n, tile, J, sched_width, d_info, dWork, work_bytes, stream)) != GP_OK) return rc;
        if ((rc = gp_mixed_slice_column(dKL, n, tile, J, dWork, work_bytes, stream)) != GP_OK) return rc;
    }
    return GP_OK;
}

// ---- the prediction on the same emulated contraction (continued) ---------------------------------
namespace {
struct MixedPredWs { size_t ticket, verV, invD, items, scale, Vt, planesL, planesV, total; };
MixedPredWs mixed_pred_ws(int64_t n, int64_t m) {
    // the FP64 solves run with 128-blocks or, for few test points, with 64-blocks (mixed_predict_block): counters and work
    // items for the finer grid, inverted diagonal blocks for the coarser one
    const size_t NB = (size_t)(n / 64), NBm = (size_t)(m / 64);
    MixedPredWs w;
    w.ticket = 0;
    w.verV = kHdrBytes;
    w.invD = align_up(w.verV + NBm * NB * sizeof(int), 256);
    w.items = align_up(w.invD + (size_t)n * 128 * sizeof(double), 256);
    w.scale = align_up(w.items + NBm * sizeof(Item), 256);
    w.Vt = align_up(w.scale + 256, 1024);
    w.planesL = align_up(w.Vt + (size_t)m * (size_t)n * sizeof(double), 1024);
    w.planesV = align_up(w.planesL + (size_t)oz::kPlanes * (size_t)n * (size_t)n, 1024);
    w.total = w.planesV + (size_t)oz::kPlanes * (size_t)m * (size_t)n;
    return w;
}
}  // namespace

extern "C" int gp_mixed_predict_workspace_bytes(int64_t n, int64_t m, int tile, size_t* bytes) {
    if (!bytes) return GP_ERR_NULL;
    int rc = mixed_ok(n, tile);
    if (rc != GP_OK) return rc;
    if (m <= 0 || m > 65536) return GP_ERR_SIZE;
    if ((rc = tile_ok(m, tile)) != GP_OK) return rc;
    *bytes = mixed_pred_ws(n, m).total;
    return GP_OK;
}

namespace {
// dSigma: full covariance (V^T solve + W on the emulated contraction); dVar (dSigma null): variances only, the V^T solve alone
int predict_mixed_impl(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m, gp_hyper h, int tile, int sched_width,
                       double* dSigma, double* dVar, void* dWork, size_t work_bytes, void* stream) {
    if (!dL || !dX || !dXs || (!dSigma && !dVar) || !dWork) return GP_ERR_NULL;
    int rc = mixed_ok(n, tile);
    if (rc != GP_OK) return rc;
    if (m <= 0 || m > 65536 || D <= 0) return GP_ERR_SIZE;
    if ((rc = tile_ok(m, tile)) != GP_OK) return rc;
    if (!hyper_ok(h)) return GP_ERR_HYPER;
    const MixedPredWs w = mixed_pred_ws(n, m);
    if (work_bytes < w.total) return GP_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    // one chain per block row of V^T and tile column: m / b independent chains of tile / b dependent steps.  With few test
    // points (c3: 32 rows of 128-blocks on 148 SMs, 0.75 ms per tile column) 64-blocks give twice the chains and cheaper steps.
    const int b = (m / 128 <= 104) ? 64 : 128;
    const int M = (int)(n / tile), nbt = tile / b, NB = (int)(n / b), NBm = (int)(m / b);
    char* ws = (char*)dWork;
    double* Vt = (double*)(ws + w.Vt);
    double* invD = (double*)(ws + w.invD);
    double* scale = (double*)(ws + w.scale);                          // [sL, sV, sL sV, sV sV], then the bits of max |L|
    unsigned long long* maxbits = (unsigned long long*)(scale + 8);
    int8_t* planesL = (int8_t*)(ws + w.planesL);
    int8_t* planesV = (int8_t*)(ws + w.planesV);
    Item* items = (Item*)(ws + w.items);
    const HyperDev hd = to_dev(h);
    if (cudaMemsetAsync(ws, 0, w.invD, st) != cudaSuccess) return GP_ERR_CUDA;
    if (cudaMemsetAsync(scale, 0, 256, st) != cudaSuccess) return GP_ERR_CUDA;
    // a9: K_{X^,X} straight into V^T, the prior K_{X^,X^} straight into Sigma (as gp_predict_full_cov)
    if ((rc = launch_assemble(dXs, m, dX, n, D, hd, tile, 0, Vt, st)) != GP_OK) return rc;
    if (dSigma) {
        const int sb = (int)((m + kAsmBlk - 1) / kAsmBlk);
        const size_t smem = 2 * (size_t)kAsmMaxD * kAsmBlk * sizeof(double);
        assemble_tiles_kernel<<<(unsigned)(sb * sb), 256, smem, st>>>(dXs, dXs, D, hd, (int)m, 1, 0, dSigma);
        if (cudaGetLastError() != cudaSuccess) return GP_ERR_CUDA;
    }
    if ((rc = launch_trtri_any(b, dL, tile, NB, invD, st)) != GP_OK) return rc;
    // fixed-point scales: |L_ij| <= max |L| (read from the factor), |V_ia| <= sqrt(k(x^_a, x^_a)) = sqrt(v)
    const double sv = std::ldexp(1.0, (int)std::ceil(std::log2(std::sqrt(h.vertical) / 0.98)) + 1);   // |V_ia| <= sqrt(v) <= 0.49 sv
    const int64_t lcount = (int64_t)M * (M + 1) / 2 * tile * tile;
    oz::absmax_lower_tiles_kernel<<<sm_count() * 8, 256, 0, st>>>(dL, lcount, maxbits);
    oz::finish_scales_kernel<<<1, 1, 0, st>>>(maxbits, sv, scale);
    for (int J = 0; J + 1 < M; ++J) {                                 // digit planes of the factor (tiles below the diagonal tiles)
        const int64_t total = (n - (int64_t)(J + 1) * tile) * (tile / 4);
        const unsigned grid = (unsigned)std::min<int64_t>((total + 255) / 256, (int64_t)sm_count() * 16);
        oz::slice_tile_column_kernel<<<grid, 256, 0, st>>>(dL, n, tile, J, scale, planesL);
    }
    ExecParams p;
    memset(&p, 0, sizeof(p));
    p.L = const_cast<double*>(dL);
    p.Vt = Vt;
    p.invD = invD;
    p.verV = (int*)(ws + w.verV);
    p.verS = p.verV;
    p.items = items;
    p.nitems = NBm;
    p.stats = (unsigned long long*)(ws + kStatsOff);
    p.t = tile;
    p.nbt = nbt;
    p.snbt = nbt;
    p.NB = NB;
    p.NBm = NBm;
    p.Mt = M;
    p.m = m;
    p.L_final = 1;
    ExecMaps mp;
    if ((rc = make_exec_maps(&mp, p, b, m)) != GP_OK) return rc;
    for (int P = 0; P < M; ++P) {
        if (P > 0) {
            // left-looking: V^T(:, P) -= V^T(:, 0:P) L(P, 0:P)^T, one emulated contraction of depth P * tile
            oz::OzParams q;
            memset(&q, 0, sizeof(q));
            q.C = Vt;
            q.tiles_m = (int)(m / oz::kTileM);
            q.kchunks = (int)((int64_t)P * tile / oz::kChunk);
            q.w_last = std::ldexp(1.0, -oz::kDigitBits * (oz::kPlanes + 1));
            q.scale = scale + 2;
            q.tiled = 2;
            q.t = tile;
            q.J = P;
            q.Mt = M;
            q.row0a = 0;
            q.row0b = P * tile;
            if ((rc = launch_ozaki(q, planesV, (uint64_t)m, planesL, (uint64_t)n, (uint64_t)n, tile, (uint64_t)m * (uint64_t)M, st)) != GP_OK) return rc;
        }
        // the FP64 half of step P: V^T(:, P) <- V^T(:, P) L(P,P)^-T, one ROW_V chain per block row, on the executor
        oz::set_general_column_versions_kernel<<<(NBm * nbt + 255) / 256, 256, 0, st>>>(p.verV, NBm, NB, nbt, P, kConsumerWarps);
        cov_row_items_kernel<<<(NBm + 255) / 256, 256, 0, st>>>((uint4*)items, NBm, 0, 1, 0, (unsigned)OP_ROW_V);
        row_items_set_column_kernel<<<(NBm + 255) / 256, 256, 0, st>>>((uint4*)items, NBm, (unsigned)(P * nbt));
        p.ticket = (unsigned int*)(ws + w.ticket) + P;
        rc = b == 64 ? launch_exec<64>(p, mp, workers_for(sched_width), st) : launch_exec<128>(p, mp, workers_for(sched_width), st);
        if (rc != GP_OK) return rc;
        if (dSigma || P + 1 < M) {              // the last column's planes only feed W
            const int64_t total = m * (tile / 4);
            const unsigned grid = (unsigned)std::min<int64_t>((total + 255) / 256, (int64_t)sm_count() * 16);
            oz::slice_general_column_kernel<<<grid, 256, 0, st>>>(Vt, m, n, tile, P, scale + 1, planesV);
        }
    }
    if (!dSigma) {
        // var_a = k(x^_a, x^_a) - sum_i V_ia^2, as gp_predict_variance
        posterior_var_kernel<<<(unsigned)((m + 7) / 8), 256, 0, st>>>(Vt, m, n, tile, hd.vertical, dVar);
        return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
    }
    {   // a12: Sigma -= V^T (V^T)^T over the lower triangle, one emulated contraction of depth n; then the mirror
        oz::OzParams q;
        memset(&q, 0, sizeof(q));
        q.C = dSigma;
        q.ldc = m;
        q.tiles_m = (int)(m / oz::kTileM);
        q.kchunks = (int)(n / oz::kChunk);
        q.w_last = std::ldexp(1.0, -oz::kDigitBits * (oz::kPlanes + 1));
        q.scale = scale + 3;
        q.tiled = 3;
        if ((rc = launch_ozaki(q, planesV, (uint64_t)m, planesV, (uint64_t)m, (uint64_t)n, m, (uint64_t)m, st)) != GP_OK) return rc;
    }
    dim3 mg((unsigned)(m / 32), (unsigned)(m / 32));
    mirror_lower_kernel<<<mg, dim3(32, 8), 0, st>>>(dSigma, m);
    return cudaGetLastError() == cudaSuccess ? GP_OK : GP_ERR_CUDA;
}
}  // namespace

extern "C" int gp_predict_full_cov_mixed(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m, gp_hyper h,
                                         int tile, int sched_width, double* dSigma, void* dWork, size_t work_bytes, void* stream) {
    if (!dSigma) return GP_ERR_NULL;
    return predict_mixed_impl(dL, dX, n, D, dXs, m, h, tile, sched_width, dSigma, nullptr, dWork, work_bytes, stream);
}

extern "C" int gp_predict_variance_mixed(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m, gp_hyper h,
                                         int tile, int sched_width, double* dVar, void* dWork, size_t work_bytes, void* stream) {
    if (!dVar) return GP_ERR_NULL;
    return predict_mixed_impl(dL, dX, n, D, dXs, m, h, tile, sched_width, nullptr, dVar, dWork, work_bytes, stream);
}

extern "C" int gp_panel_schedule_selfcheck(int64_t n, int tile, int J) {
    const int rc = mixed_ok(n, tile);
    if (rc != GP_OK) return rc;
    const int M = (int)(n / tile), nbt = tile / 128;
    if (J < 0 || J >= M) return GP_ERR_SIZE;
    std::vector<SchedItem> items;
    build_panel_schedule(M, nbt, J, 148, items, 128);
    return validate_panel_schedule(items, M, nbt, J) ? (int)items.size() : GP_ERR_SIZE;
}

extern "C" int gp_exec_stats(const void* dWork, uint64_t* h_stats, int max_workers, void* stream) {
    if (!dWork || !h_stats) return GP_ERR_NULL;
    if (max_workers <= 0) return GP_ERR_SIZE;
    const int w = max_workers < kMaxWorkers ? max_workers : kMaxWorkers;
    cudaStream_t st = (cudaStream_t)stream;
    if (cudaMemcpyAsync(h_stats, (const char*)dWork + kStatsOff, (size_t)w * kStatsBytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return GP_ERR_CUDA;
    return cudaStreamSynchronize(st) == cudaSuccess ? w : GP_ERR_CUDA;
}

static int schedule_selfcheck(int64_t n, int64_t m, int tile, int workers, bool with_sigma, double* stats5) {
    if (n <= 0 || m < 0) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    if (m > 0 && (rc = tile_ok(m, tile)) != GP_OK) return rc;
    if (workers <= 0) workers = 148;
    const int b = pick_block(tile, n), NB = (int)(n / b), NBm = (int)(m / b), nbt = pick_sched_blocks(NB, NBm);
    const int M = NB / nbt, Mm = NBm / nbt;
    std::vector<SchedItem> items;
    SchedStats st;
    if (m == 0) build_cholesky_schedule(M, nbt, workers, items, b, &st, true);
    else build_predict_schedule(M, Mm, nbt, workers, items, b, &st, true, with_sigma);
    if (stats5) {
        stats5[0] = (double)items.size();
        stats5[1] = (double)st.edges;
        stats5[2] = st.makespan_us;
        stats5[3] = st.work_us;
        stats5[4] = st.critical_path_us;
    }
    const char* why = nullptr;
    return validate_schedule(items, M, Mm, nbt, m > 0, &why, with_sigma) ? GP_OK : GP_ERR_SIZE;
}

extern "C" int gp_schedule_fingerprint(int64_t n, int64_t m, int tile, int workers, int with_sigma, uint64_t* fingerprint) {
    if (!fingerprint) return GP_ERR_NULL;
    if (n <= 0 || m < 0) return GP_ERR_SIZE;
    int rc = tile_ok(n, tile);
    if (rc != GP_OK) return rc;
    if (m > 0 && (rc = tile_ok(m, tile)) != GP_OK) return rc;
    if (workers <= 0) workers = 148;
    const int b = pick_block(tile, n), NB = (int)(n / b), NBm = (int)(m / b), g = pick_sched_blocks(NB, NBm);
    std::vector<SchedItem> items;
    if (m == 0) build_cholesky_schedule(NB / g, g, workers, items, b);
    else build_predict_schedule(NB / g, NBm / g, g, workers, items, b, nullptr, true, with_sigma != 0);
    *fingerprint = schedule_fingerprint(items);
    return GP_OK;
}

extern "C" int gp_schedule_selfcheck(int64_t n, int64_t m, int tile, int workers, double* stats5) {
    return schedule_selfcheck(n, m, tile, workers, true, stats5);
}

extern "C" int gp_schedule_selfcheck_variance(int64_t n, int64_t m, int tile, int workers, double* stats5) {
    if (m <= 0) return GP_ERR_SIZE;
    return schedule_selfcheck(n, m, tile, workers, false, stats5);
}
