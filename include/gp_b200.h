/*
 * gp_b200.h -- C ABI of the B200-native (sm_100a, FP64) GP prediction pipeline of
 * arxiv/paper_2602_19683 "GPU-Resident Gaussian Process Regression Leveraging Asynchronous
 * Tasks with HPX".  Citations are PAPER.md:<line> (the text in /root/reference) and the
 * readings A1..A12 listed in DESIGN.md.
 *
 * Conventions for every entry point
 *   - All `d*` pointers are DEVICE pointers to FP64 (or int where stated), 16-byte aligned,
 *     owned by the caller.  The library never frees or keeps caller memory.  Its only state is
 *     a per-process cache of device-resident task schedules (16 bytes per work item: 2.4 MB for
 *     the n = 32768 / tile 1024 factorisation, 9.4 MB for n = 65536 / tile 2048), keyed by
 *     (device, kind, n/tile, m/tile, tile/block, block); it never evicts, and
 *     gp_release_cached_schedules() drops it.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Every
 *     call is stream-ordered and does not synchronise the host, with ONE exception: the first
 *     gp_cholesky_tiled / gp_predict_full_cov / gp_predict_variance call for a shape that is not in
 *     the schedule cache builds the schedule on the host (0.2 s at n = 32768 / tile 1024, 1.3 s at
 *     n = 65536 / tile 2048), allocates device memory for it and uploads it with a synchronous
 *     copy.  Call gp_prepare() first to take that cost up front; after it (or after the first call)
 *     those entry points only enqueue work and are safe to capture into a CUDA graph.
 *   - Matrices are row-major, 0-based.  n = training points, m = test points
 *     (n-hat in the paper), D = regressors per point, tile = tile edge t with
 *     M = n/tile tiles per dimension.
 *   - Tile sizes: tile > 0, tile % 32 == 0, n % tile == 0 and (where m is tiled) m % tile == 0;
 *     anything else is GP_ERR_TILE (reading A7: the paper has no remainder case).
 *   - Return value: GP_OK (0) or a negative GP_ERR_* reported synchronously before any work
 *     is enqueued.  Numerical failure is reported through *d_info (see gp_cholesky_tiled).
 *
 * Tile layouts
 *   GP_SYM_LOWER  lower-packed: only tiles (I,J) with J <= I are stored,
 *                 tile (I,J) starts at ((I*(I+1)/2 + J) * tile*tile) doubles; element (r,c) of
 *                 a tile is at r*tile + c.  Diagonal tiles are stored whole; after the
 *                 factorisation their strict upper triangle is unspecified (reading A8).
 *   GP_GENERAL    (na/tile) x (nb/tile) tiles, tile (a,b) at ((a*(nb/tile) + b) * tile*tile).
 */
#ifndef GP_B200_H_
#define GP_B200_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    GP_OK = 0,
    GP_ERR_NULL = -1,        /* a required pointer is NULL */
    GP_ERR_SIZE = -2,        /* n, m, na, nb or D <= 0, or beyond what the index arithmetic supports */
    GP_ERR_TILE = -3,        /* tile <= 0, tile % 32 != 0, or a size not divisible by tile */
    GP_ERR_HYPER = -4,       /* lengthscale <= 0, vertical <= 0, noise < 0, or non-finite */
    GP_ERR_WORKSPACE = -5,   /* work_bytes smaller than gp_workspace_bytes() reports */
    GP_ERR_CUDA = -6,        /* a CUDA runtime call failed (launch, memset, schedule upload) */
    GP_ERR_MODE = -7,        /* unknown layout mode */
    GP_ERR_LIMIT = -8        /* the problem exceeds the fixed scratch of a no-allocation entry point (gp_solve_noalloc) */
};

enum { GP_SYM_LOWER = 0, GP_GENERAL = 1 };

/* Hyperparameters of the squared-exponential kernel, PAPER.md:63 (Eq. 1) and PAPER.md:66:
 *   k(xi,xj) = vertical * exp(-r2 / den) + delta_ij * noise,  r2 = sum_d (xi_d - xj_d)^2,
 *   den = 2*lengthscale as printed in Eq. 1 (ell_squared == 0, the default), or
 *   den = 2*lengthscale^2, the textbook form (ell_squared != 0) -- reading A1.
 * The noise term is added ONLY on the diagonal of the training matrix K (reading A2). */
typedef struct {
    double lengthscale;
    double vertical;
    double noise;
    int ell_squared;
} gp_hyper;

/* Covariance assembly in tiles -- PAPER.md:68 ("assemble multiple covariance matrices where each
 * entry (i,j) corresponds to the kernel evaluation k(a_i, b_j)"), Eq. 1; steps a1/a9.
 *   dA [na x D], dB [nb x D] row-major feature matrices.
 *   mode GP_SYM_LOWER: requires dA == dB and na == nb; writes the M(M+1)/2 lower tiles of
 *        K = K_{X,X} and adds h.noise on the global diagonal.
 *   mode GP_GENERAL:   writes all (na/tile) x (nb/tile) tiles of K_{A,B}; never adds noise.
 *   dTiles: output, (number of tiles) * tile^2 doubles in the layout above. */
int gp_assemble_tiles(const double* dA, int64_t na, const double* dB, int64_t nb, int D, gp_hyper h,
                      int tile, int mode, double* dTiles, void* stream);

/* Tiled right-looking Cholesky K = L L^T, in place -- PAPER.md:83-139 (section 4.2, Fig. 1):
 * POTRF on diagonal tiles, TRSM on panel tiles, SYRK / GEMM on trailing tiles (tile formulas per
 * reading A3, loop nest per reading A4); steps a2-a6.
 *   dKL: lower-packed tiles of K on entry, of L on exit (GP_SYM_LOWER layout).
 *   sched_width: number of persistent worker CTAs that execute the tile-task DAG, the analogue
 *        of the paper's CUDA-stream pool size; 0 = auto (one per SM).
 *   d_info: device int. 0 = success; k > 0 = 1-based global column of the first non-positive
 *        pivot (K not positive definite; reading A6).  After a failure the remaining tasks still
 *        terminate and dKL is unspecified.
 *   dWork/work_bytes: scratch, at least the `chol` size from gp_workspace_bytes(). On exit it
 *        holds the inverted diagonal blocks of L that gp_predict_full_cov recomputes for itself,
 *        so it may be freed or reused immediately.
 *   Limits: n <= 2^22 and n / gp_block_size(tile) <= 65535 (GP_ERR_SIZE otherwise). */
int gp_cholesky_tiled(double* dKL, int64_t n, int tile, int sched_width, int* d_info, void* dWork,
                      size_t work_bytes, void* stream);

/* Forward and backward substitution -- PAPER.md:72: L beta = y, then L^T alpha = beta; steps a7-a8.
 *   dL: lower-packed tiles of L.  dY [n].  dAlpha [n] <- K^-1 y.
 *   dBeta [n] <- L^-1 y; may be NULL, then dWork must hold n doubles more (see gp_workspace_bytes).
 *   dAlpha may be the same buffer as dY (y is consumed before alpha is written); dBeta must not overlap dY or dAlpha
 *   (it is marked "not yet computed" before y is read: the pieces of a solution are published by their values).
 *   dWork/work_bytes: scratch, at least the `solve` size from gp_workspace_bytes(). */
int gp_solve(const double* dL, int64_t n, int tile, const double* dY, double* dAlpha, double* dBeta,
             void* dWork, size_t work_bytes, void* stream);

/* gp_solve for callers that cannot allocate or carry scratch (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): same arguments and results as gp_solve, but the scratch (ticket counters, beta when dBeta is NULL,
 * the inverted diagonal blocks) lives in a file-scope `static __device__` array of the library, GP_SOLVE_NOALLOC_BYTES =
 * 4.5 MB, which every GPU that loads the library holds until exit.  Its device address is taken once per device with
 * cudaGetSymbolAddress.  The call allocates nothing: no cudaMalloc / cudaFree, no allocating library routine.
 *   Limit: the scratch gp_solve would need must fit the array: n <= GP_SOLVE_NOALLOC_MAX_N = 8192 with the block edge the
 *   library picks for such n (64 or 32); anything larger is rejected with GP_ERR_LIMIT before any work is enqueued.
 *   Every call on a device shares the ONE array (it keeps the previous call's contents; the call clears what must start at
 *   zero): calls that overlap on the GPU (different streams, or graph branches that run concurrently) RACE -- serialise them. */
#define GP_SOLVE_NOALLOC_MAX_N 8192
#define GP_SOLVE_NOALLOC_BYTES 4718592
int gp_solve_noalloc(const double* dL, int64_t n, int tile, const double* dY, double* dAlpha, double* dBeta, void* stream);

/* Predictive mean -- PAPER.md:70 (Eq. 2) through PAPER.md:72: y^ = K_{X^,X} alpha; steps a9-a10.
 * The cross-covariance is evaluated on the fly and never stored.
 *   dX [n x D], dAlpha [n], dXs [m x D]; dMean [m] output.  No tiling constraint on n or m. */
int gp_predict_mean(const double* dX, int64_t n, int D, const double* dAlpha, const double* dXs, int64_t m,
                    gp_hyper h, double* dMean, void* stream);

/* Full predictive covariance -- PAPER.md:76 (Eq. 3) computed as PAPER.md:79 prescribes:
 * solve L V = K_{X,X^}, W = V^T V, Sigma = K_{X^,X^} - W; steps a9, a11, a12.
 * V is held transposed (V^T = K_{X^,X} L^-T, m x n, GP_GENERAL tiles) in dWork.
 *   dL: lower-packed tiles of L; dX [n x D]; dXs [m x D].
 *   dSigma [m x m] dense row-major output; both triangles are written and are exactly symmetric.
 *   sched_width as in gp_cholesky_tiled.
 *   dWork/work_bytes: scratch, at least the `full_cov` size from gp_workspace_bytes(). */
int gp_predict_full_cov(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m,
                        gp_hyper h, int tile, int sched_width, double* dSigma, void* dWork,
                        size_t work_bytes, void* stream);

/* Scratch sizes in bytes for the three calls that need scratch; any output pointer may be NULL.
 * m may be 0 when only chol/solve are wanted. */
int gp_workspace_bytes(int64_t n, int64_t m, int D, int tile, size_t* chol, size_t* solve, size_t* full_cov);

/* Unpack tiles to a dense row-major matrix (testing/inspection helper, not on the hot path).
 *   lower_packed != 0: GP_SYM_LOWER tiles of an n x n matrix -> dDense [n x n] with the strict
 *        upper triangle zeroed (reading A8);  nb is ignored.
 *   lower_packed == 0: GP_GENERAL tiles of an n x nb matrix -> dDense [n x nb]. */
int gp_tiles_to_dense(const double* dTiles, int64_t n, int64_t nb, int tile, int lower_packed,
                      double* dDense, void* stream);

/* SURVEY.md 8(f) row 1, "predict with uncertainty" ("the diagonal elements of Sigma
 * represent the predictive variances"): dVar[m] <- diag(Sigma) = k(x^,x^) - sum_i V_i^2 without the
 * n m^2 contraction W = V^T V and without the m x m output.  Same arguments, workspace (the m x n
 * V^T buffer; size = full_cov of gp_workspace_bytes) and error behaviour as gp_predict_full_cov;
 * the prior variance is noise-free (reading A2), so 0 <= dVar[a] <= v. */
int gp_predict_variance(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m,
                        gp_hyper h, int tile, int sched_width, double* dVar, void* dWork, size_t work_bytes,
                        void* stream);

/* Prediction sharded by test-point tile rows (V and the mean are independent per block of
 * test points, Sigma needs V of all of them once).  The two halves a multi-GPU driver needs
 * (paper_2602_19683_b200/multi_gpu.py, ShardedPredictor: all-gather of V^T between them):
 *   gp_predict_vt        dVt [m x n as GP_GENERAL tiles]  <-  V^T = K_{X^,X} L^-T for the m test points given (a11);
 *                        arguments and workspace as gp_predict_full_cov.
 *   gp_predict_cov_rows  dSigmaRows [rows x m] dense row-major  <-  K_{X^_r, X^} - V_r^T (V^T)^T  for the test points
 *                        [row0, row0 + rows) against ALL m (a12), from the complete dVtAll [m x n, GP_GENERAL tiles] and
 *                        dXsAll [m x D].  Full block rows are computed (no symmetry across callers); row0 % tile == 0,
 *                        rows % tile == 0.  dWork: at least gp_cov_rows_workspace_bytes(). */
int gp_predict_vt(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m, gp_hyper h, int tile,
                  int sched_width, double* dVt, void* dWork, size_t work_bytes, void* stream);
int gp_cov_rows_workspace_bytes(int64_t n, int64_t m, int64_t rows, int tile, size_t* bytes);
int gp_predict_cov_rows(const double* dVtAll, const double* dXsAll, int64_t n, int64_t m, int D, int64_t row0, int64_t rows,
                        gp_hyper h, int tile, int sched_width, double* dSigmaRows, void* dWork, size_t work_bytes, void* stream);

/* SURVEY.md 8(f) row 4 (hyperparameters "are typically subject to optimization"): the
 * objective of that optimisation, *d_out (device double) <- log p(y) = -1/2 y^T alpha - sum_i log L_ii
 * - n/2 log(2 pi), from the factor of gp_cholesky_tiled and the alpha of gp_solve.  One CTA, fixed
 * summation order (bitwise reproducible). */
int gp_log_marginal_likelihood(const double* dL, int64_t n, int tile, const double* dY, const double* dAlpha,
                               double* d_out, void* stream);

/* Number of tile tasks (POTRF + TRSM + SYRK + GEMM) and of CTA-sized work items the scheduler
 * runs for an n x n factorisation with this tile size (a6 bookkeeping; host only). */
int gp_cholesky_task_counts(int64_t n, int tile, int64_t* tile_tasks, int64_t* work_items);

/* Whole pipeline with HOST buffers -- PAPER.md:143 ("explicit H2D of X, y, X^; only results are
 * copied back"): the call a user with data in host memory makes.  Copies hX [n x D], hY [n] and
 * hXs [m x D] to the device, runs a1-a12 (gp_assemble_tiles, gp_cholesky_tiled, gp_solve,
 * gp_predict_mean, gp_predict_full_cov) on `stream`, copies the results back and SYNCHRONISES the
 * stream before returning (the only entry point that does; its outputs are host memory).
 *   hMean [m], hSigma [m x m] (may be NULL: mean only), hAlpha [n] (may be NULL): host outputs;
 *   pinned host memory makes the copies asynchronous DMA, pageable memory also works.
 *   h_info: host int, as d_info of gp_cholesky_tiled.
 *   dWork/work_bytes: DEVICE scratch of at least gp_pipeline_workspace_bytes(); holds X, y, X^,
 *        the K/L tiles, alpha, beta, mean, Sigma and the per-call scratch. */
int gp_pipeline_workspace_bytes(int64_t n, int64_t m, int D, int tile, size_t* bytes);
int gp_pipeline_host(const double* hX, const double* hY, const double* hXs, int64_t n, int64_t m, int D,
                     gp_hyper h, int tile, int sched_width, double* hMean, double* hSigma, double* hAlpha,
                     int* h_info, void* dWork, size_t work_bytes, void* stream);
/* The same call with the O(n^3) contractions emulated on the int8 tensor cores: gp_cholesky_tiled_mixed
 * and gp_predict_full_cov_mixed in place of gp_cholesky_tiled and gp_predict_full_cov; same arguments, same outputs within
 * the oracle tolerances, tile % 128 == 0, and a larger scratch (gp_pipeline_mixed_workspace_bytes: the digit planes). */
int gp_pipeline_mixed_workspace_bytes(int64_t n, int64_t m, int D, int tile, size_t* bytes);
int gp_pipeline_host_mixed(const double* hX, const double* hY, const double* hXs, int64_t n, int64_t m, int D,
                           gp_hyper h, int tile, int sched_width, double* hMean, double* hSigma, double* hAlpha,
                           int* h_info, void* dWork, size_t work_bytes, void* stream);

/* FP64 peak microbenchmark launch (measurement support; north_star: "FP64 peak also measured by a
 * microbenchmark").  Enqueues one launch of independent register-resident chains on every SM:
 * mode 0 = DMMA.8x8x4 (mma.sync.m8n8k4.f64), mode 1 = DFMA.  *flops (host, may be NULL) receives
 * the floating-point operations one launch performs; the caller times the launch with events.
 *   d_sink: device double[1], never actually written. */
int gp_fp64_peak_launch(int mode, int iters, double* d_sink, double* flops, void* stream);

/* Steady-state rate of the contraction path alone (measurement support): the persistent executor
 * runs SMs x reps independent work items C(128x128) -= A(128xK) B(128xK)^T on a synthetic
 * lower-packed matrix (tile edge K) with every dependency wait switched off, so TMA streaming,
 * DMMA main loop, epilogue and version-counter signalling are all exercised but nothing waits on
 * the DAG.  The gap to the DMMA peak is the kernel's own overhead; the gap from the Cholesky rate
 * to this is the DAG's.
 *   K: multiple of 128, <= 8192.  d_buf/buf_bytes: device scratch, contents arbitrary finite
 *   doubles (overwritten); *need_bytes (host, may be NULL) receives the size required, and with
 *   d_buf == NULL the call only reports it.  *flops (host, may be NULL): flop of one launch.
 *   Performs one synchronous cudaMemcpy of the item list. */
int gp_contraction_bench_launch(int K, int reps, void* d_buf, size_t buf_bytes, double* flops, size_t* need_bytes,
                                void* stream);

/* SURVEY.md 8(f) row 3 ("we plan to introduce mixed-precision calculations to take advantage of modern
 * hardware capabilities"): the building block of a tensor-core route past the FP64 pipe -- the contraction
 * C -= A B^T in FP64 accuracy EMULATED on the int8 tensor cores (tcgen05.mma kind::i8, int32 accumulators in TMEM)
 * by the split-operand (Ozaki) scheme.  Every operand entry is written in fixed point with one global scale,
 *     x / scale = sum_{p=0}^{S-1} d_p 2^(-b (p + 1)),   d_p in [-2^(b-1), 2^(b-1) - 1]   (S planes of balanced b-bit digits;
 *     S = gp_ozaki_planes() = 7, b = gp_ozaki_digit_bits() = 8: 56 bits of fixed point),
 * the S (S + 1) / 2 = 28 plane products with p + q <= S - 1 are exact integer GEMMs, and only their recombination rounds
 * (FP64).  The truncation is 2^-(b (S + 1)) scaleA scaleB per term, below the FP64 rounding of a result of that size.
 *   gp_ozaki_plane_bytes: size of the plane array of a rows x k operand (S rows k bytes).
 *   gp_ozaki_slice: dX [rows x k] row-major FP64 with leading dimension ld  ->  dPlanes [S][rows][k] int8.
 *        Requires |x| <= 0.498 scale for every entry (the top digit must fit); *d_overflow (device int) is set to 1 otherwise, else 0.
 *        k % 32 == 0.
 *   gp_ozaki_contract: dC [ma x nb] row-major FP64, leading dimension ldc (even)  -=  A B^T from the planes of
 *        A [ma x k] and B [nb x k].  ma % 128 == 0, nb % 64 == 0, k % 32 == 0.  An int32 level accumulator takes a
 *        contraction depth of 16384; deeper contractions run as consecutive launches over k segments.
 * Both calls are stream-ordered.  bench.py reports the FP64-equivalent rate of the emulated contraction beside the DMMA
 * contraction; gp_cholesky_tiled does not use it (gp_cholesky_tiled_mixed does). */
int gp_ozaki_planes(void);
int gp_ozaki_digit_bits(void);
int gp_ozaki_plane_bytes(int64_t rows, int64_t k, size_t* bytes);
/* Output-tile shape of the emulated contraction: 0 = auto (the 128 x 128 two-pass kernel whenever the column count and
 * the k range are multiples of 128, else the 128 x 64 kernel with all level sums resident in tensor memory), 64 = always
 * the 128 x 64 kernel, 128 = same as auto.  Measurement support: an MMA of 128 x 64 x 32 takes 48 cycles (shared-memory
 * operand read), one of 128 x 128 x 32 takes 64, which is the tensor core's full rate. */
int gp_set_ozaki_tile_n(int n);
int gp_ozaki_slice(const double* dX, int64_t rows, int64_t k, int64_t ld, double scale, int8_t* dPlanes, int* d_overflow,
                   void* stream);
int gp_ozaki_contract(const int8_t* dAplanes, int64_t ma, const int8_t* dBplanes, int64_t nb, int64_t k, double scaleA,
                      double scaleB, double* dC, int64_t ldc, void* stream);

/* Measurement support for the emulated contraction (bench.py --ozaki-probe; profiles/r02_ozaki_bounds.md).
 *   gp_int8_mma_peak_launch: one thread per SM issues 16 * iters tcgen05.mma kind::i8 of 128 x n_cols x 32 (n_cols = 64,
 *        128 or 256) on whatever shared memory holds; d_cycles (device, 1 entry, may be NULL) receives the clock64 ticks of
 *        CTA 0's loop, *ops (host, may be NULL) the int8 operations of the launch (2 per multiply-add).  The caller times
 *        the launch with events: the rate at n_cols = 128 is the int8 tensor peak bench.py holds the contraction against.
 *   gp_ozaki_probe_launch: the 128 x 128 two-pass kernel on dense C [ma x nb] (ma, nb, k multiples of 128, k <= 16384,
 *        scales 1) with one of its parts switched off: probe 0 = nothing (the product kernel), 1 = no TMA loads (the MMAs
 *        run on whatever the slots hold: C is garbage), 2 = no MMAs (loads only), 4 = no reductions into C.
 *   gp_ozaki_probe_stamps: after a launch with probe > 0 (and a synchronise), 8 clock64 stamps of the second tile of CTA 0:
 *        pass 0 issue start / end, pass 1 issue start / end, epilogue of pass 0 start / end, epilogue of pass 1 start / end. */
int gp_int8_mma_peak_launch(int n_cols, int iters, long long* d_cycles, double* ops, void* stream);
int gp_ozaki_probe_launch(int probe, const int8_t* dAplanes, int64_t ma, const int8_t* dBplanes, int64_t nb, int64_t k, double* dC,
                          int64_t ldc, void* stream);
int gp_ozaki_probe_stamps(long long* h_stamps8);

/* SURVEY.md 8(f) row 3, end to end: the tiled Cholesky of gp_cholesky_tiled with its trailing updates (SYRK / GEMM tile
 * tasks: > 95 % of the flops) EMULATED on the int8 tensor cores and everything on the critical path
 * (POTRF and TRSM tile tasks) in FP64 as before.  Opt-in: gp_cholesky_tiled itself is unchanged.
 *   Left-looking over tile columns: column J first receives all its updates in ONE emulated contraction of depth J * tile
 *   (tile (I,J) -= L(I,0:J) L(J,0:J)^T from the digit planes of the finished columns), then its FP64 panel step runs on
 *   the persistent executor (POTRF tile task + TRSM tile tasks), then its tiles are sliced into digit planes.  The
 *   fixed-point scale is found on the device from max_i K_ii (|L_ij| <= sqrt(K_ii)).  Everything is stream-ordered.
 *   Accuracy: the emulation truncates below 2^-56 of the scale; measured |L - L_oracle| / |L_oracle| ~ 1e-13 (tests).
 *   Same arguments and *d_info semantics as gp_cholesky_tiled; additionally tile % 128 == 0, n / tile <= 60, n <= 65536.
 *   dWork: at least gp_mixed_workspace_bytes() (dominated by the dense digit planes, 7 n^2 bytes). */
int gp_mixed_workspace_bytes(int64_t n, int tile, size_t* bytes);
int gp_cholesky_tiled_mixed(double* dKL, int64_t n, int tile, int sched_width, int* d_info, void* dWork, size_t work_bytes,
                            void* stream);
/* The steps of gp_cholesky_tiled_mixed as separate stream-ordered calls, so that a driver can interleave them with
 * communication ("extend the library to distributed multi-GPU environments":
 * paper_2602_19683_b200/multi_gpu.py distributes the tile columns block-cyclically and broadcasts each finished panel):
 *   gp_mixed_begin          zero the counters, find the fixed-point scale from diag(K) (dKL must hold K's diagonal tiles);
 *   gp_mixed_update_column  tile column J (tiles (I,J), I >= J)  -=  L(J:, k0:k1) L(J, k0:k1)^T  over the tile columns
 *                           [k_tile0, k_tile1), k_tile1 <= J, from the digit planes (which must hold those columns);
 *   gp_mixed_panel          FP64 POTRF tile task of (J,J) + TRSM tile tasks below it; column J must have received the
 *                           updates of ALL tile columns < J;
 *   gp_mixed_slice_column   digit planes of the tiles (I,J), I > J, of the FINAL factor (computed here or received).
 * Same dWork (gp_mixed_workspace_bytes) for every call of one factorisation. */
int gp_mixed_begin(const double* dKL, int64_t n, int tile, int* d_info, void* dWork, size_t work_bytes, void* stream);
int gp_mixed_update_column(double* dKL, int64_t n, int tile, int J, int k_tile0, int k_tile1, void* dWork, size_t work_bytes,
                           void* stream);
int gp_mixed_panel(double* dKL, int64_t n, int tile, int J, int sched_width, int* d_info, void* dWork, size_t work_bytes,
                   void* stream);
int gp_mixed_slice_column(const double* dKL, int64_t n, int tile, int J, void* dWork, size_t work_bytes, void* stream);
/* gp_mixed_panel with the panel broadcast FUSED into it ("per step the owner factors the panel and
 * broadcasts ... fused as the epilogue of the TRSM kernel"): every block of tile column J that the step finishes (the
 * diagonal blocks by POTRF, the blocks below by their solve) is stored not only into dKL but also at the same offset of
 * peers[0 .. npeers-1] (host array of DEVICE addresses, npeers <= 7): the other ranks' copies of the tile array, mapped into
 * this GPU's address space (NVLink peer memory after cudaIpcOpenMemHandle + cudaDeviceEnablePeerAccess; other buffers of
 * the same device in the one-GPU emulation of tests/test_gpu_multi.py).  The transfer rides on the panel step block by
 * block instead of following it as a collective; the stores are complete when the call's work on `stream` is, so the
 * receivers need one barrier after it and no copy.  The strict upper part of the diagonal tile is not transferred
 * (it is never read).  npeers = 0 is gp_mixed_panel. */
int gp_mixed_panel_bcast(double* dKL, int64_t n, int tile, int J, int sched_width, int* d_info, void* dWork, size_t work_bytes,
                         double* const* peers, int npeers, void* stream);

/* The full-covariance prediction on the same emulated contraction (opt-in; gp_predict_full_cov is unchanged): the
 * V^T solve left-looking over tile columns (column P gets V^T(:,0:P) L(P,0:P)^T in one emulated contraction, then its FP64
 * TRSM with the diagonal tile on the executor, then its digit planes), and W = V^T (V^T)^T in ONE emulated contraction of
 * depth n over the lower triangle of Sigma, mirrored.  Arguments as gp_predict_full_cov; additionally tile % 128 == 0,
 * n / tile <= 60, n <= 65536, m <= 65536.  dWork: gp_mixed_predict_workspace_bytes() (V^T and the digit planes of L and
 * of V^T: 8 m n + 7 (n^2 + m n) bytes). */
int gp_mixed_predict_workspace_bytes(int64_t n, int64_t m, int tile, size_t* bytes);
int gp_predict_full_cov_mixed(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m, gp_hyper h,
                              int tile, int sched_width, double* dSigma, void* dWork, size_t work_bytes, void* stream);
/* Variances only on the emulated contraction (SURVEY.md 8(f) rows 1 and 3 together): the V^T solve of
 * gp_predict_full_cov_mixed without W, then var_a = v - sum_i V_ia^2 as gp_predict_variance.  dVar [m]; same scratch. */
int gp_predict_variance_mixed(const double* dL, const double* dX, int64_t n, int D, const double* dXs, int64_t m, gp_hyper h,
                              int tile, int sched_width, double* dVar, void* dWork, size_t work_bytes, void* stream);

/* Host-only replay check of the panel schedule of step J (returns the number of work items, or a negative GP_ERR_*). */
int gp_panel_schedule_selfcheck(int64_t n, int tile, int J);

/* Executor statistics of the LAST gp_cholesky_tiled / gp_predict_full_cov call that used dWork
 * (tracing support; the analogue of the paper's per-step APEX timers).  Copies
 * to h_stats (host) 8 uint64 per worker CTA:
 *   [0] SM cycles its producer warp spent polling dependency counters,
 *   [1] SM cycles from kernel start to the producer's exit,  [2] work items run,  [3] SM id,
 *   [4] SM cycles consumer warp 0 waited for a job descriptor (nothing runnable was handed over),
 *   [5] reserved,  [6] jobs (GEMM / POTRF block operations) run,  [7] reserved;
 * synchronises the stream.  Returns the number of worker slots copied (<= max_workers) or a
 * negative GP_ERR_*. */
int gp_exec_stats(const void* dWork, uint64_t* h_stats, int max_workers, void* stream);

/* Host-only self-check of the static work-item schedule the persistent executor consumes (a6):
 * builds the schedule for (n, m, tile) with `workers` virtual SMs (m == 0: Cholesky schedule,
 * m > 0: predictor schedule) and replays it against the dependency rules of the device code.
 * Returns GP_OK if every wait of every item is satisfied by earlier items and every block ends at
 * its final version, GP_ERR_SIZE otherwise.  stats (may be NULL) receives
 * {items, dependency edges, simulated makespan us, total work us, critical path us}. */
int gp_schedule_selfcheck(int64_t n, int64_t m, int tile, int workers, double* stats5);
/* The same for the schedule of gp_predict_variance (m > 0; no W = V^T V items). */
int gp_schedule_selfcheck_variance(int64_t n, int64_t m, int tile, int workers, double* stats5);

/* Build and upload, on the current device, the static work-item schedules that gp_cholesky_tiled
 * (GP_PREPARE_CHOLESKY), gp_predict_full_cov (GP_PREPARE_FULL_COV) and gp_predict_variance
 * (GP_PREPARE_VARIANCE) need for this shape (step a6: the host-side half of the tile-task scheduler,
 * PAPER.md:45, 145-147).  Synchronous: blocks the host for the list-scheduling simulation and a
 * cudaMalloc + cudaMemcpy per schedule.  Idempotent; later compute calls for the same shape find the
 * schedules in the cache and do not touch the host again.  `what` is an OR of GP_PREPARE_*; m may be 0
 * for GP_PREPARE_CHOLESKY alone.  *build_ms (host, may be NULL) receives the wall time spent. */
enum { GP_PREPARE_CHOLESKY = 1, GP_PREPARE_FULL_COV = 2, GP_PREPARE_VARIANCE = 4 };
int gp_prepare(int64_t n, int64_t m, int tile, int what, double* build_ms);

/* 64-bit fingerprint (FNV-1a over the item list) of the schedule the executor would run for this shape
 * (m == 0: Cholesky; m > 0: predictor, with or without the Sigma items).  Host only.  Measurements that
 * depend on the order of work items (the DRAM traffic recorded under profiles/) store it so that
 * bench.py can tell whether they still describe the current build. */
int gp_schedule_fingerprint(int64_t n, int64_t m, int tile, int workers, int with_sigma, uint64_t* fingerprint);

/* Scheduling granularity (step a6; the analogue of the paper's "tiles per dimension" knob).
 * The tile tasks of Fig. 1 are formed over scheduling tiles of g x g blocks (block = gp_block_size(tile)); g is
 * independent of the storage tile.  gp_schedule_granularity() returns the g the library uses for a shape:
 * auto = 1 up to 96 block columns (short serial chains while the critical path bounds the run), else about 32
 * scheduling tiles per dimension (long work items whose panels are shared in L2).  Results do not depend on g
 * beyond rounding order.  gp_set_schedule_granularity(blocks) overrides the choice for later calls of this
 * process (0 = auto again; the largest divisor of the block counts <= blocks is used): measurement support
 * for bench.py --sweep, not needed in normal use. */
int gp_set_schedule_granularity(int blocks);
int gp_schedule_granularity(int64_t n, int64_t m, int tile);

/* Drop the cached device-resident schedules (synchronises the device). */
void gp_release_cached_schedules(void);

/* Edge (in doubles) of the largest CTA-level block this tile size admits: 128 if tile % 128 == 0, else 64 if
 * tile % 64 == 0, else 32. */
int gp_block_size(int tile);
/* Edge of the block the library actually splits the tile tasks into for an n x n problem with this tile size:
 * the largest admissible edge up to 64 for n <= 8192 (short serial chains while the critical path bounds the run),
 * up to 128 beyond (full contraction rate).  The storage tile only fixes the addressing; results do not depend on
 * the block edge beyond rounding order.  gp_set_block_edge(b) (b in {0 = auto, 32, 64, 128}) overrides the cap for
 * later calls of this process -- call it before gp_workspace_bytes, whose sizes depend on the block edge;
 * measurement support for bench.py --sweep. */
int gp_block_size_for(int64_t n, int tile);
int gp_set_block_edge(int b);

const char* gp_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* GP_B200_H_ */
