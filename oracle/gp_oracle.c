/*
 * gp_oracle.c -- the CPU FP64 ORACLE for the GP prediction pipeline of
 * arxiv/paper_2602_19683 (section 4.1, Eq. 1-3).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code,
 * header, table or helper with the CUDA path under paper_2602_19683_b200/csrc/, and
 * neither includes the other.
 *
 * Everything here is the plain textbook definition written out, untiled, in index
 * order, in IEEE double.  No BLAS/LAPACK, no blocking, no fusion, no reordering; the
 * only parallelism is an OpenMP "parallel for" over independent outputs (rows of a
 * column, columns of a right-hand side), which does not change any summation order.
 * All matrices are dense row-major, 0-based.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): the 40-digit worked examples
 * A, B, B' under tests/golden/ (SURVEY.md section 8(c)(i)), n=1 and far-apart closed
 * forms, brute-force Gauss-Jordan inversion for n<=64 (Eq. 2 and Eq. 3 literally),
 * numpy.linalg.cholesky, ||LL^T-K||_F/||K||_F <= 1e-12, the X^=X identities,
 * scaling/permutation/leading-block invariants, Sigma symmetric PSD with
 * 0 <= Sigma_ii <= v.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int t)
{
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

/*
 * PAPER.md:63, Eq. 1 (squared-exponential kernel), and PAPER.md:68 (the covariance
 * matrices are kernel evaluations k(a_i, b_j)).
 *   K[i][j] = v * exp(-r2 / den) + (add_noise_diag && i == j ? noise : 0),
 *   r2 = sum_{d=0}^{D-1} (A[i][d] - B[j][d])^2, summed in index order,
 *   den = 2*ell as printed in Eq. 1 (ell_squared == 0), or 2*ell^2 (ell_squared != 0).
 * DESIGN.md readings A1 (denominator) and A2 (noise only on the training diagonal:
 * the caller sets add_noise_diag = 1 only for K = K_{X,X}).
 * A is na x D, B is nb x D, K is na x nb.
 */
void oracle_assemble(const double *A, int64_t na, const double *B, int64_t nb, int D,
                     double ell, double v, double noise, int ell_squared,
                     int add_noise_diag, double *K)
{
    const double den = ell_squared ? 2.0 * ell * ell : 2.0 * ell;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < na; ++i) {
        for (int64_t j = 0; j < nb; ++j) {
            double r2 = 0.0;
            for (int d = 0; d < D; ++d) {
                const double diff = A[i * D + d] - B[j * D + d];
                r2 += diff * diff;
            }
            double k = v * exp(-r2 / den);
            if (add_noise_diag && i == j) k += noise;
            K[i * nb + j] = k;
        }
    }
}

/*
 * K = L L^T with L lower triangular (positive diagonal, so L is unique
 * when K is positive definite -- DESIGN.md reading A6).  Unblocked column-by-column
 * (Cholesky-Crout) form of the definition:
 *   L[j][j] = sqrt(K[j][j] - sum_{p<j} L[j][p]^2)
 *   L[i][j] = (K[i][j] - sum_{p<j} L[i][p] L[j][p]) / L[j][j],  i > j
 * with every sum taken in index order p = 0..j-1.  The strict upper triangle of L is
 * set to 0 (reading A8).  Only the lower triangle of K is read.
 * Returns 0 on success, or the 1-based column of the first non-positive (or NaN) pivot.
 */
int64_t oracle_cholesky(const double *K, int64_t n, double *L)
{
    for (int64_t j = 0; j < n; ++j) {
        double s = K[j * n + j];
        for (int64_t p = 0; p < j; ++p) s -= L[j * n + p] * L[j * n + p];
        if (!(s > 0.0)) return j + 1;
        const double ljj = sqrt(s);
        L[j * n + j] = ljj;
#pragma omp parallel for schedule(static)
        for (int64_t i = j + 1; i < n; ++i) {
            double t = K[i * n + j];
            for (int64_t p = 0; p < j; ++p) t -= L[i * n + p] * L[j * n + p];
            L[i * n + j] = t / ljj;
            L[j * n + i] = 0.0; /* strict upper triangle */
        }
    }
    return 0;
}

/*
 * PAPER.md:72 "solving L beta = y (forward substitution)":
 *   x[i] = (b[i] - sum_{p<i} L[i][p] x[p]) / L[i][i],  i = 0..n-1.
 */
void oracle_forward_subst(const double *L, int64_t n, const double *b, double *x)
{
    for (int64_t i = 0; i < n; ++i) {
        double s = b[i];
        for (int64_t p = 0; p < i; ++p) s -= L[i * n + p] * x[p];
        x[i] = s / L[i * n + i];
    }
}

/*
 * PAPER.md:72 "followed by L^T alpha = beta (backward substitution)":
 *   x[i] = (b[i] - sum_{p>i} L[p][i] x[p]) / L[i][i],  i = n-1..0,
 * the sum taken in index order p = i+1..n-1.
 */
void oracle_backward_subst(const double *L, int64_t n, const double *b, double *x)
{
    for (int64_t i = n - 1; i >= 0; --i) {
        double s = b[i];
        for (int64_t p = i + 1; p < n; ++p) s -= L[p * n + i] * x[p];
        x[i] = s / L[i * n + i];
    }
}

/*
 * PAPER.md:70 Eq. 2 via PAPER.md:72: y^ = K_{X^,X} alpha.
 * Kxs is the m x n cross-covariance (row a = test point a), mean has m entries;
 * each is the dot product in index order.
 */
void oracle_matvec(const double *Kxs, int64_t m, int64_t n, const double *alpha, double *mean)
{
#pragma omp parallel for schedule(static)
    for (int64_t a = 0; a < m; ++a) {
        double s = 0.0;
        for (int64_t i = 0; i < n; ++i) s += Kxs[a * n + i] * alpha[i];
        mean[a] = s;
    }
}

/*
 * "solving L V = K_{X,X^} for V": forward substitution applied to each
 * of the m columns of the n x m right-hand side B.  V is n x m.  Columns are
 * independent, so the OpenMP loop runs over columns; each column is the same
 * recurrence as oracle_forward_subst.
 */
void oracle_forward_subst_cols(const double *L, int64_t n, const double *B, int64_t m, double *V)
{
#pragma omp parallel
    {
        double *x = (double *)malloc((size_t)n * sizeof(double));
#pragma omp for schedule(static)
        for (int64_t c = 0; c < m; ++c) {
            for (int64_t i = 0; i < n; ++i) {
                double s = B[i * m + c];
                for (int64_t p = 0; p < i; ++p) s -= L[i * n + p] * x[p];
                x[i] = s / L[i * n + i];
            }
            for (int64_t i = 0; i < n; ++i) V[i * m + c] = x[i];
        }
        free(x);
    }
}

/*
 * W := V^T V and Sigma = K_{X^,X^} - W  (Eq. 3).
 *   Sigma[a][b] = Kss[a][b] - sum_{i=0}^{n-1} V[i][a] V[i][b]
 * for ALL m^2 entries (no symmetry shortcut -- DESIGN.md reading A12), each sum in
 * index order.  V is n x m, Kss and Sigma are m x m.
 */
void oracle_posterior_cov(const double *V, int64_t n, int64_t m, const double *Kss, double *Sigma)
{
#pragma omp parallel for schedule(static)
    for (int64_t a = 0; a < m; ++a) {
        for (int64_t b = 0; b < m; ++b) {
            double w = 0.0;
            for (int64_t i = 0; i < n; ++i) w += V[i * m + a] * V[i * m + b];
            Sigma[a * m + b] = Kss[a * m + b] - w;
        }
    }
}

/*
 * PAPER.md:72 "followed by L^T alpha = beta (backward substitution)" applied to each of the m
 * columns of the n x m right-hand side B (used by the O(n^2) full-size parity probe of Eq. 3,
 * Sigma z = K_{X^,X^} z - K_{X^,X} K^-1 K_{X,X^} z with K^-1 applied as two
 * triangular solves).  Columns are independent, so the OpenMP loop runs over columns; each
 * column is exactly the recurrence of oracle_backward_subst.  X is n x m.
 */
void oracle_backward_subst_cols(const double *L, int64_t n, const double *B, int64_t m, double *X)
{
#pragma omp parallel
    {
        double *x = (double *)malloc((size_t)n * sizeof(double));
#pragma omp for schedule(static)
        for (int64_t c = 0; c < m; ++c) {
            for (int64_t i = n - 1; i >= 0; --i) {
                double s = B[i * m + c];
                for (int64_t p = i + 1; p < n; ++p) s -= L[p * n + i] * x[p];
                x[i] = s / L[i * n + i];
            }
            for (int64_t i = 0; i < n; ++i) X[i * m + c] = x[i];
        }
        free(x);
    }
}

/*
 * "The diagonal elements of Sigma represent the predictive
 * variances".  The diagonal of Eq. 3 written out, without forming W:
 *   var[a] = kss_diag[a] - sum_{i=0}^{n-1} V[i][a]^2,   kss_diag[a] = k(x^_a, x^_a) (noise-free, A2),
 * each sum in index order.  V is n x m.
 */
void oracle_posterior_var(const double *V, int64_t n, int64_t m, const double *kss_diag, double *var)
{
#pragma omp parallel for schedule(static)
    for (int64_t a = 0; a < m; ++a) {
        double w = 0.0;
        for (int64_t i = 0; i < n; ++i) w += V[i * m + a] * V[i * m + a];
        var[a] = kss_diag[a] - w;
    }
}

/*
 * SURVEY.md 8(f) row 4 ("hyperparameters are typically subject to optimization"): the
 * objective of that optimisation, the log marginal likelihood of y ~ N(0, K), K = L L^T, alpha = K^-1 y:
 *   log p(y) = -1/2 y^T alpha - sum_i log L_ii - n/2 log(2 pi)
 * (log det K = 2 sum_i log L_ii).  Sums in index order, serial.
 */
double oracle_log_marginal_likelihood(const double *L, int64_t n, const double *y, const double *alpha)
{
    double quad = 0.0, logdiag = 0.0;
    for (int64_t i = 0; i < n; ++i) quad += y[i] * alpha[i];
    for (int64_t i = 0; i < n; ++i) logdiag += log(L[i * n + i]);
    return -0.5 * quad - logdiag - 0.5 * (double)n * log(2.0 * 3.14159265358979323846264338327950288);
}
