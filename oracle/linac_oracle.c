/*
 * linac_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of what the Linac hot path computes
 * (arxiv/paper_2605_25863; line numbers are /root/reference/PAPER.md).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this
 * library.  It shares NO code, header, table or trick with the CUDA path under
 * paper_2605_25863_b200/csrc: every reduction is the C `%` operator on uint64_t, the
 * inverse is extended Euclid on signed 64-bit, the schedule is the paper's one-column-
 * at-a-time Gauss-Jordan loop.  No blocking, no Barrett/Montgomery, no limb splitting.
 *
 * What is defined here and which passage each function follows:
 *   oracle_inv_modp / oracle_pow_modp  -- field inverse (K7 "rescales it to a 1");
 *                                          the paper does not say how (reading Q7)
 *   oracle_rref_modp     -- partially pivoted row reduction to REDUCED echelon form over F_p:
 *                           PAPER.md:153 (RREF in the original shape, zero rows at the bottom),
 *                           :225 (row permutations only), :239 (one pass per column, any shape),
 *                           :241 (pivot located in column j among the rows left to reduce),
 *                           :243 (head (i,j); rescale the head to 1 if non-zero),
 *                           :245-249 (row k -= head_k * pivot row; head of row k becomes 0),
 *                           :251 (j always advances, i only on a non-zero pivot)
 *   oracle_det_modp      -- determinant as product of pivots times permutation sign (same loop)
 *   oracle_nullspace_modp-- canonical kernel basis from the RREF, PAPER.md:403-415 (eq. 8-9):
 *                           free columns are the free variables, "fixes their coefficients to
 *                           minus the identity matrix"
 *   oracle_matmul_modp   -- plain triple loop (used to check A.K = 0, eq. 9, and A = C.R, eq. 7)
 *   oracle_solve_f64     -- row rescaling (K1/K2), partial pivoting on the
 *                           column maximum, tolerance test on the head
 *                           (PAPER.md:243), Gauss-Jordan elimination of (A B) -> (I X)
 *                           (eq. 10-12)
 *   oracle_backward_error-- the acceptance metric of BASELINE.json (inf-norm, long double)
 *
 * Threading: `nthreads` > 1 only splits the independent "for every row k != i" loop of one
 * pivot step across OpenMP threads; the arithmetic and its order per element are unchanged,
 * so results are bit-identical to nthreads == 1.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PIVOT_FIRST 0 /* lowest row index >= i with a non-zero entry (north_star)     */
#define ORACLE_PIVOT_LAST 1  /* highest such row index                                      */
#define ORACLE_PIVOT_MAX 2   /* largest integer representative (what the paper does, :241)  */

int oracle_version(void) { return 1; }

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* a^{-1} mod p by the extended Euclidean algorithm on signed 64-bit; a in [1, p). */
uint32_t oracle_inv_modp(uint32_t a, uint32_t p) {
    int64_t r0 = (int64_t)p, r1 = (int64_t)(a % p);
    int64_t t0 = 0, t1 = 1;
    while (r1 != 0) {
        int64_t q = r0 / r1;
        int64_t r2 = r0 - q * r1;
        int64_t t2 = t0 - q * t1;
        r0 = r1; r1 = r2;
        t0 = t1; t1 = t2;
    }
    /* r0 == gcd == 1 for prime p and a != 0 */
    t0 %= (int64_t)p;
    if (t0 < 0) t0 += (int64_t)p;
    return (uint32_t)t0;
}

/* a^e mod p by square-and-multiply (Fermat inverse is e = p-2); second, independent route. */
uint32_t oracle_pow_modp(uint32_t a, uint64_t e, uint32_t p) {
    uint64_t result = 1 % p, base = a % p;
    while (e) {
        if (e & 1) result = result * base % p;
        base = base * base % p;
        e >>= 1;
    }
    return (uint32_t)result;
}

static void swap_rows_u32(uint32_t *A, int64_t ld, int64_t cols, int64_t r1, int64_t r2) {
    if (r1 == r2) return;
    uint32_t *x = A + r1 * ld, *y = A + r2 * ld;
    for (int64_t c = 0; c < cols; ++c) { uint32_t t = x[c]; x[c] = y[c]; y[c] = t; }
}

/*
 * In place: A (rows x cols, row-major, leading dimension ld >= cols, in elements) becomes its
 * reduced row-echelon form over F_p with canonical representatives in [0,p).  Columns >= cols
 * of each row are never touched (reading Q8).  Entries >= p are first reduced (reading Q5).
 * *rank = number of non-zero rows; pivot_cols[0..rank) = pivot columns, ascending (may be NULL).
 * det_out (may be NULL): for square A, the determinant mod p (0 if rank < rows).
 * Returns 0, or -1 on bad arguments.
 */
static int rref_core(uint32_t *A, int64_t rows, int64_t cols, int64_t ld, uint32_t p, int pivot_rule,
                     int nthreads, int64_t *rank, int32_t *pivot_cols, uint32_t *det_out) {
    if (rows < 0 || cols < 0 || ld < cols || p < 2 || (rows > 0 && cols > 0 && !A)) return -1;
    const uint64_t P = p;
    for (int64_t r = 0; r < rows; ++r)
        for (int64_t c = 0; c < cols; ++c) A[r * ld + c] %= p;

    int64_t i = 0;       /* next pivot row  ("the row index may be lower")   */
    uint64_t det = 1 % p;
    int negate = 0;
    (void)nthreads;
    for (int64_t j = 0; j < cols && i < rows; ++j) {       /* PAPER.md:239; reading Q2 */
        /* pivot search in column j among rows >= i */
        int64_t k = -1;
        if (pivot_rule == ORACLE_PIVOT_FIRST) {
            for (int64_t r = i; r < rows; ++r) if (A[r * ld + j] != 0) { k = r; break; }
        } else if (pivot_rule == ORACLE_PIVOT_LAST) {
            for (int64_t r = rows - 1; r >= i; --r) if (A[r * ld + j] != 0) { k = r; break; }
        } else {
            uint32_t best = 0;
            for (int64_t r = i; r < rows; ++r) if (A[r * ld + j] > best) { best = A[r * ld + j]; k = r; }
        }
        if (k < 0) continue;                                 /* zero head: j advances, i does not (:251) */
        if (k != i) { swap_rows_u32(A, ld, cols, k, i); negate ^= 1; }   /* CudaSwitchRows (:241) */
        uint32_t *pi = A + i * ld;
        const uint64_t head = pi[j];
        det = det * head % P;
        const uint64_t inv = oracle_inv_modp((uint32_t)head, p);
        for (int64_t c = j; c < cols; ++c) pi[c] = (uint32_t)((uint64_t)pi[c] * inv % P);  /* (:243) */
        /* every other row k: row_k -= head_k * row_i, head_k becomes 0 (all k != i, reading Q3) */
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads) if (nthreads > 1)
#endif
        for (int64_t r = 0; r < rows; ++r) {
            if (r == i) continue;
            uint32_t *pr = A + r * ld;
            const uint64_t h = pr[j];
            if (h == 0) continue;                            /* conditional skip */
            for (int64_t c = j; c < cols; ++c)
                pr[c] = (uint32_t)(((uint64_t)pr[c] + P - (h * (uint64_t)pi[c] % P)) % P);
        }
        if (pivot_cols) pivot_cols[i] = (int32_t)j;
        ++i;                                                 /* (:251) */
    }
    if (rank) *rank = i;
    if (det_out) {
        if (rows != cols || i < rows) det = 0;
        else if (negate) det = (P - det) % P;
        *det_out = (uint32_t)det;
    }
    return 0;
}

int oracle_rref_modp(uint32_t *A, int64_t rows, int64_t cols, int64_t ld, uint32_t p, int pivot_rule,
                     int nthreads, int64_t *rank, int32_t *pivot_cols) {
    return rref_core(A, rows, cols, ld, p, pivot_rule, nthreads, rank, pivot_cols, NULL);
}

/* Determinant of the n x n matrix A mod p (A is destroyed: it is left in RREF). */
int oracle_det_modp(uint32_t *A, int64_t n, int64_t ld, uint32_t p, uint32_t *det) {
    int64_t rank;
    return rref_core(A, n, n, ld, p, ORACLE_PIVOT_FIRST, 1, &rank, NULL, det);
}

/*
 * Canonical kernel basis.  R is an RREF (rows x cols, ld), `rank` pivots at
 * pivot_cols (ascending).  K is cols x nullity (row-major, ldk), nullity = cols - rank; column t
 * belongs to the t-th free column f_t (ascending):  K[f_t, t] = p-1  ("minus the identity"),
 * K[c_k, t] = R[k, f_t] for every pivot row k, all other entries 0 (reading Q9).
 */
int oracle_nullspace_modp(const uint32_t *R, int64_t rows, int64_t cols, int64_t ld, uint32_t p,
                          int64_t rank, const int32_t *pivot_cols, uint32_t *K, int64_t ldk) {
    (void)rows;
    const int64_t d = cols - rank;
    if (d < 0 || ldk < d) return -1;
    char *is_pivot = (char *)calloc((size_t)(cols > 0 ? cols : 1), 1);
    if (!is_pivot) return -2;
    for (int64_t k = 0; k < rank; ++k) is_pivot[pivot_cols[k]] = 1;
    for (int64_t r = 0; r < cols; ++r) for (int64_t t = 0; t < d; ++t) K[r * ldk + t] = 0;
    int64_t t = 0;
    for (int64_t f = 0; f < cols; ++f) {
        if (is_pivot[f]) continue;
        K[f * ldk + t] = (p - 1) % p;
        for (int64_t k = 0; k < rank; ++k) K[(int64_t)pivot_cols[k] * ldk + t] = R[k * ld + f] % p;
        ++t;
    }
    free(is_pivot);
    return 0;
}

/* C (m x n, ldc) = A (m x k, lda) . B (k x n, ldb) mod p, plain triple loop. */
int oracle_matmul_modp(const uint32_t *A, int64_t lda, const uint32_t *B, int64_t ldb, uint32_t *C, int64_t ldc,
                       int64_t m, int64_t k, int64_t n, uint32_t p, int nthreads) {
    const uint64_t P = p;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads) if (nthreads > 1)
#endif
    for (int64_t r = 0; r < m; ++r)
        for (int64_t c = 0; c < n; ++c) {
            uint64_t acc = 0;
            for (int64_t t = 0; t < k; ++t)
                acc = (acc + (uint64_t)(A[r * lda + t] % p) * (uint64_t)(B[t * ldb + c] % p) % P) % P;
            C[r * ldc + c] = (uint32_t)acc;
        }
    return 0;
}

/*
 * fp64: solve A X = B.  A is n x n (lda), B is n x nrhs (ldb); both overwritten: A by the
 * reduced matrix (identity), B by X.  Steps, in the paper's order:
 *   1. row scales s_r = max_c |A[r,c]| over A's columns only (reading Q11), A[r,:] /= s_r,
 *      B[r,:] /= s_r  (CudaSetRowScales / CudaRescaleRows); s_r == 0 -> singular
 *   2. for j = 0..n-1: pivot = arg max_{k>=j} |A[k,j]|, lowest index on ties (
 *      reading Q12); if |pivot| <= tol: return 1 with *info = j+1; swap rows;
 *      rescale the pivot row to head 1 (:243); every other row k: row_k -= head_k * row_j (:245)
 *   3. X is read off the augmented block (eq. 12).
 * tol < 0 selects the default n * 2^-52 (reading Q10; the scaled matrix has max-norm 1 rows).
 * Returns 0 (ok, *info = 0), 1 (singular, *info = 1-based column), -1 (bad arguments).
 */
int oracle_solve_f64(double *A, int64_t n, int64_t lda, double *B, int64_t nrhs, int64_t ldb, double tol,
                     int nthreads, int64_t *info) {
    if (n < 0 || nrhs < 0 || lda < n || ldb < nrhs) return -1;
    if (info) *info = 0;
    if (tol < 0) tol = (double)n * ldexp(1.0, -52);
    (void)nthreads;
    for (int64_t r = 0; r < n; ++r) {
        double s = 0.0;
        for (int64_t c = 0; c < n; ++c) { double v = fabs(A[r * lda + c]); if (v > s) s = v; }
        if (s == 0.0) { if (info) *info = 1; return 1; }
        for (int64_t c = 0; c < n; ++c) A[r * lda + c] /= s;
        for (int64_t c = 0; c < nrhs; ++c) B[r * ldb + c] /= s;
    }
    for (int64_t j = 0; j < n; ++j) {
        int64_t k = j;
        double best = fabs(A[j * lda + j]);
        for (int64_t r = j + 1; r < n; ++r) { double v = fabs(A[r * lda + j]); if (v > best) { best = v; k = r; } }
        if (!(best > tol)) { if (info) *info = j + 1; return 1; }
        if (k != j) {
            for (int64_t c = 0; c < n; ++c) { double t = A[j * lda + c]; A[j * lda + c] = A[k * lda + c]; A[k * lda + c] = t; }
            for (int64_t c = 0; c < nrhs; ++c) { double t = B[j * ldb + c]; B[j * ldb + c] = B[k * ldb + c]; B[k * ldb + c] = t; }
        }
        const double head = A[j * lda + j];
        for (int64_t c = j; c < n; ++c) A[j * lda + c] /= head;
        for (int64_t c = 0; c < nrhs; ++c) B[j * ldb + c] /= head;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads) if (nthreads > 1)
#endif
        for (int64_t r = 0; r < n; ++r) {
            if (r == j) continue;
            const double h = A[r * lda + j];
            if (h == 0.0) continue;
            for (int64_t c = j; c < n; ++c) A[r * lda + c] -= h * A[j * lda + c];
            for (int64_t c = 0; c < nrhs; ++c) B[r * ldb + c] -= h * B[j * ldb + c];
        }
    }
    return 0;
}

/*
 * eta = max over right-hand-side columns of ||A0 x - b||_inf / (||A0||_inf ||x||_inf + ||b||_inf)
 * on the ORIGINAL data, residual accumulated in long double (BASELINE.json; reading Q13).
 */
double oracle_backward_error(const double *A0, int64_t n, int64_t lda, const double *X, int64_t ldx,
                             const double *B0, int64_t ldb, int64_t nrhs, int nthreads) {
    long double norm_a = 0.0L;
    for (int64_t r = 0; r < n; ++r) {
        long double s = 0.0L;
        for (int64_t c = 0; c < n; ++c) s += fabsl((long double)A0[r * lda + c]);
        if (s > norm_a) norm_a = s;
    }
    if (nrhs <= 0) return 0.0;
    long double *norm_r = (long double *)calloc((size_t)nrhs, sizeof(long double));
    long double *norm_x = (long double *)calloc((size_t)nrhs, sizeof(long double));
    long double *norm_b = (long double *)calloc((size_t)nrhs, sizeof(long double));
    (void)nthreads;
    /* rows of the residual are independent; each thread keeps the column maxima of its rows */
#ifdef _OPENMP
#pragma omp parallel num_threads(nthreads) if (nthreads > 1)
#endif
    {
        long double *ax = (long double *)malloc((size_t)nrhs * sizeof(long double));
        long double *mx = (long double *)calloc((size_t)nrhs, sizeof(long double));
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int64_t r = 0; r < n; ++r) {
            for (int64_t q = 0; q < nrhs; ++q) ax[q] = 0.0L;
            for (int64_t c = 0; c < n; ++c) {
                const long double a = (long double)A0[r * lda + c];
                for (int64_t q = 0; q < nrhs; ++q) ax[q] += a * (long double)X[c * ldx + q];
            }
            for (int64_t q = 0; q < nrhs; ++q) {
                long double res = fabsl(ax[q] - (long double)B0[r * ldb + q]);
                if (res > mx[q]) mx[q] = res;
            }
        }
#ifdef _OPENMP
#pragma omp critical
#endif
        for (int64_t q = 0; q < nrhs; ++q) if (mx[q] > norm_r[q]) norm_r[q] = mx[q];
        free(ax); free(mx);
    }
    double eta = 0.0;
    for (int64_t q = 0; q < nrhs; ++q) {
        for (int64_t r = 0; r < n; ++r) {
            long double xv = fabsl((long double)X[r * ldx + q]);
            if (xv > norm_x[q]) norm_x[q] = xv;
            long double bv = fabsl((long double)B0[r * ldb + q]);
            if (bv > norm_b[q]) norm_b[q] = bv;
        }
        long double den = norm_a * norm_x[q] + norm_b[q];
        double e = den > 0.0L ? (double)(norm_r[q] / den) : (norm_r[q] > 0.0L ? INFINITY : 0.0);
        if (e > eta) eta = e;
    }
    free(norm_r); free(norm_x); free(norm_b);
    return eta;
}

/* =====================================================================================================
 * the 64-bit backend ("uint32 is used for p <= 2^32 - 1 and uint64 for
 * 2^32 - 1 < p <= ..."; the upper bound is lost in the extraction -- DESIGN.md reading Q18
 * takes p < 2^63).  The SAME one-column-at-a-time loop as rref_core above (same passages: PAPER.md:153,
 * 225, 239-251), with uint64_t storage and every reduction the C `%` operator on unsigned __int128.
 * oracle_rref_modp (32-bit storage) is already valid for every p <= 2^32 - 1: its temporaries are
 * uint64_t and (a + P - x) < 2^33.
 * ===================================================================================================== */
typedef unsigned __int128 u128;

/* a^{-1} mod p by the extended Euclidean algorithm on signed 128-bit; a in [1, p), p < 2^64. */
uint64_t oracle_inv_modp64(uint64_t a, uint64_t p) {
    __int128 r0 = (__int128)p, r1 = (__int128)(a % p);
    __int128 t0 = 0, t1 = 1;
    while (r1 != 0) {
        __int128 q = r0 / r1;
        __int128 r2 = r0 - q * r1;
        __int128 t2 = t0 - q * t1;
        r0 = r1; r1 = r2;
        t0 = t1; t1 = t2;
    }
    t0 %= (__int128)p;
    if (t0 < 0) t0 += (__int128)p;
    return (uint64_t)t0;
}

int oracle_rref_modp64(uint64_t *A, int64_t rows, int64_t cols, int64_t ld, uint64_t p, int pivot_rule,
                       int nthreads, int64_t *rank, int32_t *pivot_cols) {
    if (rows < 0 || cols < 0 || ld < cols || p < 2 || (rows > 0 && cols > 0 && !A)) return -1;
    const u128 P = p;
    for (int64_t r = 0; r < rows; ++r)
        for (int64_t c = 0; c < cols; ++c) A[r * ld + c] %= p;
    int64_t i = 0;
    (void)nthreads;
    for (int64_t j = 0; j < cols && i < rows; ++j) {
        int64_t k = -1;
        if (pivot_rule == ORACLE_PIVOT_FIRST) {
            for (int64_t r = i; r < rows; ++r) if (A[r * ld + j] != 0) { k = r; break; }
        } else if (pivot_rule == ORACLE_PIVOT_LAST) {
            for (int64_t r = rows - 1; r >= i; --r) if (A[r * ld + j] != 0) { k = r; break; }
        } else {
            uint64_t best = 0;
            for (int64_t r = i; r < rows; ++r) if (A[r * ld + j] > best) { best = A[r * ld + j]; k = r; }
        }
        if (k < 0) continue;
        if (k != i) {
            uint64_t *x = A + k * ld, *y = A + i * ld;
            for (int64_t c = 0; c < cols; ++c) { uint64_t t = x[c]; x[c] = y[c]; y[c] = t; }
        }
        uint64_t *pi = A + i * ld;
        const u128 inv = oracle_inv_modp64(pi[j], p);
        for (int64_t c = j; c < cols; ++c) pi[c] = (uint64_t)((u128)pi[c] * inv % P);
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads) if (nthreads > 1)
#endif
        for (int64_t r = 0; r < rows; ++r) {
            if (r == i) continue;
            uint64_t *pr = A + r * ld;
            const u128 h = pr[j];
            if (h == 0) continue;
            for (int64_t c = j; c < cols; ++c)
                pr[c] = (uint64_t)(((u128)pr[c] + P - (h * (u128)pi[c] % P)) % P);
        }
        if (pivot_cols) pivot_cols[i] = (int32_t)j;
        ++i;
    }
    if (rank) *rank = i;
    return 0;
}

/* C = A.B mod p with 64-bit storage, plain triple loop (checks of the 64-bit results). */
int oracle_matmul_modp64(const uint64_t *A, int64_t lda, const uint64_t *B, int64_t ldb, uint64_t *C, int64_t ldc,
                         int64_t m, int64_t k, int64_t n, uint64_t p, int nthreads) {
    const u128 P = p;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads) if (nthreads > 1)
#endif
    for (int64_t r = 0; r < m; ++r)
        for (int64_t c = 0; c < n; ++c) {
            u128 acc = 0;
            for (int64_t t = 0; t < k; ++t)
                acc = (acc + (u128)(A[r * lda + t] % p) * (u128)(B[t * ldb + c] % p) % P) % P;
            C[r * ldc + c] = (uint64_t)acc;
        }
    return 0;
}

/* =====================================================================================================
 * the paper's ORIGINAL floating-point mode: row reduction of a rectangular,
 * possibly rank-deficient matrix to reduced echelon form with an explicit threshold deciding "which small
 * quantities are treated as zero".  Steps, in the paper's order:
 *   1. CudaSetRowScales / CudaRescaleRows: s_r = max_c |A[r,c]|, A[r,:] /= s_r
 *      (a zero row stays zero).
 *   2. for every column j, while rows are left (reading Q2):
 *        k = arg max_{r >= i} |A[r,j]|, lowest index on ties (reading Q12); swap rows k and i
 *        ("At this point, the maximum may still be a zero", :241);
 *        head = A[i,j]; if |head| <= tol: nothing else happens, j advances (CudaCompareHeadToTolerance, :243, :251);
 *        else row i /= head (:243); every other row r: row_r -= head_r * row_i on the columns from j on, and the
 *        head of row r is SET to zero (:245-249); i advances (:251).
 *   3. Reading Q19: what the thresholds declared zero is written as zero, so that the result is an
 *      exact reduced echelon STRUCTURE ("zero rows possibly appearing at the bottom"): rows >= rank
 *      become 0, and so do the entries of a pivot row left of its pivot (free-column residue below tol).
 * tol < 0 selects max(rows, cols) * 2^-52 (reading Q10; the rescaled rows have max-norm 1).
 * Returns 0, or -1 on bad arguments.
 * ===================================================================================================== */
int oracle_rref_f64(double *A, int64_t rows, int64_t cols, int64_t ld, double tol, int nthreads, int64_t *rank,
                    int32_t *pivot_cols) {
    if (rows < 0 || cols < 0 || ld < cols || (rows > 0 && cols > 0 && !A)) return -1;
    if (tol < 0) tol = (double)(rows > cols ? rows : cols) * ldexp(1.0, -52);
    (void)nthreads;
    for (int64_t r = 0; r < rows; ++r) {
        double s = 0.0;
        for (int64_t c = 0; c < cols; ++c) { double v = fabs(A[r * ld + c]); if (v > s) s = v; }
        if (s == 0.0) continue;
        for (int64_t c = 0; c < cols; ++c) A[r * ld + c] /= s;
    }
    int64_t i = 0;
    for (int64_t j = 0; j < cols && i < rows; ++j) {
        int64_t k = i;
        double best = fabs(A[i * ld + j]);
        for (int64_t r = i + 1; r < rows; ++r) { double v = fabs(A[r * ld + j]); if (v > best) { best = v; k = r; } }
        if (k != i)
            for (int64_t c = 0; c < cols; ++c) { double t = A[i * ld + c]; A[i * ld + c] = A[k * ld + c]; A[k * ld + c] = t; }
        const double head = A[i * ld + j];
        if (!(fabs(head) > tol)) continue;
        double *pi = A + i * ld;
        for (int64_t c = j; c < cols; ++c) pi[c] /= head;
        pi[j] = 1.0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads) if (nthreads > 1)
#endif
        for (int64_t r = 0; r < rows; ++r) {
            if (r == i) continue;
            double *pr = A + r * ld;
            const double h = pr[j];
            if (h == 0.0) continue;
            for (int64_t c = j + 1; c < cols; ++c) pr[c] -= h * pi[c];
            pr[j] = 0.0;
        }
        if (pivot_cols) pivot_cols[i] = (int32_t)j;
        ++i;
    }
    if (rank) *rank = i;
    /* step 3: flush what the thresholds declared zero */
    for (int64_t r = i; r < rows; ++r)
        for (int64_t c = 0; c < cols; ++c) A[r * ld + c] = 0.0;
    if (pivot_cols)
        for (int64_t r = 0; r < i; ++r)
            for (int64_t c = 0; c < pivot_cols[r]; ++c) A[r * ld + c] = 0.0;
    return 0;
}

/* =====================================================================================================
 * SURVEY.md 8(f) rank 3, complex128 ("complex128" is one of the data types the reduction is
 * instantiated for): the same loop as oracle_rref_f64 on double _Complex entries (row-major, ld in elements).
 *   1. row scale: s_r = max_c max(|Re A[r,c]|, |Im A[r,c]|)  -- reading Q21: the
 *      paper does not say which absolute value a complex row is rescaled by; the largest real or imaginary part
 *      keeps the scale a real number that depends on the row only, within sqrt(2) of the largest modulus;
 *   2. pivot = arg max_{r >= i} |A[r,j]| (modulus), lowest index on ties; |head| <= tol => free column;
 *      row i /= head; every other row r: row_r -= head_r * row_i on the columns from j on, head of row r set to 0;
 *   3. what the thresholds declared zero is written as zero (reading Q19).
 * tol < 0 selects max(rows, cols) * 2^-52.  Returns 0, or -1 on bad arguments.
 * ===================================================================================================== */
#include <complex.h>
int oracle_rref_c128(double _Complex *A, int64_t rows, int64_t cols, int64_t ld, double tol, int nthreads, int64_t *rank,
                     int32_t *pivot_cols) {
    if (rows < 0 || cols < 0 || ld < cols || (rows > 0 && cols > 0 && !A)) return -1;
    if (tol < 0) tol = (double)(rows > cols ? rows : cols) * ldexp(1.0, -52);
    (void)nthreads;
    for (int64_t r = 0; r < rows; ++r) {
        double s = 0.0;
        for (int64_t c = 0; c < cols; ++c) {
            const double re = fabs(creal(A[r * ld + c])), im = fabs(cimag(A[r * ld + c]));
            if (re > s) s = re;
            if (im > s) s = im;
        }
        if (s == 0.0) continue;
        for (int64_t c = 0; c < cols; ++c) A[r * ld + c] /= s;
    }
    int64_t i = 0;
    for (int64_t j = 0; j < cols && i < rows; ++j) {
        int64_t k = i;
        double best = cabs(A[i * ld + j]);
        for (int64_t r = i + 1; r < rows; ++r) { double v = cabs(A[r * ld + j]); if (v > best) { best = v; k = r; } }
        if (k != i)
            for (int64_t c = 0; c < cols; ++c) { double _Complex t = A[i * ld + c]; A[i * ld + c] = A[k * ld + c]; A[k * ld + c] = t; }
        const double _Complex head = A[i * ld + j];
        if (!(cabs(head) > tol)) continue;
        double _Complex *pi = A + i * ld;
        for (int64_t c = j; c < cols; ++c) pi[c] /= head;
        pi[j] = 1.0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads) if (nthreads > 1)
#endif
        for (int64_t r = 0; r < rows; ++r) {
            if (r == i) continue;
            double _Complex *pr = A + r * ld;
            const double _Complex h = pr[j];
            if (h == 0.0) continue;
            for (int64_t c = j + 1; c < cols; ++c) pr[c] -= h * pi[c];
            pr[j] = 0.0;
        }
        if (pivot_cols) pivot_cols[i] = (int32_t)j;
        ++i;
    }
    if (rank) *rank = i;
    for (int64_t r = i; r < rows; ++r)
        for (int64_t c = 0; c < cols; ++c) A[r * ld + c] = 0.0;
    if (pivot_cols)
        for (int64_t r = 0; r < i; ++r)
            for (int64_t c = 0; c < pivot_cols[r]; ++c) A[r * ld + c] = 0.0;
    return 0;
}
