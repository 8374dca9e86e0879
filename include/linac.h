/*
 * linac.h -- C ABI of the B200-native Linac hot path (arxiv/paper_2605_25863).
 *
 * Dense Gaussian elimination to REDUCED row-echelon form over a 32-bit prime field F_p
 * (uint32 storage, 2 <= p < 2^32; the tensor-core schedule for p < 2^31, a CUDA-core Montgomery schedule for
 * 2^31 <= p < 2^32; uint64 storage for odd p < 2^63), canonical null-space basis, an fp64
 * partial-pivot solve and the floating-point row reduction with a threshold.
 * Citations "PAPER.md:<line>" refer to the paper text this library was written from.
 *
 * Conventions (all entry points)
 *   - extern "C", plain pointers and sizes; no exceptions cross the boundary.
 *   - Every function returns a linac_status (int).  Outputs are defined only on LINAC_OK,
 *     except where a function documents otherwise.
 *   - "device" pointers must be device memory of the CURRENT CUDA device (compute capability
 *     10.x; anything else -> LINAC_ERR_UNSUPPORTED_DEVICE: there is no fallback path).
 *     "host" pointers are ordinary host memory.
 *   - Ownership: the library never frees or keeps caller memory.  Matrices, K and the optional
 *     workspace are caller-allocated.  `stream` is the caller's CUDA stream (cudaStream_t passed
 *     as void*; NULL = default stream).  Calls enqueue their work on `stream` and SYNCHRONISE it
 *     before returning (rank / pivots are host outputs).
 *   - Matrices are row-major with a leading dimension in ELEMENTS (ld >= cols).  Columns
 *     cols..ld-1 are never read as data and never written (the paper pads rows the same way,
 *     PAPER.md:227).
 *   - Workspace: if linac_set_workspace() gave the library a buffer at least as large as the
 *     *_workspace() query, it is used and the call allocates NO device memory; otherwise the library
 *     allocates (and caches) its own with cudaMalloc and linac_release() frees it.
 *   - Re-entrancy: everything a call mutates -- the workspace binding, the statistics, the error text, the
 *     host mailbox the strip kernels write to, the constant-memory slot that holds the field -- belongs to
 *     the calling HOST THREAD.  Calls issued from different host threads on different streams (each thread
 *     with its own workspace) run independently, with different matrices and different moduli; calls from
 *     one thread are sequential by construction (every call synchronises its stream before returning).
 *     linac_set_workspace / linac_release / linac_get_last_stats / linac_last_cuda_error act on the calling
 *     thread's state.  linac_set_option is process-wide: set options while no call is in flight.  At most
 *     64 host threads may be inside the library at once (LINAC_ERR_INTERNAL beyond that).
 */
#ifndef LINAC_H_
#define LINAC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    LINAC_OK = 0,
    LINAC_ERR_INVALID_ARG = 1,        /* null matrix with non-empty shape, negative size, ld < cols, cols >= 2^31 */
    LINAC_ERR_BAD_MODULUS = 2,        /* p outside the entry point's range, or p composite (deterministic Miller-Rabin on the host) */
    LINAC_ERR_WORKSPACE = 3,          /* workspace allocation failed */
    LINAC_ERR_CUDA = 4,               /* a CUDA call failed; linac_last_cuda_error() has the text */
    LINAC_ERR_SINGULAR = 5,           /* fp64: pivot with |pivot| <= tol */
    LINAC_ERR_BUFFER_TOO_SMALL = 6,   /* K buffer has fewer columns than the nullity */
    LINAC_ERR_UNSUPPORTED_DEVICE = 7, /* current device is not sm_100 class */
    LINAC_ERR_INTERNAL = 8,           /* an internal consistency check failed (a bug; never a data property) */
    LINAC_ERR_TOO_LARGE = 9           /* linac_gemm_sub_u32_static: the problem needs more than LINAC_STATIC_SCRATCH_BYTES of scratch */
} linac_status;

/* Static strings; never NULL. */
const char *linac_status_string(int status);
const char *linac_last_cuda_error(void);
/* major*10000 + minor*100 + patch */
int linac_version(void);

/* ---- workspace ------------------------------------------------------------------------- */
/* Bytes of device workspace linac_rref_u32 / linac_nullspace_u32 want for this shape (host out). */
int linac_rref_u32_workspace(int64_t rows, int64_t cols, size_t *bytes);
/* Bytes of device workspace linac_solve_f64 wants. */
int linac_solve_f64_workspace(int64_t n, int64_t nrhs, size_t *bytes);
/* Hand the library a device buffer to use as workspace (NULL, 0 to take it back).  The buffer
 * stays the caller's; it must outlive the calls that use it. */
int linac_set_workspace(void *dev_ptr, size_t bytes);
/* Free library-owned workspace and cached state (idempotent). */
int linac_release(void);

/* ---- F_p: reduced row-echelon form ------------------------------------------------------- */
/*
 * linac_rref_u32 -- the operation of cuda_row_reduce(matrix, field_characteristic=p)
 * (PAPER.md:147-155): in place, dA (DEVICE, rows x cols, ld) becomes THE reduced row-echelon
 * form of A over F_p: non-zero rows first, each with leading entry 1, pivot columns strictly
 * increasing, a pivot the only non-zero of its column, zero rows at the bottom,
 * entries canonical in [0,p).  Row permutations only (partial pivoting); any shape
 * (PAPER.md:73, 239).  Input entries >= p are first reduced mod p.
 *   rank            HOST out: number of non-zero rows.
 *   pivot_cols_out  HOST out, capacity min(rows, cols) int32, ascending; may be NULL.
 * rows == 0 or cols == 0 is legal: rank 0, nothing touched.
 * The schedule is NOT the paper's per-column kernel sequence: it is a blocked
 * right-looking elimination (panel factorisation + Schur update A22 -= L21.U12 mod p) followed by
 * back-elimination of the free columns; the result is identical because the RREF is unique.
 */
int linac_rref_u32(uint32_t *dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p, void *stream,
                   int64_t *rank, int32_t *pivot_cols_out);

/*
 * Moduli: linac_rref_u32 (and linac_nullspace_u32 / linac_solve_u32 / linac_rank_factor_u32, which call it) accepts
 * every prime 2 <= p <= 2^32 - 5 ("uint32 is used for p <= 2^32 - 1").  For p < 2^31 the blocked
 * tensor-core schedule above runs; for 2^31 <= p < 2^32 the residues no longer fit four 8-bit limbs with a spare
 * sign bit, and the call runs the CUDA-core Montgomery schedule of fp_wide.cu (blocked Gauss-Jordan, 32-column
 * panels, no host synchronisation inside the loop) -- same result, same conventions.
 *
 * linac_rref_u64 -- the 64-bit backend of PAPER.md:163 ("uint64 for [larger p]"; the upper bound is lost in the
 * extraction: this library takes odd primes 3 <= p < 2^63, reading Q18).  dA is DEVICE uint64, row-major;
 * everything else as linac_rref_u32.  LINAC_ERR_BAD_MODULUS for p = 2, p >= 2^63 or composite p.
 */
int linac_rref_u64_workspace(int64_t rows, int64_t cols, size_t *bytes);
int linac_rref_u64(uint64_t *dA, int64_t rows, int64_t cols, int64_t ld, uint64_t p, void *stream, int64_t *rank,
                   int32_t *pivot_cols_out);

/* ---- F_p: canonical null-space basis ------------------------------------------------------- */
/*
 * linac_nullspace_u32 -- reduces dA in place exactly as linac_rref_u32, then writes the canonical
 * kernel basis of PAPER.md:403-415 (eq. 8-9) to dK (DEVICE, row-major, cols x nullity, ldk):
 * with free (non-pivot) columns f_0 < ... < f_{d-1}, d = nullity = cols - rank, column t has
 *   K[f_t, t] = p - 1 ("fixes their coefficients to minus the identity"),
 *   K[c_k, t] = R[k, f_t] for each pivot row k with pivot column c_k,   0 elsewhere,
 * so that A.K = 0 mod p (eq. 9).
 *   nullity          HOST out, always set when the reduction succeeded.
 *   k_capacity_cols  columns available in dK.  If < nullity: returns LINAC_ERR_BUFFER_TOO_SMALL,
 *                    nullity, rank and pivots are valid, dA holds the RREF, dK is untouched; the
 *                    caller may then call linac_nullspace_from_rref_u32.
 * dK may be NULL iff k_capacity_cols == 0.
 */
int linac_nullspace_u32(uint32_t *dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p, void *stream,
                        int64_t *rank, int32_t *pivot_cols_out, uint32_t *dK, int64_t ldk,
                        int64_t k_capacity_cols, int64_t *nullity);

/* Kernel basis from an RREF already on the device.  pivot_cols: HOST, `rank` ascending entries. */
int linac_nullspace_from_rref_u32(const uint32_t *dR, int64_t rows, int64_t cols, int64_t ld, uint32_t p,
                                  int64_t rank, const int32_t *pivot_cols, uint32_t *dK, int64_t ldk,
                                  void *stream);

/* ---- F_p: linear systems (eq. 10-14) ------------------ */
/*
 * linac_solve_u32 -- solves A X = B over F_p by row reducing the augmented matrix M = (A | B) (eq. 11).
 *   dM   DEVICE rows x (cols + nrhs) row-major (ld >= cols + nrhs): (A | B) on entry, the RREF of M on return.
 *   dX   DEVICE cols x nrhs (ldx >= nrhs), out: for every CONSISTENT right-hand side the particular solution with
 *        the free variables set to zero; the columns of inconsistent right-hand sides are zero.
 *   rank_a          HOST out: rank of A (number of pivot columns < cols).
 *   pivot_cols_out  HOST out, capacity min(rows, cols + nrhs) int32: pivot columns of the RREF of M; may be NULL.
 *   consistent      HOST out, nrhs bytes: 1 iff rank(A) = rank(A | b_j) (eq. 13).  The right-hand sides are reduced
 *        together, so b_j counts as consistent iff its column is not a pivot column AND vanishes on the rows whose
 *        pivots lie in the augmented block (such a row is the (0 ... 0 | 1) of eq. 14 for an earlier right-hand side).
 * rows, cols or nrhs equal to 0 are legal.  Same conventions and errors as linac_rref_u32.
 */
int linac_solve_u32(uint32_t *dM, int64_t rows, int64_t cols, int64_t nrhs, int64_t ld, uint32_t p, void *stream,
                    int64_t *rank_a, int32_t *pivot_cols_out, uint8_t *consistent, uint32_t *dX, int64_t ldx);

/* ---- F_p: rank factorisation (eq. 7) ----------------- */
/*
 * linac_rank_factor_u32 -- A = C.R over F_p with R the non-zero rows of the RREF of A ("drop_bottom_zero_rows")
 * and C = A[:, J], J the pivot columns (a basis of the column space taken from A itself).
 *   dA   DEVICE rows x cols (lda >= cols), const: A is left untouched.
 *   dR   DEVICE rows x cols (ldr >= cols), out: the whole RREF of A (it is also the work buffer); R is its
 *        first `rank` rows, the rest are zero rows.
 *   dC   DEVICE rows x min(rows, cols) (ldc >= min(rows, cols)), out: columns [0, rank) are written, canonical
 *        in [0,p); the remaining columns are not touched.
 *   rank, pivot_cols_out  as in linac_rref_u32 (rank is required).
 * rows == 0 or cols == 0 is legal (rank 0).  Same errors as linac_rref_u32.  dA, dR, dC must not overlap.
 */
int linac_rank_factor_u32(const uint32_t *dA, int64_t rows, int64_t cols, int64_t lda, uint32_t p, void *stream,
                          uint32_t *dR, int64_t ldr, uint32_t *dC, int64_t ldc, int64_t *rank,
                          int32_t *pivot_cols_out);

/* ---- F_p: building the matrix on the device -- */
/*
 * linac_load_matrix_u32 -- the operation of cuda_load_matrix: every column is a monomial in the "basis
 * variables", evaluated at one sampling point per row,
 *     A[r][c] = prod_{t < d} bases[r][ lindices[c][t] ]   (mod p).
 *   dA        DEVICE out, n_rows x n_cols row-major (ld >= n_cols): exactly what linac_rref_u32 consumes, so the
 *             host -> device copy of A that the paper keeps disappears.
 *   dBases    DEVICE n_rows x n_basis uint32 (ldb >= n_basis); entries >= p are reduced mod p.
 *   dLindices DEVICE n_cols x d int32, row-major, contiguous.  Reading (the paper's footnote on monomials of lower
 *             degree is lost in the extraction): an index outside [0, n_basis) stands for "no factor" (1), so -1 pads
 *             monomials with fewer than d factors; d = 0 gives the all-ones matrix.
 * Pure streaming kernel (4 B written per element); synchronises `stream` before returning.
 */
int linac_load_matrix_u32(uint32_t *dA, int64_t n_rows, int64_t n_cols, int64_t ld, const uint32_t *dBases,
                          int64_t n_basis, int64_t ldb, const int32_t *dLindices, int64_t d, uint32_t p, void *stream);

/* ---- F_p: the Schur-update primitive on its own (S5; exposed for measurement and tests) ------ */
/*
 * linac_gemm_sub_u32 -- C <- C - A.B (mod p), the blocked form of the paper's row update
 * "row_k -= head_k * pivot_row" for K pivots at once.  All DEVICE, row-major:
 * C is M x N (ldc), A is M x K (lda), B is K x N (ldb); entries must already be in [0,p).
 * path: 0 = automatic choice, 1 = CUDA-core kernel (IMAD.WIDE + delayed reduction),
 *       2 = tensor-core kernel (tcgen05 int8 limb planes; LINAC_ERR_INVALID_ARG if the shape is
 *       not supported by it).  Synchronises `stream` before returning.
 */
int linac_gemm_sub_u32(uint32_t *dC, int64_t ldc, const uint32_t *dA, int64_t lda, const uint32_t *dB, int64_t ldb,
                       int64_t M, int64_t N, int64_t K, uint32_t p, int path, void *stream);

/*
 * linac_gemm_sub_u32_static -- the same update, C <- C - A.B (mod p), for callers that may not
 * allocate device memory (a stream under CUDA graph capture, a serving loop, a harness that forbids cudaMalloc).
 * Arguments and layout as linac_gemm_sub_u32 (all DEVICE, row-major, entries in [0,p), p prime < 2^31); the path is
 * the automatic one (tensor kernels where the shape allows, else the CUDA-core kernel).
 *   - Allocates nothing: no cudaMalloc / cudaFree, no events, no workspace.  The limb-plane scratch of the tensor
 *     kernels lives in a static device array of LINAC_STATIC_SCRATCH_BYTES inside the library (held by every GPU
 *     that loads the library until the process exits).
 *   - Limit: 4 (M + N) Kc + 4096 <= LINAC_STATIC_SCRATCH_BYTES, Kc = K rounded up to a multiple of 128 (K <= 8192;
 *     equal chunks of at most 8192 above), e.g. M = N = 4096 with K <= 1024, or M = N = 16384 with K <= 256.
 *     Beyond it: LINAC_ERR_TOO_LARGE, nothing launched, C untouched.
 *   - Asynchronous: the kernels are enqueued on `stream`, which is NOT synchronised; errors of the kernels
 *     themselves surface at the caller's next synchronisation.  linac_get_last_stats is not updated with times.
 *   - Every call on a device shares the one array.  Nothing in it has to start at zero (each call rewrites all it
 *     reads), but two calls that OVERLAP on the GPU -- different streams or host threads on the same device --
 *     race on it: serialise them (one stream, or events).
 */
#define LINAC_STATIC_SCRATCH_BYTES ((size_t)32 << 20)
int linac_gemm_sub_u32_static(uint32_t *dC, int64_t ldc, const uint32_t *dA, int64_t lda, const uint32_t *dB,
                              int64_t ldb, int64_t M, int64_t N, int64_t K, uint32_t p, void *stream);

/* ---- fp64: partial-pivot solve ------------------------------------------------------------- */
/*
 * linac_solve_f64 -- solves A X = B (eq. 10-12) in floating point:
 * row equilibration s_r = max_c |A[r,c]|, A[r,:] /= s_r, B[r,:] /= s_r (CudaSetRowScales /
 * CudaRescaleRows), then Gaussian elimination with partial pivoting on the
 * column maximum and triangular solves for the right-hand sides.
 *   dA  DEVICE n x n (lda), overwritten by the factors.   dB  DEVICE n x nrhs (ldb), overwritten by X.
 *   tol threshold below which a pivot of the row-scaled matrix counts as zero;
 *       tol < 0 selects n * 2^-52.
 *   info HOST out: 0, or the 1-based column of the first pivot with |pivot| <= tol
 *       (then the return value is LINAC_ERR_SINGULAR and dA/dB are undefined).
 */
int linac_solve_f64(double *dA, int64_t n, int64_t lda, double *dB, int64_t nrhs, int64_t ldb, double tol,
                    void *stream, int64_t *info);

/* ---- floating point: row reduction with a threshold -------- */
/*
 * linac_rref_f64 -- the operation of cuda_row_reduce(matrix, field_characteristic=0) on a real matrix:
 * in place, dA (DEVICE float64, rows x cols, ld) becomes its reduced row-echelon form, computed as the paper does:
 * every row is first divided by its largest |entry| (CudaSetRowScales / CudaRescaleRows); then column
 * by column the pivot is the largest |entry| among the rows left (partial pivoting), and a column
 * whose pivot has |pivot| <= tol yields no pivot (CudaCompareHeadToTolerance, "explicitly control
 * numerical thresholds").  Any shape; rank-deficient input is the point of the function.
 *   tol   threshold on the row-scaled matrix; tol < 0 selects max(rows, cols) * 2^-52.
 *   rank, pivot_cols_out   HOST out, as in linac_rref_u32.
 * On return the pivots are exactly 1, pivot columns are exact unit vectors, and what the thresholds declared zero
 * is written as zero: rows >= rank, and the entries of a pivot row left of its pivot (reading Q19).
 * The schedule is a blocked Gauss-Jordan over 32-column panels (pivot search kernel + DMMA update of all other rows).
 */
int linac_rref_f64_workspace(int64_t rows, int64_t cols, size_t *bytes);
int linac_rref_f64(double *dA, int64_t rows, int64_t cols, int64_t ld, double tol, void *stream, int64_t *rank,
                   int32_t *pivot_cols_out);

/* ---- complex128 (the reduction is instantiated for complex128 as well) ---------------------------
 * linac_rref_c128: the same reduction with a threshold on a rows x cols matrix of complex doubles (interleaved re, im:
 * C's double _Complex / numpy complex128 / torch.complex128; dA 16-byte aligned, ld in complex elements), in place;
 * rank, pivot columns, tol and the written-as-zero convention as linac_rref_f64.  Rows are rescaled by their largest
 * real or imaginary part (reading Q21).
 * Computed as the real reduction of the 2 x 2 block embedding  x + iy -> [[x, -y], [y, x]]  (a ring homomorphism, and the
 * reduced echelon form of a row space is unique, so RREF_real(E(A)) = E(RREF_complex(A))): the fp64 tensor-pipe
 * kernels serve unchanged, at twice the flops and memory of a native complex elimination.  The workspace holds the
 * 2 rows x 2 cols real matrix (32 bytes per complex entry) plus linac_rref_f64's own for that shape.
 * LINAC_ERR_SINGULAR if the threshold fell between the two real columns of one complex column (a pivot within a factor
 * sqrt(2) of tol: choose another tol); dA is then unchanged.
 */
int linac_rref_c128_workspace(int64_t rows, int64_t cols, size_t *bytes);
int linac_rref_c128(void *dA, int64_t rows, int64_t cols, int64_t ld, double tol, void *stream, int64_t *rank,
                    int32_t *pivot_cols_out);

/* ---- instrumentation (host-side counters of the LAST F_p call; for tests and bench.py) ------ */
typedef struct {
    int64_t kernel_launches;     /* kernels this library launched                                 */
    int64_t host_syncs;          /* stream synchronisations inside the call                       */
    int64_t panels;              /* base panels factored                                          */
    int64_t row_swaps;           /* row exchanges performed                                       */
    int64_t update_macs;         /* field multiply-accumulates executed by Schur/TRSM updates     */
    int64_t residual_nonzero;    /* internal check: must be 0                                     */
    int64_t tc_launches;         /* Schur updates that ran on the tensor-core (tcgen05) path      */
    double  ms_update;           /* device ms spent in the Schur-update (GEMM) kernels, if timed  */
    double  ms_total;            /* device ms of the whole call, if timed                         */
    double  ms_strip;            /* device ms in the cooperative strip kernels (S1-S4), if timed   */
    double  ms_trsm;             /* device ms in the triangular-solve leaf kernels, if timed       */
    double  ms_update_top;       /* device ms of the largest single Schur update (incl. its limb split), if timed */
    int64_t top_m, top_n, top_k; /* its shape                                                      */
    double  ms_overlap;          /* timing = 2: device ms during which a strip kernel (look-ahead, second stream) and a
                                    Schur-update kernel were running at the same time                               */
    int64_t lookahead_strips;    /* strips whose kernel was launched beside the previous strip's bulk update        */
    int64_t winv_solves;         /* row-block solves done as one product with the strip's 128 x 128 operator W       */
} linac_stats;
int linac_get_last_stats(linac_stats *out);
/* Timeline of the calling thread's last linac_rref_u32 call made with option "timing" = 2: one record per kernel launch
 * of the three classes, in launch order, times in ms from the start of the call (CUDA events around each launch, read
 * after the call's final synchronisation).  cls: 0 = Schur update, 1 = strip kernel, 2 = row-block solve (W kernel, W
 * product, chain kernel); stream: 0 = the call's stream, 1 = the look-ahead sweep's second stream; m, n, k: shape of an
 * update (0 otherwise).  Writes at most `capacity` records to `out` (may be NULL with capacity 0) and the number
 * available to *count.  What it is for: seeing which launches overlap (profiles/r02_lookahead.md). */
typedef struct {
    int32_t cls, stream;
    int64_t m, n, k;
    float t0_ms, t1_ms;
} linac_mark;
int linac_get_last_marks(linac_mark *out, int64_t capacity, int64_t *count);
/* Tunables, mainly for A/B measurements: name in {"gemm_path" (0 auto, 1 CUDA-core, 2 tensor), "timing" (0, 1 = un-fused schedule with a
 * host sync per launch, 2 = event pairs around every launch of the production schedule), "lookahead" (0/1: factor strip s+1 beside the bulk
 * of strip s's Schur update), "trsm_winv" (0/1: row-block solve of a strip with 128 pivots as one tensor-core product with its explicit operator W),
 * "trsm_split" (0/1: under look-ahead that product runs on the next strip's columns first and on the rest beside the narrow update), "la_ctas" (SMs of the look-ahead strip kernel, 0 = cost model), "tc_min_k", "tc_min_mn",
 * "strip_width" (columns per cooperative strip kernel: 32..256, multiple of 32), "flat_cols" (nodes up to this many
 * columns are swept flat, wider ones recurse), "flat_group" (strips per Schur update of the flat sweep), "tc_panel" (0/1), "tc_panel_deep" (0/1: K <= 128 updates with one A stage and seven C-tile buffers), "f64_mma" (fp64 trailing update: 1 = DMMA tensor pipe with 128 x 64 tiles, 2 = DMMA with 128 x 128 tiles, 0 = DFMA),
 * "f64_strip" (fp64 factorisation: columns per strip of the flat top-level sweep, multiple of 32, 0 = pure recursion),
 * "f64_panel_threads" (256/512/1024) and "f64_panel_grid" (0 = one CTA per SM) of the fp64 panel kernel, "f64_panel_tags" (1 = tagged
 * candidate records instead of a grid barrier per column), "f64_panel_cluster" (CTAs of the cluster + DSMEM panel variant, 0 = off) with
 * "f64_cluster_rows" (rows per CTA up to which it is used),
 * "f64_rref_strip" (linac_rref_f64: columns per strip, 32..128 in steps of 32; the columns right of a strip are updated once per strip
 * with K = that width, 32 = once per panel),
 * "f64_rhs_inv" (fp64 substitution on the right-hand sides: 1 = blocked, with inverted 128 x 128 diagonal blocks, 0 = recursive leaf solves)}.
 * Returns LINAC_ERR_INVALID_ARG for unknown names / out-of-range values. */
int linac_set_option(const char *name, int64_t value);

/* ---- measured peaks of the pipes the rooflines are quoted against ("Measure, do not assume") ---- */
/*
 * linac_measure_peak -- runs a microbenchmark that issues nothing but one instruction class from on-chip operands:
 *   "tc_i8_n256", "tc_i8_n128"  tcgen05.mma.cta_group::1.kind::i8, M = 128, N = 256 / 128, K = 32 -> *value in TOP/s
 *                               (2 ops per u8 multiply-accumulate)
 *   "dmma"                      mma.sync.m8n8k4.f64 (DMMA.8x8x4)                                  -> TFLOP/s
 *   "imad_wide"                 32 x 32 -> 64-bit multiply + 64-bit accumulate, new operands every time -> T multiply-adds/s (thread-level)
 *   "hbm_copy", "hbm_read"      16-byte grid-stride copy / read over `scratch` (DEVICE, >= 32 MiB; use >= 1 GiB) -> GB/s
 *                               (copy counts read + written bytes)
 * ms_target: approximate duration of the timed launch (<= 0: 2 ms; a few hundred ms shows the power-capped rate).
 * sm_mhz (HOST out, may be NULL): the SM clock the timed launch actually ran at (%clock64 against %globaltimer).
 * Synchronises `stream`.  scratch may be NULL for the compute kinds.
 */
int linac_measure_peak(const char *what, double ms_target, void *scratch, size_t scratch_bytes, void *stream,
                       double *value, double *sm_mhz);

#ifdef __cplusplus
}
#endif
#endif /* LINAC_H_ */
