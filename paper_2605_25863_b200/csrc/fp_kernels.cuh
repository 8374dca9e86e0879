// fp_kernels.cuh -- the small kernels of the F_p path (everything except the Schur-update GEMM).
//
// Storage convention of the forward phase (in place).  Base panel b covers columns [32b, 32b+w).
// Its pivots (global pivot indices t in [pstart[b], pstart[b+1])) live in ROWS t after the panel's
// row exchanges; pivcols[t] is the pivot column.  With P the pivot rows and Jp the pivot columns of
// the panel, T_b = (A[P, Jp])^{-1} is kept in a side buffer; the reduced pivot rows are U = T_b A[P, :]
// (identity on Jp).  Because U is the identity on the panel's pivot columns, the multiplier of any
// other row k against reduced pivot row t is simply the stored entry A[k, pivcols[t]] -- the panel
// columns of the rows below are never rewritten:
//   (row k >= pstart[b+1], col pivcols[t])   raw value = multiplier L[k][t]
//   (row t, col c right of the panel)        U[t][c] once the enclosing recursion node has applied T
//   (row t of panel b, free column of b)     U[t][c]   (written by panel_finish_kernel when r < w)
//   (row k >= pstart[b+1], free column of b) mathematically 0; storage holds garbage that the
//                                            gather / finalise kernels replace by 0
// The finalise kernel overwrites every pivot column with a unit vector and the garbage with zeros,
// which makes the result the RREF of PAPER.md:153.
#pragma once
#include <climits>

#include "linac_internal.h"

namespace linac {

// ------------------------------------------------------------------------------------------
// S0 ingest: a <- a mod p over the rows x cols window (reading Q5: entries >= p are reduced).
__global__ void reduce_mod_p_kernel(uint32_t* __restrict__ A, int64_t rows, int64_t cols, int64_t ld, uint32_t p) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cols) return;
    for (int64_t r = blockIdx.y; r < rows; r += gridDim.y) {
        uint32_t v = A[r * ld + c];
        if (v >= p) A[r * ld + c] = v % p;
    }
}

// The same for 16-byte aligned rows (base and ld): four columns per thread, 128-bit loads, a store only where a
// residue changed.  cols4 = cols / 4; the caller runs the scalar kernel on the remaining cols % 4 columns.
__global__ void reduce_mod_p_vec4_kernel(uint32_t* __restrict__ A, int64_t rows, int64_t cols4, int64_t ld, uint32_t p) {
    const int64_t c4 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c4 >= cols4) return;
    for (int64_t r = blockIdx.y; r < rows; r += gridDim.y) {
        uint4* q = reinterpret_cast<uint4*>(A + r * ld) + c4;
        uint4 v = *q;
        if (v.x >= p || v.y >= p || v.z >= p || v.w >= p) {
            v.x %= p; v.y %= p; v.z %= p; v.w %= p;
            *q = v;
        }
    }
}

// ------------------------------------------------------------------------------------------
// Free-column gather / scatter for the back-elimination workspace: F[k][t] = A[k][freecols[t]] for
// k below the column's threshold row (the number of pivots found up to and including the column's
// panel); rows at or beyond it are mathematically zero there (storage may hold garbage).
__global__ void gather_cols_kernel(const uint32_t* __restrict__ A, int64_t ld, int64_t nrows,
                                   const int32_t* __restrict__ colidx, const int32_t* __restrict__ thresh, int64_t ncols,
                                   uint32_t* __restrict__ F, int64_t ldf) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ncols) return;
    const int64_t c = colidx[t];
    const int64_t th = thresh[t];
    for (int64_t k = blockIdx.y; k < nrows; k += gridDim.y) F[k * ldf + t] = k < th ? A[k * ld + c] : 0u;
}
__global__ void scatter_cols_kernel(uint32_t* __restrict__ A, int64_t ld, int64_t nrows,
                                    const int32_t* __restrict__ colidx, int64_t ncols, const uint32_t* __restrict__ F,
                                    int64_t ldf) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ncols) return;
    const int64_t c = colidx[t];
    for (int64_t k = blockIdx.y; k < nrows; k += gridDim.y) A[k * ld + c] = F[k * ldf + t];
}

// S7 finalise.  colinfo[c] >= 0: column c is the pivot column of pivot t = colinfo[c]; it becomes the
// unit vector e_t over ALL rows (removes multipliers and raw pivot blocks).  colinfo[c] < 0: free
// column whose entries in rows >= -(colinfo[c]+1) become 0.  Rows >= rank end up zero.
__global__ void finalize_kernel(uint32_t* __restrict__ A, int64_t ld, int64_t rows, int64_t cols,
                                const int32_t* __restrict__ colinfo) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cols) return;
    const int32_t ci = colinfo[c];
    if (ci >= 0) {
        for (int64_t k = blockIdx.y; k < rows; k += gridDim.y) A[k * ld + c] = (k == ci) ? 1u : 0u;
    } else {
        const int64_t th = -((int64_t)ci + 1);
        for (int64_t k = th + blockIdx.y; k < rows; k += gridDim.y) A[k * ld + c] = 0u;
    }
}

// ------------------------------------------------------------------------------------------
// S8 null space.  colmap[c] = pivot index of column c, or -(t+1) if c is the
// t-th free column.  K is cols x d: K[c][t] = R[colmap[c]][free[t]] for pivot columns c,
// p-1 at (free[t], t), 0 elsewhere.
__global__ void nullspace_kernel(const uint32_t* __restrict__ R, int64_t ld, int64_t cols, int64_t d,
                                 const int32_t* __restrict__ colmap, const int32_t* __restrict__ freecols,
                                 uint32_t* __restrict__ K, int64_t ldk, uint32_t p) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= d) return;
    const int64_t fc = freecols[t];
    for (int64_t c = blockIdx.y; c < cols; c += gridDim.y) {
        const int32_t m = colmap[c];
        uint32_t v;
        if (m >= 0) v = R[(int64_t)m * ld + fc];
        else v = (-(int64_t)m - 1 == t) ? p - 1 : 0u;
        K[c * ldk + t] = v;
    }
}

// ------------------------------------------------------------------------------------------
// Solutions of A X = B from the RREF R of (A | B).  Rows [0, rank_a) have their pivots in
// A's columns (colrow[c] = that row, or -1 for a free column c), rows [rank_a, rank_m) in the augmented block.
// One thread per right-hand side j: consistent iff column cols+j vanishes on rows [rank_a, rank_m) (this
// includes "is not a pivot column"); then X[c][j] = R[colrow[c]][cols+j] for pivot columns, 0 for free ones.
__global__ void solve_extract_kernel(const uint32_t* __restrict__ R, int64_t ld, int64_t cols, int64_t nrhs,
                                     int64_t rank_a, int64_t rank_m, const int32_t* __restrict__ colrow,
                                     uint32_t* __restrict__ X, int64_t ldx, uint8_t* __restrict__ consistent) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nrhs) return;
    bool ok = true;
    for (int64_t k = rank_a; k < rank_m; ++k) ok = ok && R[k * ld + cols + j] == 0u;
    if (blockIdx.y == 0) consistent[j] = ok ? 1 : 0;
    for (int64_t c = blockIdx.y; c < cols; c += gridDim.y) {
        const int32_t k = colrow[c];
        X[c * ldx + j] = (ok && k >= 0) ? R[(int64_t)k * ld + cols + j] : 0u;
    }
}

// ------------------------------------------------------------------------------------------
// Column basis of a rank factorisation A = C.R (eq. 7): C = A[:, J] with J the pivot columns,
// entries reduced to [0,p).  Thread per pivot (J ascending, so a warp's reads fall in few sectors), grid.y over rows.
__global__ void gather_columns_kernel(const uint32_t* __restrict__ A, int64_t lda, int64_t rows, int64_t rank,
                                      const int32_t* __restrict__ piv, uint32_t* __restrict__ Cm, int64_t ldc, uint32_t p) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= rank) return;
    const int64_t c = piv[k];
    for (int64_t r = blockIdx.y; r < rows; r += gridDim.y) {
        const uint32_t v = A[r * lda + c];
        Cm[r * ldc + k] = v >= p ? v % p : v;
    }
}

// ------------------------------------------------------------------------------------------
// cuda_load_matrix: A[r][c] = prod_t bases[r][lind[c][t]] mod p.  A CTA owns 256 columns
// (their index lists staged once in shared memory) and walks over its share of the rows; the row of basis values is
// staged per row, the 256 products are written as one coalesced row segment.  Bound: the 4 B written per element.
constexpr int LM_COLS = 256;
constexpr int LM_ROWS = 8;           // rows per pass: the index tile is read once per factor for all of them
// MONT: the staged basis values are put in Montgomery form (one Barrett product each, shared by 256 columns), every
// factor then costs a 4-instruction Montgomery product instead of a 14-instruction Barrett one (p odd).
template <bool MONT>
__global__ void __launch_bounds__(LM_COLS) load_matrix_kernel(uint32_t* __restrict__ A, int64_t n_rows, int64_t n_cols,
                                                              int64_t ld, const uint32_t* __restrict__ bases, int64_t n_basis,
                                                              int64_t ldb, const int32_t* __restrict__ lind, int d,
                                                              int basis_cap, ModP f) {
    extern __shared__ __align__(16) unsigned char lm_smem[];
    int32_t* L = reinterpret_cast<int32_t*>(lm_smem);                          // index tile, stored [t][col]
    uint32_t* Bv = reinterpret_cast<uint32_t*>(lm_smem + (size_t)LM_COLS * d * 4);   // [LM_ROWS][basis_cap]
    const int tid = threadIdx.x;
    const int64_t c0 = (int64_t)blockIdx.x * LM_COLS, c = c0 + tid;
    for (int e = tid; e < LM_COLS * d; e += LM_COLS) {                        // coalesced read of the index tile
        const int cl = e / d, t = e - cl * d;
        const int32_t v = c0 + cl < n_cols ? lind[(c0 + cl) * d + t] : -1;
        L[t * LM_COLS + cl] = (v >= 0 && v < n_basis) ? v : -1;
    }
    const bool staged = n_basis <= basis_cap;
    auto prep = [&](uint32_t v) {                                              // canonical residue, Montgomery form if MONT
        v = v >= f.p ? v % f.p : v;
        return MONT ? reduce64((uint64_t)v * f.c32, f) : v;
    };
    for (int64_t r0 = (int64_t)blockIdx.y * LM_ROWS; r0 < n_rows; r0 += (int64_t)gridDim.y * LM_ROWS) {
        const int nr = (int)min((int64_t)LM_ROWS, n_rows - r0);
        __syncthreads();
        if (staged)
            for (int rr = 0; rr < nr; ++rr)
                for (int bb = tid; bb < (int)n_basis; bb += LM_COLS)
                    Bv[(size_t)rr * basis_cap + bb] = prep(bases[(r0 + rr) * ldb + bb]);
        __syncthreads();
        if (c < n_cols) {
            uint32_t acc[LM_ROWS];
            const uint32_t one = MONT ? f.c32 % f.p : 1u % f.p;
#pragma unroll
            for (int rr = 0; rr < LM_ROWS; ++rr) acc[rr] = one;
            for (int t = 0; t < d; ++t) {
                const int32_t i = L[t * LM_COLS + tid];
                if (i < 0) continue;
#pragma unroll
                for (int rr = 0; rr < LM_ROWS; ++rr) {
                    if (rr < nr) {
                        const uint32_t v = staged ? Bv[(size_t)rr * basis_cap + i] : prep(bases[(r0 + rr) * ldb + i]);
                        acc[rr] = MONT ? mulredc(acc[rr], v, f) : mulmod(acc[rr], v, f);
                    }
                }
            }
#pragma unroll
            for (int rr = 0; rr < LM_ROWS; ++rr)
                if (rr < nr) A[(r0 + rr) * ld + c] = MONT ? redc(acc[rr], f) : acc[rr];
        }
    }
}

}  // namespace linac
