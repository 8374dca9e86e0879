// fp_kernels.cuh -- the small kernels of the F_p path (everything except the Schur-update GEMM).
//
// Storage convention of the forward phase (in place, LAPACK-like).  Pivot t (global pivot index)
// lives in ROW t and column pivcols[t].  After a panel is factored:
//   (row t, col pivcols[t])            holds d_t^{-1}  (d_t = the pivot value before normalisation;
//                                      the echelon row's leading 1 is implicit)
//   (row t, col c > pivcols[t])        holds E_t[c], the normalised echelon row
//   (row k > t, col pivcols[t])        holds the multiplier L[k][t]  (row_k = sum_t L[k][t] E_t)
//   (row k, non-pivot col c of a finished panel, k >= #pivots left of c) holds a true 0
// The finalise kernel overwrites every pivot column with a unit vector, which removes the L
// entries and the stored d^{-1} -- that is what makes the result the RREF of PAPER.md:153.
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

// ------------------------------------------------------------------------------------------
// S1 + S2 (decision part): pivot search for one base panel (columns [j0, j0+w), rows >= i0).
//
// One CTA.  Works on a shared-memory copy, so global memory still holds the original strip when
// it ends.  Rows are scanned in chunks of CH; each chunk is first reduced against the echelon rows
// found so far, then searched column by column for the FIRST row with a non-zero entry (warp
// ballot / atomicMin; for F_p any non-zero pivot will do).  Elimination inside the
// chunk is division-free (row_k <- d*row_k - h*row_q), so no modular inverse sits on the
// column-to-column dependency chain; the new pivot rows are normalised together at the end of
// the chunk, one warp per row, inverses computed in parallel.
// Stops as soon as w pivots are known; otherwise it has looked at every row, which is what
// proves that the remaining columns of the panel are free columns.
__global__ void __launch_bounds__(256) panel_pivots_kernel(const uint32_t* __restrict__ A, int64_t ld, int64_t rows,
                                                           int64_t i0, int64_t j0, int w, ModP f,
                                                           PanelInfo* __restrict__ info, uint32_t* __restrict__ Eout,
                                                           int32_t* __restrict__ pivcols_global) {
    __shared__ uint32_t X[CH][PW + 1];
    __shared__ uint32_t E[PW][PW + 1];     // normalised echelon rows, discovery order
    __shared__ int epc[PW];                // pivot column of E[t]
    __shared__ long long esrc[PW];         // source row (absolute) of E[t]
    __shared__ int urow[PW];               // chunk-local row that became pivot t (this chunk)
    __shared__ int ord[PW];                // E rows sorted by pivot column
    __shared__ int found[PW];
    __shared__ int any_nz;

    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    int r = 0;

    for (int64_t cs = i0; cs < rows && r < w; cs += CH) {
        const int nh = (int)min((int64_t)CH, rows - cs);
        if (tid < PW) found[tid] = INT_MAX;
        if (tid == 0) any_nz = 0;
        __syncthreads();
        // load + reduce against the current echelon rows (ascending pivot column)
        int nz = 0;
        for (int k = wq; k < CH; k += 8) {
            uint32_t s = 0;
            if (k < nh && lane < w) {
                s = A[(cs + k) * ld + j0 + lane];
                if (s >= f.p) s %= f.p;
            }
            for (int a = 0; a < r; ++a) {
                const int t = ord[a];
                const uint32_t l = __shfl_sync(0xffffffffu, s, epc[t]);
                if (l) s = submulmod(s, l, E[t][lane], f);
            }
            X[k][lane] = s;
            nz |= (s != 0);
        }
        if (__any_sync(0xffffffffu, nz) && lane == 0) any_nz = 1;
        __syncthreads();
        if (!any_nz) continue;          // the whole chunk lies in the span found so far

        const int r_start = r;
        unsigned usedmask = 0;          // bit t: my warp's row wq + 8t is already a pivot row
        for (int c = 0; c < w && r < w; ++c) {
            // lanes 0..7 test this warp's 8 rows
            if (lane < 8) {
                const int k = wq + 8 * lane;
                if (!((usedmask >> lane) & 1u) && X[k][c] != 0) atomicMin(&found[c], k);
            }
            __syncthreads();
            const int q = found[c];
            if (q == INT_MAX) continue;
            const uint32_t d = X[q][c];
            const uint32_t pv = X[q][lane];
            for (int t = 0; t < 8; ++t) {
                const int k = wq + 8 * t;
                if (k == q) { usedmask |= 1u << t; continue; }
                if ((usedmask >> t) & 1u) continue;
                const uint32_t h = X[k][c];
                if (h == 0) continue;
                // division-free: scales row k by d != 0, which changes neither its span nor its zeros
                X[k][lane] = submod(mulmod(d, X[k][lane], f), mulmod(h, pv, f), f);
            }
            if (tid == 0) { epc[r] = c; esrc[r] = cs + q; urow[r] = q; }
            ++r;
            __syncwarp();               // lanes 0..7 read what other lanes of this warp just wrote
        }
        __syncthreads();
        // normalise the new pivot rows (parallel inverses), one warp per row
        for (int t = r_start + wq; t < r; t += 8) {
            const int q = urow[t];
            const uint32_t dinv = invmod(X[q][epc[t]], f);
            E[t][lane] = mulmod(X[q][lane], dinv, f);
        }
        if (tid == 0) {                 // insertion sort of <= 32 pivot columns
            for (int t = r_start; t < r; ++t) {
                int a = t;
                while (a > 0 && epc[ord[a - 1]] > epc[t]) { ord[a] = ord[a - 1]; --a; }
                ord[a] = t;
            }
        }
        __syncthreads();
    }

    // outputs
    __syncthreads();
    for (int a = wq; a < r; a += 8) Eout[a * PW + lane] = E[ord[a]][lane];
    if (tid == 0) {
        info->r = r;
        info->residual = 0;
        // Row i0+a must receive source row esrc[ord[a]]: turn that into sequential exchanges.
        long long pos_of[PW];   // where the row that originally sat at i0+b is now (only b < r matter)
        for (int b = 0; b < r; ++b) pos_of[b] = i0 + b;
        int nsw = 0;
        for (int a = 0; a < r; ++a) {
            long long src = esrc[ord[a]];
            // current position of the original row `src`: it moved only if it was one of the top rows
            long long cur = src;
            if (src < i0 + r) cur = pos_of[src - i0];
            info->swp[a] = cur;
            info->pc[a] = epc[ord[a]];
            pivcols_global[i0 + a] = (int32_t)(j0 + epc[ord[a]]);
            if (cur != i0 + a) {
                ++nsw;
                // the row now at i0+a goes to `cur`; find which original top row that is
                for (int b = 0; b < r; ++b)
                    if (pos_of[b] == i0 + a) { pos_of[b] = cur; break; }
                if (src < i0 + r) pos_of[src - i0] = i0 + a;
            }
        }
        info->nswaps = nsw;
    }
}

// ------------------------------------------------------------------------------------------
// K5 CudaSwitchRows for a whole panel: the exchanges are applied to complete
// rows, one thread per column (so the sequence of exchanges needs no inter-thread ordering).
__global__ void apply_swaps_kernel(uint32_t* __restrict__ A, int64_t ld, int64_t cols, int64_t i0,
                                   const PanelInfo* __restrict__ info) {
    if (info->nswaps == 0) return;
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cols) return;
    const int r = info->r;
    for (int a = 0; a < r; ++a) {
        const int64_t s = info->swp[a];
        if (s != i0 + a) {
            uint32_t x = A[(i0 + a) * ld + c], y = A[s * ld + c];
            A[(i0 + a) * ld + c] = y;
            A[s * ld + c] = x;
        }
    }
}

// ------------------------------------------------------------------------------------------
// S2 + S3: with the panel's echelon rows E known, every row k >= i0 of the strip is rewritten in
// place from its ORIGINAL values: forward substitution against E gives the multipliers L[k][t]
// (stored at the pivot columns); pivot rows additionally get normalised (K7) and keep
// their echelon entries.  One warp per row, lane = panel column; rows are independent.
__global__ void __launch_bounds__(256) panel_apply_kernel(uint32_t* __restrict__ A, int64_t ld, int64_t rows, int64_t i0,
                                                          int64_t j0, int w, ModP f, PanelInfo* __restrict__ info,
                                                          const uint32_t* __restrict__ Eg) {
    __shared__ uint32_t E[PW][PW + 1];
    __shared__ int pc[PW];
    const int r = info->r;
    if (r == 0) return;
    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    for (int a = wq; a < r; a += 8) E[a][lane] = Eg[a * PW + lane];
    if (tid < r) pc[tid] = info->pc[tid];
    __syncthreads();
    unsigned pivmask = 0;                       // bit c: local column c is a pivot column
    for (int t = 0; t < r; ++t) pivmask |= 1u << pc[t];

    const int64_t k = i0 + (int64_t)blockIdx.x * 8 + wq;
    if (k >= rows) return;
    uint32_t s = 0;
    if (lane < w) {
        s = A[k * ld + j0 + lane];
        if (s >= f.p) s %= f.p;
    }
    const int64_t a = k - i0;
    const int steps = a < r ? (int)a : r;
    for (int t = 0; t < steps; ++t) {
        const uint32_t l = __shfl_sync(0xffffffffu, s, pc[t]);
        if (lane == pc[t]) s = l;                            // keep the multiplier where the zero would be
        else if (lane > pc[t] && l) s = submulmod(s, l, E[t][lane], f);
    }
    if (a < r) {
        // pivot row: what is left is d_a * E_a; normalise, store d_a^{-1} on the (implicit-1) pivot
        const int pa = pc[a];
        const uint32_t d = __shfl_sync(0xffffffffu, s, pa);
        const uint32_t dinv = d ? invmod(d, f) : 0;
        if (d == 0 && lane == 0) atomicAdd(&info->residual, 1);
        if (lane == pa) s = dinv;
        else if (lane > pa) s = mulmod(s, dinv, f);
        else if (!((pivmask >> lane) & 1u) && s != 0) atomicAdd(&info->residual, 1);
    } else {
        // a row below the pivots must have been reduced to zero on the non-pivot columns
        if (lane < w && !((pivmask >> lane) & 1u) && s != 0) atomicAdd(&info->residual, 1);
    }
    if (lane < w) A[k * ld + j0 + lane] = s;
}

// ------------------------------------------------------------------------------------------
// S4 row-block solve, base case: X <- L11^{-1} X for nb <= 32 pivots (global pivot indices
// t0..t0+nb), X = A[t0 : t0+nb, c0 : c0+ncols].  L11[a][b] = A[t0+a][pivcols[t0+b]] (b < a), the
// diagonal position holds d_a^{-1}.  One thread per column of X, the column kept in shared memory.
constexpr int TRSM_THREADS = 128;
__global__ void __launch_bounds__(TRSM_THREADS) trsm_lower_base_kernel(uint32_t* __restrict__ X, int64_t ldx,
                                                                       int64_t ncols, const uint32_t* __restrict__ A,
                                                                       int64_t lda, const int32_t* __restrict__ pivcols,
                                                                       int64_t t0, int nb, ModP f) {
    __shared__ uint32_t L[PW][PW + 1];
    __shared__ uint32_t Xs[PW][TRSM_THREADS];
    const int tid = threadIdx.x;
    for (int e = tid; e < nb * nb; e += TRSM_THREADS) {
        const int a = e / nb, b = e % nb;
        L[a][b] = b <= a ? A[(t0 + a) * lda + pivcols[t0 + b]] : 0;
    }
    const int64_t c = (int64_t)blockIdx.x * TRSM_THREADS + tid;
    const bool on = c < ncols;
    for (int a = 0; a < nb; ++a) Xs[a][tid] = on ? X[(int64_t)a * ldx + c] : 0;
    __syncthreads();
    if (!on) return;
    for (int a = 0; a < nb; ++a) {
        uint64_t acc = 0;
        for (int b = 0; b < a; ++b) {
            acc += (uint64_t)L[a][b] * Xs[b][tid];
            if (b & 1) acc = fold64(acc, f);
        }
        const uint32_t v = submod(Xs[a][tid], reduce64(acc, f), f);
        const uint32_t y = mulmod(v, L[a][a], f);
        Xs[a][tid] = y;
        X[(int64_t)a * ldx + c] = y;
    }
}

// S6 back-elimination, base case: X <- T^{-1} X, T unit upper triangular nb x nb with
// T[a][b] = A[t0+a][pivcols[t0+b]] for b > a (the echelon rows' entries above later pivots).
__global__ void __launch_bounds__(TRSM_THREADS) trsm_upper_base_kernel(uint32_t* __restrict__ X, int64_t ldx,
                                                                       int64_t ncols, const uint32_t* __restrict__ A,
                                                                       int64_t lda, const int32_t* __restrict__ pivcols,
                                                                       int64_t t0, int nb, ModP f) {
    __shared__ uint32_t T[PW][PW + 1];
    __shared__ uint32_t Xs[PW][TRSM_THREADS];
    const int tid = threadIdx.x;
    for (int e = tid; e < nb * nb; e += TRSM_THREADS) {
        const int a = e / nb, b = e % nb;
        T[a][b] = b > a ? A[(t0 + a) * lda + pivcols[t0 + b]] : 0;
    }
    const int64_t c = (int64_t)blockIdx.x * TRSM_THREADS + tid;
    const bool on = c < ncols;
    for (int a = 0; a < nb; ++a) Xs[a][tid] = on ? X[(int64_t)a * ldx + c] : 0;
    __syncthreads();
    if (!on) return;
    for (int a = nb - 2; a >= 0; --a) {
        uint64_t acc = 0;
        for (int b = a + 1; b < nb; ++b) {
            acc += (uint64_t)T[a][b] * Xs[b][tid];
            if ((b - a) % 2 == 0) acc = fold64(acc, f);
        }
        const uint32_t y = submod(Xs[a][tid], reduce64(acc, f), f);
        Xs[a][tid] = y;
        X[(int64_t)a * ldx + c] = y;
    }
}

// ------------------------------------------------------------------------------------------
// Free-column gather / scatter for the back-elimination workspace: F[k][t] = A[k][freecols[t]].
__global__ void gather_cols_kernel(const uint32_t* __restrict__ A, int64_t ld, int64_t nrows,
                                   const int32_t* __restrict__ colidx, int64_t ncols, uint32_t* __restrict__ F,
                                   int64_t ldf) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ncols) return;
    const int64_t c = colidx[t];
    for (int64_t k = blockIdx.y; k < nrows; k += gridDim.y) F[k * ldf + t] = A[k * ld + c];
}
__global__ void scatter_cols_kernel(uint32_t* __restrict__ A, int64_t ld, int64_t nrows,
                                    const int32_t* __restrict__ colidx, int64_t ncols, const uint32_t* __restrict__ F,
                                    int64_t ldf) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ncols) return;
    const int64_t c = colidx[t];
    for (int64_t k = blockIdx.y; k < nrows; k += gridDim.y) A[k * ld + c] = F[k * ldf + t];
}

// S7 finalise: every pivot column becomes a unit vector over ALL rows (removes the multipliers
// and the stored inverses); rows >= rank are zero rows.
__global__ void finalize_pivot_cols_kernel(uint32_t* __restrict__ A, int64_t ld, int64_t rows,
                                           const int32_t* __restrict__ pivcols, int64_t rank) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= rank) return;
    const int64_t c = pivcols[t];
    for (int64_t k = blockIdx.y; k < rows; k += gridDim.y) A[k * ld + c] = (k == t) ? 1u : 0u;
}

// Internal check used by tests: counts non-zeros in rows >= rank (must be 0).
__global__ void count_nonzero_tail_kernel(const uint32_t* __restrict__ A, int64_t ld, int64_t rows, int64_t cols,
                                          int64_t rank, unsigned long long* __restrict__ count) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cols) return;
    unsigned long long n = 0;
    for (int64_t k = rank + blockIdx.y; k < rows; k += gridDim.y) n += A[k * ld + c] != 0;
    if (n) atomicAdd(count, n);
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

}  // namespace linac
