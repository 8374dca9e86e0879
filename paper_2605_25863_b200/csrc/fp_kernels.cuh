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

// d*x - h*y mod p with one reduction: d*x + (p-h)*y < 2^63.
__device__ __forceinline__ uint32_t lincomb(uint32_t d, uint32_t x, uint32_t h, uint32_t y, const ModP& f) {
    return reduce64((uint64_t)d * x + (uint64_t)(f.p - h) * y, f);
}

// ------------------------------------------------------------------------------------------
// S1 + S2 + S3 for one base panel (columns [j0, j0+w), rows >= i0), one CTA of 256 threads.
//
// Phase 1 (pivot search, K3/K4/K6 of PAPER.md:241-243): rows are scanned in chunks of CH = 32 held in
// shared memory; a chunk is first reduced against the pivot rows found so far, then searched column
// by column for the FIRST row with a non-zero entry (warp ballot; for F_p any non-zero pivot will do,
// PAPER.md:241).  Elimination is division-free (row_k <- d*row_k - h*row_q), so no modular inverse
// sits on the column-to-column dependency chain.  The scan stops once w pivots are known; otherwise
// it has looked at every row, which is what proves the remaining columns are free columns.
// Phase 2 (K7 "rescale the head to 1", done for the whole panel at once): Gauss-Jordan
// on [D | I], D = A[pivot rows, pivot columns] in ascending pivot-column order (no search needed:
// pivot rows with a larger leading column vanish on the smaller columns, so D has an LU factorisation
// without pivoting), division-free, followed by r independent extended-Euclid inverses.
// Outputs: rec (r, local pivot columns, LAPACK-style exchange list), T (32x32, zero padded),
// E = T A[P, panel] when r < w (the free columns' entries of the reduced pivot rows), pivcols.
__global__ void __launch_bounds__(256) panel_factor_kernel(const uint32_t* __restrict__ A, int64_t ld, int64_t rows,
                                                           int64_t i0, int64_t j0, int w, ModP f,
                                                           PanelRec* __restrict__ rec, uint32_t* __restrict__ Tout,
                                                           uint32_t* __restrict__ Eout,
                                                           int32_t* __restrict__ pivcols_global,
                                                           const int* __restrict__ fail_flag, int panel_index) {
    __shared__ uint32_t X[CH][PW + 1];
    __shared__ uint32_t Ep[PW][PW + 1];        // pivot rows as selected (unnormalised), discovery order
    __shared__ uint32_t G[PW][2 * PW + 1];     // phase 2: [D | I]
    __shared__ int epc[PW];                    // pivot column of pivot t (discovery order)
    __shared__ long long esrc[PW];             // source row (absolute) of pivot t
    __shared__ int ord[PW];                    // pivots sorted by pivot column
    __shared__ uint32_t ginv[PW];
    __shared__ long long pos_of[PW];           // absolute position of the row that started at i0 + b
    __shared__ int at[PW];                     // which of those rows sits at top position a
    __shared__ int s_nsw;

    if (fail_flag && *fail_flag < panel_index) return;      // an earlier panel left the optimistic schedule

    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    int r = 0;                 // uniform over the CTA
    unsigned pcmask = 0;       // pivot columns so far (uniform)

    for (int64_t cs = i0; cs < rows && r < w; cs += CH) {
        const int nh = (int)min((int64_t)CH, rows - cs);
        int nz = 0;
#pragma unroll
        for (int t = 0; t < CH / 8; ++t) {
            const int k = wq * (CH / 8) + t;
            uint32_t s = 0;
            if (k < nh && lane < w) s = A[(cs + k) * ld + j0 + lane];
            for (int a = 0; a < r; ++a) {          // ascending pivot column
                const int tt = ord[a];
                const int c = epc[tt];
                const uint32_t l = __shfl_sync(0xffffffffu, s, c);
                if (l) s = lane > c ? lincomb(Ep[tt][c], s, l, Ep[tt][lane], f) : (lane == c ? 0u : mulmod(Ep[tt][c], s, f));
            }
            X[k][lane] = s;
            nz |= (s != 0);
        }
        if (!__syncthreads_or(nz)) continue;       // the whole chunk lies in the span found so far

        unsigned used = 0;                         // chunk rows that became pivot rows (uniform)
        for (int c = 0; c < w && r < w; ++c) {
            if ((pcmask >> c) & 1u) continue;
            const unsigned cand = __ballot_sync(0xffffffffu, X[lane][c] != 0) & ~used;
            if (!cand) continue;
            const int q = __ffs(cand) - 1;
            const uint32_t d = X[q][c];
            const uint32_t pv = X[q][lane];
#pragma unroll
            for (int t = 0; t < CH / 8; ++t) {
                const int k = wq * (CH / 8) + t;
                if (k == q || ((used >> k) & 1u)) continue;
                const uint32_t h = X[k][c];
                if (h == 0) continue;
                if (lane > c) X[k][lane] = lincomb(d, X[k][lane], h, pv, f);   // column c itself is not rewritten
            }
            if (wq == 0) Ep[r][lane] = ((pcmask >> lane) & 1u) ? 0u : pv;      // stale entries at earlier pivot columns are zeros
            if (tid == 0) { epc[r] = c; esrc[r] = cs + q; }
            used |= 1u << q;
            pcmask |= 1u << c;
            ++r;
            __syncthreads();
        }
        // rank sort of the pivots by column (needed to reduce the next chunk, and at the end)
        if (wq == 0) {
            const int mine = lane < r ? epc[lane] : INT_MAX;
            int pos = 0;
            for (int s = 0; s < r; ++s) pos += (epc[s] < mine);
            if (lane < r) ord[pos] = lane;
        }
        __syncthreads();
    }

    // ---- exchange list: row i0+a must receive source row esrc[ord[a]]
    if (wq == 0) {
        const bool inplace = lane >= r || esrc[ord[lane]] == i0 + lane;
        const bool all_inplace = __all_sync(0xffffffffu, inplace);
        if (lane < r) { pos_of[lane] = i0 + lane; at[lane] = lane; }
        __syncwarp();
        if (lane == 0) {
            int nsw = 0;
            if (all_inplace) {
                for (int a = 0; a < r; ++a) rec->swp[a] = i0 + a;
            } else {
                for (int a = 0; a < r; ++a) {
                    const long long src = esrc[ord[a]];
                    const long long cur = src < i0 + r ? pos_of[(int)(src - i0)] : src;
                    rec->swp[a] = cur;
                    if (cur != i0 + a) {
                        ++nsw;
                        const int x = at[a];                 // top-origin row now sitting at position a
                        pos_of[x] = cur;
                        if (cur < i0 + r) at[(int)(cur - i0)] = x;
                    }
                }
            }
            s_nsw = nsw;
        }
    }
    // ---- phase 2: T = D^{-1}
    for (int e = tid; e < PW * 2 * PW; e += 256) {
        const int a = e / (2 * PW), b = e % (2 * PW);
        uint32_t v = 0;
        if (a < r) {
            if (b < PW) { if (b < r) v = A[esrc[ord[a]] * ld + j0 + epc[ord[b]]]; }
            else v = (b - PW == a) ? 1u : 0u;
        }
        G[a][b] = v;
    }
    __syncthreads();
    for (int t = 0; t < r; ++t) {
        const uint32_t d = G[t][t];
        const uint32_t pl = lane > t ? G[t][lane] : 0u;
        const uint32_t pr = lane <= t ? G[t][PW + lane] : 0u;
#pragma unroll
        for (int u = 0; u < PW / 8; ++u) {
            const int s = wq * (PW / 8) + u;
            if (s == t || s >= r) continue;
            const uint32_t h = G[s][t];
            if (h == 0) continue;
            if (lane > t || lane == s) G[s][lane] = lincomb(d, G[s][lane], h, pl, f);
            if (lane <= t || lane == s) G[s][PW + lane] = lincomb(d, G[s][PW + lane], h, pr, f);
        }
        __syncthreads();
    }
    if (wq == 0 && lane < r) ginv[lane] = invmod(G[lane][lane], f);
    __syncthreads();
    for (int e = tid; e < PW * PW; e += 256) {
        const int a = e / PW, b = e % PW;
        const uint32_t v = (a < r && b < r) ? mulmod(ginv[a], G[a][PW + b], f) : 0u;
        Tout[e] = v;
        G[a][b] = v;                  // keep T in shared memory for E below (left half is dead now)
    }
    if (r < w && r > 0) {
        // E = T . A[P, panel]: reduced pivot rows restricted to the panel (identity on the pivot columns)
        for (int e = tid; e < PW * PW; e += 256) {
            const int a = e / PW, b = e % PW;
            X[a][b] = (a < r && b < w) ? A[esrc[ord[a]] * ld + j0 + b] : 0u;
        }
        __syncthreads();
#pragma unroll
        for (int u = 0; u < PW / 8; ++u) {
            const int a = wq * (PW / 8) + u;
            uint64_t acc = 0;
            for (int b = 0; b < r; ++b) {
                acc += (uint64_t)G[a][b] * X[b][lane];
                if (b & 1) acc = fold64(acc, f);
            }
            Eout[a * PW + lane] = a < r ? reduce64(acc, f) : 0u;
        }
    }
    if (tid < PW) {
        rec->pc[tid] = tid < r ? epc[ord[tid]] : -1;
        if (tid < r) pivcols_global[i0 + tid] = (int32_t)(j0 + epc[ord[tid]]);
    }
    __syncthreads();
    if (tid == 0) {
        rec->r = r;
        rec->w = w;
        rec->nswaps = s_nsw;
    }
}

// ------------------------------------------------------------------------------------------
// K5 CudaSwitchRows for a whole panel: the exchanges are applied to complete rows,
// one thread per column (so the sequence of exchanges needs no inter-thread ordering).  When the
// panel is rank deficient the same thread then stores the reduced pivot rows' panel entries E.
__global__ void panel_finish_kernel(uint32_t* __restrict__ A, int64_t ld, int64_t cols, int64_t i0, int64_t j0,
                                    const PanelRec* __restrict__ rec, const uint32_t* __restrict__ E,
                                    const int* __restrict__ fail_flag, int panel_index) {
    if (fail_flag && *fail_flag < panel_index) return;
    const int r = rec->r, ns = rec->nswaps, w = rec->w;
    if (r == 0 || (ns == 0 && r == w)) return;
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cols) return;
    if (ns > 0) {
        for (int a = 0; a < r; ++a) {
            const int64_t s = rec->swp[a];
            if (s != i0 + a) {
                const uint32_t x = A[(i0 + a) * ld + c], y = A[s * ld + c];
                A[(i0 + a) * ld + c] = y;
                A[s * ld + c] = x;
            }
        }
    }
    if (r < w && c >= j0 && c < j0 + w)
        for (int a = 0; a < r; ++a) A[(i0 + a) * ld + c] = E[a * PW + (int)(c - j0)];
}

// ------------------------------------------------------------------------------------------
// S4 row-block solve, base case: X <- T X for one base panel (r <= 32 pivot rows i0..i0+r),
// X = A[i0 : i0+r, c0 : c0+ncols].  A 32x32 tile of X per CTA; thread = (4 output rows, 1 column).
__global__ void __launch_bounds__(256) apply_t_kernel(uint32_t* __restrict__ X, int64_t ldx, int64_t ncols,
                                                      const uint32_t* __restrict__ T, int r, ModP f,
                                                      const int* __restrict__ fail_flag, int epoch) {
    if (fail_flag && *fail_flag <= epoch) return;
    __shared__ uint32_t Ts[PW][PW + 1];
    __shared__ uint32_t Xs[PW][PW + 1];
    const int tid = threadIdx.x, lane = tid & 31, g = tid >> 5;
    const int64_t c = (int64_t)blockIdx.x * PW + lane;
    for (int e = tid; e < PW * PW; e += 256) Ts[e / PW][e % PW] = T[e];
#pragma unroll
    for (int u = 0; u < PW / 8; ++u) {
        const int a = g * (PW / 8) + u;
        Xs[a][lane] = (a < r && c < ncols) ? X[(int64_t)a * ldx + c] : 0u;
    }
    __syncthreads();
    if (c >= ncols) return;
#pragma unroll
    for (int u = 0; u < PW / 8; ++u) {
        const int a = g * (PW / 8) + u;
        if (a >= r) continue;
        uint64_t acc = 0;
#pragma unroll 8
        for (int b = 0; b < PW; b += 2) {
            acc += (uint64_t)Ts[a][b] * Xs[b][lane];
            acc += (uint64_t)Ts[a][b + 1] * Xs[b + 1][lane];
            acc = fold64(acc, f);
        }
        X[(int64_t)a * ldx + c] = reduce64(acc, f);
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

}  // namespace linac
