// f64_solve.cu -- linac_solve_f64: row-equilibrated LU with partial pivoting + triangular solves.
//
// F1  row scales (CudaSetRowScales / CudaRescaleRows)
// F2  blocked right-looking LU, partial pivoting on the column maximum:
//       * 32-column panels factored by ONE cooperative kernel (grid of one CTA per SM, the strip
//         resident in shared memory, one grid-wide sync per column: warp-shuffle arg-max inside
//         each CTA, candidates exchanged through global memory)
//       * row exchanges applied to whole rows of A and B (CudaSwitchRows)
//       * row-block solves and trailing updates A22 -= L21.U12 as DGEMMs (DMMA m8n8k4), organised recursively
//     B rides along as extra trailing columns, which performs the forward substitution
//     (the paper reduces the augmented matrix (A b)).
// F3  back substitution with U on the right-hand sides (blocked, GEMM for the off-diagonal part).
// A pivot with |pivot| <= tol marks the matrix singular (CudaCompareHeadToTolerance).
#include <cooperative_groups.h>

#include <algorithm>
#include <climits>
#include <mutex>
#include <vector>

#include "linac_internal.h"

namespace cg = cooperative_groups;

namespace linac {
namespace {

constexpr int FW = 32;              // panel width

// ---------------------------------------------------------------- F1
// One block per row: s = max_c |A[r,c]| over A's columns (reading Q11), then A[r,:] /= s, B[r,:] /= s.
// The row is kept in shared memory between the two passes when it fits (n <= 24576 doubles), so the matrix is read
// once and written once: 16 B per element, the algorithmic minimum (the first version read it twice: 24 B).
constexpr int RS_THREADS = 512;
__global__ void __launch_bounds__(RS_THREADS) row_scale_kernel(double* __restrict__ A, int64_t n, int64_t lda,
                                                               double* __restrict__ B, int64_t nrhs, int64_t ldb,
                                                               int* __restrict__ info, int cache_n) {
    extern __shared__ __align__(16) double rs_row[];
    __shared__ double red[RS_THREADS / 32];
    const int64_t r = blockIdx.x;
    double* row = A + r * lda;
    const bool vec = ((reinterpret_cast<uintptr_t>(row) & 15) == 0) && (n % 2 == 0);
    double m = 0.0;
    if (vec) {
        const double2* row2 = reinterpret_cast<const double2*>(row);
        for (int64_t c = threadIdx.x; c < n / 2; c += blockDim.x) {
            const double2 v = row2[c];
            if (2 * c + 1 < cache_n) reinterpret_cast<double2*>(rs_row)[c] = v;
            m = fmax(m, fmax(fabs(v.x), fabs(v.y)));
        }
    } else {
        for (int64_t c = threadIdx.x; c < n; c += blockDim.x) {
            const double v = row[c];
            if (c < cache_n) rs_row[c] = v;
            m = fmax(m, fabs(v));
        }
    }
    for (int o = 16; o; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    m = red[0];
    for (int w = 1; w < RS_THREADS / 32; ++w) m = fmax(m, red[w]);
    if (m == 0.0) {
        if (threadIdx.x == 0) atomicMin(info, 1);      // a zero row: singular at the very first column
        return;
    }
    if (vec) {
        double2* row2 = reinterpret_cast<double2*>(row);
        for (int64_t c = threadIdx.x; c < n / 2; c += blockDim.x) {
            double2 v = 2 * c + 1 < cache_n ? reinterpret_cast<const double2*>(rs_row)[c] : row2[c];
            v.x = v.x / m;
            v.y = v.y / m;
            row2[c] = v;
        }
    } else {
        for (int64_t c = threadIdx.x; c < n; c += blockDim.x) row[c] = (c < cache_n ? rs_row[c] : row[c]) / m;
    }
    for (int64_t c = threadIdx.x; c < nrhs; c += blockDim.x) B[r * ldb + c] = B[r * ldb + c] / m;
}

// Launch helper: the row cache takes what is left of one SM's shared memory for two resident CTAs.
int launch_row_scale(double* A, int64_t rows, int64_t n, int64_t lda, double* B, int64_t nrhs, int64_t ldb, int* info,
                     cudaStream_t s) {
    static PerDeviceOnce once;
    const int rc = once.run([]() -> int {
        LINAC_CUDA(cudaFuncSetAttribute(row_scale_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
        return LINAC_OK;
    });
    if (rc) return rc;
    const int cache_n = (int)std::min<int64_t>(n / 2 * 2, 100 * 1024 / 8);
    row_scale_kernel<<<(unsigned)rows, RS_THREADS, (size_t)cache_n * 8, s>>>(A, n, lda, B, nrhs, ldb, info, cache_n);
    LINAC_CUDA(cudaGetLastError());
    return LINAC_OK;
}

// ---------------------------------------------------------------- F2 panel
struct Cand {                 // one CTA's arg-max candidate for a column, with the row's content
    double absval;
    long long row;            // absolute row index, -1 if the CTA owns no eligible row
    double2 content[FW];      // .x = the row's panel entries; .y = the column's tag (tagged mode: every 16-byte word validates itself)
};

// Tagged records: {payload, tag} travel as ONE 128-bit scalar memory operation (.b128, PTX ISA 8.3; SASS
// STG/LDG.E.128.STRONG.GPU), relaxed at gpu scope.  A scalar access is a single operation of the memory model (a
// .v2 vector access is modelled as two), so a reader sees either the old or the new 16 bytes, never a mix: the tag
// validates the payload without a fence.
__device__ __forceinline__ void st_b128(void* p, unsigned long long w0, unsigned long long w1) {
    asm volatile("{ .reg .b128 t; mov.b128 t, {%0, %1}; st.relaxed.gpu.global.b128 [%2], t; }" ::"l"(w0), "l"(w1), "l"(p) : "memory");
}
__device__ __forceinline__ void ld_b128(const void* p, unsigned long long& w0, unsigned long long& w1) {
    asm volatile("{ .reg .b128 t; ld.relaxed.gpu.global.b128 t, [%2]; mov.b128 {%0, %1}, t; }" : "=l"(w0), "=l"(w1) : "l"(p) : "memory");
}
__device__ __forceinline__ void st_tagged(double2* p, double v, unsigned tag) {
    st_b128(p, (unsigned long long)__double_as_longlong(v), (unsigned long long)tag);
}
__device__ __forceinline__ double ld_tagged(const double2* p, unsigned tag) {      // spins until the word carries `tag`
    unsigned long long w0, w1;
    do {
        ld_b128(p, w0, w1);
    } while ((unsigned)w1 != tag);
    return __longlong_as_double((long long)w0);
}

// Warp arg-max of non-negative doubles with the lowest index winning ties, on the redux.sync unit: the bit pattern of
// a non-negative double orders like the number, so the maximum is two 32-bit max-reductions (high word, then low word
// among the lanes that hold the maximal high word) and the tie-break one min-reduction -- about ten instructions
// instead of five shuffle rounds on three 64-bit values.  A lane takes part iff idx >= 0 (then v >= 0); every lane
// returns the winner's (v, idx, aux), idx = -1 if no lane took part.
__device__ __forceinline__ void warp_argmax(double& v, int& idx, int& aux) {
    const bool has = idx >= 0;
    const unsigned hi = has ? (unsigned)__double2hiint(v) : 0u;
    const unsigned lo = has ? (unsigned)__double2loint(v) : 0u;
    const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
    const unsigned ml = __reduce_max_sync(0xffffffffu, hi == mh ? lo : 0u);
    const unsigned key = (has && hi == mh && lo == ml) ? (unsigned)idx : 0xffffffffu;
    const unsigned mk = __reduce_min_sync(0xffffffffu, key);
    if (mk == 0xffffffffu) { v = -1.0; idx = -1; aux = -1; return; }
    const int who = __ffs(__ballot_sync(0xffffffffu, key == mk)) - 1;
    v = __hiloint2double((int)mh, (int)ml);
    idx = (int)mk;
    aux = __shfl_sync(0xffffffffu, aux, who);
}

// What the panel kernel reports in RREF mode (device-resident: the host never reads it inside the loop).
struct F64Rec {
    long long i0;             // first pivot row of the panel
    int r;                    // pivots found (<= FW)
    int pad;
    int pc[FW];               // local pivot columns, ascending (-1 beyond r)
};

// CLUSTER = false: cooperative kernel, one CTA per SM, grid barrier and candidate records in global memory (L2).
// CLUSTER = true: ONE thread-block cluster of up to 16 CTAs holds the strip; the per-column barrier is the hardware
// cluster barrier and the candidate records are read from the peers' shared memory (DSMEM), which cuts the
// per-column latency from two L2 round trips and a grid barrier to about a microsecond.
// RREF = false (linac_solve_f64): factors A[j0:n, j0:j0+w) in place (unit-lower L below, U on and above the
// diagonal), records the exchanges in ipiv[j0..j0+w).  CTA b owns rows [j0 + b*R, j0 + (b+1)*R).
// RREF = true (linac_rref_f64): the same elimination on the rows from i0 = *state on, as a pivot SEARCH only -- the
// strip is not written back.  A column whose largest remaining entry is <= tol yields no pivot (CudaCompareHeadTo-
// Tolerance) and the row counter does not advance; the pivot of ordinal t goes to row
// i0 + t.  Outputs: ipiv[i0 + t] (exchanges), rec (i0, r, pivot columns), *state += r.
template <int FTHREADS, bool CLUSTER, bool RREF>
__global__ void __launch_bounds__(FTHREADS) f64_panel_kernel(double* __restrict__ A, int64_t n, int64_t lda, int64_t j0,
                                                              int w, int rows_per_cta, double tol,
                                                              Cand* __restrict__ cand /* [2][gridDim] */,
                                                              double2* __restrict__ target /* [2][FW] */,
                                                              long long* __restrict__ ipiv, int* __restrict__ info,
                                                              unsigned tag0, long long* __restrict__ state,
                                                              F64Rec* __restrict__ rec, int32_t* __restrict__ pivcols) {
    extern __shared__ __align__(16) double S[];         // rows_per_cta x LDS
    constexpr int NE = FTHREADS / 32 * 4;               // arg-max entries per column: 4 row groups per warp
    __shared__ double s_val[NE];
    __shared__ int s_idx[NE];
    __shared__ __align__(16) double pv_al[FW];
    __shared__ Cand l_cand[2];                          // CLUSTER: this CTA's records, read by the peers
    __shared__ double2 l_target[2][FW];
    __shared__ int s_pc[FW];                            // RREF: pivot columns in discovery (= ascending) order
    __shared__ int s_flag;                              // RREF: 1 iff the current column yields a pivot
    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    int G = gridDim.x, b = blockIdx.x;
    if constexpr (CLUSTER) { G = (int)cg::this_cluster().num_blocks(); b = (int)cg::this_cluster().block_rank(); }
    auto group_sync = [&]() {
        if constexpr (CLUSTER) cg::this_cluster().sync(); else cg::this_grid().sync();
    };
    auto cand_of = [&](int c, int q) -> const Cand* {   // CTA q's record for column c
        if constexpr (CLUSTER) return cg::this_cluster().map_shared_rank(&l_cand[c & 1], q);
        else return cand + (size_t)(c & 1) * G + q;
    };
    auto ld_f = [&](const double* p) { if constexpr (CLUSTER) return *p; else return __ldcg(p); };
    auto ld_i = [&](const long long* p) { if constexpr (CLUSTER) return *p; else return __ldcg(p); };
    const int64_t i0 = RREF ? (int64_t)*state : j0;     // first row of the strip
    if constexpr (RREF) {
        if (i0 >= n) {                                  // no rows left: every remaining column is free (uniform exit)
            if (b == 0 && tid == 0) { rec->i0 = i0; rec->r = 0; }
            if (b == 0 && tid < FW) rec->pc[tid] = -1;
            return;
        }
    }
    const int64_t r0 = i0 + (int64_t)b * rows_per_cta;
    const int nr = (int)max((int64_t)0, min((int64_t)rows_per_cta, n - r0));
    constexpr int LDS = FW + 2;                         // even: the update reads rows as 16-byte pairs
    double* pv = pv_al;

    for (int k = wq; k < nr; k += FTHREADS / 32) S[k * LDS + lane] = lane < w ? A[(r0 + k) * lda + j0 + lane] : 0.0;
    __syncthreads();

    // second half of publishing column c: the warps' arg-max values are in s_val/s_idx (after a __syncthreads);
    // jc = the row the column's pivot will go to (its present content travels to the winner's owner)
    auto publish_tail = [&](int c, int64_t jc) {
        if (wq == 0) {
            double best = -1.0;
            int bi = -1, none = 0;
            for (int e = lane; e < NE; e += 32) {
                const double v = s_val[e];
                const int i = s_idx[e];
                if (i >= 0 && (bi < 0 || v > best || (v == best && i < bi))) { best = v; bi = i; }
            }
            warp_argmax(best, bi, none);
            Cand* cd = CLUSTER ? &l_cand[c & 1] : cand + (size_t)(c & 1) * G + b;
            const bool tagged = !CLUSTER && tag0 != 0;
            const unsigned tag = tag0 + (unsigned)c;
            double2* tgt = CLUSTER ? l_target[c & 1] : target + (c & 1) * FW;
            if (tagged) {
                // tagged records instead of a grid barrier and fences: every 16-byte word {value, tag} validates itself,
                // so the stores need no order among themselves; the head word is {|value|, tag : row}
                if (bi >= 0) st_tagged(&cd->content[lane], S[bi * LDS + lane], tag);
                if (jc >= r0 && jc < r0 + nr) st_tagged(&tgt[lane], S[(int)(jc - r0) * LDS + lane], tag);
                if (lane == 0) {
                    const unsigned long long w0 = (unsigned long long)__double_as_longlong(best);
                    const unsigned long long w1 = ((unsigned long long)tag << 32) | (unsigned)(bi >= 0 ? (int)(r0 + bi) : -1);
                    st_b128(&cd->absval, w0, w1);
                }
            } else {
                if (bi >= 0) cd->content[lane] = make_double2(S[bi * LDS + lane], 0.0);
                if (jc >= r0 && jc < r0 + nr) tgt[lane] = make_double2(S[(int)(jc - r0) * LDS + lane], 0.0);
                if (lane == 0) { cd->absval = best; cd->row = bi >= 0 ? r0 + bi : -1; }
            }
        }
    };                                                      // always followed by group_sync(), which is a block barrier too

    // publish the candidate for column c among own rows with absolute index >= jc, and row jc itself
    auto publish = [&](int c, int64_t jc) {
        double best = -1.0;
        int bi = -1;
        for (int k = tid; k < nr; k += FTHREADS) {
            if (r0 + k < jc) continue;
            const double v = fabs(S[k * LDS + c]);
            if (v > best) { best = v; bi = k; }          // strict >: lowest index wins inside a thread
        }
        int none = 0;
        warp_argmax(best, bi, none);
        if (lane < 4) { s_val[wq * 4 + lane] = best; s_idx[wq * 4 + lane] = lane == 0 ? bi : -1; }
        __syncthreads();
        publish_tail(c, jc);
    };

    int npiv = 0;                                           // RREF: pivots found so far (uniform over the grid)
    publish(0, i0);
    for (int c = 0; c < w; ++c) {
        const bool tagged = !CLUSTER && tag0 != 0;
        if (!tagged) group_sync();
        const int64_t jc = RREF ? i0 + npiv : j0 + c;       // the row this column's pivot goes to
        if constexpr (RREF) {
            if (jc >= n) break;                             // every row holds a pivot: the remaining columns are free
        }
        // every CTA reduces the G candidates identically: largest |value|, lowest row on ties (reading Q12).
        // Warp 0 alone: up to CPL candidates per lane, their loads all in flight together (one round trip), one
        // warp arg-max, then the winner's row content (the second round trip).
        if (wq == 0) {
            constexpr int CPL = 5;                         // 160 candidates per pass (148 CTAs on a B200)
            double best = -1.0;
            int brow = -1, bcta = -1;
            for (int q0 = 0; q0 < G; q0 += 32 * CPL) {
                double v[CPL];
                int rr[CPL];
                if (tagged) {                              // poll until every record of this pass carries the column's tag
                    const unsigned tag = tag0 + (unsigned)c;
                    bool ok;
                    do {
                        ok = true;
#pragma unroll
                        for (int u = 0; u < CPL; ++u) {
                            const int q = q0 + u * 32 + lane;
                            v[u] = -1.0;
                            rr[u] = -1;
                            if (q < G) {
                                unsigned long long w0, w1;
                                ld_b128(&cand_of(c, q)->absval, w0, w1);
                                ok = ok && (unsigned)(w1 >> 32) == tag;
                                v[u] = __longlong_as_double((long long)w0);
                                rr[u] = (int)(unsigned)w1;
                            }
                        }
                    } while (!__all_sync(0xffffffffu, ok));
                } else {
#pragma unroll
                    for (int u = 0; u < CPL; ++u) {
                        const int q = q0 + u * 32 + lane;
                        v[u] = -1.0;
                        rr[u] = -1;
                        if (q < G) {
                            const Cand* cd = cand_of(c, q);
                            v[u] = ld_f(&cd->absval);
                            rr[u] = (int)ld_i(&cd->row);
                        }
                    }
                }
#pragma unroll
                for (int u = 0; u < CPL; ++u)
                    if (rr[u] >= 0 && (brow < 0 || v[u] > best || (v[u] == best && rr[u] < brow))) {
                        best = v[u]; brow = rr[u]; bcta = q0 + u * 32 + lane;
                    }
            }
            warp_argmax(best, brow, bcta);
            const bool is_pivot = best > tol;
            if (RREF && lane == 0) s_flag = is_pivot ? 1 : 0;   // next written after the block barriers of publish / update
            if (!RREF || is_pivot) {
                // the winner's row content; no candidate (a column of NaNs): flagged below
                const double x = bcta < 0 ? 0.0 : tagged ? ld_tagged(&cand_of(c, bcta)->content[lane], tag0 + (unsigned)c) : ld_f(&cand_of(c, bcta)->content[lane].x);
                if (brow < 0) brow = (int)jc;
                if (lane == 0 && b == 0) {
                    ipiv[jc] = brow;
                    if (!RREF && !is_pivot) atomicMin(info, (int)min((int64_t)INT_MAX, jc + 1));
                }
                // exchange rows jc and g = brow (content of row jc comes from `target`, the pivot row from `pv`)
                const long long g = brow;
                if (g != jc && g >= r0 && g < r0 + nr) {
                    const double2* tg = target + (c & 1) * FW;
                    if constexpr (CLUSTER) tg = cg::this_cluster().map_shared_rank(&l_target[c & 1][0], (int)((jc - i0) / rows_per_cta));
                    S[(int)(g - r0) * LDS + lane] = tagged ? ld_tagged(tg + lane, tag0 + (unsigned)c) : ld_f(&tg[lane].x);
                }
                if (jc >= r0 && jc < r0 + nr) S[(int)(jc - r0) * LDS + lane] = x;
                pv[lane] = x;
            }
        }
        __syncthreads();
        if constexpr (RREF) {
            if (s_flag == 0) {                              // no pivot in this column: the row counter stays
                if (c + 1 < w) publish(c + 1, jc);
                continue;
            }
            if (tid == 0) s_pc[npiv] = c;
            ++npiv;
        }
        double piv = pv[c];
        if (!RREF && !(fabs(piv) > tol)) piv = 1.0;     // singular: flagged above; keep the arithmetic finite
        const double rp = __drcp_rn(piv);
        // multipliers and rank-1 update of own rows below jc: a warp takes four rows per pass, eight lanes per row,
        // four columns per lane (two 16-byte accesses each way).  The lane that holds column c+1 sees the new
        // entries of the next column as they are made and keeps their arg-max (lowest row on ties).
        const int seg = lane & 7, rg = lane >> 3, jb = seg * 4;
        const int cs = c >> 2, ns = (c + 1) >> 2, ne = (c + 1) & 3;
        const double2 pa = *reinterpret_cast<const double2*>(pv + jb), pb = *reinterpret_cast<const double2*>(pv + jb + 2);
        double best = -1.0;
        int bi = -1;
        const int kmin = (int)max((int64_t)0, min((int64_t)nr, jc + 1 - r0));   // own rows below the pivot row
#pragma unroll 2
        for (int k = kmin + wq * 4 + rg; k < nr; k += FTHREADS / 32 * 4) {
            double* row = S + k * LDS;
            const double l = row[c] * rp;
            if (seg >= cs) {                               // columns >= w hold zeros in S and in pv: no bound needed
                double2 xa = *reinterpret_cast<double2*>(row + jb), xb = *reinterpret_cast<double2*>(row + jb + 2);
                xa.x = jb + 0 > c ? xa.x - l * pa.x : (jb + 0 == c ? l : xa.x);
                xa.y = jb + 1 > c ? xa.y - l * pa.y : (jb + 1 == c ? l : xa.y);
                xb.x = jb + 2 > c ? xb.x - l * pb.x : (jb + 2 == c ? l : xb.x);
                xb.y = jb + 3 > c ? xb.y - l * pb.y : (jb + 3 == c ? l : xb.y);
                *reinterpret_cast<double2*>(row + jb) = xa;
                *reinterpret_cast<double2*>(row + jb + 2) = xb;
                if (seg == ns) {
                    const double v = fabs(ne == 0 ? xa.x : ne == 1 ? xa.y : ne == 2 ? xb.x : xb.y);
                    if (v > best) { best = v; bi = k; }
                }
            }
        }
        if (c + 1 < w) {
            if (seg == ns) { s_val[wq * 4 + rg] = best; s_idx[wq * 4 + rg] = bi; }
            __syncthreads();
            publish_tail(c + 1, jc + 1);
        }
    }
    __syncthreads();                                        // the last column's updates (rows change warps per column)
    if constexpr (RREF) {
        if (b == 0) {
            if (tid < FW) {
                const int pc = tid < npiv ? s_pc[tid] : -1;
                rec->pc[tid] = pc;
                if (tid < npiv) pivcols[i0 + tid] = (int32_t)(j0 + pc);
            }
            if (tid == 0) { rec->i0 = i0; rec->r = npiv; *state = i0 + npiv; }
        }
    } else {
        for (int k = wq; k < nr; k += FTHREADS / 32)
            if (lane < w) A[(r0 + k) * lda + j0 + lane] = S[k * LDS + lane];
    }
    if constexpr (CLUSTER) cg::this_cluster().sync();   // no CTA may leave while a peer can still read its records
}

// Row exchanges of one panel applied to whole rows outside the panel columns; one thread per column.
__global__ void f64_swap_kernel(double* __restrict__ M, int64_t ld, int64_t c_begin, int64_t c_end, int64_t skip0,
                                int64_t skip1, const long long* __restrict__ ipiv, int64_t j0, int w) {
    int64_t c = c_begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= c_end || (c >= skip0 && c < skip1)) return;
    for (int a = 0; a < w; ++a) {
        const int64_t s = ipiv[j0 + a];
        if (s != j0 + a && s >= 0) {
            const double x = M[(j0 + a) * ld + c], y = M[s * ld + c];
            M[(j0 + a) * ld + c] = y;
            M[s * ld + c] = x;
        }
    }
}

// X <- L11^{-1} X, L11 unit lower nb x nb at A[t0:t0+nb, t0:t0+nb]; one thread per column of X.
constexpr int FT = 128;
__global__ void __launch_bounds__(FT) f64_trsm_lower_kernel(double* __restrict__ X, int64_t ldx, int64_t ncols,
                                                            const double* __restrict__ A, int64_t lda, int64_t t0, int nb) {
    __shared__ double L[FW][FW + 1];
    __shared__ double Xs[FW][FT];
    const int tid = threadIdx.x;
    for (int e = tid; e < nb * nb; e += FT) L[e / nb][e % nb] = A[(t0 + e / nb) * lda + t0 + e % nb];
    const int64_t c = (int64_t)blockIdx.x * FT + tid;
    const bool on = c < ncols;
    for (int a = 0; a < nb; ++a) Xs[a][tid] = on ? X[(int64_t)a * ldx + c] : 0.0;
    __syncthreads();
    if (!on) return;
    for (int a = 1; a < nb; ++a) {
        double s = Xs[a][tid];
        for (int q = 0; q < a; ++q) s -= L[a][q] * Xs[q][tid];
        Xs[a][tid] = s;
        X[(int64_t)a * ldx + c] = s;
    }
}

// The full-width leaf (nb = 32) with the column of X in registers: right-looking order, so the 31 - q updates that
// follow x[q] are independent (the dot-product order above is one dependent chain per entry), L read as broadcasts.
constexpr int FT2 = 64;
__global__ void __launch_bounds__(FT2) f64_trsm_lower32_kernel(double* __restrict__ X, int64_t ldx, int64_t ncols,
                                                               const double* __restrict__ A, int64_t lda, int64_t t0) {
    __shared__ __align__(16) double Lt[FW][FW + 2];        // Lt[q][a] = L[a][q]
    const int tid = threadIdx.x;
    for (int e = tid; e < FW * FW; e += FT2) Lt[e & 31][e >> 5] = A[(t0 + (e >> 5)) * lda + t0 + (e & 31)];
    __syncthreads();
    const int64_t c = (int64_t)blockIdx.x * FT2 + tid;
    if (c >= ncols) return;
    double x[FW];
#pragma unroll
    for (int a = 0; a < FW; ++a) x[a] = X[(int64_t)a * ldx + c];
#pragma unroll
    for (int q = 0; q < FW - 1; ++q) {
#pragma unroll
        for (int a = q + 1; a < FW; ++a) x[a] -= Lt[q][a] * x[q];
    }
#pragma unroll
    for (int a = 1; a < FW; ++a) X[(int64_t)a * ldx + c] = x[a];
}

// X <- U11^{-1} X, U11 upper nb x nb (non-unit) at A[t0:t0+nb, t0:t0+nb].
__global__ void __launch_bounds__(FT) f64_trsm_upper_kernel(double* __restrict__ X, int64_t ldx, int64_t ncols,
                                                            const double* __restrict__ A, int64_t lda, int64_t t0, int nb) {
    __shared__ double U[FW][FW + 1];
    __shared__ double Xs[FW][FT];
    const int tid = threadIdx.x;
    for (int e = tid; e < nb * nb; e += FT) U[e / nb][e % nb] = A[(t0 + e / nb) * lda + t0 + e % nb];
    const int64_t c = (int64_t)blockIdx.x * FT + tid;
    const bool on = c < ncols;
    for (int a = 0; a < nb; ++a) Xs[a][tid] = on ? X[(int64_t)a * ldx + c] : 0.0;
    __syncthreads();
    if (!on) return;
    for (int a = nb - 1; a >= 0; --a) {
        double s = Xs[a][tid];
        for (int q = a + 1; q < nb; ++q) s -= U[a][q] * Xs[q][tid];
        s /= U[a][a];
        Xs[a][tid] = s;
        X[(int64_t)a * ldx + c] = s;
    }
}

// ---------------------------------------------------------------- F2 trailing update: C -= A.B (DFMA)
constexpr int DM = 128, DN = 128, DK = 8, DTM = 8, DTN = 8;
constexpr int DTHREADS = (DM / DTM) * (DN / DTN);      // 256
__global__ void __launch_bounds__(DTHREADS) dgemm_sub_kernel(double* __restrict__ C, int64_t ldc,
                                                             const double* __restrict__ A, int64_t lda,
                                                             const double* __restrict__ B, int64_t ldb, int64_t M,
                                                             int64_t N, int64_t K) {
    __shared__ __align__(16) double As[2][DK][DM + 2];
    __shared__ __align__(16) double Bs[2][DK][DN];
    const int tid = threadIdx.x, tx = tid % (DN / DTN), ty = tid / (DN / DTN);
    const int64_t m0 = (int64_t)blockIdx.y * DM, n0 = (int64_t)blockIdx.x * DN;
    double acc[DTM][DTN];
#pragma unroll
    for (int i = 0; i < DTM; ++i)
#pragma unroll
        for (int j = 0; j < DTN; ++j) acc[i][j] = 0.0;

    // each thread stages 4 A elements (128x8) and 4 B elements (8x128) per k-block
    double ra[4], rb[4];
    auto gload = [&](int64_t k0) {
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            const int idx = tid + t * DTHREADS;
            const int kk = idx % DK, mm = idx / DK;
            const int64_t m = m0 + mm, k = k0 + kk;
            ra[t] = (m < M && k < K) ? A[m * lda + k] : 0.0;
            const int nn = idx % DN, kb = idx / DN;
            const int64_t n = n0 + nn, k2 = k0 + kb;
            rb[t] = (n < N && k2 < K) ? B[k2 * ldb + n] : 0.0;
        }
    };
    auto sstore = [&](int buf) {
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            const int idx = tid + t * DTHREADS;
            As[buf][idx % DK][idx / DK] = ra[t];
            Bs[buf][idx / DN][idx % DN] = rb[t];
        }
    };
    gload(0);
    sstore(0);
    __syncthreads();
    int buf = 0;
    for (int64_t k0 = 0; k0 < K; k0 += DK) {
        const bool more = k0 + DK < K;
        if (more) gload(k0 + DK);
#pragma unroll
        for (int kk = 0; kk < DK; ++kk) {
            double a[DTM], bb[DTN];
#pragma unroll
            for (int i = 0; i < DTM; i += 2)
                *reinterpret_cast<double2*>(&a[i]) = *reinterpret_cast<const double2*>(&As[buf][kk][ty * DTM + i]);
#pragma unroll
            for (int j = 0; j < DTN; j += 2)
                *reinterpret_cast<double2*>(&bb[j]) = *reinterpret_cast<const double2*>(&Bs[buf][kk][tx * DTN + j]);
#pragma unroll
            for (int i = 0; i < DTM; ++i)
#pragma unroll
                for (int j = 0; j < DTN; ++j) acc[i][j] = fma(a[i], bb[j], acc[i][j]);
        }
        if (more) {
            sstore(buf ^ 1);
            __syncthreads();
            buf ^= 1;
        }
    }
#pragma unroll
    for (int i = 0; i < DTM; ++i) {
        const int64_t m = m0 + ty * DTM + i;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < DTN; ++j) {
            const int64_t n = n0 + tx * DTN + j;
            if (n < N) C[m * ldc + n] -= acc[i][j];
        }
    }
}

// The same update on the FP64 tensor pipe (DMMA m8n8k4, the only FP64 MMA shape sm_100 has): 128 x 128 tile, 8 warps
// as 2 x 4, a 64 x 32 warp tile = 8 x 4 MMA tiles.  Operands come from shared memory one double per thread and
// per fragment, so a k-step costs 12 LDS.64 per 32 MMAs: five times less shared-memory traffic per flop than the
// 8 x 8 register tile of the DFMA kernel above, which was co-bound by the shared-memory pipe.
constexpr int QK = 16;                    // k per shared-memory stage (the A copy mapping below assumes 16)
constexpr int QLD = DM + 4;               // row stride in doubles: = 4 mod 16, conflict-free fragment loads
constexpr int QNS = 3;                    // cp.async stages
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc, bool valid) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    const int bytes = valid ? 8 : 0;                   // src-size 0: the 8 bytes are zero-filled, nothing is read
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d), "l"(gsrc), "r"(bytes) : "memory");
}
__device__ __forceinline__ void dmma_8x8x4(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
// TN = 128 (8 warps as 2 x 4, 64 x 32 warp tiles) or 64 (64 x 16 warp tiles: the skinny right-hand-side updates).
// ASSIGN: C = A.B instead of C -= A.B; a CTA reads every B element of its column range before its epilogue, so
// C may alias B when one CTA covers all M rows (the diagonal-block step of the blocked substitution).
// Shape taken from device memory (linac_rref_f64, which never syncs with the host inside its loop): K and M are clipped
// to *kact / *mact and the rows of C and A start at *row0.  All null for the ordinary call.
struct DevShape {
    const int* kact;
    const int* mact;
    const long long* row0;
};
template <int TN, bool ASSIGN, int NW>
__global__ void __launch_bounds__(NW * 32, TN == 64 ? 2 : 1) dgemm_sub_mma_kernel(double* C, int64_t ldc,
                                                            const double* __restrict__ A, int64_t lda,
                                                            const double* B, int64_t ldb, int64_t M,
                                                            int64_t N, int64_t K, DevShape ds) {
    if (ds.kact != nullptr) {                              // the panel's pivot count
        K = min(K, (int64_t)*ds.kact);
        if (K <= 0) return;
    }
    if (ds.mact != nullptr) {
        M = min(M, (int64_t)*ds.mact);
        if (M <= 0) return;
    }
    if (ds.row0 != nullptr) {
        C += *ds.row0 * ldc;
        A += *ds.row0 * lda;
    }
    constexpr int NJ = TN / 32;                            // MMA tiles per warp along n
    constexpr int NT = NW * 32;                            // threads: 8 warps as 2 x 4 (16 as 4 x 4 measured no faster)
    constexpr int MI = 64 / NW;                            // MMA tiles per warp along m (warp tile 64 or 32 rows)
    constexpr int BL = QK * TN / NT;                       // B elements per thread and stage
    extern __shared__ __align__(16) double dq_smem[];
    double (*As)[QK][QLD] = reinterpret_cast<double (*)[QK][QLD]>(dq_smem);                       // [QNS], k-major
    double (*Bs)[QK][TN + 4] = reinterpret_cast<double (*)[QK][TN + 4]>(dq_smem + QNS * QK * QLD);  // [QNS]
    constexpr int AL = QK * DM / NT;                      // A elements per thread and stage
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm0 = (warp >> 2) * (MI * 8), wn0 = (warp & 3) * (TN / 4);
    const int g = lane >> 2, q = lane & 3;                // fragment coordinates (PTX ISA, m8n8k4 .f64)
    // Tile order: bands of RB column tiles, row tiles fastest inside a band, so that the CTAs in flight together share
    // few B panels (a plain row-major order re-read all of B from DRAM on every wave: 4x the algorithmic traffic)
    int tx = blockIdx.x, ty = blockIdx.y;
    {
        constexpr int RB = 16;
        const int gx = gridDim.x, gy = gridDim.y;
        const int lin = blockIdx.y * gx + blockIdx.x;
        const int band = lin / (RB * gy);
        const int bw = min(RB, gx - band * RB);            // the last band may be narrower
        const int within = lin - band * RB * gy;
        ty = within / bw;
        tx = band * RB + within - ty * bw;
    }
    const int64_t m0 = (int64_t)ty * DM, n0 = (int64_t)tx * TN;
    if (m0 >= M) return;                                   // only when *mact clipped M below the grid
    double acc[MI][NJ][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NJ; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    // QNS-stage cp.async ring: 8-byte copies scatter A into the k-major tile, zero-fill outside the matrix
    auto issue = [&](int64_t k0, int buf) {
#pragma unroll
        for (int t = 0; t < AL; ++t) {
            // a warp copies 8 rows x 4 consecutive k (one 32-byte sector per row): its 32 scattered 8-byte writes
            // into the k-major tile then fall on every bank pair exactly twice (QLD = 4 mod 16), the minimum
            const int idx = tid + t * NT;
            const int kk = 4 * ((idx >> 5) & 3) + (idx & 3), mm = 8 * (idx >> 7) + ((idx >> 2) & 7);
            const int64_t m = m0 + mm, k = k0 + kk;
            const bool ok = m < M && k < K;
            cp_async8(&As[buf][kk][mm], ok ? A + m * lda + k : A, ok);
        }
#pragma unroll
        for (int t = 0; t < BL; ++t) {
            const int idx = tid + t * NT;
            const int nn = idx % TN, kb = idx / TN;
            const int64_t n = n0 + nn, k2 = k0 + kb;
            const bool ok = n < N && k2 < K;
            cp_async8(&Bs[buf][kb][nn], ok ? B + k2 * ldb + n : B, ok);
        }
    };
    if constexpr (!ASSIGN) {                               // the C tile is wanted at the end: start moving it into L2 now
#pragma unroll
        for (int i = 0; i < MI; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int64_t m = m0 + wm0 + i * 8 + g, n = n0 + wn0 + j * 8 + q * 2;
                if (m < M && n < N) asm volatile("prefetch.global.L2 [%0];" ::"l"(C + m * ldc + n));
            }
    }
    const int64_t nk = (K + QK - 1) / QK;
#pragma unroll
    for (int st = 0; st < QNS - 1; ++st) {
        if (st < nk) issue((int64_t)st * QK, st);
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    for (int64_t kt = 0; kt < nk; ++kt) {
        asm volatile("cp.async.wait_group %0;" ::"n"(QNS - 2) : "memory");
        __syncthreads();                                   // stage kt has landed; stage kt-1's buffer is free
        if (kt + QNS - 1 < nk) issue((kt + QNS - 1) * QK, (int)((kt + QNS - 1) % QNS));
        asm volatile("cp.async.commit_group;" ::: "memory");
        const int buf = (int)(kt % QNS);
#pragma unroll
        for (int ks = 0; ks < QK; ks += 4) {
            double a[MI], b[NJ];
#pragma unroll
            for (int i = 0; i < MI; ++i) a[i] = As[buf][ks + q][wm0 + i * 8 + g];
#pragma unroll
            for (int j = 0; j < NJ; ++j) b[j] = Bs[buf][ks + q][wn0 + j * 8 + g];
#pragma unroll
            for (int i = 0; i < MI; ++i)
#pragma unroll
                for (int j = 0; j < NJ; ++j) dmma_8x8x4(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if constexpr (ASSIGN) {
        __syncthreads();                                   // every read of B (possibly = C) is done
#pragma unroll
        for (int i = 0; i < MI; ++i) {
            const int64_t m = m0 + wm0 + i * 8 + g;
            if (m >= M) continue;
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int64_t n = n0 + wn0 + j * 8 + q * 2;
                double* pc = C + m * ldc + n;
                if (n < N) pc[0] = acc[i][j][0];
                if (n + 1 < N) pc[1] = acc[i][j][1];
            }
        }
    } else {
        // C -= acc in batches of four tile rows: all the loads of a batch are issued before the first store, so the
        // epilogue costs one DRAM round trip per batch instead of one per element pair (load -> subtract -> store
        // chains were 15 % of the warp samples of the largest update)
        constexpr int EB = 4;
#pragma unroll
        for (int ib = 0; ib < MI; ib += EB) {
            double2 cv[EB][NJ];
            bool fast[EB][NJ];
#pragma unroll
            for (int ii = 0; ii < EB; ++ii)
#pragma unroll
                for (int j = 0; j < NJ; ++j) {
                    const int64_t m = m0 + wm0 + (ib + ii) * 8 + g, n = n0 + wn0 + j * 8 + q * 2;
                    const double* pc = C + m * ldc + n;
                    fast[ii][j] = m < M && n + 1 < N && ((reinterpret_cast<uintptr_t>(pc) & 15) == 0);
                    cv[ii][j] = fast[ii][j] ? __ldcg(reinterpret_cast<const double2*>(pc)) : make_double2(0.0, 0.0);
                }
#pragma unroll
            for (int ii = 0; ii < EB; ++ii)
#pragma unroll
                for (int j = 0; j < NJ; ++j) {
                    const int64_t m = m0 + wm0 + (ib + ii) * 8 + g, n = n0 + wn0 + j * 8 + q * 2;
                    if (m >= M) continue;
                    double* pc = C + m * ldc + n;
                    if (fast[ii][j]) {
                        cv[ii][j].x -= acc[ib + ii][j][0];
                        cv[ii][j].y -= acc[ib + ii][j][1];
                        *reinterpret_cast<double2*>(pc) = cv[ii][j];
                    } else {
                        if (n < N) pc[0] -= acc[ib + ii][j][0];
                        if (n + 1 < N) pc[1] -= acc[ib + ii][j][1];
                    }
                }
        }
    }
}

// ---------------------------------------------------------------- F3: inverses of the diagonal blocks
// Blocked substitution on the right-hand sides (F3) with explicit inverses of the TB x TB diagonal blocks of L and
// U: X_t = inv(D_t).B_t is then a tensor-pipe product instead of a chain of dependent leaf solves.  One CTA per
// block, thread j owns column j of the inverse (kept in shared memory), L/U entries are warp-uniform loads.
constexpr int TB = 128;
template <bool LOWER>
__global__ void __launch_bounds__(TB) f64_tri_inv_kernel(const double* __restrict__ A, int64_t n, int64_t lda,
                                                         double* __restrict__ inv /* [blocks][TB][TB] */) {
    extern __shared__ double XS[];                        // [TB][TB + 1]
    constexpr int LX = TB + 1;
    const int j = threadIdx.x;
    const int64_t t0 = (int64_t)blockIdx.x * TB;
    const int nb = (int)min((int64_t)TB, n - t0);
    const double* D = A + t0 * lda + t0;
    double* out = inv + (size_t)blockIdx.x * TB * TB;
    if (LOWER) {
        if (j < nb) {
            XS[j * LX + j] = 1.0;
            for (int i = j + 1; i < nb; ++i) {
                double s0 = 0.0, s1 = 0.0;
                int qq = j;
                for (; qq + 1 < i; qq += 2) {
                    s0 += D[(int64_t)i * lda + qq] * XS[qq * LX + j];
                    s1 += D[(int64_t)i * lda + qq + 1] * XS[(qq + 1) * LX + j];
                }
                if (qq < i) s0 += D[(int64_t)i * lda + qq] * XS[qq * LX + j];
                XS[i * LX + j] = -(s0 + s1);
            }
        }
    } else {
        if (j < nb) {
            XS[j * LX + j] = 1.0 / D[(int64_t)j * lda + j];
            for (int i = j - 1; i >= 0; --i) {
                double s0 = 0.0, s1 = 0.0;
                int qq = i + 1;
                for (; qq + 1 <= j; qq += 2) {
                    s0 += D[(int64_t)i * lda + qq] * XS[qq * LX + j];
                    s1 += D[(int64_t)i * lda + qq + 1] * XS[(qq + 1) * LX + j];
                }
                if (qq <= j) s0 += D[(int64_t)i * lda + qq] * XS[qq * LX + j];
                XS[i * LX + j] = -(s0 + s1) / D[(int64_t)i * lda + i];
            }
        }
    }
    __syncthreads();
    for (int e = j; e < TB * TB; e += TB) {
        const int r = e / TB, c = e % TB;
        const bool tri = LOWER ? (c <= r) : (c >= r);
        out[e] = (r < nb && c < nb && tri) ? XS[r * LX + c] : 0.0;
    }
}

constexpr size_t dmma_smem_bytes(int tn) { return (size_t)(QNS * QK * QLD + QNS * QK * (tn + 4)) * sizeof(double); }

struct F64 {
    double* A; int64_t n, lda;
    double* B; int64_t nrhs, ldb;
    double tol;
    cudaStream_t s;
    Cand* cand; double2* target; long long* ipiv; int* info;
    double* inv;                // inverted diagonal blocks of L and U (F3)
    int grid, rows_cap;         // cooperative grid size and the smem row capacity per CTA
    int panel_threads;
    int cluster_ctas;           // CTAs of the panel cluster (0: cluster launch not available)
    size_t smem_max;
};

int dgemm_sub(F64& c, double* C, int64_t ldc, const double* A, int64_t lda, const double* B, int64_t ldb, int64_t M,
              int64_t N, int64_t K, bool assign = false, const int* kact = nullptr, const int* mact = nullptr,
              const long long* row0 = nullptr) {
    if (M <= 0 || N <= 0 || K <= 0) return LINAC_OK;
    const DevShape ds{kact, mact, row0};
    // 128 x 64 tiles with two CTAs per SM (16 warps in flight) beat one 128 x 128 CTA per SM on every shape measured
    // (c4: 225 -> 217 ms); option f64_mma = 2 keeps the 128 x 128 tile for A/B runs
    const bool skinny = N <= 64 || assign || options().f64_mma != 2;
    const int tn = skinny ? 64 : DN;
    dim3 grid((unsigned)((N + tn - 1) / tn), (unsigned)((M + DM - 1) / DM));
    if (assign)
        dgemm_sub_mma_kernel<64, true, 8><<<grid, 256, dmma_smem_bytes(64), c.s>>>(C, ldc, A, lda, B, ldb, M, N, K, ds);
    else if (options().f64_mma == 0 && kact == nullptr)
        dgemm_sub_kernel<<<grid, DTHREADS, 0, c.s>>>(C, ldc, A, lda, B, ldb, M, N, K);
    else if (skinny)
        dgemm_sub_mma_kernel<64, false, 8><<<grid, 256, dmma_smem_bytes(64), c.s>>>(C, ldc, A, lda, B, ldb, M, N, K, ds);
    else
        dgemm_sub_mma_kernel<128, false, 8><<<grid, 256, dmma_smem_bytes(128), c.s>>>(C, ldc, A, lda, B, ldb, M, N, K, ds);
    LINAC_CUDA(cudaGetLastError());
    stats().kernel_launches++;
    stats().update_macs += M * N * K;
    return LINAC_OK;
}

// F3: B <- U^{-1} L^{-1} B by blocks of TB rows with the inverted diagonal blocks: X_t = inv(D_t).B_t (one CTA per 64
// right-hand sides, in place), then B_rest -= A[rest, t].X_t on the tensor pipe.
int solve_rhs_f64(F64& c) {
    const int64_t nblk = (c.n + TB - 1) / TB;
    const size_t smem = (size_t)TB * (TB + 1) * sizeof(double);
    LINAC_CUDA(cudaFuncSetAttribute(f64_tri_inv_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    LINAC_CUDA(cudaFuncSetAttribute(f64_tri_inv_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    double* invL = c.inv;
    double* invU = c.inv + (size_t)nblk * TB * TB;
    f64_tri_inv_kernel<true><<<(unsigned)nblk, TB, smem, c.s>>>(c.A, c.n, c.lda, invL);
    f64_tri_inv_kernel<false><<<(unsigned)nblk, TB, smem, c.s>>>(c.A, c.n, c.lda, invU);
    LINAC_CUDA(cudaGetLastError());
    stats().kernel_launches += 2;
    for (int64_t t = 0; t < nblk; ++t) {                                  // forward: L
        const int64_t t0 = t * TB, nb = std::min<int64_t>(TB, c.n - t0);
        double* Bt = c.B + t0 * c.ldb;
        int rc = dgemm_sub(c, Bt, c.ldb, invL + (size_t)t * TB * TB, TB, Bt, c.ldb, nb, c.nrhs, nb, true);
        if (rc) return rc;
        rc = dgemm_sub(c, Bt + nb * c.ldb, c.ldb, c.A + (t0 + nb) * c.lda + t0, c.lda, Bt, c.ldb, c.n - t0 - nb, c.nrhs, nb);
        if (rc) return rc;
    }
    for (int64_t t = nblk - 1; t >= 0; --t) {                             // backward: U
        const int64_t t0 = t * TB, nb = std::min<int64_t>(TB, c.n - t0);
        double* Bt = c.B + t0 * c.ldb;
        int rc = dgemm_sub(c, Bt, c.ldb, invU + (size_t)t * TB * TB, TB, Bt, c.ldb, nb, c.nrhs, nb, true);
        if (rc) return rc;
        rc = dgemm_sub(c, c.B, c.ldb, c.A + t0, c.lda, Bt, c.ldb, t0, c.nrhs, nb);
        if (rc) return rc;
    }
    return LINAC_OK;
}

// X <- L^{-1} X for the unit-lower block at [t0, t0+nb) on an arbitrary row-major X (ldx, ncols).
int trsm_lower_f64(F64& c, double* X, int64_t ldx, int64_t ncols, int64_t t0, int64_t nb) {
    if (nb <= 0 || ncols <= 0) return LINAC_OK;
    if (nb <= FW) {
        if (nb == FW)
            f64_trsm_lower32_kernel<<<(unsigned)((ncols + FT2 - 1) / FT2), FT2, 0, c.s>>>(X, ldx, ncols, c.A, c.lda, t0);
        else
            f64_trsm_lower_kernel<<<(unsigned)((ncols + FT - 1) / FT), FT, 0, c.s>>>(X, ldx, ncols, c.A, c.lda, t0, (int)nb);
        LINAC_CUDA(cudaGetLastError());
        stats().kernel_launches++;
        return LINAC_OK;
    }
    const int64_t h = std::max<int64_t>(FW, nb / 2 / FW * FW);
    int rc = trsm_lower_f64(c, X, ldx, ncols, t0, h);
    if (rc) return rc;
    rc = dgemm_sub(c, X + h * ldx, ldx, c.A + (t0 + h) * c.lda + t0, c.lda, X, ldx, nb - h, ncols, h);
    if (rc) return rc;
    return trsm_lower_f64(c, X + h * ldx, ldx, ncols, t0 + h, nb - h);
}

int trsm_upper_f64(F64& c, double* X, int64_t ldx, int64_t ncols, int64_t t0, int64_t nb) {
    if (nb <= 0 || ncols <= 0) return LINAC_OK;
    if (nb <= FW) {
        f64_trsm_upper_kernel<<<(unsigned)((ncols + FT - 1) / FT), FT, 0, c.s>>>(X, ldx, ncols, c.A, c.lda, t0, (int)nb);
        LINAC_CUDA(cudaGetLastError());
        stats().kernel_launches++;
        return LINAC_OK;
    }
    const int64_t h = std::max<int64_t>(FW, nb / 2 / FW * FW);
    int rc = trsm_upper_f64(c, X + h * ldx, ldx, ncols, t0 + h, nb - h);
    if (rc) return rc;
    rc = dgemm_sub(c, X, ldx, c.A + t0 * c.lda + t0 + h, c.lda, X + h * ldx, ldx, h, ncols, nb - h);
    if (rc) return rc;
    return trsm_upper_f64(c, X, ldx, ncols, t0, h);
}

int panel_f64(F64& c, int64_t j0, int w) {
    const int64_t m = c.n - j0;
    int rows_per_cta = (int)((m + c.grid - 1) / c.grid);
    rows_per_cta = std::max(rows_per_cta, 1);
    if (rows_per_cta > c.rows_cap) return LINAC_ERR_INVALID_ARG;
    size_t smem = (size_t)rows_per_cta * (FW + 2) * sizeof(double);
    double* A = c.A; int64_t n = c.n, lda = c.lda; double tol = c.tol;
    Cand* cand = c.cand; double2* target = c.target; long long* ipiv = c.ipiv; int* info = c.info;
    unsigned tag0 = options().f64_panel_tags != 0 ? (unsigned)(j0 + 1) : 0u;   // column j carries tag j + 1 within a solve
    long long* state = nullptr; F64Rec* rec = nullptr; int32_t* pivcols = nullptr;      // RREF mode only
    void* args[] = {&A, &n, &lda, &j0, &w, &rows_per_cta, &tol, &cand, &target, &ipiv, &info, &tag0, &state, &rec, &pivcols};
    if (c.cluster_ctas > 0 && m <= (int64_t)c.cluster_ctas * std::min<int64_t>(c.rows_cap, options().f64_cluster_rows)) {
        rows_per_cta = std::max(1, (int)((m + c.cluster_ctas - 1) / c.cluster_ctas));
        smem = (size_t)rows_per_cta * (FW + 2) * sizeof(double);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(c.cluster_ctas);
        cfg.blockDim = dim3(512);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = c.s;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)c.cluster_ctas;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        LINAC_CUDA(cudaLaunchKernelEx(&cfg, f64_panel_kernel<512, true, false>, A, n, lda, j0, w, rows_per_cta, tol, cand, target, ipiv, info, 0u, state, rec, pivcols));
    } else if (c.panel_threads == 1024)
        LINAC_CUDA(cudaLaunchCooperativeKernel((void*)f64_panel_kernel<1024, false, false>, dim3(c.grid), dim3(1024), args, smem, c.s));
    else if (c.panel_threads == 512)
        LINAC_CUDA(cudaLaunchCooperativeKernel((void*)f64_panel_kernel<512, false, false>, dim3(c.grid), dim3(512), args, smem, c.s));
    else
        LINAC_CUDA(cudaLaunchCooperativeKernel((void*)f64_panel_kernel<256, false, false>, dim3(c.grid), dim3(256), args, smem, c.s));
    // exchanges on the rest of A (left L part and right trailing part) and on B
    const int64_t ncol = c.n;
    f64_swap_kernel<<<(unsigned)((ncol + 255) / 256), 256, 0, c.s>>>(c.A, c.lda, 0, ncol, j0, j0 + w, c.ipiv, j0, w);
    LINAC_CUDA(cudaGetLastError());
    if (c.nrhs > 0) {
        f64_swap_kernel<<<(unsigned)((c.nrhs + 255) / 256), 256, 0, c.s>>>(c.B, c.ldb, 0, c.nrhs, -1, -1, c.ipiv, j0, w);
        LINAC_CUDA(cudaGetLastError());
    }
    stats().kernel_launches += 3;
    stats().panels++;
    return LINAC_OK;
}

// LU of columns [j0, j1) (square part: rows >= j0), right-looking recursion inside the range.
int factor_f64(F64& c, int64_t j0, int64_t j1) {
    const int64_t w = j1 - j0;
    if (w <= 0) return LINAC_OK;
    if (w <= FW) return panel_f64(c, j0, (int)w);
    const int64_t h = std::max<int64_t>(FW, w / 2 / FW * FW);
    const int64_t jm = j0 + h;
    int rc = factor_f64(c, j0, jm);
    if (rc) return rc;
    rc = trsm_lower_f64(c, c.A + j0 * c.lda + jm, c.lda, j1 - jm, j0, h);
    if (rc) return rc;
    rc = dgemm_sub(c, c.A + jm * c.lda + jm, c.lda, c.A + jm * c.lda + j0, c.lda, c.A + j0 * c.lda + jm, c.lda,
                   c.n - jm, j1 - jm, h);
    if (rc) return rc;
    return factor_f64(c, jm, j1);
}

// Top level: a flat right-looking sweep over strips of `f64_strip` columns (each factored by the recursion above, then
// one U12 solve and ONE full-size trailing update with K = strip width), so that the bulk of the flops runs in
// square, many-tile DMMA launches instead of the recursion's skinny mid-level products.
int factor_flat_f64(F64& c) {
    const int64_t W = options().f64_strip;
    if (W <= 0 || c.n <= W) return factor_f64(c, 0, c.n);
    for (int64_t s0 = 0; s0 < c.n; s0 += W) {
        const int64_t s1 = std::min(c.n, s0 + W);
        int rc = factor_f64(c, s0, s1);
        if (rc) return rc;
        if (s1 >= c.n) break;
        rc = trsm_lower_f64(c, c.A + s0 * c.lda + s1, c.lda, c.n - s1, s0, s1 - s0);
        if (rc) return rc;
        rc = dgemm_sub(c, c.A + s1 * c.lda + s1, c.lda, c.A + s1 * c.lda + s0, c.lda, c.A + s0 * c.lda + s1, c.lda,
                       c.n - s1, c.n - s1, s1 - s0);
        if (rc) return rc;
    }
    return LINAC_OK;
}

// ---------------------------------------------------------------- floating-point RREF
// linac_rref_f64: the paper's original mode -- a rectangular, possibly rank-deficient
// matrix reduced to echelon form with a threshold.  Blocked Gauss-Jordan over 32-column panels, no host
// synchronisation inside the loop (row counter and panel records live on the device):
//   f64_panel_kernel<RREF>     pivot search with partial pivoting and the threshold test on the updated column
//   f64_rref_swap_kernel       row exchanges (K5)
//   f64_rref_pivot_rows_kernel U = D^-1 . A[pivot rows, j0:], D = the panel's pivot block (Gauss-Jordan without
//                              further pivoting: the rows are in the order partial pivoting chose them), exactly the
//                              identity on the pivot columns
//   f64_rref_tinv_kernel       T = D^-1
//   f64_rref_lcopy_kernel      L[k][t] = A[k][pivot column t], zero for the pivot rows themselves
//   dgemm_sub_mma_kernel       A -= L . U for ALL rows (above too, as in the paper's RowReduce), on DMMA: at once on the
//                              columns of the panel's 128-column strip, once per strip (K = 128) right of it
// so the matrix ends as the RREF without a back-elimination pass.
// The panel's exchanges (ipiv[i0 + a] <-> i0 + a, a = 0 .. r-1, in that order) touch at most 2 r rows: thread 0 composes
// them into one permutation of those rows, then a CTA moves 32 columns of them through shared memory -- two memory round
// trips instead of r dependent ones.
__global__ void __launch_bounds__(256) f64_rref_swap_kernel(double* __restrict__ M, int64_t ld, int64_t c0, int64_t cols,
                                                           const F64Rec* __restrict__ rec, const long long* __restrict__ ipiv) {
    __shared__ long long s_row[2 * FW];                     // the touched rows: the panel's pivot rows, then their partners
    __shared__ long long s_piv[FW];
    __shared__ int s_cur[2 * FW];                           // s_cur[k] = the slot whose ORIGINAL content ends in slot k
    __shared__ int s_n;
    __shared__ double tile[2 * FW][33];
    const int r = rec->r;
    if (r == 0) return;
    const int64_t i0 = rec->i0;
    const int tid = threadIdx.x;
    if (tid < r) s_piv[tid] = ipiv[i0 + tid];
    __syncthreads();
    if (tid < 32) {                                         // warp 0: lane k keeps partner slot r + k
        long long ext = -1;
        int n = r;
        bool any = false;
        if (tid < r) { s_row[tid] = i0 + tid; s_cur[tid] = tid; }
        __syncwarp();
        for (int a = 0; a < r; ++a) {
            const long long sr = s_piv[a];
            if (sr == i0 + a) continue;
            any = true;
            int k;
            if (sr < i0 + r) k = (int)(sr - i0);
            else {
                const unsigned m = __ballot_sync(0xffffffffu, ext == sr);
                if (m) k = r + __ffs(m) - 1;
                else {
                    k = n;
                    if (tid == n - r) { ext = sr; s_row[n] = sr; s_cur[n] = n; }
                    ++n;
                    __syncwarp();
                }
            }
            if (tid == 0) {
                const int t = s_cur[a];
                s_cur[a] = s_cur[k];
                s_cur[k] = t;
            }
            __syncwarp();
        }
        if (tid == 0) s_n = any ? n : 0;
    }
    __syncthreads();
    const int n = s_n;
    if (n == 0) return;
    const int cx = tid & 31, g = tid >> 5;
    const int64_t c = c0 + (int64_t)blockIdx.x * 32 + cx;
    if (c < cols)
        for (int k = g; k < n; k += 8) tile[k][cx] = M[s_row[k] * ld + c];
    __syncthreads();
    if (c < cols)
        for (int k = g; k < n; k += 8)
            if (s_cur[k] != k) M[s_row[k] * ld + c] = tile[s_cur[k]][cx];
}

// T = D^-1, D = A[i0 : i0+r, pivot columns] after the exchanges (one CTA; its own launch, so that the kernel below can
// overwrite the pivot rows while every CTA of it reads the same T).
__global__ void __launch_bounds__(128) f64_rref_tinv_kernel(const double* __restrict__ A, int64_t ld, int64_t j0,
                                                           const F64Rec* __restrict__ rec, double* __restrict__ Tout) {
    __shared__ double G[FW][2 * FW + 1];
    __shared__ int s_pc[FW];
    const int r = rec->r;
    const int tid = threadIdx.x;
    if (r == 0) return;
    const int64_t i0 = rec->i0;
    if (tid < FW) s_pc[tid] = rec->pc[tid];
    __syncthreads();
    for (int e = tid; e < FW * 2 * FW; e += 128) {
        const int a = e / (2 * FW), b = e % (2 * FW);
        double v = 0.0;
        if (a < r) {
            if (b < FW) { if (b < r) v = A[(i0 + a) * ld + j0 + s_pc[b]]; }
            else v = (b - FW == a) ? 1.0 : 0.0;
        }
        G[a][b] = v;
    }
    __syncthreads();
    // Gauss-Jordan on [D | I]: thread = (row a, 16 columns); two phases per step so nobody reads a half-updated row t
    const int a = tid & 31, cg0 = (tid >> 5) * 16;          // a warp = 32 rows x the same 16 columns: conflict-free
    for (int t = 0; t < r; ++t) {
        // one reciprocal per step: a division per entry took the slow path of the double-precision division on every
        // zero of [D | I] (116 us per panel)
        const double rd = 1.0 / G[t][t], h = G[a][t];
        double pt[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) pt[q] = G[t][cg0 + q] * rd;
        __syncthreads();
        if (a < r) {
#pragma unroll
            for (int q = 0; q < 16; ++q) G[a][cg0 + q] = a == t ? pt[q] : G[a][cg0 + q] - h * pt[q];
        }
        __syncthreads();
    }
    for (int e = tid; e < FW * FW; e += 128) Tout[e] = G[e / FW][FW + e % FW];
}

// U = T . A[i0 : i0+r, c] for the columns c >= j0 (thread per column); written to the pivot rows and to the U buffer.
__global__ void __launch_bounds__(128) f64_rref_pivot_rows_kernel(double* __restrict__ A, int64_t ld, int64_t j0, int64_t cols,
                                                                 const F64Rec* __restrict__ rec, const double* __restrict__ Tin,
                                                                 double* __restrict__ U, int64_t ldu) {
    __shared__ double Ts[FW][FW + 1];
    __shared__ int s_pc[FW];
    const int r = rec->r;
    const int tid = threadIdx.x;
    if (r == 0) return;
    const int64_t i0 = rec->i0;
    if (tid < FW) s_pc[tid] = rec->pc[tid];
    for (int e = tid; e < FW * FW; e += 128) Ts[e / FW][e % FW] = Tin[e];
    __syncthreads();
    const int64_t c = j0 + (int64_t)blockIdx.x * 128 + tid;
    if (c >= cols) return;
    int piv_ord = -1;                                       // is c one of the panel's pivot columns?
    if (c - j0 < FW)
        for (int t = 0; t < r; ++t) if (s_pc[t] == (int)(c - j0)) piv_ord = t;
    double x[FW];
#pragma unroll
    for (int b = 0; b < FW; ++b) x[b] = b < r ? A[(i0 + b) * ld + c] : 0.0;
    for (int q = 0; q < FW; ++q) {
        double acc = 0.0;
        if (q < r) {
#pragma unroll
            for (int b = 0; b < FW; ++b) acc += Ts[q][b] * x[b];
            if (piv_ord >= 0) acc = piv_ord == q ? 1.0 : 0.0;      // exactly the identity on the pivot columns
            A[(i0 + q) * ld + c] = acc;
        }
        U[(int64_t)q * ldu + c] = acc;
    }
}

// L[k][col_off + t] = A[k][pivot column t] (the raw entries ARE the multipliers once the pivot rows hold T . rows);
// for the panel's own pivot rows the whole row of L up to col_off + 32 is zeroed: this panel's multipliers, and those
// of the strip's earlier panels, which the catch-up product has just applied to these rows.
__global__ void f64_rref_lcopy_kernel(const double* __restrict__ A, int64_t ld, int64_t rows, int64_t j0,
                                      const F64Rec* __restrict__ rec, double* __restrict__ L, int ldl, int col_off) {
    const int r = rec->r;
    if (r == 0) return;
    const int t = threadIdx.x & 31;
    const int64_t i0 = rec->i0;
    const int pc = rec->pc[t];
    for (int64_t k = (int64_t)blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5); k < rows; k += (int64_t)gridDim.x * (blockDim.x / 32)) {
        const bool pivot_row = k >= i0 && k < i0 + r;
        if (pivot_row) {
            for (int q = t; q < col_off + FW; q += 32) L[k * ldl + q] = 0.0;
        } else {
            L[k * ldl + col_off + t] = pc >= 0 ? A[k * ld + j0 + pc] : 0.0;
        }
    }
}

// Reading Q19: what the thresholds declared zero is written as zero -- rows >= rank, and the entries of a pivot row
// left of its pivot (sub-threshold residue in free columns).  One CTA per row.
__global__ void f64_rref_finalize_kernel(double* __restrict__ A, int64_t ld, int64_t rows, int64_t cols,
                                         const long long* __restrict__ state, const int32_t* __restrict__ pivcols) {
    const int64_t k = blockIdx.x;
    const int64_t rank = *state;
    const int64_t end = k < rank ? pivcols[k] : cols;
    for (int64_t c = threadIdx.x; c < end; c += blockDim.x) A[k * ld + c] = 0.0;
}

constexpr int RW = 128;                   // strip width of linac_rref_f64: the wide update's K
size_t f64_rref_workspace_bytes(int64_t rows, int64_t cols) {
    const int64_t ldu = (cols + 63) / 64 * 64;
    return 16384 + 2 * 1024 * sizeof(Cand) + 2 * FW * sizeof(double2) + (size_t)std::max<int64_t>(rows, 1) * 8 +
           (size_t)RW * ldu * 8 + (size_t)rows * RW * 8 + (size_t)std::max<int64_t>(1, std::min(rows, cols)) * 4;
}

size_t f64_workspace_bytes(int64_t n) {
    (void)n;
    const size_t inv = 2 * (size_t)((n + TB - 1) / TB) * TB * TB * sizeof(double);
    return 8192 + 2 * 1024 * sizeof(Cand) + 2 * FW * sizeof(double2) + (size_t)std::max<int64_t>(n, 1) * 8 + 1024 + inv;
}

}  // namespace
}  // namespace linac

using namespace linac;

extern "C" {

int linac_solve_f64_workspace(int64_t n, int64_t nrhs, size_t* bytes) {
    if (!bytes || n < 0 || nrhs < 0) return LINAC_ERR_INVALID_ARG;
    *bytes = n == 0 ? 0 : f64_workspace_bytes(n);
    return LINAC_OK;
}

int linac_solve_f64(double* dA, int64_t n, int64_t lda, double* dB, int64_t nrhs, int64_t ldb, double tol, void* stream,
                    int64_t* info_out) {
    linac_stats& st = stats();
    st = linac_stats{};
    if (n < 0 || nrhs < 0 || !info_out) return LINAC_ERR_INVALID_ARG;
    *info_out = 0;
    if (n == 0) return LINAC_OK;
    if (!dA || lda < n || (nrhs > 0 && (!dB || ldb < nrhs))) return LINAC_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    Arena arena;
    rc = acquire_workspace(f64_workspace_bytes(n), &arena);
    if (rc) return rc;

    F64 c;
    c.A = dA; c.n = n; c.lda = lda; c.B = dB; c.nrhs = nrhs; c.ldb = ldb; c.s = s;
    c.tol = tol < 0 ? (double)n * 2.220446049250313e-16 : tol;
    int dev = 0, sms = 0, smem_optin = 0;
    LINAC_CUDA(cudaGetDevice(&dev));
    LINAC_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    LINAC_CUDA(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    c.grid = std::min(sms, 1024);
    c.panel_threads = (int)options().f64_panel_threads;
    if (options().f64_panel_grid > 0) c.grid = (int)std::min<int64_t>(sms, options().f64_panel_grid);
    c.smem_max = (size_t)smem_optin - 4096;
    c.rows_cap = (int)(c.smem_max / ((FW + 2) * sizeof(double)));
    if ((n + c.grid - 1) / c.grid > c.rows_cap) return LINAC_ERR_INVALID_ARG;   // n > ~118k: strip no longer fits on chip
    LINAC_CUDA(cudaFuncSetAttribute(f64_panel_kernel<256, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem_max));
    LINAC_CUDA(cudaFuncSetAttribute(f64_panel_kernel<512, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem_max));
    LINAC_CUDA(cudaFuncSetAttribute(f64_panel_kernel<1024, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem_max));
    c.cluster_ctas = 0;
    if (options().f64_panel_cluster > 0) {                 // one cluster of up to 16 CTAs (non-portable size), if the device places it
        const int want = (int)options().f64_panel_cluster;
        cudaError_t ce = cudaFuncSetAttribute(f64_panel_kernel<512, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem_max);
        if (ce == cudaSuccess && want > 8)
            ce = cudaFuncSetAttribute(f64_panel_kernel<512, true, false>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (ce == cudaSuccess) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(want);
            cfg.blockDim = dim3(512);
            cfg.dynamicSmemBytes = c.smem_max;
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = (unsigned)want;
            at[0].val.clusterDim.y = 1;
            at[0].val.clusterDim.z = 1;
            cfg.attrs = at;
            cfg.numAttrs = 1;
            int nclusters = 0;
            ce = cudaOccupancyMaxActiveClusters(&nclusters, f64_panel_kernel<512, true, false>, &cfg);
            if (ce == cudaSuccess && nclusters >= 1) c.cluster_ctas = want;
        }
        if (ce != cudaSuccess) (void)cudaGetLastError();    // not available: the cooperative kernel does every panel
    }
    LINAC_CUDA(cudaFuncSetAttribute(dgemm_sub_mma_kernel<128, false, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dmma_smem_bytes(128)));
    LINAC_CUDA(cudaFuncSetAttribute(dgemm_sub_mma_kernel<64, false, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dmma_smem_bytes(64)));
    LINAC_CUDA(cudaFuncSetAttribute(dgemm_sub_mma_kernel<64, true, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dmma_smem_bytes(64)));
    c.cand = (Cand*)arena.take(2 * 1024 * sizeof(Cand));
    c.target = (double2*)arena.take(2 * FW * sizeof(double2));
    c.ipiv = (long long*)arena.take((size_t)n * 8);
    c.info = (int*)arena.take(256);
    c.inv = nrhs > 0 ? (double*)arena.take(2 * (size_t)((n + TB - 1) / TB) * TB * TB * sizeof(double)) : nullptr;
    if (!c.cand || !c.target || !c.ipiv || !c.info || (nrhs > 0 && !c.inv)) return LINAC_ERR_WORKSPACE;
    const int big = INT_MAX;
    LINAC_CUDA(cudaMemcpyAsync(c.info, &big, sizeof(int), cudaMemcpyHostToDevice, s));
    LINAC_CUDA(cudaMemsetAsync(c.cand, 0, 2 * 1024 * sizeof(Cand), s));        // tags of an earlier solve must not match
    LINAC_CUDA(cudaMemsetAsync(c.target, 0, 2 * FW * sizeof(double2), s));

    CallEvents evs;
    rc = evs.create();
    if (rc) return rc;
    cudaEvent_t e0 = evs.ev0, e1 = evs.ev1;
    cudaEventRecord(e0, s);
    rc = launch_row_scale(dA, n, n, lda, dB, nrhs, ldb, c.info, s);                            // F1
    if (rc) return rc;
    st.kernel_launches++;
    // F2 with B as trailing columns: factor A in outer blocks so B's forward substitution is blocked too
    rc = factor_flat_f64(c);
    if (rc == LINAC_OK && nrhs > 0) {
        if (options().f64_rhs_inv != 0) rc = solve_rhs_f64(c);                                // F3, blocked with inverses
        else {
            rc = trsm_lower_f64(c, dB, ldb, nrhs, 0, n);                                      // forward substitution (L)
            if (rc == LINAC_OK) rc = trsm_upper_f64(c, dB, ldb, nrhs, 0, n);                  // back substitution (U)
        }
    }
    int h_info = INT_MAX;
    if (rc == LINAC_OK) {
        cudaEventRecord(e1, s);
        LINAC_CUDA(cudaMemcpyAsync(&h_info, c.info, sizeof(int), cudaMemcpyDeviceToHost, s));
    }
    cudaError_t e = cudaStreamSynchronize(s);
    st.host_syncs++;
    if (e != cudaSuccess) { set_cuda_error(e, "cudaStreamSynchronize(solve_f64)", __FILE__, __LINE__); rc = rc ? rc : LINAC_ERR_CUDA; }
    float ms = 0;
    if (rc == LINAC_OK) cudaEventElapsedTime(&ms, e0, e1);
    st.ms_total = ms;
    if (rc) return rc;
    if (h_info != INT_MAX) {
        *info_out = h_info;
        return LINAC_ERR_SINGULAR;
    }
    return LINAC_OK;
}

int linac_rref_f64_workspace(int64_t rows, int64_t cols, size_t* bytes) {
    if (!bytes || rows < 0 || cols < 0) return LINAC_ERR_INVALID_ARG;
    *bytes = (rows == 0 || cols == 0) ? 0 : f64_rref_workspace_bytes(rows, cols);
    return LINAC_OK;
}

// The reduction proper; `arena` already holds f64_rref_workspace_bytes(rows, cols) beyond what the caller took from it.
static int rref_f64_impl(double* dA, int64_t rows, int64_t cols, int64_t ld, double tol, cudaStream_t s, int64_t* rank_out,
                         int32_t* pivot_cols_out, Arena& arena) {
    linac_stats& st = stats();
    int rc = LINAC_OK;
    F64 c{};
    c.A = dA; c.n = rows; c.lda = ld; c.B = nullptr; c.nrhs = 0; c.ldb = 0; c.s = s;
    c.tol = tol < 0 ? (double)std::max(rows, cols) * 2.220446049250313e-16 : tol;
    int dev = 0, sms = 0, smem_optin = 0;
    LINAC_CUDA(cudaGetDevice(&dev));
    LINAC_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    LINAC_CUDA(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    c.grid = std::min(sms, 1024);
    c.smem_max = (size_t)smem_optin - 4096;
    c.rows_cap = (int)(c.smem_max / ((FW + 2) * sizeof(double)));
    int rows_per_cta = (int)((rows + c.grid - 1) / c.grid);
    if (rows_per_cta > c.rows_cap) return LINAC_ERR_INVALID_ARG;          // rows > ~118k: the strip no longer fits on chip
    LINAC_CUDA(cudaFuncSetAttribute(f64_panel_kernel<512, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem_max));
    LINAC_CUDA(cudaFuncSetAttribute(dgemm_sub_mma_kernel<128, false, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dmma_smem_bytes(128)));
    LINAC_CUDA(cudaFuncSetAttribute(dgemm_sub_mma_kernel<64, false, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dmma_smem_bytes(64)));
    const int64_t mn = std::min(rows, cols), ldu = (cols + 63) / 64 * 64;
    Cand* cand = (Cand*)arena.take(2 * 1024 * sizeof(Cand));
    double2* target = (double2*)arena.take(2 * FW * sizeof(double2));
    long long* ipiv = (long long*)arena.take((size_t)rows * 8);
    long long* state = (long long*)arena.take(256);
    int* dummy_info = (int*)(state + 8);
    F64Rec* rec = (F64Rec*)arena.take(sizeof(F64Rec));
    double* U = (double*)arena.take((size_t)RW * ldu * 8);
    double* L = (double*)arena.take((size_t)rows * RW * 8);
    int32_t* d_piv = (int32_t*)arena.take((size_t)mn * 4);
    double* Tb = (double*)arena.take(FW * FW * 8);
    if (!cand || !target || !ipiv || !state || !rec || !U || !L || !d_piv || !Tb) return LINAC_ERR_WORKSPACE;
    LINAC_CUDA(cudaMemsetAsync(state, 0, 256, s));
    LINAC_CUDA(cudaMemsetAsync(cand, 0, 2 * 1024 * sizeof(Cand), s));
    LINAC_CUDA(cudaMemsetAsync(target, 0, 2 * FW * sizeof(double2), s));
    rc = launch_row_scale(dA, rows, cols, ld, nullptr, 0, 0, dummy_info, s);                         // K1/K2; zero rows stay zero
    if (rc) return rc;
    st.kernel_launches++;
    const size_t smem = (size_t)rows_per_cta * (FW + 2) * sizeof(double);
    double tolv = c.tol;
    int* info = dummy_info;
    // Strips of RW columns, panels of FW inside.  A panel's multipliers L_p (all rows) and normalised pivot rows U_p go
    // to column block p of L and row block p of U; the panel updates the strip's own columns at once (K = 32) and the
    // columns right of the strip once per strip (K = RW): A[:, right] -= L . U.  Before a panel's pivot rows are
    // normalised their right part is brought up to date with the strip's earlier panels (the catch-up product, row
    // offset and count read from the panel record on the device), and their rows of L are zeroed so the strip-wide
    // product does not apply those panels twice.  Row exchanges move the rows of L with the rows of A.
    const int rw = (int)std::max<int64_t>(FW, std::min<int64_t>(RW, options().f64_rref_strip / FW * FW));
    for (int64_t s0 = 0; s0 < cols; s0 += rw) {
        const int64_t s1 = std::min<int64_t>(cols, s0 + rw), nright = cols - s1;
        if (nright > 0 && rw > FW) {
            LINAC_CUDA(cudaMemsetAsync(L, 0, (size_t)rows * RW * 8, s));
            LINAC_CUDA(cudaMemsetAsync(U, 0, (size_t)RW * ldu * 8, s));
        }
        const bool deferred = nright > 0 && rw > FW;       // else every panel updates all the columns right of it at once
        for (int64_t j0 = s0; j0 < s1; j0 += FW) {
            int w = (int)std::min<int64_t>(FW, cols - j0);
            const int poff = (int)(j0 - s0);
            int64_t j0v = j0, nv = rows, ldv = ld;
            const int64_t nc = (deferred ? s1 : cols) - j0;
            unsigned tag0 = options().f64_panel_tags != 0 ? (unsigned)(j0 + 1) : 0u;
            void* args[] = {&dA, &nv, &ldv, &j0v, &w, &rows_per_cta, &tolv, &cand, &target, &ipiv, &info, &tag0, &state, &rec, &d_piv};
            LINAC_CUDA(cudaLaunchCooperativeKernel((void*)f64_panel_kernel<512, false, true>, dim3(c.grid), dim3(512), args, smem, s));
            f64_rref_swap_kernel<<<(unsigned)((cols - j0 + 31) / 32), 256, 0, s>>>(dA, ld, j0, cols, rec, ipiv);
            st.kernel_launches += 2;
            double* Up = deferred ? U + (size_t)poff * ldu : U;
            if (deferred && poff > 0) {
                f64_rref_swap_kernel<<<(unsigned)((poff + 31) / 32), 256, 0, s>>>(L, RW, 0, poff, rec, ipiv);
                st.kernel_launches++;
                rc = dgemm_sub(c, dA + s1, ld, L, RW, U + s1, ldu, FW, nright, poff, false, nullptr, &rec->r, &rec->i0);
                if (rc) return rc;
            }
            f64_rref_tinv_kernel<<<1, 128, 0, s>>>(dA, ld, j0, rec, Tb);
            f64_rref_pivot_rows_kernel<<<(unsigned)((cols - j0 + 127) / 128), 128, 0, s>>>(dA, ld, j0, cols, rec, Tb, Up, ldu);
            f64_rref_lcopy_kernel<<<(unsigned)std::min<int64_t>((rows + 7) / 8, 148 * 8), 256, 0, s>>>(dA, ld, rows, j0, rec,
                                                                                                      L, deferred ? RW : FW, deferred ? poff : 0);
            LINAC_CUDA(cudaGetLastError());
            st.kernel_launches += 3;
            st.panels++;
            rc = dgemm_sub(c, dA + j0, ld, deferred ? L + poff : L, deferred ? RW : FW, Up + j0, ldu, rows, nc, FW, false, &rec->r);
            if (rc) return rc;
        }
        if (deferred) {
            rc = dgemm_sub(c, dA + s1, ld, L, RW, U + s1, ldu, rows, nright, s1 - s0);
            if (rc) return rc;
        }
    }
    f64_rref_finalize_kernel<<<(unsigned)rows, 256, 0, s>>>(dA, ld, rows, cols, state, d_piv);
    LINAC_CUDA(cudaGetLastError());
    st.kernel_launches++;
    long long h_rank = 0;
    std::vector<int32_t> piv((size_t)mn);
    LINAC_CUDA(cudaMemcpyAsync(&h_rank, state, 8, cudaMemcpyDeviceToHost, s));
    LINAC_CUDA(cudaMemcpyAsync(piv.data(), d_piv, (size_t)mn * 4, cudaMemcpyDeviceToHost, s));
    LINAC_CUDA(cudaStreamSynchronize(s));
    st.host_syncs++;
    if (h_rank < 0 || h_rank > mn) return LINAC_ERR_INTERNAL;
    *rank_out = h_rank;
    if (pivot_cols_out) std::copy(piv.begin(), piv.begin() + h_rank, pivot_cols_out);
    return LINAC_OK;
}

int linac_rref_f64(double* dA, int64_t rows, int64_t cols, int64_t ld, double tol, void* stream, int64_t* rank_out,
                   int32_t* pivot_cols_out) {
    stats() = linac_stats{};
    if (rows < 0 || cols < 0 || rows >= (1ll << 31) || cols >= (1ll << 31) || !rank_out) return LINAC_ERR_INVALID_ARG;
    *rank_out = 0;
    if (rows == 0 || cols == 0) return LINAC_OK;
    if (!dA || ld < cols) return LINAC_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    Arena arena;
    rc = acquire_workspace(f64_rref_workspace_bytes(rows, cols), &arena);
    if (rc) return rc;
    return rref_f64_impl(dA, rows, cols, ld, tol, (cudaStream_t)stream, rank_out, pivot_cols_out, arena);
}

// ---------------------------------------------------------------- complex128 through the real embedding
// z = x + iy  ->  [[x, -y], [y, x]] is a ring homomorphism E from complex m x n matrices into real 2m x 2n ones: E(M A) =
// E(M) E(A), E of an invertible matrix is invertible, so E(A) and E(RREF(A)) have the same row space; E(RREF(A)) IS a
// reduced echelon matrix (a pivot 1 in (i, j) becomes the 2 x 2 identity in rows 2i, 2i+1 and columns 2j, 2j+1), and
// the reduced echelon form of a row space is unique: RREF_real(E(A)) = E(RREF_complex(A)).  The complex reduction is
// therefore the real one on the embedding -- the DMMA kernels above, unchanged -- between two element-wise kernels.
// It costs twice the flops of a native complex elimination (8 real multiply-adds per complex one instead of 4) and
// twice the memory; in exchange every kernel of the real path (tensor-pipe updates, device-resident control) serves.
// Rows 2i and 2i+1 of E(A) hold the same set of absolute values, so the real row rescaling gives both the scale
// max_c max(|Re|, |Im|) of complex row i (reading Q21) and the embedding survives it.
}  // extern "C"

namespace linac {
namespace {
__global__ void c128_expand_kernel(const double2* __restrict__ A, int64_t rows, int64_t cols, int64_t ld, double* __restrict__ E,
                                   int64_t lde) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cols) return;
    for (int64_t r = blockIdx.y; r < rows; r += gridDim.y) {
        const double2 z = A[r * ld + c];
        *reinterpret_cast<double2*>(E + (2 * r) * lde + 2 * c) = make_double2(z.x, -z.y);
        *reinterpret_cast<double2*>(E + (2 * r + 1) * lde + 2 * c) = make_double2(z.y, z.x);
    }
}
__global__ void c128_contract_kernel(double2* __restrict__ A, int64_t rows, int64_t cols, int64_t ld, const double* __restrict__ E,
                                     int64_t lde) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cols) return;
    for (int64_t r = blockIdx.y; r < rows; r += gridDim.y)
        A[r * ld + c] = make_double2(E[(2 * r) * lde + 2 * c], E[(2 * r + 1) * lde + 2 * c]);
}

}  // namespace
}  // namespace linac

extern "C" {

int linac_rref_c128_workspace(int64_t rows, int64_t cols, size_t* bytes) {
    if (!bytes || rows < 0 || cols < 0 || rows >= (1ll << 30) || cols >= (1ll << 30)) return LINAC_ERR_INVALID_ARG;
    *bytes = (rows == 0 || cols == 0) ? 0 : (size_t)2 * rows * 2 * cols * 8 + 1024 + f64_rref_workspace_bytes(2 * rows, 2 * cols);
    return LINAC_OK;
}

int linac_rref_c128(void* dA, int64_t rows, int64_t cols, int64_t ld, double tol, void* stream, int64_t* rank_out,
                    int32_t* pivot_cols_out) {
    stats() = linac_stats{};
    if (rows < 0 || cols < 0 || rows >= (1ll << 30) || cols >= (1ll << 30) || !rank_out) return LINAC_ERR_INVALID_ARG;
    *rank_out = 0;
    if (rows == 0 || cols == 0) return LINAC_OK;
    if (!dA || ld < cols || ((uintptr_t)dA & 15)) return LINAC_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    size_t need = 0;
    linac_rref_c128_workspace(rows, cols, &need);
    Arena arena;
    rc = acquire_workspace(need, &arena);
    if (rc) return rc;
    const int64_t lde = 2 * cols;
    double* E = (double*)arena.take((size_t)2 * rows * lde * 8, 1024);
    if (!E) return LINAC_ERR_WORKSPACE;
    const dim3 grid((unsigned)((cols + 127) / 128), (unsigned)std::min<int64_t>(rows, 8192));
    c128_expand_kernel<<<grid, 128, 0, s>>>((const double2*)dA, rows, cols, ld, E, lde);
    LINAC_CUDA(cudaGetLastError());
    int64_t rank2 = 0;
    std::vector<int32_t> piv2((size_t)2 * std::min(rows, cols) + 1);
    // the threshold defaults to the COMPLEX shape's max(rows, cols) * 2^-52, as the oracle's
    const double tolv = tol < 0 ? (double)std::max(rows, cols) * 2.220446049250313e-16 : tol;
    rc = rref_f64_impl(E, 2 * rows, 2 * cols, lde, tolv, s, &rank2, piv2.data(), arena);
    if (rc) return rc;
    // the real pivots must come in pairs (2j, 2j+1): anything else means the threshold fell between the two real
    // columns of one complex column (a head within a factor sqrt(2) of tol)
    if (rank2 & 1) return LINAC_ERR_SINGULAR;
    for (int64_t t = 0; t < rank2; t += 2)
        if ((piv2[t] & 1) || piv2[t + 1] != piv2[t] + 1) return LINAC_ERR_SINGULAR;
    c128_contract_kernel<<<grid, 128, 0, s>>>((double2*)dA, rows, cols, ld, E, lde);
    LINAC_CUDA(cudaGetLastError());
    LINAC_CUDA(cudaStreamSynchronize(s));
    stats().kernel_launches += 2;
    stats().host_syncs++;
    *rank_out = rank2 / 2;
    if (pivot_cols_out)
        for (int64_t t = 0; t < rank2; t += 2) pivot_cols_out[t / 2] = piv2[t] / 2;
    return LINAC_OK;
}

}  // extern "C"
