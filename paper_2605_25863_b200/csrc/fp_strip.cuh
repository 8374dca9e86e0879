// fp_strip.cuh -- S1-S4 of the F_p path for one STRIP of up to 8 base panels: a cooperative kernel, and the
// column-parallel triangular-solve leaf that follows it.
//
// One launch factors columns [j0, j0+ws) (ws <= SW_MAX) over the active rows >= i0, base panel by base panel
// (PW = 32 columns each), with the whole grid resident (one CTA of 1024 threads per SM).  Per base panel, between
// two grid barriers (strip_factor_kernel below has the details):
//
//   CTA 0        ahead update of the next panel's 32 candidate rows, then pivot search + T = (pivot block)^-1
//                of the NEXT panel from them                                       (S1, S2)
//   CTAs 1..     U12 = T.A12 on the pivot rows and A22 -= L21.U12 on the rows below, restricted to the
//                strip's columns right of the panel                               (S3/S4 inside the strip)
//   (if needed)  row exchanges on complete rows (K5); general-path factorisation by CTA 0
//
// so the ~10 dependent launches and the host round trip per base panel of a launch-per-step schedule become one
// grid barrier.  Everything right of the strip is updated afterwards by the row-block solve (trsm_strip_kernel)
// and the tensor-core Schur update.
//
// Storage convention: see fp_kernels.cuh (multipliers are the raw entries at the pivot columns).
#pragma once
#include <climits>
#include <cooperative_groups.h>

#include "linac_internal.h"

namespace linac {
namespace cg = cooperative_groups;

// The fields of the running calls: one slot per host thread inside the library (Context::slot), written once per
// call by the host (cudaMemcpyToSymbolAsync on the call's stream) and read through the constant bank, so no device
// function carries the descriptor in registers or on the stack.  The strip kernel keeps its slot in shared memory.
__constant__ ModP c_f[FIELD_SLOTS];

constexpr int SW_MAX = 256;                 // widest strip (columns)
constexpr int SNT = 1024;                   // threads per CTA of the strip kernel (32 warps)
constexpr int SRB = 256;                    // rows of one P2 tile
constexpr int MAXBP = SW_MAX / PW;          // base panels per strip

// d*x - h*y mod p with one reduction: d*x + (p-h)*y < 2^63.
__device__ __forceinline__ uint32_t lincomb(uint32_t d, uint32_t x, uint32_t h, uint32_t y, const ModP& f) {
    return reduce64((uint64_t)d * x + (uint64_t)(f.p - h) * y, f);
}

struct UPending {
    long long row0;                  // first pivot row (absolute), or -1 if nothing is pending
    long long col0;
    int r, nc;
};

struct StripSmem {
    int slot;                        // this launch's entry of c_f
    // ---- P1
    uint32_t W[2][PW][PW + 1];       // fast path: double-buffered block; general path: W[0] = chunk X, W[1] = Ep
    uint32_t G[PW][2 * PW + 1];      // general path phase 2: [D | I]
    uint32_t gs[2][PW];              // fast path: per-row scale / pivot value
    int epc[PW];                     // pivot column of pivot t (discovery order)
    long long esrc[PW];              // source row (absolute) of pivot t
    int ord[PW];                     // pivots sorted by pivot column
    uint32_t ginv[PW];
    long long pos_of[PW];
    int at[PW];
    int nsw;
    int fast_ok;
    int r_out;
    int last_r, last_nsw;            // CTA 0's own copy of the record it wrote last (saves it a round trip to L2)
    unsigned last_pcm;
    // ---- P2
    uint32_t Ts[PW][PW + 1];
    uint32_t Ar[PW][PW + 1];
    __align__(16) uint32_t Us[2][PW][PW];    // this CTA's U12 slices (slot 0: next panel's columns, slot 1: the rest)
    __align__(16) uint32_t Lk[PW][SRB + 4];  // L tile, k-major (pivot index, row)
    UPending pend[2];                // deferred write-back of Us[slot]
    // ---- CTA 0 running ahead: T and the candidate rows' multipliers with 16-byte aligned rows
    __align__(16) uint32_t Bt[PW][PW + 4];
    __align__(16) uint32_t Bl[PW][PW + 4];
};

// ------------------------------------------------------------------------------------------------
// P1, fast path: the 32 candidate rows i0..i0+31 and the 32 panel columns as one block, inverted IN
// PLACE by division-free Gauss-Jordan with row pivoting (first non-zero among the unused rows; for
// F_p any non-zero pivot will do).  Warp = block row (kept in registers), lane = column.
// Step c: every row k != q becomes d*row_k - h_k*row_q with d the pivot; the slot of column c then
// holds the column of the accumulated transform that belongs to source row q, and g_k tracks the
// scalar each row has been multiplied by (for q: the pivot value).  At the end
//   T[a][b] = g_{q_a}^-1 * W[q_a][b],   q_a = the row that pivoted column a,
// is the inverse of D = A[pivot rows in column order, panel].  Every product here is a Montgomery product
// (a*b*2^-32 mod p, four instructions instead of Barrett's fourteen): the extra factor 2^-32 only rescales
// rows, which a division-free elimination does not care about, and the tracked scales absorb it.  Fails (returns false, nothing
// written) as soon as a column has no pivot among the unused rows: the caller then runs the general
// path, which handles rank-deficient and multi-chunk panels.
// Block rows per working warp of the fast panel: 8 (4 warps, one per scheduler) or 4 (8 warps).
#ifndef FAST_RPW
#define FAST_RPW 4
#endif
#if FAST_RPW == 8
#define FAST_IF8(...) __VA_ARGS__
#else
#define FAST_IF8(...)
#endif
__device__ __forceinline__ bool panel_fast(StripSmem& sm, const uint32_t* A, int64_t ld, int64_t i0, int64_t j0) {
    const ModP& f = c_f[sm.slot];
    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    constexpr int FW = PW / FAST_RPW, RPW = FAST_RPW;          // working warps, block rows per warp (registers)
    uint32_t x0 = 0, x1 = 0, x2 = 0, x3 = 0, x4 = 0, x5 = 0, x6 = 0, x7 = 0;
    const int row0 = wq * RPW;
#define FAST_EACH_ROW(M) M(x0, 0) M(x1, 1) M(x2, 2) M(x3, 3) FAST_IF8(M(x4, 4) M(x5, 5) M(x6, 6) M(x7, 7))
    if (wq < FW) {
#define FAST_LOAD(X, I) X = A[(i0 + row0 + I) * ld + j0 + lane];
        FAST_EACH_ROW(FAST_LOAD)
#undef FAST_LOAD
#define FAST_PUT(X, I) sm.W[0][row0 + I][lane] = X;
        FAST_EACH_ROW(FAST_PUT)
#undef FAST_PUT
    }
    __syncthreads();
    if (wq < FW) {
        unsigned used = 0;
        uint32_t dtot = 1u;                       // product of the pivots so far (the scale of every unused row)
        bool ok = true;
#pragma unroll 1
        for (int c = 0; c < PW; ++c) {
            const int buf = c & 1;
            const unsigned cand = __ballot_sync(0xffffffffu, sm.W[buf][lane][c] != 0) & ~used;
            if (!cand) { ok = false; break; }                 // uniform over the working warps
            const int q = __ffs(cand) - 1;
            const uint32_t pv = sm.W[buf][q][lane];
            const uint32_t d = __shfl_sync(0xffffffffu, pv, c);
            const bool atc = lane == c;
            const uint32_t y = atc ? dtot : pv;               // slot c of the pivot row holds its scale
            // row <- d (x) row - h (x) pivot row for the rows that are not the pivot row; the pivot row keeps its
            // entries and receives its scale in slot c
#define FAST_ROW(X, I)                                                                                   \
            {                                                                                            \
                const uint32_t h = __shfl_sync(0xffffffffu, X, c);                                       \
                const uint32_t upd = redc((uint64_t)d * (atc ? 0u : X) + (uint64_t)(f.p - h) * y, f);    \
                X = (row0 + I) != q ? upd : (atc ? dtot : X);                                            \
                sm.W[buf ^ 1][row0 + I][lane] = X;                                                       \
            }
            FAST_EACH_ROW(FAST_ROW)
#undef FAST_ROW
            if (tid == 0) { sm.esrc[c] = i0 + q; sm.gs[0][c] = dtot; }    // gs[0][c] = prefix product BEFORE step c
            dtot = mulredc(dtot, d, f);
            used |= 1u << q;
            asm volatile("bar.sync 1, %0;" ::"n"(FW * 32) : "memory");
        }
        if (tid == 0) { sm.fast_ok = ok ? 1 : 0; sm.gs[1][0] = dtot; }
    }
    __syncthreads();
    return sm.fast_ok != 0;     // on success the final block is in W[0] (32 steps); gs[1][0] = product of all pivots
}

// ------------------------------------------------------------------------------------------------
// P1, general path (any width w <= 32, any number of rows): rows are scanned in chunks of 32 held in
// shared memory (warp = chunk row, lane = column); a chunk is first reduced against the pivot rows
// found so far, then searched column by column for the FIRST row with a non-zero entry (warp ballot).
// Elimination is division-free (row_k <- d*row_k - h*row_q), so no modular inverse sits on the
// column-to-column dependency chain.  The scan stops once w pivots are known; otherwise it has looked
// at every row, which is what proves the remaining columns are free columns.  Returns r.
__device__ __noinline__ int panel_scan(StripSmem& sm, const uint32_t* A, int64_t ld, int64_t rows, int64_t i0, int64_t j0, int w) {
    const ModP& f = c_f[sm.slot];
    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    uint32_t (*X)[PW + 1] = sm.W[0];
    uint32_t (*Ep)[PW + 1] = sm.W[1];          // pivot rows as selected (unnormalised), discovery order
    int r = 0;
    unsigned pcmask = 0;
    for (int64_t cs = i0; cs < rows && r < w; cs += PW) {
        const int nh = (int)min((int64_t)PW, rows - cs);
        uint32_t s = 0;
        if (wq < nh && lane < w) s = A[(cs + wq) * ld + j0 + lane];
        for (int a = 0; a < r; ++a) {              // ascending pivot column
            const int tt = sm.ord[a];
            const int c = sm.epc[tt];
            const uint32_t l = __shfl_sync(0xffffffffu, s, c);
            if (l) s = lane > c ? lincomb(Ep[tt][c], s, l, Ep[tt][lane], f) : (lane == c ? 0u : mulmod(Ep[tt][c], s, f));
        }
        X[wq][lane] = s;
        if (!__syncthreads_or(s != 0)) continue;   // the whole chunk lies in the span found so far

        unsigned used = 0;
        for (int c = 0; c < w && r < w; ++c) {
            if ((pcmask >> c) & 1u) continue;
            const unsigned cand = __ballot_sync(0xffffffffu, X[lane][c] != 0) & ~used;
            if (!cand) continue;
            const int q = __ffs(cand) - 1;
            const uint32_t d = X[q][c];
            const uint32_t pv = X[q][lane];
            if (wq != q && !((used >> wq) & 1u)) {
                const uint32_t h = X[wq][c];
                if (h != 0 && lane > c) X[wq][lane] = lincomb(d, X[wq][lane], h, pv, f);   // column c itself is not rewritten
            }
            if (wq == 0) Ep[r][lane] = ((pcmask >> lane) & 1u) ? 0u : pv;   // entries at earlier pivot columns are zeros
            if (tid == 0) { sm.epc[r] = c; sm.esrc[r] = cs + q; }
            used |= 1u << q;
            pcmask |= 1u << c;
            ++r;
            __syncthreads();
        }
        if (wq == 0) {                             // rank sort of the pivots by column
            const int mine = lane < r ? sm.epc[lane] : INT_MAX;
            int pos = 0;
            for (int t = 0; t < r; ++t) pos += (sm.epc[t] < mine);
            if (lane < r) sm.ord[pos] = lane;
        }
        __syncthreads();
    }
    return r;
}

// T = D^-1 for the general path: Gauss-Jordan on [D | I], D = A[pivot rows, pivot columns] in ascending
// pivot-column order (no search needed: pivot rows with a larger leading column vanish on the smaller
// columns, so D has an LU factorisation without pivoting), division-free; leaves g (diagonal) and the
// transform in G.  Also E = T.A[P, panel] when r < w.
__device__ __noinline__ void panel_invert_general(StripSmem& sm, const uint32_t* A, int64_t ld, int64_t j0, int w, int r,
                                                  uint32_t* Tout, uint32_t* Eout) {
    const ModP& f = c_f[sm.slot];
    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    for (int e = tid; e < PW * 2 * PW; e += SNT) {
        const int a = e / (2 * PW), b = e % (2 * PW);
        uint32_t v = 0;
        if (a < r) {
            if (b < PW) { if (b < r) v = A[sm.esrc[sm.ord[a]] * ld + j0 + sm.epc[sm.ord[b]]]; }
            else v = (b - PW == a) ? 1u : 0u;
        }
        sm.G[a][b] = v;
    }
    __syncthreads();
    for (int t = 0; t < r; ++t) {
        const uint32_t d = sm.G[t][t];
        const uint32_t pl = lane > t ? sm.G[t][lane] : 0u;
        const uint32_t pr = lane <= t ? sm.G[t][PW + lane] : 0u;
        if (wq != t && wq < r) {
            const uint32_t h = sm.G[wq][t];
            if (h != 0) {
                if (lane > t || lane == wq) sm.G[wq][lane] = lincomb(d, sm.G[wq][lane], h, pl, f);
                if (lane <= t || lane == wq) sm.G[wq][PW + lane] = lincomb(d, sm.G[wq][PW + lane], h, pr, f);
            }
        }
        __syncthreads();
    }
    if (wq == 0 && lane < r) sm.ginv[lane] = invmod(sm.G[lane][lane], f);
    __syncthreads();
    {
        const int a = wq, b = lane;
        const uint32_t v = (a < r && b < r) ? mulmod(sm.ginv[a], sm.G[a][PW + b], f) : 0u;
        Tout[a * PW + b] = v;
        sm.Ts[a][b] = v;
    }
    if (r < w && r > 0) {
        // E = T . A[P, panel]: reduced pivot rows restricted to the panel (identity on the pivot columns)
        sm.Ar[wq][lane] = (wq < r && lane < w) ? A[sm.esrc[sm.ord[wq]] * ld + j0 + lane] : 0u;
        __syncthreads();
        uint64_t acc = 0;
        for (int b = 0; b < r; ++b) {
            acc += (uint64_t)sm.Ts[wq][b] * sm.Ar[b][lane];
            if (b & 1) acc = fold64(acc, f);
        }
        Eout[wq * PW + lane] = wq < r ? reduce64(acc, f) : 0u;
    }
}

// Exchange list (LAPACK style): row i0+a must receive source row esrc[ord[a]].  Warp 0 only.
__device__ void panel_exchange_list(StripSmem& sm, int64_t i0, int r, PanelRec* rec) {
    const int lane = threadIdx.x & 31;
    const bool inplace = lane >= r || sm.esrc[sm.ord[lane]] == i0 + lane;
    const bool all_inplace = __all_sync(0xffffffffu, inplace);
    if (lane < r) { sm.pos_of[lane] = i0 + lane; sm.at[lane] = lane; }
    __syncwarp();
    if (all_inplace) {
        if (lane < r) rec->swp[lane] = i0 + lane;
        if (lane == 0) sm.nsw = 0;
    } else if (lane == 0) {
        int nsw = 0;
        for (int a = 0; a < r; ++a) {
            const long long src = sm.esrc[sm.ord[a]];
            const long long cur = src < i0 + r ? sm.pos_of[(int)(src - i0)] : src;
            rec->swp[a] = cur;
            if (cur != i0 + a) {
                ++nsw;
                const int x = sm.at[a];                 // top-origin row now sitting at position a
                sm.pos_of[x] = cur;
                if (cur < i0 + r) sm.at[(int)(cur - i0)] = x;
            }
        }
        sm.nsw = nsw;
    }
}

// P1 for one base panel (columns [j0, j0+w), rows >= i0), executed by ONE CTA of SNT threads.
// Outputs: rec (r, local pivot columns, exchange list), T (32x32, zero padded), E = T A[P, panel] when
// r < w (the free columns' entries of the reduced pivot rows), pivcols.
// With allow_general = false only the fast path is tried (the caller has not finished updating the rows beyond
// the 32 candidates); returns whether the panel was factored.
__device__ bool panel_factor(StripSmem& sm, const uint32_t* A, int64_t ld, int64_t rows, int64_t i0, int64_t j0, int w,
                             PanelRec* rec, uint32_t* Tout, uint32_t* Eout, int32_t* pivcols_global,
                             bool allow_general = true) {
    const ModP& f = c_f[sm.slot];
    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    int r = 0;
    bool fast = false;
    if (w == PW && rows - i0 >= PW && f.ninv != 0) fast = panel_fast(sm, A, ld, i0, j0);
    if (fast) {
        // row q_a that pivoted column a has been scaled by g = (all pivots) / (pivots before step a), so
        // 1/g = prefix[a] / (all pivots): ONE modular inverse for the panel (K7)
        r = PW;
        if (tid < PW) { sm.epc[tid] = tid; sm.ord[tid] = tid; }
        // (with Montgomery products the identity reads 1/g_a = prefix[a] (x) 1/(all pivots))
        if (wq == 0) sm.ginv[lane] = mulredc(sm.gs[0][lane], invmod_fermat(sm.gs[1][0], f), f);
        __syncthreads();
        if (wq == 0) panel_exchange_list(sm, i0, r, rec);
        const int qa = (int)(sm.esrc[wq] - i0);
        Tout[wq * PW + lane] = mulmod(sm.ginv[wq], sm.W[0][qa][lane], f);
    } else {
        if (!allow_general) return false;
        __syncthreads();
        r = panel_scan(sm, A, ld, rows, i0, j0, w);
        if (wq == 0) panel_exchange_list(sm, i0, r, rec);
        __syncthreads();
        panel_invert_general(sm, A, ld, j0, w, r, Tout, Eout);
    }
    if (tid < PW) {
        const int pc = tid < r ? sm.epc[sm.ord[tid]] : -1;
        rec->pc[tid] = pc;
        if (tid < r) pivcols_global[i0 + tid] = (int32_t)(j0 + pc);
        const unsigned pcm = __reduce_or_sync(0xffffffffu, pc >= 0 ? 1u << pc : 0u);
        if (tid == 0) sm.last_pcm = pcm;
    }
    __syncthreads();
    if (tid == 0) {
        rec->r = r;
        rec->w = w;
        rec->nswaps = sm.nsw;
        sm.r_out = r;
        sm.last_r = r;
        sm.last_nsw = sm.nsw;
    }
    return true;
}

// What the host needs of a strip's records (r, nswaps, pc[32] per panel), posted to mapped pinned host memory --
// PCIe writes, no copy engine, so a large transfer the caller has in flight cannot delay the host's next launches.
// Every 64-bit word carries the launch's sequence number in its upper half, so no system-wide fence is needed: the
// host waits until every word shows the tag.  Called by all threads of ONE CTA.
constexpr int MAIL_WORDS = 2 + PW;          // per panel: r, nswaps, pc[32]
__device__ __forceinline__ void mail_records(volatile unsigned long long* dst, unsigned long long seq, const PanelRec* rec,
                                             int nbp) {
    for (int e = threadIdx.x; e < nbp * MAIL_WORDS; e += blockDim.x) {
        const PanelRec* rc = rec + e / MAIL_WORDS;
        const int k = e % MAIL_WORDS;
        const uint32_t v = k == 0 ? (uint32_t)rc->r : (k == 1 ? (uint32_t)rc->nswaps : (uint32_t)rc->pc[k - 2]);
        dst[e] = (seq << 32) | v;
    }
}

// ------------------------------------------------------------------------------------------------
// The strip kernel.  Panel metadata arrays are indexed by the GLOBAL base panel number b = j0/PW + i.
// pstart[b+1] (device) receives the number of pivots found left of panel b+1.
struct StripArgs {
    uint32_t* A;
    int64_t ld, rows, cols;
    int64_t i0;              // first active row
    int64_t j0;              // first column of the strip (multiple of PW)
    int ws;                  // strip width in columns
    PanelRec* rec;           // [nb]
    uint32_t* T;             // [nb][PW*PW]
    uint32_t* E;             // [nb][PW*PW]
    int32_t* pivcols;        // [min(rows, cols)]
    int32_t* pstart;         // [nb+1]
    uint8_t* Aq;             // optional: receives the u8 limb planes of L21 (rows below the strip x its pivot columns)
    int kp;                  //   Aq[limb][m][kp], k-major, zero padded to kp (what the Schur update's TMA loads expect)
    unsigned long long* host_mail;  // mapped pinned host memory: MAXBP * MAIL_WORDS tagged words, written by CTA 0
    unsigned long long seq;         // tag of this launch (32 significant bits)
    int slot;                       // entry of c_f that holds this call's field
    int64_t swap_c0, swap_c1;       // columns on which row exchanges are applied at once ([0, cols) normally; the strip's own
                                    // columns under look-ahead, where the previous strip's bulk update is still writing the
                                    // other columns of the same rows: deferred_swaps_kernel applies the rest afterwards)
};

// Deferred write-back of a U12 slice: the raw entries it replaces are read by every row worker of
// the column block, so the owner (row worker 0) keeps the slice in shared memory until the next
// grid barrier has passed.
__device__ __forceinline__ void strip_flush_u(StripSmem& sm, int slot, uint32_t* A, int64_t ld) {
    const UPending& u = sm.pend[slot];
    if (u.row0 < 0) return;
    const int lane = threadIdx.x & 31, wq = threadIdx.x >> 5;
    if (wq < u.r && lane < u.nc) A[(u.row0 + wq) * ld + u.col0 + lane] = sm.Us[slot][wq][lane];
}

// One CTA's share of the in-strip update behind a factored base panel (pivot rows pr0..pr0+r, panel
// columns jp.., T at Tb, pivot columns in rec):
//   U = T . A[pr0 : pr0+r, cc0 : cc0+nc]                                   (kept in Us[slot])
//   A[m, cc0 : cc0+nc] -= sum_k A[m, pivot column k] * U[k, :]   for this worker's rows m in [my0, my1)
// Tiles of 32*RPT rows: the L tile goes to shared memory k-major, the C tile stays in registers (thread =
// RPT consecutive rows x 1 column: L by one broadcast vector LDS per k, U by one LDS per k).  RPT is chosen
// from the number of rows the worker owns, so that a short share still spreads over all 32 warps.
template <int RPT>
__device__ __noinline__ void strip_update_t(StripSmem& sm, int slot, uint32_t* A, int64_t ld, const uint32_t* Tb,
                                            unsigned pcm, int64_t jp, int64_t pr0, int r, int64_t cc0, int nc,
                                            int64_t my0, int64_t my1, bool owner) {
    const ModP& f = c_f[sm.slot];
    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    constexpr int TR = 32 * RPT;
    // pivot index of panel column `lane` (pcm = mask of the panel's pivot columns, ascending), or -1
    const int kcol = ((pcm >> lane) & 1u) ? __popc(pcm & ((1u << lane) - 1u)) : -1;
    uint32_t cv[RPT];
    auto load_tile = [&](int64_t m0) {
        uint32_t lreg[RPT];
#pragma unroll
        for (int t = 0; t < RPT; ++t) {
            const int64_t m = m0 + wq + 32 * t;
            lreg[t] = (kcol >= 0 && m < my1) ? A[m * ld + jp + lane] : 0u;
        }
#pragma unroll
        for (int t = 0; t < RPT; ++t) {
            const int64_t m = m0 + wq * RPT + t;
            cv[t] = (lane < nc && m < my1) ? A[m * ld + cc0 + lane] : 0u;
        }
        if (kcol >= 0) {
#pragma unroll
            for (int t = 0; t < RPT; ++t) sm.Lk[kcol][wq + 32 * t] = lreg[t];
        }
    };
    const uint32_t tval = Tb[wq * PW + lane];
    const uint32_t aval = (wq < r && lane < nc) ? A[(pr0 + wq) * ld + cc0 + lane] : 0u;
    if (my0 < my1) load_tile(my0);
    sm.Ts[wq][lane] = tval;
    sm.Ar[wq][lane] = aval;
    __syncthreads();
    {
        uint64_t acc = 0;
#pragma unroll 8
        for (int k = 0; k < PW; k += 2) {
            acc += (uint64_t)sm.Ts[wq][k] * sm.Ar[k][lane];
            acc += (uint64_t)sm.Ts[wq][k + 1] * sm.Ar[k + 1][lane];
            acc = fold64(acc, f);
        }
        sm.Us[slot][wq][lane] = wq < r ? reduce64(acc, f) : 0u;
    }
    if (owner && tid == 0) { UPending& u = sm.pend[slot]; u.row0 = pr0; u.col0 = cc0; u.r = r; u.nc = nc; }
    for (int64_t m0 = my0; m0 < my1; m0 += TR) {
        if (m0 != my0) {
            __syncthreads();             // previous tile's readers of Lk are done
            load_tile(m0);
        }
        __syncthreads();
        if (m0 + wq * RPT < my1) {
            uint64_t acc[RPT];
#pragma unroll
            for (int t = 0; t < RPT; ++t) acc[t] = 0;
            auto mac = [&](int k) {
                const uint32_t u = sm.Us[slot][k][lane];
                uint32_t l[RPT];
                if constexpr (RPT == 1) {
                    l[0] = sm.Lk[k][wq];
                } else if constexpr (RPT == 2) {
                    const uint2 v = *reinterpret_cast<const uint2*>(&sm.Lk[k][wq * 2]);
                    l[0] = v.x; l[1] = v.y;
                } else {
#pragma unroll
                    for (int h = 0; h < RPT / 4; ++h) {
                        const uint4 v = *reinterpret_cast<const uint4*>(&sm.Lk[k][wq * RPT + 4 * h]);
                        l[4 * h] = v.x; l[4 * h + 1] = v.y; l[4 * h + 2] = v.z; l[4 * h + 3] = v.w;
                    }
                }
#pragma unroll
                for (int t = 0; t < RPT; ++t) acc[t] += (uint64_t)l[t] * u;
            };
#pragma unroll 1
            for (int k = 0; k + 1 < r; k += 2) {
                mac(k);
                mac(k + 1);
#pragma unroll
                for (int t = 0; t < RPT; ++t) acc[t] = fold64(acc[t], f);
            }
            if (r & 1) {
                mac(r - 1);
#pragma unroll
                for (int t = 0; t < RPT; ++t) acc[t] = fold64(acc[t], f);
            }
#pragma unroll
            for (int t = 0; t < RPT; ++t) {
                const int64_t m = m0 + wq * RPT + t;
                if (lane < nc && m < my1) A[m * ld + cc0 + lane] = submod(cv[t], reduce64(acc[t], f), f);
            }
        }
    }
    __syncthreads();                     // Ts / Ar / Lk may be reused by the caller's next phase
}

// CTA 0 running ahead of the others: U = T . A[pr0 : pr0+r, cc0 : cc0+32] (kept in Us[0], written back after the
// next barrier) and the update of the 32 candidate rows c0row.. of the next panel, one output per thread
// (warp = row, lane = column), the row operand read by LDS.128.  Latency matters here, not throughput: this
// sits between two panel factorisations on the pivot-to-pivot chain.
__device__ __noinline__ void strip_ahead_update(StripSmem& sm, uint32_t* A, int64_t ld, const uint32_t* Tb, unsigned pcm,
                                                int64_t jp, int64_t pr0, int r, int64_t cc0, int64_t c0row) {
    const ModP& f = c_f[sm.slot];
    const int tid = threadIdx.x, lane = tid & 31, a = tid >> 5;
    const int kcol = ((pcm >> lane) & 1u) ? __popc(pcm & ((1u << lane) - 1u)) : -1;
    const uint32_t t = Tb[a * PW + lane];
    const uint32_t ar = a < r ? A[(pr0 + a) * ld + cc0 + lane] : 0u;
    const uint32_t l = A[(c0row + a) * ld + jp + lane];
    uint32_t c = A[(c0row + a) * ld + cc0 + lane];
    sm.Bt[a][lane] = t;                                   // zero beyond r (T is stored zero padded)
    sm.Ar[a][lane] = ar;
    if (kcol >= 0) sm.Bl[a][kcol] = l;
    if (lane >= r) sm.Bl[a][lane] = 0u;                   // the r pivot indices fill 0..r-1
    __syncthreads();
    auto dot = [&](const uint32_t* row, const uint32_t (*col)[PW + 1]) {
        uint64_t acc = 0;
#pragma unroll
        for (int k = 0; k < PW; k += 4) {
            const uint4 v = *reinterpret_cast<const uint4*>(row + k);
            acc += (uint64_t)v.x * col[k][lane];
            acc += (uint64_t)v.y * col[k + 1][lane];
            acc = fold64(acc, f);
            acc += (uint64_t)v.z * col[k + 2][lane];
            acc += (uint64_t)v.w * col[k + 3][lane];
            acc = fold64(acc, f);
        }
        return reduce64(acc, f);
    };
    const uint32_t u = dot(sm.Bt[a], sm.Ar);
    __syncthreads();                                      // every reader of Ar is done: Ar now carries U
    sm.Ar[a][lane] = a < r ? u : 0u;
    sm.Us[0][a][lane] = a < r ? u : 0u;
    if (tid == 0) { UPending& p = sm.pend[0]; p.row0 = pr0; p.col0 = cc0; p.r = r; p.nc = PW; }
    __syncthreads();
    c = submod(c, dot(sm.Bl[a], sm.Ar), f);
    A[(c0row + a) * ld + cc0 + lane] = c;
    __syncthreads();                                      // the panel factorisation that follows reads these rows
}

// Row worker rw of nrw: its rows, then the variant whose tile matches them.
__device__ __forceinline__ void strip_update(StripSmem& sm, int slot, uint32_t* A, int64_t ld, int64_t rows,
                                             const uint32_t* Tb, unsigned pcm, int64_t jp, int64_t pr0, int r,
                                             int64_t cc0, int nc, int rw, int nrw, int skip, bool owner) {
    const int64_t mb0 = min(rows, pr0 + r + skip);       // `skip` rows right below the pivots belong to someone else
    const int64_t mrem = rows - mb0;
    int64_t rpw = (mrem + nrw - 1) / nrw;
    rpw = (rpw + 7) / 8 * 8;
    const int64_t my0 = min(rows, mb0 + (int64_t)rw * rpw), my1 = min(rows, my0 + rpw);
    const int64_t n = my1 - my0;
    if (n <= 32) strip_update_t<1>(sm, slot, A, ld, Tb, pcm, jp, pr0, r, cc0, nc, my0, my1, owner);
    else if (n <= 64) strip_update_t<2>(sm, slot, A, ld, Tb, pcm, jp, pr0, r, cc0, nc, my0, my1, owner);
    else if (n <= 128) strip_update_t<4>(sm, slot, A, ld, Tb, pcm, jp, pr0, r, cc0, nc, my0, my1, owner);
    else strip_update_t<8>(sm, slot, A, ld, Tb, pcm, jp, pr0, r, cc0, nc, my0, my1, owner);
}

// The strip kernel, software-pipelined so that ONE grid barrier per base panel sits on the pivot-to-pivot
// dependency chain.  Loop invariant at the top of iteration i: panel i is factored (record, T, pivot columns
// published and a barrier passed) and every update of the panels before i has been applied everywhere.  Then,
// between two barriers,
//   CTA 0        updates the 32 candidate rows of panel i+1 (its own U slice, a 32-row tile) and factors panel
//                i+1 from them by the fast path;
//   CTAs 1..G-1  apply panel i's update to all the other rows below and all strip columns to the right
//                (2-D split: column block x row worker; U = T.A12 recomputed per CTA, written back by the
//                owners after the barrier because every row worker reads the raw entries).
// If the fast path does not apply or fails (rank-deficient candidates), CTA 0 factors panel i+1 by the general
// path after the barrier, when all rows are up to date, and one more barrier follows.
__global__ void __launch_bounds__(SNT, 1) strip_factor_kernel(const StripArgs a) {
    extern __shared__ __align__(16) unsigned char strip_smem_raw[];
    StripSmem& sm = *reinterpret_cast<StripSmem*>(strip_smem_raw);
    cg::grid_group grid = cg::this_grid();
    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    const int G = gridDim.x, cta = blockIdx.x;
    uint32_t* A = a.A;
    const int64_t ld = a.ld;
    const int nbp = (a.ws + PW - 1) / PW;
    const int64_t b0 = a.j0 / PW;
    const int64_t cu1 = a.j0 + a.ws;               // end of the strip
    int64_t cur = a.i0;

    // CTA 0, once it has written the record of the strip's LAST panel, mails the records to the host -- unless the
    // row-block solve launched right behind this kernel does it (host_mail == nullptr): there the PCIe drain hides
    // under 40 us of work instead of sitting in front of this kernel's last grid barrier.
    auto mail = [&]() {
        if (a.host_mail == nullptr) return;
        __syncthreads();
        mail_records(a.host_mail, a.seq, a.rec + b0, nbp);
    };
    const int64_t blast = b0 + nbp - 1;

    // CTA 0: factor panel bb (columns jpp.., width ww) from row `row` on, fast path first, general path otherwise.
    auto factor_full = [&](int64_t bb, int64_t jpp, int ww, int64_t row) {
        if (cta != 0) return;
        if (row < a.rows) {
            panel_factor(sm, A, ld, a.rows, row, jpp, ww, a.rec + bb, a.T + bb * PW * PW, a.E + bb * PW * PW, a.pivcols);
            if (tid == 0) a.pstart[bb + 1] = (int32_t)(row + sm.r_out);
        } else if (tid == 0) {                     // no rows left: the panel's columns are free
            a.rec[bb].r = 0; a.rec[bb].nswaps = 0; a.rec[bb].w = ww;
            sm.last_r = 0; sm.last_nsw = 0; sm.last_pcm = 0;
            a.pstart[bb + 1] = (int32_t)row;
        }
        if (bb == blast) mail();
    };
    auto flush_all = [&]() {                       // U slices whose readers all passed the last grid barrier
        strip_flush_u(sm, 0, A, ld);
        strip_flush_u(sm, 1, A, ld);
        __syncthreads();
        if (tid == 0) { sm.pend[0].row0 = -1; sm.pend[1].row0 = -1; }
    };

    if (tid == 0) { sm.pend[0].row0 = -1; sm.pend[1].row0 = -1; sm.slot = a.slot; }
    __syncthreads();
    factor_full(b0, a.j0, (int)min((int64_t)PW, cu1 - a.j0), cur);
    grid.sync();
    for (int i = 0; i < nbp; ++i) {
        const int64_t b = b0 + i;
        const int64_t jp = a.j0 + (int64_t)i * PW;
        const int w = (int)min((int64_t)PW, cu1 - jp);
        const int64_t cu0 = jp + w;                // first strip column right of panel i
        const int wn = (int)min((int64_t)PW, cu1 - cu0);      // width of panel i+1 (<= 0: panel i is the last)
        flush_all();
        // everything the updates need from the panel record, in ONE round trip to L2
        const PanelRec* rec = a.rec + b;
        int r, nsw;
        unsigned pcm;
        if (cta == 0) {                            // CTA 0 wrote the record itself
            r = sm.last_r; nsw = sm.last_nsw; pcm = sm.last_pcm;
        } else {
            const int pcl = rec->pc[lane];
            r = rec->r; nsw = rec->nswaps;
            pcm = __reduce_or_sync(0xffffffffu, pcl >= 0 ? 1u << pcl : 0u);
        }
        if (r == 0) {                              // free panel: nothing to apply, the next panel is factored as is
            if (wn > 0) {
                factor_full(b + 1, cu0, wn, cur);
                grid.sync();
            }
            continue;
        }
        // ---- row exchanges on complete rows, one thread per column (so the sequence of exchanges
        // needs no inter-thread ordering)
        if (nsw > 0) {
            for (int64_t c = a.swap_c0 + (int64_t)cta * SNT + tid; c < a.swap_c1; c += (int64_t)G * SNT) {
                for (int t = 0; t < r; ++t) {
                    const int64_t s = rec->swp[t];
                    if (s != cur + t) {
                        const uint32_t x = A[(cur + t) * ld + c], y = A[s * ld + c];
                        A[(cur + t) * ld + c] = y;
                        A[s * ld + c] = x;
                    }
                }
            }
            grid.sync();
        }
        // reduced pivot rows' entries inside a rank-deficient panel (nobody reads these during the updates)
        if (r < w && cta == G - 1)
            if (wq < r && lane < w) A[(cur + wq) * ld + jp + lane] = a.E[b * PW * PW + wq * PW + lane];
        if (wn <= 0) { cur += r; continue; }       // last panel of the strip: nothing to its right
        const int ncu = (int)(cu1 - cu0);
        const int ncb = (ncu + PW - 1) / PW;
        const uint32_t* Tb = a.T + b * PW * PW;
        // CTA 0 runs ahead on the next panel if its 32 candidate rows exist and the fast path can take them
        const bool ahead = G >= 2 && G - 1 >= ncb && wn == PW && cur + r + PW <= a.rows && c_f[a.slot].ninv != 0;
        if (G == 1 || G - 1 < ncb) {
            // degenerate grids: the column blocks in turn (sole reader and writer: the slice goes back at once)
            for (int cb = (G == 1 ? 0 : cta - 1); cb >= 0 && cb < ncb; cb += (G == 1 ? 1 : G - 1)) {
                const int64_t cc0 = cu0 + (int64_t)cb * PW;
                strip_update(sm, 1, A, ld, a.rows, Tb, pcm, jp, cur, r, cc0, (int)min((int64_t)PW, cu1 - cc0), 0, 1, 0, true);
                strip_flush_u(sm, 1, A, ld);
                __syncthreads();
                if (tid == 0) sm.pend[1].row0 = -1;
                __syncthreads();
            }
            if (cta == 0 && tid == 0) a.rec[b + 1].pad = 0;
        } else if (cta == 0) {
            if (ahead) {
                strip_ahead_update(sm, A, ld, Tb, pcm, jp, cur, r, cu0, cur + r);
                const bool got = panel_factor(sm, A, ld, a.rows, cur + r, cu0, wn, a.rec + b + 1, a.T + (b + 1) * PW * PW,
                                              a.E + (b + 1) * PW * PW, a.pivcols, false);
                if (tid == 0) {
                    if (got) a.pstart[b + 2] = (int32_t)(cur + r + sm.r_out);
                    a.rec[b + 1].pad = got ? 1 : 0;
                }
                if (got && b + 1 == blast) mail();
            } else if (tid == 0) {
                a.rec[b + 1].pad = 0;
            }
        } else {
            const int nrw = (G - 1) / ncb, job = cta - 1, cb = job % ncb, rw = job / ncb;
            if (rw < nrw) {
                const int64_t cc0 = cu0 + (int64_t)cb * PW;
                const bool shared0 = cb == 0 && ahead;           // CTA 0 owns the candidate rows of block 0 and its U slice
                strip_update(sm, 1, A, ld, a.rows, Tb, pcm, jp, cur, r, cc0, (int)min((int64_t)PW, cu1 - cc0), rw, nrw,
                             shared0 ? PW : 0, rw == 0 && !shared0);
            }
        }
        grid.sync();
        cur += r;
        // rec.pad is written ONLY between the barriers above (by CTA 0), never by the factorisation that may follow,
        // so every CTA reads the same value however late it gets here
        if (a.rec[b + 1].pad != 1) {
            factor_full(b + 1, cu0, wn, cur);      // every row is up to date now (pending U slices are rows < cur)
            grid.sync();
        }
    }
    strip_flush_u(sm, 0, A, ld);
    strip_flush_u(sm, 1, A, ld);
    // Tail: every pivot column of the strip is known and the rows below are final in those columns, so the whole
    // grid writes the limb planes of L21 for the Schur update that follows (saves that update its own split pass).
    if (a.Aq != nullptr) {
        const int K = (int)(cur - a.i0);
        const int64_t M = a.rows - cur;
        const int64_t plane = M * a.kp;
        const int nword = a.kp / 4;                       // 4 k per 32-bit word
        for (int wd = lane; wd < nword; wd += 32) {
            int32_t pc[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) pc[e] = wd * 4 + e < K ? a.pivcols[a.i0 + wd * 4 + e] : -1;
            for (int64_t m = (int64_t)cta * (SNT / 32) + wq; m < M; m += (int64_t)G * (SNT / 32)) {
                const uint32_t* row = A + (cur + m) * ld;
                uint32_t v[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) v[e] = pc[e] >= 0 ? row[pc[e]] : 0u;
#pragma unroll
                for (int l = 0; l < 4; ++l) {
                    const uint32_t packed = ((v[0] >> (8 * l)) & 0xFF) | (((v[1] >> (8 * l)) & 0xFF) << 8) |
                                            (((v[2] >> (8 * l)) & 0xFF) << 16) | (((v[3] >> (8 * l)) & 0xFF) << 24);
                    *reinterpret_cast<uint32_t*>(a.Aq + l * plane + m * a.kp + wd * 4) = packed;
                }
            }
        }
    }
}

// Row exchanges of a whole strip on the columns a look-ahead strip kernel left out ([0, skip0) and [skip1, cols)), in
// the order the strip performed them; one thread per column.  Exits at once when the strip exchanged nothing.
__global__ void deferred_swaps_kernel(uint32_t* __restrict__ A, int64_t ld, int64_t cols, int64_t skip0, int64_t skip1,
                                      const PanelRec* __restrict__ rec, const int32_t* __restrict__ pstart, int b0, int nbp) {
    bool any = false;
    for (int b = b0; b < b0 + nbp; ++b) any = any || (rec[b].r > 0 && rec[b].nswaps > 0);
    if (!any) return;
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= skip0) c += skip1 - skip0;
    if (c >= cols) return;
    for (int b = b0; b < b0 + nbp; ++b) {
        const int r = rec[b].r;
        if (r == 0 || rec[b].nswaps == 0) continue;
        const int64_t cur = pstart[b];
        for (int t = 0; t < r; ++t) {
            const int64_t s = rec[b].swp[t];
            if (s != cur + t) {
                const uint32_t x = A[(cur + t) * ld + c], y = A[s * ld + c];
                A[(cur + t) * ld + c] = y;
                A[s * ld + c] = x;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S4 / S6 leaf: triangular solve against ONE strip's pivots, column-parallel (a CTA owns 32 columns
// of X and keeps them in shared memory, so the sequential dependence between base panels never
// leaves the CTA).  X has K = pstart[bs1] - pstart[bs0] rows (the strip's pivot rows, in order).
//   LOWER (row-block solve, U12 = L11^-1 A12):  for each base panel b, ascending:
//           X_b <- T_b X_b ;  X_t -= sum_k L[t][k] X_b[k]  for the strip's pivot rows t after b
//   UPPER (back-elimination of the free columns): for each base panel b, descending:
//           X_t -= sum_k U[t][k] X_b[k]  for the strip's pivot rows t before b
// with L[t][k] = U[t][k] = A[row t][pivcols[first pivot of b + k]] (fp_kernels.cuh storage convention).
constexpr int TNT = 512;       // threads per CTA (16 warps)
constexpr int TLS = PW + 4;    // row stride of the staged L block (16-byte aligned rows, conflict-free stores)
constexpr int TLR = SW_MAX - PW;                       // most rows an L block can have
constexpr int TNL = (TLR * PW + TNT - 1) / TNT;        // prefetch registers per thread for one L block

__host__ __device__ inline size_t trsm_smem_bytes(int64_t K) {
    return (size_t)K * PW * 4 + (size_t)PW * TLS * 4 + (size_t)TLR * TLS * 4;
}

// sum_k row[k] * x[k] over a full 32-pivot panel: the row (16-byte aligned in shared memory) by LDS.128, the column of
// X from registers, one fold per two products (fold64 keeps the accumulator below 2^63 + 2^32).
__device__ __forceinline__ uint64_t dot32_pair(const uint32_t* __restrict__ row, const uint32_t (&x)[PW], const ModP& f) {
    uint64_t acc = 0;
#pragma unroll
    for (int k = 0; k < PW; k += 4) {
        const uint4 v = *reinterpret_cast<const uint4*>(row + k);
        acc = fold64(acc + (uint64_t)v.x * x[k] + (uint64_t)v.y * x[k + 1], f);
        acc = fold64(acc + (uint64_t)v.z * x[k + 2] + (uint64_t)v.w * x[k + 3], f);
    }
    return acc;
}

template <bool LOWER>
__global__ void __launch_bounds__(TNT, 2) trsm_strip_kernel(const uint32_t* __restrict__ A, int64_t ld,
                                                         uint32_t* __restrict__ X, int64_t ldx, int64_t ncols,
                                                         const int32_t* __restrict__ pstart, int bs0, int bs1,
                                                         const uint32_t* __restrict__ T,
                                                         const int32_t* __restrict__ pivcols, ModP f,
                                                         uint8_t* __restrict__ Bq, int kp,
                                                         unsigned long long* host_mail, unsigned long long seq,
                                                         const PanelRec* rec, int64_t bq_col0, int64_t bq_total) {
    extern __shared__ __align__(16) unsigned char trsm_smem_raw[];
    if (host_mail != nullptr && blockIdx.x == 0) mail_records(host_mail, seq, rec + bs0, bs1 - bs0);
    const int t0 = pstart[bs0], K = pstart[bs1] - t0;
    uint32_t (*Xs)[PW] = reinterpret_cast<uint32_t (*)[PW]>(trsm_smem_raw);                                 // [K][32]
    uint32_t (*Ts)[TLS] = reinterpret_cast<uint32_t (*)[TLS]>(trsm_smem_raw + (size_t)K * PW * 4);           // [32][36]
    uint32_t (*Lp)[TLS] = reinterpret_cast<uint32_t (*)[TLS]>(trsm_smem_raw + (size_t)K * PW * 4 + PW * TLS * 4);
    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    constexpr int NW = TNT / 32;
    const int64_t c = (int64_t)blockIdx.x * PW + lane;
    const bool cok = c < ncols;
    const int nbp = bs1 - bs0;

    // The L (or U) block and T of a base panel are fetched into registers one panel ahead, so their global
    // latency hides under the previous panel's arithmetic instead of sitting on the panel-to-panel chain.
    uint32_t lpre[TNL], tpre[2];
    int nxt = 0;                                       // next panel (in processing order) to prefetch
    auto panel_of = [&](int ii) { return LOWER ? bs0 + ii : bs1 - 1 - ii; };
    auto prefetch = [&]() {
        while (nxt < nbp && pstart[panel_of(nxt) + 1] == pstart[panel_of(nxt)]) ++nxt;     // skip empty panels
        if (nxt >= nbp) return;
        const int b = panel_of(nxt);
        const int s = pstart[b] - t0, e = pstart[b + 1] - t0, r = e - s;
        const int lo = LOWER ? e : 0, nrow = LOWER ? K - e : s;
        if (LOWER) {
            tpre[0] = T[(int64_t)b * PW * PW + tid];
            tpre[1] = T[(int64_t)b * PW * PW + TNT + tid];
        }
        const int32_t pc = lane < r ? pivcols[t0 + s + lane] : -1;
#pragma unroll
        for (int j = 0; j < TNL; ++j) {
            const int row = wq + NW * j;
            lpre[j] = (row < nrow && pc >= 0) ? A[(int64_t)(t0 + lo + row) * ld + pc] : 0u;
        }
    };
    prefetch();
    for (int t = wq; t < K; t += NW) Xs[t][lane] = cok ? X[(int64_t)t * ldx + c] : 0u;

    for (int ii = 0; ii < nbp; ++ii) {
        const int b = panel_of(ii);
        const int s = pstart[b] - t0, e = pstart[b + 1] - t0, r = e - s;
        if (r == 0) continue;
        const int lo = LOWER ? e : 0, nrow = LOWER ? K - e : s;
        // registers -> shared memory (the previous panel's readers passed the barrier that ended its update)
        if (LOWER) {
            Ts[tid / PW][tid % PW] = tpre[0];
            Ts[(TNT + tid) / PW][tid % PW] = tpre[1];
        }
#pragma unroll
        for (int j = 0; j < TNL; ++j) {
            const int row = wq + NW * j;
            if (row < nrow) Lp[row][lane] = lpre[j];
        }
        __syncthreads();
        nxt = ii + 1;
        prefetch();
        if (r == PW) {
            // Full panel (the common case): the 32 entries of this thread's column of X_b live in registers for the whole
            // panel, rows of T / L come in by LDS.128, everything is unrolled -- about 2.5 instructions per multiply-
            // accumulate against 10 in the general loops below (run-time r, scalar shared-memory operands).
            uint32_t x[PW];
            if (LOWER) {
#pragma unroll
                for (int k = 0; k < PW; ++k) x[k] = Xs[s + k][lane];
                const uint32_t y0 = reduce64(dot32_pair(Ts[wq], x, f), f);
                const uint32_t y1 = reduce64(dot32_pair(Ts[wq + NW], x, f), f);
                __syncthreads();
                Xs[s + wq][lane] = y0;
                Xs[s + wq + NW][lane] = y1;
                __syncthreads();
            }
            if (nrow > 0) {
#pragma unroll
                for (int k = 0; k < PW; ++k) x[k] = Xs[s + k][lane];
                for (int row = wq; row < nrow; row += 2 * NW) {
                    const bool two = row + NW < nrow;
                    const uint64_t a0 = dot32_pair(Lp[row], x, f);
                    const uint64_t a1 = dot32_pair(Lp[two ? row + NW : row], x, f);
                    Xs[lo + row][lane] = submod(Xs[lo + row][lane], reduce64(a0, f), f);
                    if (two) Xs[lo + row + NW][lane] = submod(Xs[lo + row + NW][lane], reduce64(a1, f), f);
                }
            }
            __syncthreads();
            continue;
        }
        if (LOWER) {
            // two outputs per thread (rows wq and wq + 16 of T) share the X loads
            static_assert(PW / NW == 2, "the T product below is written for two rows per warp");
            uint32_t y[2];
            {
                uint64_t a0 = 0, a1 = 0;
                const uint32_t* t0r = Ts[wq];
                const uint32_t* t1r = Ts[wq + NW];
                for (int k = 0; k + 1 < r; k += 2) {
                    const uint32_t x0 = Xs[s + k][lane], x1 = Xs[s + k + 1][lane];
                    a0 = fold64(a0 + (uint64_t)t0r[k] * x0 + (uint64_t)t0r[k + 1] * x1, f);
                    a1 = fold64(a1 + (uint64_t)t1r[k] * x0 + (uint64_t)t1r[k + 1] * x1, f);
                }
                if (r & 1) {
                    const uint32_t x0 = Xs[s + r - 1][lane];
                    a0 = fold64(a0 + (uint64_t)t0r[r - 1] * x0, f);
                    a1 = fold64(a1 + (uint64_t)t1r[r - 1] * x0, f);
                }
                y[0] = reduce64(a0, f);
                y[1] = reduce64(a1, f);
            }
            __syncthreads();
#pragma unroll
            for (int u = 0; u < PW / NW; ++u)
                if (wq + NW * u < r) Xs[s + wq + NW * u][lane] = y[u];
            __syncthreads();
        }
        // rows in pairs (row, row + 16) sharing the X loads; L by LDS.128 along k
        for (int row = wq; row < nrow; row += 2 * NW) {
            const bool two = row + NW < nrow;
            const uint32_t* l0 = Lp[row];
            const uint32_t* l1 = Lp[two ? row + NW : row];
            uint64_t a0 = 0, a1 = 0;
            int k = 0;
            for (; k + 3 < r; k += 4) {
                const uint4 p = *reinterpret_cast<const uint4*>(l0 + k);
                const uint4 q = *reinterpret_cast<const uint4*>(l1 + k);
                const uint32_t x0 = Xs[s + k][lane], x1 = Xs[s + k + 1][lane], x2 = Xs[s + k + 2][lane], x3 = Xs[s + k + 3][lane];
                a0 = fold64(a0 + (uint64_t)p.x * x0 + (uint64_t)p.y * x1, f);
                a1 = fold64(a1 + (uint64_t)q.x * x0 + (uint64_t)q.y * x1, f);
                a0 = fold64(a0 + (uint64_t)p.z * x2 + (uint64_t)p.w * x3, f);
                a1 = fold64(a1 + (uint64_t)q.z * x2 + (uint64_t)q.w * x3, f);
            }
            for (; k < r; ++k) {
                const uint32_t x0 = Xs[s + k][lane];
                a0 = fold64(a0 + (uint64_t)l0[k] * x0, f);
                a1 = fold64(a1 + (uint64_t)l1[k] * x0, f);
            }
            Xs[lo + row][lane] = submod(Xs[lo + row][lane], reduce64(a0, f), f);
            if (two) Xs[lo + row + NW][lane] = submod(Xs[lo + row + NW][lane], reduce64(a1, f), f);
        }
        __syncthreads();
    }
    if (cok)
        for (int t = wq; t < K; t += NW) X[(int64_t)t * ldx + c] = Xs[t][lane];
    // Optionally hand the result to the Schur update already split into its four u8 limb planes
    // (Bq[limb][column][kp], k-major, zero padded to kp): saves the update its own pass over U12.
    // The planes may belong to a wider row block than this launch solves (look-ahead splits the solve into the next
    // strip's columns and the rest): bq_total columns per plane, this launch starts at column bq_col0.
    if (Bq != nullptr && cok) {
        const int64_t plane = bq_total * (int64_t)kp;
        for (int job = wq; job < 4 * (kp / 16); job += NW) {          // (limb, 16 consecutive k) per warp, lane = column
            const int l = job / (kp / 16), k0 = (job % (kp / 16)) * 16;
            uint32_t w[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                uint32_t packed = 0;
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int k = k0 + 4 * q + e;
                    const uint32_t v = k < K ? Xs[k][lane] : 0u;
                    packed |= ((v >> (8 * l)) & 0xFFu) << (8 * e);
                }
                w[q] = packed;
            }
            *reinterpret_cast<uint4*>(Bq + (int64_t)l * plane + (bq_col0 + c) * kp + k0) = make_uint4(w[0], w[1], w[2], w[3]);
        }
    }
}

}  // namespace linac
