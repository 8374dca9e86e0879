// fp_wide.cu -- SURVEY.md 8(f) rank 4: the moduli the tensor-core path does not cover (PAPER.md:163:
// "uint32 is used for p <= 2^32 - 1 and uint64 for [larger p]").
//
//   * uint32 storage, 2^31 <= p < 2^32   (linac_rref_u32 routes here)
//   * uint64 storage, odd p < 2^63       (linac_rref_u64)
//
// Schedule: the paper's Gauss-Jordan loop, blocked by PANELS of 32 columns and, like the
// paper's, with NO host involvement ("the device will not be aware of the state of the matrix"):
// the running row index lives in device memory, every kernel of a round reads the panel's record from there
// and exits at once when the panel produced no pivot, so the host only enqueues cols/32 identical rounds:
//
//   wide_panel_kernel      pivot search (warp ballot, first non-zero; K3/K4/K6) among the rows
//                          left, chunk by chunk, with a division-free elimination inside the panel; the pivot
//                          block D = A[pivot rows, pivot columns] is inverted (Gauss-Jordan on [D | I], one
//                          Fermat inverse per pivot; K7)
//   wide_swap_kernel       row exchanges on the columns from the panel on (K5)
//   wide_pivot_rows_kernel U = D^-1 . A[pivot rows, j0:]: the reduced pivot rows, the identity on the panel's pivot
//                          columns (K7's "rescales it to a 1" for 32 pivots at once)
//   wide_lcopy_kernel      L[k][t] = A[k][pivot column t] for every other row k (the "heads")
//   wide_update_kernel     A[k][j0:] -= L[k][:] . U for ALL rows k that are not pivot rows of the panel -- rows
//                          above too, as in the paper's RowReduce (reading Q3) -- so the matrix ends as the RREF
//                          with no separate back-elimination; the pivot columns become unit vectors exactly
//
// Arithmetic: Montgomery form throughout (the matrix is converted on ingest and back at the end), R = 2^32 for
// 32-bit storage and R = 2^64 for 64-bit storage; CUDA cores only (IMAD / IMAD.WIDE).  A limb-plane tensor-core
// formulation would need 5 planes (25 products) for 33-bit residues and 64 products for 64-bit ones.
#include <algorithm>
#include <mutex>
#include <vector>

#include "linac_internal.h"

namespace linac {
namespace {

constexpr int WP = 32;           // panel width

// ---- the two fields ---------------------------------------------------------------------------------------
struct F32W {                    // uint32 storage, odd p < 2^32, R = 2^32
    using T = uint32_t;
    uint32_t p, ninv, one, r2;   // -p^-1 mod R, R mod p, R^2 mod p
    __device__ __forceinline__ T mul(T a, T b) const {
        const uint64_t t = (uint64_t)a * b;
        const uint32_t m = (uint32_t)t * ninv;
        // (t + m p) / 2^32: the low words cancel to 0 or 2^32 (a carry iff the low word of t is non-zero)
        const uint64_t u = (t >> 32) + (((uint64_t)m * p) >> 32) + ((uint32_t)t != 0u ? 1u : 0u);
        return (T)(u >= p ? u - p : u);
    }
    __device__ __forceinline__ T add(T a, T b) const { const uint64_t s = (uint64_t)a + b; return (T)(s >= p ? s - p : s); }
    __device__ __forceinline__ T sub(T a, T b) const { return a >= b ? a - b : a + (p - b); }   // a + (p - b) < p
    __device__ __forceinline__ T canon(T a) const { return a >= p ? a % p : a; }
    // Lazy dot product: the raw 64-bit products are summed in a 96-bit accumulator (two instructions per term: an
    // IMAD.WIDE with carry-out and the carry into the top word -- what the compiler makes of the 128-bit sum, whose
    // top 32 bits are never read) and reduced once -- sum_t mul(l_t, u_t) without a reduction per term.
    struct Acc { unsigned __int128 v; };
    __device__ __forceinline__ void acc_zero(Acc& c) const { c.v = 0; }
    __device__ __forceinline__ void acc_mac(Acc& c, T a, T b) const { c.v += (uint64_t)a * b; }
    // (a2 2^64 + a1 2^32 + a0) R^-1 mod p, R = 2^32: one Montgomery step on (a1 : a0) leaves u < 2^33, and
    // u mod p = mul(mul(u_lo, R^2), 1), 2^32 k mod p = mul(k, R^2) for the small k = a2 + (u >> 32)
    __device__ __forceinline__ T acc_reduce(const Acc& c) const {
        const uint32_t a0 = (uint32_t)c.v, a1 = (uint32_t)(c.v >> 32), a2 = (uint32_t)(c.v >> 64);
        const uint32_t m = a0 * ninv;
        const uint64_t u = (uint64_t)a1 + (((uint64_t)m * p) >> 32) + (a0 != 0u ? 1u : 0u);
        const T x = mul(mul((T)u, r2), 1u);
        const T w = mul((T)(a2 + (uint32_t)(u >> 32)), r2);
        return add(x, w);
    }
};
struct F64M {                    // uint64 storage, odd p < 2^63, R = 2^64
    using T = unsigned long long;
    unsigned long long p, ninv, one, r2;
    __device__ __forceinline__ T mul(T a, T b) const {
        const T lo = a * b, hi = __umul64hi(a, b);
        const T m = lo * ninv;
        const T u = hi + __umul64hi(m, p) + (lo != 0ull ? 1ull : 0ull);      // < 2p < 2^64
        return u >= p ? u - p : u;
    }
    __device__ __forceinline__ T add(T a, T b) const { const T s = a + b; return s >= p ? s - p : s; }   // p < 2^63
    __device__ __forceinline__ T sub(T a, T b) const { return a >= b ? a - b : a + (p - b); }
    __device__ __forceinline__ T canon(T a) const { return a >= p ? a % p : a; }
    // Lazy dot product in a 192-bit accumulator (see F32W), R = 2^64.
    struct Acc { unsigned long long a0, a1, a2; };
    __device__ __forceinline__ void acc_zero(Acc& c) const { c.a0 = c.a1 = c.a2 = 0ull; }
    __device__ __forceinline__ void acc_mac(Acc& c, T a, T b) const {
        const T lo = a * b, hi = __umul64hi(a, b);
        asm("add.cc.u64 %0, %0, %3;\n\taddc.cc.u64 %1, %1, %4;\n\taddc.u64 %2, %2, 0;"
            : "+l"(c.a0), "+l"(c.a1), "+l"(c.a2) : "l"(lo), "l"(hi));
    }
    __device__ __forceinline__ T acc_reduce(const Acc& c) const {
        const T m = c.a0 * ninv;
        T u = c.a1 + __umul64hi(m, p);                     // (a1 : a0 + m p) / 2^64, up to 65 bits
        unsigned long long ov = u < c.a1 ? 1ull : 0ull;
        if (c.a0 != 0ull) { u += 1ull; ov += u == 0ull ? 1ull : 0ull; }
        const T x = mul(mul(u, r2), 1ull);                 // u mod p (mul takes any 64-bit first factor)
        const T w = mul(c.a2 + ov, r2);                    // 2^64 k mod p
        return add(x, w);
    }
};
template <class F> __device__ __forceinline__ typename F::T to_mont(const F& f, typename F::T a) { return f.mul(f.canon(a), f.r2); }
template <class F> __device__ __forceinline__ typename F::T from_mont(const F& f, typename F::T a) { return f.mul(a, 1); }
// d*x - h*y (Montgomery products: the common factor R^-1 only rescales the row)
template <class F> __device__ __forceinline__ typename F::T lincomb(const F& f, typename F::T d, typename F::T x, typename F::T h, typename F::T y) {
    return f.sub(f.mul(d, x), f.mul(h, y));
}
// a^-1 (a and the result in Montgomery form): Fermat, a^(p-2), square-and-multiply
template <class F> __device__ typename F::T inv_mont(const F& f, typename F::T a) {
    typename F::T acc = f.one, base = a;
    for (typename F::T e = f.p - 2; e; e >>= 1) {
        if (e & 1) acc = f.mul(acc, base);
        base = f.mul(base, base);
    }
    return acc;
}

// ---- device-resident control state (the host never reads it during the loop) -----------------------------
struct WideRec {
    long long i0;                // first pivot row of this panel
    int r;                       // pivots found (<= 32)
    int nswaps;
    int pc[WP];                  // local pivot columns, ascending (-1 beyond r)
    long long swp[WP];           // LAPACK style: at step a exchange rows i0+a and swp[a]
};
struct WideState {
    long long i;                 // next pivot row (the paper's row counter)
};

template <class F>
struct WideSmem {
    typename F::T X[WP][WP + 1];
    typename F::T Ep[WP][WP + 1];
    typename F::T G[WP][2 * WP + 1];
    typename F::T ginv[WP];
    int epc[WP];
    long long esrc[WP];
    int ord[WP];
    long long pos_of[WP];
    int at[WP];
    int nsw;
};

template <class F>
__global__ void wide_ingest_kernel(typename F::T* __restrict__ A, int64_t rows, int64_t cols, int64_t ld, F f, bool to) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cols) return;
    for (int64_t r = blockIdx.y; r < rows; r += gridDim.y) {
        const typename F::T v = A[r * ld + c];
        A[r * ld + c] = to ? to_mont(f, v) : from_mont(f, v);
    }
}

// One CTA of 1024 threads (warp = chunk row, lane = panel column).
template <class F>
__global__ void __launch_bounds__(1024, 1) wide_panel_kernel(typename F::T* __restrict__ A, int64_t ld, int64_t rows, int64_t j0,
                                                              int w, WideState* st, WideRec* rec, typename F::T* __restrict__ Tout,
                                                              int32_t* __restrict__ pivcols, F f) {
    using T = typename F::T;
    __shared__ WideSmem<F> sm;
    const int tid = threadIdx.x, lane = tid & 31, wq = tid >> 5;
    const int64_t i0 = st->i;
    int r = 0;
    unsigned pcmask = 0;
    for (int64_t cs = i0; cs < rows && r < w; cs += WP) {
        const int nh = (int)min((int64_t)WP, rows - cs);
        T s = 0;
        if (wq < nh && lane < w) s = A[(cs + wq) * ld + j0 + lane];
        for (int a = 0; a < r; ++a) {                          // against the pivots found so far, ascending column
            const int tt = sm.ord[a];
            const int c = sm.epc[tt];
            const T l = __shfl_sync(0xffffffffu, s, c);
            if (l) s = lane > c ? lincomb(f, sm.Ep[tt][c], s, l, sm.Ep[tt][lane]) : (lane == c ? (T)0 : f.mul(sm.Ep[tt][c], s));
        }
        sm.X[wq][lane] = s;
        if (!__syncthreads_or(s != 0)) continue;               // the whole chunk lies in the span found so far
        unsigned used = 0;
        for (int c = 0; c < w && r < w; ++c) {
            if ((pcmask >> c) & 1u) continue;
            const unsigned cand = __ballot_sync(0xffffffffu, sm.X[lane][c] != 0) & ~used;   // first non-zero
            if (!cand) continue;
            const int q = __ffs(cand) - 1;
            const T d = sm.X[q][c];
            const T pv = sm.X[q][lane];
            if (wq != q && !((used >> wq) & 1u)) {
                const T h = sm.X[wq][c];
                if (h != 0 && lane > c) sm.X[wq][lane] = lincomb(f, d, sm.X[wq][lane], h, pv);   // column c itself is not rewritten
            }
            if (wq == 0) sm.Ep[r][lane] = ((pcmask >> lane) & 1u) ? (T)0 : pv;
            if (tid == 0) { sm.epc[r] = c; sm.esrc[r] = cs + q; }
            used |= 1u << q;
            pcmask |= 1u << c;
            ++r;
            __syncthreads();
        }
        if (wq == 0) {                                         // rank sort of the pivots by column
            const int mine = lane < r ? sm.epc[lane] : INT_MAX;
            int pos = 0;
            for (int t = 0; t < r; ++t) pos += (sm.epc[t] < mine);
            if (lane < r) sm.ord[pos] = lane;
        }
        __syncthreads();
    }
    // exchange list: row i0+a must receive source row esrc[ord[a]]
    if (wq == 0) {
        if (lane < r) { sm.pos_of[lane] = i0 + lane; sm.at[lane] = lane; }
        __syncwarp();
        if (lane == 0) {
            int nsw = 0;
            for (int a = 0; a < r; ++a) {
                const long long src = sm.esrc[sm.ord[a]];
                const long long cur = src < i0 + r ? sm.pos_of[(int)(src - i0)] : src;
                rec->swp[a] = cur;
                if (cur != i0 + a) {
                    ++nsw;
                    const int x = sm.at[a];
                    sm.pos_of[x] = cur;
                    if (cur < i0 + r) sm.at[(int)(cur - i0)] = x;
                }
            }
            sm.nsw = nsw;
        }
    }
    __syncthreads();
    // T = D^-1, D = A[pivot rows, pivot columns] in ascending pivot-column order: Gauss-Jordan on [D | I], division-free
    for (int e = tid; e < WP * 2 * WP; e += 1024) {
        const int a = e / (2 * WP), b = e % (2 * WP);
        T v = 0;
        if (a < r) {
            if (b < WP) { if (b < r) v = A[sm.esrc[sm.ord[a]] * ld + j0 + sm.epc[sm.ord[b]]]; }
            else v = (b - WP == a) ? f.one : (T)0;
        }
        sm.G[a][b] = v;
    }
    __syncthreads();
    for (int t = 0; t < r; ++t) {
        const T d = sm.G[t][t];
        const T pl = lane > t ? sm.G[t][lane] : (T)0;
        const T pr = lane <= t ? sm.G[t][WP + lane] : (T)0;
        if (wq != t && wq < r) {
            const T h = sm.G[wq][t];
            if (h != 0) {
                if (lane > t || lane == wq) sm.G[wq][lane] = lincomb(f, d, sm.G[wq][lane], h, pl);
                if (lane <= t || lane == wq) sm.G[wq][WP + lane] = lincomb(f, d, sm.G[wq][WP + lane], h, pr);
            }
        }
        __syncthreads();
    }
    if (wq == 0 && lane < r) sm.ginv[lane] = inv_mont(f, sm.G[lane][lane]);
    __syncthreads();
    Tout[wq * WP + lane] = (wq < r && lane < r) ? f.mul(sm.ginv[wq], sm.G[wq][WP + lane]) : (T)0;
    if (tid < WP) {
        const int pc = tid < r ? sm.epc[sm.ord[tid]] : -1;
        rec->pc[tid] = pc;
        if (tid < r) pivcols[i0 + tid] = (int32_t)(j0 + pc);
    }
    if (tid == 0) {
        rec->i0 = i0;
        rec->r = r;
        rec->nswaps = sm.nsw;
        st->i = i0 + r;
    }
}

template <class T>
__global__ void wide_swap_kernel(T* __restrict__ A, int64_t ld, int64_t c0, int64_t cols, const WideRec* __restrict__ rec) {
    const int r = rec->r;
    if (r == 0 || rec->nswaps == 0) return;
    const int64_t c = c0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cols) return;
    const int64_t i0 = rec->i0;
    for (int a = 0; a < r; ++a) {
        const int64_t s = rec->swp[a];
        if (s != i0 + a) {
            const T x = A[(i0 + a) * ld + c], y = A[s * ld + c];
            A[(i0 + a) * ld + c] = y;
            A[s * ld + c] = x;
        }
    }
}

// U = T . A[i0 : i0+r, c] for the columns c >= j0: thread per column, T in shared memory.
template <class F>
__global__ void __launch_bounds__(128) wide_pivot_rows_kernel(typename F::T* __restrict__ A, int64_t ld, int64_t j0, int64_t cols,
                                                             const WideRec* __restrict__ rec, const typename F::T* __restrict__ Tin,
                                                             typename F::T* __restrict__ U, int64_t ldu, F f) {
    using T = typename F::T;
    __shared__ T Ts[WP][WP + 1];
    const int r = rec->r;
    if (r == 0) return;
    for (int e = threadIdx.x; e < WP * WP; e += 128) Ts[e / WP][e % WP] = Tin[e];
    __syncthreads();
    const int64_t c = j0 + (int64_t)blockIdx.x * 128 + threadIdx.x;
    if (c >= cols) return;
    const int64_t i0 = rec->i0;
    T x[WP];
#pragma unroll
    for (int b = 0; b < WP; ++b) x[b] = b < r ? A[(i0 + b) * ld + c] : (T)0;
    for (int a = 0; a < WP; ++a) {
        T acc = 0;
        if (a < r) {
            typename F::Acc s;
            f.acc_zero(s);
#pragma unroll
            for (int b = 0; b < WP; ++b) f.acc_mac(s, Ts[a][b], x[b]);
            acc = f.acc_reduce(s);
            A[(i0 + a) * ld + c] = acc;
        }
        U[(int64_t)a * ldu + c] = acc;
    }
}

// L[k][t] = A[k][j0 + pc[t]] for the rows that are not pivot rows of the panel (zero for those, and for t >= r).
template <class T>
__global__ void wide_lcopy_kernel(const T* __restrict__ A, int64_t ld, int64_t rows, int64_t j0, const WideRec* __restrict__ rec,
                                  T* __restrict__ L) {
    const int r = rec->r;
    if (r == 0) return;
    const int t = threadIdx.x & 31;
    const int64_t i0 = rec->i0;
    const int pc = rec->pc[t];
    for (int64_t k = (int64_t)blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5); k < rows; k += (int64_t)gridDim.x * (blockDim.x / 32)) {
        const bool pivot_row = k >= i0 && k < i0 + r;
        L[k * WP + t] = (pc >= 0 && !pivot_row) ? A[k * ld + j0 + pc] : (T)0;
    }
}

// A[k][c] -= sum_t L[k][t] U[t][c]: 64 x 64 tiles, 256 threads, 4 x 4 outputs per thread.
template <class F>
__global__ void __launch_bounds__(256) wide_update_kernel(typename F::T* __restrict__ A, int64_t ld, int64_t rows, int64_t j0, int64_t cols,
                                                         const WideRec* __restrict__ rec, const typename F::T* __restrict__ L,
                                                         const typename F::T* __restrict__ U, int64_t ldu, F f) {
    using T = typename F::T;
    __shared__ T Ls[64][WP + 1];
    __shared__ T Us[WP][64];
    const int r = rec->r;
    if (r == 0) return;
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int64_t m0 = (int64_t)blockIdx.y * 64, n0 = j0 + (int64_t)blockIdx.x * 64;
    for (int e = tid; e < 64 * WP; e += 256) {
        const int mm = e / WP, t = e % WP;
        Ls[mm][t] = m0 + mm < rows ? L[(m0 + mm) * WP + t] : (T)0;
    }
    for (int e = tid; e < WP * 64; e += 256) {
        const int t = e / 64, nn = e % 64;
        Us[t][nn] = (t < r && n0 + nn < cols) ? U[(int64_t)t * ldu + n0 + nn] : (T)0;
    }
    __syncthreads();
    typename F::Acc acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) f.acc_zero(acc[i][j]);
    bool any = false;
#pragma unroll
    for (int i = 0; i < 4; ++i)
        for (int t = 0; t < r; ++t) any = any || Ls[ty * 4 + i][t] != 0;
    if (!any) return;                                   // conditional skipping: rows with zero heads
#pragma unroll 2
    for (int t = 0; t < r; ++t) {
        T l[4], u[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) l[i] = Ls[ty * 4 + i][t];
#pragma unroll
        for (int j = 0; j < 4; ++j) u[j] = Us[t][tx + 16 * j];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) f.acc_mac(acc[i][j], l[i], u[j]);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int64_t m = m0 + ty * 4 + i;
        if (m >= rows) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int64_t c = n0 + tx + 16 * j;
            if (c < cols) A[m * ld + c] = f.sub(A[m * ld + c], f.acc_reduce(acc[i][j]));
        }
    }
}

// ---- host ------------------------------------------------------------------------------------------------
uint64_t mulmod_u64(uint64_t a, uint64_t b, uint64_t m) { return (uint64_t)((unsigned __int128)a * b % m); }

F32W make_f32w(uint32_t p) {
    F32W f; f.p = p;
    uint32_t inv = p; for (int i = 0; i < 5; ++i) inv *= 2u - p * inv;
    f.ninv = 0u - inv;
    f.one = (uint32_t)((1ull << 32) % p);
    f.r2 = (uint32_t)((uint64_t)f.one * f.one % p);
    return f;
}
F64M make_f64m(uint64_t p) {
    F64M f; f.p = p;
    uint64_t inv = p; for (int i = 0; i < 6; ++i) inv *= 2ull - p * inv;
    f.ninv = 0ull - inv;
    f.one = (uint64_t)((((unsigned __int128)1) << 64) % p);
    f.r2 = mulmod_u64(f.one, f.one, p);
    return f;
}

template <class T> size_t wide_workspace(int64_t rows, int64_t cols) {
    const int64_t ldu = (cols + 63) / 64 * 64;
    return 8192 + (size_t)cols * 12 + (size_t)WP * ldu * sizeof(T) + (size_t)rows * WP * sizeof(T) + WP * WP * sizeof(T) + sizeof(WideRec) + 256 +
           (size_t)std::max<int64_t>(1, std::min(rows, cols)) * 4 + 1024;
}

template <class F>
int rref_wide(typename F::T* dA, int64_t rows, int64_t cols, int64_t ld, const F& f, cudaStream_t s, int64_t* rank,
              int32_t* pivot_cols_out, Arena* ext_arena) {
    using T = typename F::T;
    linac_stats& st = stats();
    st = linac_stats{};
    *rank = 0;
    if (rows == 0 || cols == 0) return LINAC_OK;
    int rc = check_device();
    if (rc) return rc;
    Arena own;
    if (!ext_arena) {
        rc = acquire_workspace(wide_workspace<T>(rows, cols), &own);
        if (rc) return rc;
    }
    Arena& arena = ext_arena ? *ext_arena : own;
    const int64_t mn = std::min(rows, cols), ldu = (cols + 63) / 64 * 64;
    T* U = (T*)arena.take((size_t)WP * ldu * sizeof(T));
    T* L = (T*)arena.take((size_t)rows * WP * sizeof(T));
    T* Tb = (T*)arena.take(WP * WP * sizeof(T));
    WideRec* rec = (WideRec*)arena.take(sizeof(WideRec));
    WideState* state = (WideState*)arena.take(sizeof(WideState));
    int32_t* d_piv = (int32_t*)arena.take((size_t)mn * 4);
    if (!U || !L || !Tb || !rec || !state || !d_piv) return LINAC_ERR_WORKSPACE;
    LINAC_CUDA(cudaMemsetAsync(state, 0, sizeof(WideState), s));
    {
        dim3 grid((unsigned)((cols + 255) / 256), (unsigned)std::min<int64_t>(rows, 2048));
        wide_ingest_kernel<F><<<grid, 256, 0, s>>>(dA, rows, cols, ld, f, true);
        LINAC_CUDA(cudaGetLastError());
        st.kernel_launches++;
    }
    for (int64_t j0 = 0; j0 < cols; j0 += WP) {
        const int w = (int)std::min<int64_t>(WP, cols - j0);
        const int64_t nc = cols - j0;
        wide_panel_kernel<F><<<1, 1024, 0, s>>>(dA, ld, rows, j0, w, state, rec, Tb, d_piv, f);
        wide_swap_kernel<T><<<(unsigned)((nc + 255) / 256), 256, 0, s>>>(dA, ld, j0, cols, rec);
        wide_pivot_rows_kernel<F><<<(unsigned)((nc + 127) / 128), 128, 0, s>>>(dA, ld, j0, cols, rec, Tb, U, ldu, f);
        wide_lcopy_kernel<T><<<(unsigned)std::min<int64_t>((rows + 7) / 8, 148 * 8), 256, 0, s>>>(dA, ld, rows, j0, rec, L);
        dim3 grid((unsigned)((nc + 63) / 64), (unsigned)((rows + 63) / 64));
        wide_update_kernel<F><<<grid, 256, 0, s>>>(dA, ld, rows, j0, cols, rec, L, U, ldu, f);
        LINAC_CUDA(cudaGetLastError());
        st.kernel_launches += 5;
        st.panels++;
        st.update_macs += rows * nc * w;
    }
    {
        dim3 grid((unsigned)((cols + 255) / 256), (unsigned)std::min<int64_t>(rows, 2048));
        wide_ingest_kernel<F><<<grid, 256, 0, s>>>(dA, rows, cols, ld, f, false);
        LINAC_CUDA(cudaGetLastError());
        st.kernel_launches++;
    }
    WideState h_state{};
    std::vector<int32_t> piv((size_t)mn);
    LINAC_CUDA(cudaMemcpyAsync(&h_state, state, sizeof h_state, cudaMemcpyDeviceToHost, s));
    LINAC_CUDA(cudaMemcpyAsync(piv.data(), d_piv, (size_t)mn * 4, cudaMemcpyDeviceToHost, s));
    LINAC_CUDA(cudaStreamSynchronize(s));
    st.host_syncs++;
    if (h_state.i < 0 || h_state.i > mn) return LINAC_ERR_INTERNAL;
    *rank = h_state.i;
    if (pivot_cols_out) std::copy(piv.begin(), piv.begin() + h_state.i, pivot_cols_out);
    return LINAC_OK;
}

}  // namespace

size_t wide_workspace_u32(int64_t rows, int64_t cols) { return wide_workspace<uint32_t>(rows, cols); }

// linac_rref_u32 with 2^31 <= p < 2^32; `arena` is the caller's workspace (the consumers behind it take more from it)
int rref_u32_wide(uint32_t* dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p, cudaStream_t s, int64_t* rank,
                  int32_t* pivot_cols_out, Arena* arena) {
    return rref_wide<F32W>(dA, rows, cols, ld, make_f32w(p), s, rank, pivot_cols_out, arena);
}

}  // namespace linac

using namespace linac;

extern "C" {

int linac_rref_u64_workspace(int64_t rows, int64_t cols, size_t* bytes) {
    if (!bytes || rows < 0 || cols < 0) return LINAC_ERR_INVALID_ARG;
    *bytes = (rows == 0 || cols == 0) ? 0 : wide_workspace<unsigned long long>(rows, cols);
    return LINAC_OK;
}

int linac_rref_u64(uint64_t* dA, int64_t rows, int64_t cols, int64_t ld, uint64_t p, void* stream, int64_t* rank,
                   int32_t* pivot_cols_out) {
    if (rows < 0 || cols < 0 || cols >= (1ll << 31) || rows >= (1ll << 31) || !rank) return LINAC_ERR_INVALID_ARG;
    if (rows > 0 && cols > 0 && (dA == nullptr || ld < cols)) return LINAC_ERR_INVALID_ARG;
    if (p < 3 || p >= (1ull << 63) || !is_prime_u64(p)) return LINAC_ERR_BAD_MODULUS;
    return rref_wide<F64M>(reinterpret_cast<unsigned long long*>(dA), rows, cols, ld, make_f64m(p), (cudaStream_t)stream, rank,
                           pivot_cols_out, nullptr);
}

}  // extern "C"
