// fp_rref.cu -- host orchestration of the F_p path: linac_rref_u32 / linac_nullspace_u32.
//
// Schedule: S0 ingest -> recursive right-looking elimination
// (base panels of PW columns: pivot kernel + row exchanges + in-place multipliers; above them
// row-block solves and Schur updates C -= L21.U12 mod p as GEMMs) -> back-elimination of the free
// columns (blocked unit-upper-triangular solve, again GEMMs) -> finalise (pivot columns become
// unit vectors).  One small device->host copy per base panel tells the host how many pivots the
// panel produced; that is the only host involvement (the paper's loop has none, at
// the price of 8 launches per COLUMN).
#include <algorithm>
#include <mutex>
#include <vector>

#include "fp_kernels.cuh"

namespace linac {
extern std::mutex g_call_mutex;

namespace {

struct Fp {
    uint32_t* A;
    int64_t rows, cols, ld;
    ModP f;
    cudaStream_t s;
    // device metadata
    int32_t* d_pivcols;
    PanelInfo* d_info;
    uint32_t* d_E;
    Arena* arena;
    // host
    PanelInfo* h_info;        // pinned
    std::vector<int32_t> pivcols;
    int status = LINAC_OK;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
};

int64_t round_down(int64_t x, int64_t m) { return x / m * m; }

int run_gemm(Fp& c, const GemmArgs& g) {
    Options& o = options();
    const bool timing = o.timing != 0;
    if (timing) cudaEventRecord(c.ev0, c.s);
    int rc = -1;
    if (o.gemm_path != 1 && g.K >= o.tc_min_k && g.M >= o.tc_min_mn && g.N >= o.tc_min_mn) {
        const size_t mark = c.arena->off;
        rc = gemm_modp_tc(g, c.f, c.s, c.arena);
        c.arena->off = mark;
    }
    if (rc < 0) rc = gemm_modp_simt(g, c.f, c.s);
    if (timing && rc == LINAC_OK) {
        cudaEventRecord(c.ev1, c.s);
        cudaEventSynchronize(c.ev1);
        float ms = 0;
        cudaEventElapsedTime(&ms, c.ev0, c.ev1);
        stats().ms_update += ms;
    }
    return rc;
}

// X <- L11^{-1} X for pivots [t0, t0+nb) on columns [c0, c1) of rows t0.. (S4).
int trsm_lower(Fp& c, int64_t t0, int64_t nb, int64_t c0, int64_t c1) {
    if (nb <= 0 || c1 <= c0) return LINAC_OK;
    if (nb <= PW) {
        const int64_t ncols = c1 - c0;
        trsm_lower_base_kernel<<<(unsigned)((ncols + TRSM_THREADS - 1) / TRSM_THREADS), TRSM_THREADS, 0, c.s>>>(
            c.A + t0 * c.ld + c0, c.ld, ncols, c.A, c.ld, c.d_pivcols, t0, (int)nb, c.f);
        LINAC_CUDA(cudaGetLastError());
        stats().kernel_launches++;
        stats().update_macs += nb * nb / 2 * ncols;
        return LINAC_OK;
    }
    const int64_t h = std::max<int64_t>(PW, round_down(nb / 2, PW));
    int rc = trsm_lower(c, t0, h, c0, c1);
    if (rc) return rc;
    GemmArgs g{c.A + (t0 + h) * c.ld + c0, c.ld, c.A + (t0 + h) * c.ld, c.ld, c.d_pivcols + t0,
               c.A + t0 * c.ld + c0,       c.ld, nb - h,                c1 - c0, h};
    rc = run_gemm(c, g);
    if (rc) return rc;
    return trsm_lower(c, t0 + h, nb - h, c0, c1);
}

// One base panel: columns [j0, j0+w), rows >= i0.  Returns the number of pivots through *r.
int base_panel(Fp& c, int64_t j0, int w, int64_t i0, int64_t* r) {
    panel_pivots_kernel<<<1, 256, 0, c.s>>>(c.A, c.ld, c.rows, i0, j0, w, c.f, c.d_info, c.d_E, c.d_pivcols);
    LINAC_CUDA(cudaGetLastError());
    apply_swaps_kernel<<<(unsigned)((c.cols + 255) / 256), 256, 0, c.s>>>(c.A, c.ld, c.cols, i0, c.d_info);
    LINAC_CUDA(cudaGetLastError());
    const int64_t nrows = c.rows - i0;
    panel_apply_kernel<<<(unsigned)((nrows + 7) / 8), 256, 0, c.s>>>(c.A, c.ld, c.rows, i0, j0, w, c.f, c.d_info, c.d_E);
    LINAC_CUDA(cudaGetLastError());
    LINAC_CUDA(cudaMemcpyAsync(c.h_info, c.d_info, sizeof(PanelInfo), cudaMemcpyDeviceToHost, c.s));
    LINAC_CUDA(cudaStreamSynchronize(c.s));
    linac_stats& st = stats();
    st.kernel_launches += 3;
    st.host_syncs++;
    st.panels++;
    st.row_swaps += c.h_info->nswaps;
    st.residual_nonzero += c.h_info->residual;
    *r = c.h_info->r;
    for (int a = 0; a < c.h_info->r; ++a) c.pivcols[i0 + a] = (int32_t)(j0 + c.h_info->pc[a]);
    return LINAC_OK;
}

// Recursive factorisation of columns [j0, j1) with active rows [i0, rows).
int factor(Fp& c, int64_t j0, int64_t j1, int64_t i0, int64_t* r_out) {
    const int64_t w = j1 - j0;
    *r_out = 0;
    if (w <= 0 || i0 >= c.rows) return LINAC_OK;
    if (w <= PW) return base_panel(c, j0, (int)w, i0, r_out);
    const int64_t jm = j0 + std::max<int64_t>(PW, round_down(w / 2, PW));
    int64_t r1 = 0, r2 = 0;
    int rc = factor(c, j0, jm, i0, &r1);
    if (rc) return rc;
    if (r1 > 0) {
        rc = trsm_lower(c, i0, r1, jm, j1);
        if (rc) return rc;
        const int64_t m2 = c.rows - (i0 + r1);
        if (m2 > 0) {
            GemmArgs g{c.A + (i0 + r1) * c.ld + jm, c.ld, c.A + (i0 + r1) * c.ld, c.ld, c.d_pivcols + i0,
                       c.A + i0 * c.ld + jm,        c.ld, m2,                     j1 - jm, r1};
            rc = run_gemm(c, g);
            if (rc) return rc;
        }
    }
    rc = factor(c, jm, j1, i0 + r1, &r2);
    *r_out = r1 + r2;
    return rc;
}

// X <- T^{-1} X on the gathered free columns F (rank x nf, ldf), pivots [t0, t0+nb) (S6).
int trsm_upper(Fp& c, uint32_t* F, int64_t ldf, int64_t nf, int64_t t0, int64_t nb) {
    if (nb <= 0 || nf <= 0) return LINAC_OK;
    if (nb <= PW) {
        trsm_upper_base_kernel<<<(unsigned)((nf + TRSM_THREADS - 1) / TRSM_THREADS), TRSM_THREADS, 0, c.s>>>(
            F + t0 * ldf, ldf, nf, c.A, c.ld, c.d_pivcols, t0, (int)nb, c.f);
        LINAC_CUDA(cudaGetLastError());
        stats().kernel_launches++;
        stats().update_macs += nb * nb / 2 * nf;
        return LINAC_OK;
    }
    const int64_t h = std::max<int64_t>(PW, round_down(nb / 2, PW));   // top block [t0, t0+h), bottom the rest
    int rc = trsm_upper(c, F, ldf, nf, t0 + h, nb - h);
    if (rc) return rc;
    // X_top -= T[top, bottom pivots] . X_bottom
    GemmArgs g{F + t0 * ldf, ldf, c.A + t0 * c.ld, c.ld, c.d_pivcols + t0 + h, F + (t0 + h) * ldf, ldf, h, nf, nb - h};
    rc = run_gemm(c, g);
    if (rc) return rc;
    return trsm_upper(c, F, ldf, nf, t0, h);
}

size_t meta_bytes(int64_t rows, int64_t cols) {
    const int64_t mn = std::max<int64_t>(1, std::min(rows, cols));
    return 4096 + sizeof(PanelInfo) + PW * PW * 4 + (size_t)mn * 4 + (size_t)cols * 8 + 8 * 256;
}

// Free-column slab width for the back-elimination workspace.
int64_t backelim_slab(int64_t rows, int64_t cols) {
    (void)rows;
    return std::min<int64_t>(cols, 4096);
}

size_t workspace_bytes(int64_t rows, int64_t cols) {
    const int64_t mn = std::max<int64_t>(1, std::min(rows, cols));
    size_t b = meta_bytes(rows, cols);
    b += (size_t)mn * (size_t)backelim_slab(rows, cols) * 4 + 256;          // gathered free columns
    b += gemm_modp_tc_scratch_bytes(rows, cols, std::min<int64_t>(mn, 4096)) + 256;
    return b;
}

struct PinnedInfo {
    PanelInfo* p = nullptr;
    ~PinnedInfo() { if (p) cudaFreeHost(p); }
};

int validate(const uint32_t* dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p) {
    if (rows < 0 || cols < 0 || cols >= (1ll << 31) || rows >= (1ll << 40)) return LINAC_ERR_INVALID_ARG;
    if (rows > 0 && cols > 0 && (dA == nullptr || ld < cols)) return LINAC_ERR_INVALID_ARG;
    if (p < 2 || p >= (1u << 31) || !is_prime_u32(p)) return LINAC_ERR_BAD_MODULUS;
    return LINAC_OK;
}

// The whole reduction.  On success the device arrays d_pivcols (in the arena) stay valid until the
// arena is reused, which linac_nullspace_u32 relies on.
int rref_impl(uint32_t* dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p, cudaStream_t s, int64_t* rank,
              int32_t* pivot_cols_out, Arena* arena, int32_t** d_pivcols_out) {
    linac_stats& st = stats();
    st = linac_stats{};
    int rc = validate(dA, rows, cols, ld, p);
    if (rc) return rc;
    if (!rank) return LINAC_ERR_INVALID_ARG;
    *rank = 0;
    if (rows == 0 || cols == 0) return LINAC_OK;
    rc = check_device();
    if (rc) return rc;
    rc = acquire_workspace(workspace_bytes(rows, cols), arena);
    if (rc) return rc;

    static PinnedInfo pinned;
    if (!pinned.p) LINAC_CUDA(cudaMallocHost(&pinned.p, sizeof(PanelInfo)));

    Fp c;
    c.A = dA; c.rows = rows; c.cols = cols; c.ld = ld; c.f = make_modp(p); c.s = s; c.arena = arena;
    const int64_t mn = std::min(rows, cols);
    c.d_info = (PanelInfo*)arena->take(sizeof(PanelInfo));
    c.d_E = (uint32_t*)arena->take(PW * PW * 4);
    c.d_pivcols = (int32_t*)arena->take((size_t)mn * 4);
    if (!c.d_info || !c.d_E || !c.d_pivcols) return LINAC_ERR_WORKSPACE;
    c.h_info = pinned.p;
    c.pivcols.assign(mn, -1);
    LINAC_CUDA(cudaEventCreate(&c.ev0));
    LINAC_CUDA(cudaEventCreate(&c.ev1));
    cudaEvent_t t0, t1;
    LINAC_CUDA(cudaEventCreate(&t0));
    LINAC_CUDA(cudaEventCreate(&t1));
    LINAC_CUDA(cudaEventRecord(t0, s));

    // S0 ingest
    {
        dim3 grid((unsigned)((cols + 255) / 256), (unsigned)std::min<int64_t>(rows, 2048));
        reduce_mod_p_kernel<<<grid, 256, 0, s>>>(dA, rows, cols, ld, p);
        LINAC_CUDA(cudaGetLastError());
        st.kernel_launches++;
    }
    // forward elimination
    int64_t r = 0;
    rc = factor(c, 0, cols, 0, &r);
    if (rc == LINAC_OK && st.residual_nonzero != 0) rc = LINAC_ERR_INTERNAL;
    // S6 back-elimination of the free columns, a slab at a time
    if (rc == LINAC_OK && r > 0 && r < cols) {
        std::vector<char> is_piv(cols, 0);
        for (int64_t t = 0; t < r; ++t) is_piv[c.pivcols[t]] = 1;
        std::vector<int32_t> freec;
        for (int64_t cc = c.pivcols[0]; cc < cols; ++cc)   // free columns left of the first pivot are all zero
            if (!is_piv[cc]) freec.push_back((int32_t)cc);
        const int64_t slab = backelim_slab(rows, cols);
        int32_t* d_free = (int32_t*)arena->take((size_t)std::max<int64_t>(1, slab) * 4);
        uint32_t* F = (uint32_t*)arena->take((size_t)r * (size_t)slab * 4);
        if (!d_free || !F) rc = LINAC_ERR_WORKSPACE;
        for (size_t f0 = 0; rc == LINAC_OK && f0 < freec.size(); f0 += (size_t)slab) {
            const int64_t nf = (int64_t)std::min<size_t>((size_t)slab, freec.size() - f0);
            // only pivots whose column lies left of the slab's last free column can be affected
            LINAC_CUDA(cudaMemcpyAsync(d_free, freec.data() + f0, (size_t)nf * 4, cudaMemcpyHostToDevice, s));
            dim3 grid((unsigned)((nf + 255) / 256), (unsigned)std::min<int64_t>(r, 1024));
            gather_cols_kernel<<<grid, 256, 0, s>>>(dA, ld, r, d_free, nf, F, nf);
            LINAC_CUDA(cudaGetLastError());
            rc = trsm_upper(c, F, nf, nf, 0, r);
            if (rc) break;
            scatter_cols_kernel<<<grid, 256, 0, s>>>(dA, ld, r, d_free, nf, F, nf);
            LINAC_CUDA(cudaGetLastError());
            LINAC_CUDA(cudaStreamSynchronize(s));   // freec slab (pageable host memory) is reused next round
            st.kernel_launches += 2;
            st.host_syncs++;
        }
    }
    // S7 finalise
    if (rc == LINAC_OK && r > 0) {
        LINAC_CUDA(cudaMemcpyAsync(c.d_pivcols, c.pivcols.data(), (size_t)r * 4, cudaMemcpyHostToDevice, s));
        dim3 grid((unsigned)((r + 255) / 256), (unsigned)std::min<int64_t>(rows, 1024));
        finalize_pivot_cols_kernel<<<grid, 256, 0, s>>>(dA, ld, rows, c.d_pivcols, r);
        LINAC_CUDA(cudaGetLastError());
        st.kernel_launches++;
    }
    cudaEventRecord(t1, s);
    cudaError_t e = cudaStreamSynchronize(s);
    st.host_syncs++;
    if (e != cudaSuccess) { set_cuda_error(e, "cudaStreamSynchronize(final)", __FILE__, __LINE__); rc = rc ? rc : LINAC_ERR_CUDA; }
    float ms = 0;
    if (e == cudaSuccess) cudaEventElapsedTime(&ms, t0, t1);
    st.ms_total = ms;
    cudaEventDestroy(t0); cudaEventDestroy(t1);
    cudaEventDestroy(c.ev0); cudaEventDestroy(c.ev1);
    if (rc) return rc;
    *rank = r;
    if (pivot_cols_out) std::copy(c.pivcols.begin(), c.pivcols.begin() + r, pivot_cols_out);
    if (d_pivcols_out) *d_pivcols_out = c.d_pivcols;
    return LINAC_OK;
}

int nullspace_from_rref_impl(const uint32_t* dR, int64_t rows, int64_t cols, int64_t ld, uint32_t p, int64_t rank,
                             const int32_t* pivot_cols, uint32_t* dK, int64_t ldk, cudaStream_t s) {
    (void)rows;
    const int64_t d = cols - rank;
    if (d <= 0) return LINAC_OK;
    std::vector<int32_t> colmap(cols), freec;
    std::vector<char> is_piv(cols, 0);
    for (int64_t t = 0; t < rank; ++t) {
        if (pivot_cols[t] < 0 || pivot_cols[t] >= cols || (t && pivot_cols[t] <= pivot_cols[t - 1]))
            return LINAC_ERR_INVALID_ARG;
        is_piv[pivot_cols[t]] = 1;
        colmap[pivot_cols[t]] = (int32_t)t;
    }
    for (int64_t cc = 0; cc < cols; ++cc)
        if (!is_piv[cc]) { colmap[cc] = -(int32_t)freec.size() - 1; freec.push_back((int32_t)cc); }
    int32_t* dm = nullptr;
    LINAC_CUDA(cudaMalloc(&dm, (size_t)(cols + d) * 4));
    cudaError_t e = cudaMemcpyAsync(dm, colmap.data(), (size_t)cols * 4, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dm + cols, freec.data(), (size_t)d * 4, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) {
        dim3 grid((unsigned)((d + 255) / 256), (unsigned)std::min<int64_t>(cols, 4096));
        nullspace_kernel<<<grid, 256, 0, s>>>(dR, ld, cols, d, dm, dm + cols, dK, ldk, p);
        e = cudaGetLastError();
        stats().kernel_launches++;
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(dm);
    if (e != cudaSuccess) { set_cuda_error(e, "nullspace", __FILE__, __LINE__); return LINAC_ERR_CUDA; }
    return LINAC_OK;
}

}  // namespace
}  // namespace linac

using namespace linac;

extern "C" {

int linac_rref_u32_workspace(int64_t rows, int64_t cols, size_t* bytes) {
    if (!bytes || rows < 0 || cols < 0) return LINAC_ERR_INVALID_ARG;
    *bytes = (rows == 0 || cols == 0) ? 0 : workspace_bytes(rows, cols);
    return LINAC_OK;
}

int linac_rref_u32(uint32_t* dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p, void* stream, int64_t* rank,
                   int32_t* pivot_cols_out) {
    std::lock_guard<std::mutex> lock(g_call_mutex);
    Arena arena;
    return rref_impl(dA, rows, cols, ld, p, (cudaStream_t)stream, rank, pivot_cols_out, &arena, nullptr);
}

int linac_nullspace_u32(uint32_t* dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p, void* stream, int64_t* rank,
                        int32_t* pivot_cols_out, uint32_t* dK, int64_t ldk, int64_t k_capacity_cols, int64_t* nullity) {
    std::lock_guard<std::mutex> lock(g_call_mutex);
    if (!nullity || k_capacity_cols < 0 || (k_capacity_cols > 0 && (!dK || ldk < k_capacity_cols)))
        return LINAC_ERR_INVALID_ARG;
    Arena arena;
    std::vector<int32_t> piv((size_t)std::max<int64_t>(1, std::min(rows, cols)));
    int64_t r = 0;
    int rc = rref_impl(dA, rows, cols, ld, p, (cudaStream_t)stream, &r, piv.data(), &arena, nullptr);
    if (rc) return rc;
    if (rank) *rank = r;
    *nullity = cols - r;
    if (pivot_cols_out) std::copy(piv.begin(), piv.begin() + r, pivot_cols_out);
    if (cols - r > k_capacity_cols) return LINAC_ERR_BUFFER_TOO_SMALL;
    if (cols == 0) return LINAC_OK;
    const linac_stats keep = stats();
    rc = nullspace_from_rref_impl(dA, rows, cols, ld, p, r, piv.data(), dK, ldk, (cudaStream_t)stream);
    stats().kernel_launches = keep.kernel_launches + 1;
    return rc;
}

int linac_nullspace_from_rref_u32(const uint32_t* dR, int64_t rows, int64_t cols, int64_t ld, uint32_t p, int64_t rank,
                                  const int32_t* pivot_cols, uint32_t* dK, int64_t ldk, void* stream) {
    std::lock_guard<std::mutex> lock(g_call_mutex);
    if (rows < 0 || cols < 0 || rank < 0 || rank > std::min(rows, cols) || (rank > 0 && !pivot_cols))
        return LINAC_ERR_INVALID_ARG;
    if (cols - rank > 0 && (!dK || ldk < cols - rank)) return LINAC_ERR_INVALID_ARG;
    if (rows > 0 && cols > 0 && (!dR || ld < cols)) return LINAC_ERR_INVALID_ARG;
    if (p < 2 || p >= (1u << 31) || !is_prime_u32(p)) return LINAC_ERR_BAD_MODULUS;
    int rc = check_device();
    if (rc) return rc;
    return nullspace_from_rref_impl(dR, rows, cols, ld, p, rank, pivot_cols, dK, ldk, (cudaStream_t)stream);
}

int linac_gemm_sub_u32(uint32_t* dC, int64_t ldc, const uint32_t* dA, int64_t lda, const uint32_t* dB, int64_t ldb, int64_t M,
                       int64_t N, int64_t K, uint32_t p, int path, void* stream) {
    std::lock_guard<std::mutex> lock(g_call_mutex);
    if (M < 0 || N < 0 || K < 0 || path < 0 || path > 2) return LINAC_ERR_INVALID_ARG;
    if (p < 2 || p >= (1u << 31) || !is_prime_u32(p)) return LINAC_ERR_BAD_MODULUS;
    if (M == 0 || N == 0 || K == 0) return LINAC_OK;
    if (!dC || !dA || !dB || ldc < N || lda < K || ldb < N) return LINAC_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    stats() = linac_stats{};
    const ModP f = make_modp(p);
    cudaStream_t s = (cudaStream_t)stream;
    GemmArgs g{dC, ldc, dA, lda, nullptr, dB, ldb, M, N, K};
    cudaEvent_t e0, e1;
    LINAC_CUDA(cudaEventCreate(&e0));
    LINAC_CUDA(cudaEventCreate(&e1));
    rc = -1;
    cudaEventRecord(e0, s);
    if (path == 2 || (path == 0 && K >= options().tc_min_k && M >= options().tc_min_mn && N >= options().tc_min_mn)) {
        Arena arena;
        rc = acquire_workspace(gemm_modp_tc_scratch_bytes(M, N, K) + 4096, &arena);
        if (rc) return rc;
        rc = gemm_modp_tc(g, f, s, &arena);
        if (rc < 0 && path == 2) rc = LINAC_ERR_INVALID_ARG;
    }
    if (rc < 0) rc = gemm_modp_simt(g, f, s);
    cudaEventRecord(e1, s);
    cudaError_t e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { set_cuda_error(e, "cudaStreamSynchronize(gemm)", __FILE__, __LINE__); rc = rc ? rc : LINAC_ERR_CUDA; }
    float ms = 0;
    if (e == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
    stats().ms_update = ms;
    stats().ms_total = ms;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return rc;
}

}  // extern "C"
