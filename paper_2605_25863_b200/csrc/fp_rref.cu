// fp_rref.cu -- host orchestration of the F_p path: linac_rref_u32 / linac_nullspace_u32.
//
// Schedule: S0 ingest -> recursive right-looking elimination over
// STRIPS of `strip_width` columns.  One cooperative kernel factors a strip (fp_strip.cuh: pivot rows,
// pivot columns and T = (pivot block)^-1 per 32-column base panel, row exchanges, the in-strip updates;
// the multipliers are the stored entries themselves); between strips the row-block solves U12 = L11^-1 A12
// (column-parallel leaf kernel per strip, GEMMs between strips) and the Schur updates C -= L21.U12 mod p
// (tensor-core GEMMs) -> back-elimination of the free columns (blocked unit-upper-triangular solve with
// the same leaf kernel and GEMMs) -> finalise.  One small device->host copy per STRIP tells the host how
// many pivots it produced; that is the only host involvement (the paper's loop has none, at
// the price of 8 launches per COLUMN).
#include <algorithm>
#include <atomic>
#include <cstring>
#include <mutex>
#include <vector>

#include "fp_kernels.cuh"
#include "fp_strip.cuh"
#include "tc_ptx.cuh"
#include "fp_trsm_inv.cuh"

namespace linac {

namespace {

struct Fp {
    uint32_t* A;
    int64_t rows, cols, ld;
    ModP f;
    cudaStream_t s;
    int64_t nb;               // number of base panels = ceil(cols / PW)
    int64_t bps;              // base panels per strip
    int64_t ns;               // number of strips
    int coop_grid;            // CTAs of the cooperative strip kernel
    int slot;                 // this thread's entry of the constant field table
    // device metadata
    int32_t* d_pivcols;
    int32_t* d_pstart;        // [nb+1]
    PanelRec* d_rec;          // [nb]
    uint32_t* d_T;            // [nb][PW*PW]
    uint32_t* d_E;            // [nb][PW*PW]
    uint8_t* d_W = nullptr;   // 2 x [4][WK][WK] limb planes of a regular strip's solve operator (fp_trsm_inv.cuh); strip s uses
                              // buffer s & 1: the tail of strip s's solve (second stream) may still read W while W of s+1 is written
    int64_t winv_count = 0;
    Arena* arena;
    // host
    unsigned long long* h_mail;      // mapped pinned, MAXBP * MAIL_WORDS tagged words written by the strip kernel itself
    std::vector<int64_t> pstart;     // [nb+1] pivots found left of base panel b
    std::vector<int32_t> pivcols;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    // timing == 2: the PRODUCTION schedule with an event pair around every launch and no host synchronisation; the
    // pairs are read after the call's final sync (class 0 = Schur update, 1 = strip kernel, 2 = triangular solve)
    std::vector<cudaEvent_t>* pool = nullptr;
    struct Mark { int cls; int ev; int64_t m, n, k; cudaStream_t on; };
    std::vector<Mark> marks;
    int pool_used = 0;
    int mark_begin(int cls, int64_t m = 0, int64_t n = 0, int64_t k = 0, cudaStream_t on = nullptr) {
        if (options().timing != 2 || !pool) return -1;
        if (!on) on = s;
        if (pool_used + 2 > (int)pool->size()) {
            const size_t old = pool->size();
            pool->resize(old + 512, nullptr);
            for (size_t i = old; i < pool->size(); ++i) cudaEventCreate(&(*pool)[i]);
        }
        marks.push_back({cls, pool_used, m, n, k, on});
        cudaEventRecord((*pool)[pool_used], on);
        pool_used += 2;
        return (int)marks.size() - 1;
    }
    void mark_end(int h) { if (h >= 0) cudaEventRecord((*pool)[marks[h].ev + 1], marks[h].on); }

    int64_t sb0(int64_t s) const { return std::min(nb, s * bps); }          // first base panel of strip s
    int64_t sp(int64_t s) const { return pstart[sb0(s)]; }                  // pivots found left of strip s
};

constexpr int LINAC_EARLY_SOLVE_DONE = -1000;      // internal: factor_strip already enqueued the row-block solve

int64_t panel_col0(int64_t b) { return b * PW; }

int run_gemm(Fp& c, const GemmArgs& g, cudaStream_t stream = nullptr) {
    Options& o = options();
    if (!stream) stream = c.s;
    const bool timing = o.timing == 1;
    if (timing) cudaEventRecord(c.ev0, c.s);
    const int mk = c.mark_begin(0, g.M, g.N, g.K, stream);
    int rc = -1;
    if (o.gemm_path != 1 && g.K >= o.tc_min_k && g.M >= o.tc_min_mn && g.N >= o.tc_min_mn) {
        const size_t mark = c.arena->off;
        rc = gemm_modp_tc(g, c.f, stream, c.arena);
        c.arena->off = mark;
    }
    if (rc < 0) rc = gemm_modp_simt(g, c.f, stream);
    c.mark_end(mk);
    if (timing && rc == LINAC_OK) {
        cudaEventRecord(c.ev1, c.s);
        cudaEventSynchronize(c.ev1);
        float ms = 0;
        cudaEventElapsedTime(&ms, c.ev0, c.ev1);
        stats().ms_update += ms;
        if ((double)g.M * g.N * g.K > (double)stats().top_m * stats().top_n * stats().top_k) {
            stats().top_m = g.M; stats().top_n = g.N; stats().top_k = g.K;
            stats().ms_update_top = ms;
        }
    }
    return rc;
}

// Brackets one kernel class with events when the "timing" option is on (costs a host sync per launch).
struct Timed {
    Fp& c; double& acc; bool on; int mk;
    Timed(Fp& c_, double& acc_, int cls, cudaStream_t stream = nullptr)
        : c(c_), acc(acc_), on(options().timing == 1), mk(c_.mark_begin(cls, 0, 0, 0, stream)) {
        if (on) cudaEventRecord(c.ev0, c.s);
    }
    ~Timed() {
        c.mark_end(mk);
        if (!on) return;
        cudaEventRecord(c.ev1, c.s);
        cudaEventSynchronize(c.ev1);
        float ms = 0;
        if (cudaEventElapsedTime(&ms, c.ev0, c.ev1) == cudaSuccess) acc += ms;
    }
};


// Leaf of both triangular solves: the pivots of ONE strip against columns [0, ncols) of X.
template <bool LOWER>
int trsm_leaf(Fp& c, int64_t s, uint32_t* X, int64_t ldx, int64_t ncols) {
    const int64_t K = c.sp(s + 1) - c.sp(s);
    if (K <= 0 || ncols <= 0) return LINAC_OK;
    if (!LOWER && c.sb0(s + 1) - c.sb0(s) <= 1) return LINAC_OK;     // U is the identity inside one base panel
    Timed tm(c, stats().ms_trsm, 2);
    if (LOWER && options().trsm_winv != 0 && c.d_W != nullptr && K == WK && c.sb0(s + 1) - c.sb0(s) == WK / PW && ncols >= 4 * WTN) {
        bool regular = true;                                   // four base panels with 32 pivots each: one product with W
        for (int64_t b = c.sb0(s); b < c.sb0(s + 1); ++b) regular = regular && c.pstart[b + 1] - c.pstart[b] == PW;
        if (regular) {
            uint8_t* W = c.d_W + (size_t)((c.winv_count++) & 1) * W_A_BYTES;
            strip_winv_kernel<<<WINV_CTAS, WINV_NT, sizeof(WinvSmem), c.s>>>(c.A, c.ld, c.d_pstart, (int)c.sb0(s), c.d_T,
                                                                             (int)c.sp(s), c.f, W);
            LINAC_CUDA(cudaGetLastError());
            const int64_t ntiles = (ncols + WTN - 1) / WTN;
            trsm_winv_kernel<<<(unsigned)std::min<int64_t>(ntiles, 2 * sm_count()), WNT, WTRSM_SMEM, c.s>>>(
                W, X, ldx, ncols, c.f, nullptr, 0, 0, ncols);
            LINAC_CUDA(cudaGetLastError());
            stats().kernel_launches += 2;
            stats().winv_solves++;
            stats().update_macs += K * K / 2 * ncols;
            return LINAC_OK;
        }
    }
    trsm_strip_kernel<LOWER><<<(unsigned)((ncols + PW - 1) / PW), TNT, trsm_smem_bytes(K), c.s>>>(
        c.A, c.ld, X, ldx, ncols, c.d_pstart, (int)c.sb0(s), (int)c.sb0(s + 1), c.d_T, c.d_pivcols, c.f, nullptr, 0, nullptr, 0, nullptr,
        0, 0);
    LINAC_CUDA(cudaGetLastError());
    stats().kernel_launches++;
    stats().update_macs += K * K / 2 * ncols;
    return LINAC_OK;
}

// X <- L^{-1} X (S4) for the pivots of strips [s0, s1) on columns [c0, c1) of their rows: leaf kernel per
// strip; between blocks X_bottom -= L[bottom rows, top pivot columns] . X_top.
int trsm_lower(Fp& c, int64_t s0, int64_t s1, int64_t c0, int64_t c1) {
    const int64_t t0 = c.sp(s0), t1 = c.sp(s1);
    if (t1 <= t0 || c1 <= c0) return LINAC_OK;
    if (s1 - s0 == 1) return trsm_leaf<true>(c, s0, c.A + t0 * c.ld + c0, c.ld, c1 - c0);
    const int64_t sh = s0 + (s1 - s0) / 2, th = c.sp(sh);
    int rc = trsm_lower(c, s0, sh, c0, c1);
    if (rc) return rc;
    if (th > t0 && t1 > th) {
        GemmArgs g{c.A + th * c.ld + c0, c.ld, c.A + th * c.ld, c.ld, c.d_pivcols + t0,
                   c.A + t0 * c.ld + c0, c.ld, t1 - th,         c1 - c0, th - t0};
        rc = run_gemm(c, g);
        if (rc) return rc;
    }
    return trsm_lower(c, sh, s1, c0, c1);
}

int factor(Fp& c, int64_t s0, int64_t s1, int64_t i0, int64_t* r_out, bool allow_flat);

// A strip kernel in flight: what collect_strip needs to read its mail.
struct StripLaunch {
    unsigned long long seq = 0;
    int64_t b0 = 0, b1 = 0, j0 = 0, j1 = 0;
    cudaStream_t stream = nullptr;
    bool winv = false;        // strip_winv_kernel was enqueued behind the strip kernel (it writes W only for a regular strip)
    uint8_t* W = nullptr;     // ... into this buffer
    // filled by collect_strip
    int64_t nswaps = 0;       // row exchanges of the strip's panels that found pivots
    bool regular = false;     // four base panels with 32 pivots each
};

// Launches the cooperative strip kernel for strip s (active rows >= i0) on `stream` with `grid` CTAs.
//   self_mail  the kernel posts its records to the host mailbox itself (otherwise the solve kernel behind it does)
//   la         look-ahead launch: row exchanges are applied to the strip's own columns only (deferred_swaps_kernel
//              applies the rest once the previous strip's bulk update has finished with those rows)
int launch_strip(Fp& c, int64_t s, int64_t i0, cudaStream_t stream, int grid, bool la, bool self_mail, uint8_t* tail_Aq,
                 int kp, StripLaunch* out) {
    const int64_t b0 = c.sb0(s), b1 = c.sb0(s + 1);
    const int64_t j0 = panel_col0(b0), j1 = std::min(c.cols, panel_col0(b1));
    StripArgs a;
    a.A = c.A; a.ld = c.ld; a.rows = c.rows; a.cols = c.cols; a.i0 = i0; a.j0 = j0; a.ws = (int)(j1 - j0);
    a.rec = c.d_rec; a.T = c.d_T; a.E = c.d_E; a.pivcols = c.d_pivcols; a.pstart = c.d_pstart;
    a.Aq = tail_Aq; a.kp = kp;
    a.slot = c.slot;
    a.swap_c0 = la ? j0 : 0;
    a.swap_c1 = la ? j1 : c.cols;
    a.seq = (++ctx().seq) & 0xFFFFFFFFull;
    if (a.seq == 0) a.seq = ++ctx().seq & 0xFFFFFFFFull;        // 0 is the mailbox's initial content
    a.host_mail = self_mail ? c.h_mail : nullptr;
    void* args[] = {&a};
    {
        Timed tm(c, stats().ms_strip, 1, stream);
        LINAC_CUDA(cudaLaunchCooperativeKernel((void*)strip_factor_kernel, dim3((unsigned)grid), dim3(SNT), args, sizeof(StripSmem),
                                               stream));
    }
    stats().kernel_launches++;
    out->seq = a.seq; out->b0 = b0; out->b1 = b1; out->j0 = j0; out->j1 = j1; out->stream = stream;
    return LINAC_OK;
}

// Waits for the mail of a launched strip (it may arrive before the kernel has ended) and records its pivots.
int collect_strip(Fp& c, StripLaunch& L, int64_t i0, int64_t* r) {
    linac_stats& st = stats();
    {
        volatile unsigned long long* mailbox = c.h_mail;
        const int nw = (int)(L.b1 - L.b0) * MAIL_WORDS;
        int seen = 0;                                     // words [0, seen) already carry this launch's tag
        for (uint64_t spins = 0; seen < nw; ++spins) {
            while (seen < nw && (mailbox[seen] >> 32) == L.seq) ++seen;
            if (seen < nw && (spins & 0x3FFF) == 0x3FFF) {
                const cudaError_t q = cudaStreamQuery(L.stream);
                if (q != cudaSuccess && q != cudaErrorNotReady) { set_cuda_error(q, "strip kernel", __FILE__, __LINE__); return LINAC_ERR_CUDA; }
                if (q == cudaSuccess) {                   // stream drained: the mail must be complete by now
                    while (seen < nw && (mailbox[seen] >> 32) == L.seq) ++seen;
                    if (seen < nw) return LINAC_ERR_INTERNAL;
                }
            }
        }
        std::atomic_thread_fence(std::memory_order_acquire);
    }
    st.host_syncs++;
    int64_t cur = i0;
    L.nswaps = 0;
    L.regular = L.b1 - L.b0 == WK / PW;
    for (int64_t b = L.b0; b < L.b1; ++b) {
        const unsigned long long* m = c.h_mail + (b - L.b0) * MAIL_WORDS;
        const int32_t hr = (int32_t)(uint32_t)m[0], hns = (int32_t)(uint32_t)m[1];
        if (hr < 0 || hr > PW || cur + hr > c.rows) return LINAC_ERR_INTERNAL;
        st.panels++;
        st.row_swaps += hr > 0 ? hns : 0;
        L.nswaps += hr > 0 ? hns : 0;
        L.regular = L.regular && hr == PW;
        for (int q = 0; q < hr; ++q) c.pivcols[cur + q] = (int32_t)(panel_col0(b) + (int32_t)(uint32_t)m[2 + q]);
        cur += hr;
        c.pstart[b + 1] = cur;
    }
    *r = cur - i0;
    return LINAC_OK;
}

// Enqueues strip_winv_kernel behind a strip kernel: W = the strip's solve operator, if the strip turns out regular.
int launch_winv(Fp& c, StripLaunch& L, cudaStream_t stream, int64_t i0) {
    if (options().trsm_winv == 0 || c.d_W == nullptr || L.b1 - L.b0 != WK / PW || L.j1 - L.j0 != WK || i0 + WK > c.rows) return LINAC_OK;
    Timed tm(c, stats().ms_trsm, 2, stream);
    L.W = c.d_W + (size_t)((c.winv_count++) & 1) * W_A_BYTES;
    strip_winv_kernel<<<WINV_CTAS, WINV_NT, sizeof(WinvSmem), stream>>>(c.A, c.ld, c.d_pstart, (int)L.b0, c.d_T, (int)i0, c.f, L.W);
    LINAC_CUDA(cudaGetLastError());
    stats().kernel_launches++;
    L.winv = true;
    return LINAC_OK;
}

// The strip's row-block solve on columns [c0, c0 + ncols) of its pivot rows (S4), optionally writing the u8 limb planes
// of the result (Bq) and posting the strip's records to the host (mail != nullptr).
// bq_col0 / bq_total: position of column c0 inside the planes and the planes' total column count (0 = this launch only).
int launch_strip_solve(Fp& c, const StripLaunch& L, int64_t i0, int64_t c0, int64_t ncols, uint8_t* Bq, int kp, bool mail,
                       int64_t bq_col0 = 0, int64_t bq_total = 0, cudaStream_t stream = nullptr) {
    if (ncols <= 0) return LINAC_OK;
    if (!stream) stream = c.s;
    Timed tm(c, stats().ms_trsm, 2, stream);
    if (L.winv && L.regular && !mail && (Bq == nullptr || kp == WK)) {          // one dense product with the strip's W
        const int64_t ntiles = (ncols + WTN - 1) / WTN;
        trsm_winv_kernel<<<(unsigned)std::min<int64_t>(ntiles, 2 * sm_count()), WNT, WTRSM_SMEM, stream>>>(
            L.W, c.A + i0 * c.ld + c0, c.ld, ncols, c.f, Bq, kp, bq_col0, bq_total > 0 ? bq_total : ncols);
        LINAC_CUDA(cudaGetLastError());
        stats().kernel_launches++;
        stats().winv_solves++;
        return LINAC_OK;
    }
    trsm_strip_kernel<true><<<(unsigned)((ncols + PW - 1) / PW), TNT, trsm_smem_bytes(L.j1 - L.j0), stream>>>(
        c.A, c.ld, c.A + i0 * c.ld + c0, c.ld, ncols, c.d_pstart, (int)L.b0, (int)L.b1, c.d_T, c.d_pivcols, c.f, Bq, kp,
        mail ? c.h_mail : nullptr, L.seq, c.d_rec, bq_col0, bq_total > 0 ? bq_total : ncols);
    LINAC_CUDA(cudaGetLastError());
    stats().kernel_launches++;
    return LINAC_OK;
}

// One strip s with active rows >= i0 (one cooperative launch).  Returns the number of pivots through *r.
// If early_ncols > 0 the strip's row-block solve on columns [early_c0, early_c0 + early_ncols) is enqueued right
// behind the strip kernel (it takes the pivot counts from device memory and posts the records to the host): the
// round trip then hides under the solve instead of idling the GPU.
int factor_strip(Fp& c, int64_t s, int64_t i0, int64_t* r, int64_t early_c0 = 0, int64_t early_ncols = 0,
                 uint8_t* early_Bq = nullptr, int early_kp = 0, uint8_t* tail_Aq = nullptr) {
    const bool early = early_ncols > 0 && options().timing != 1;
    StripLaunch L;
    int rc = launch_strip(c, s, i0, c.s, c.coop_grid, false, !early, tail_Aq, early_kp, &L);
    if (rc) return rc;
    if (early) {
        rc = launch_strip_solve(c, L, i0, early_c0, early_ncols, early_Bq, early_kp, true);
        if (rc) return rc;
    }
    rc = collect_strip(c, L, i0, r);
    if (rc) return rc;
    if (early) stats().update_macs += (*r) * (*r) / 2 * early_ncols;
    return early ? LINAC_EARLY_SOLVE_DONE : LINAC_OK;
}

// Flat sweep with LOOK-AHEAD over strips [s0, s1) (columns up to jend): once strip s is factored and its row-block solve
// has run, the Schur update is split in two: the next strip's columns first (a narrow product), then -- concurrently --
// the strip kernel of s+1 on `la_ctas` SMs (second stream) and the bulk of the update on the remaining SMs.  The strip
// kernel is a latency chain that leaves most issue slots of the GPU unused; the bulk update fills them.
//   stream c.s:   ... | solve_s | update_s[next strip] | strip kernel s+1 -------| swaps_{s+1} solve_{s+1} | ...
//   second stream:                                      | update_s[rest] ---------|
// Row exchanges of a look-ahead strip touch only its own columns while the bulk update owns the rest of those rows;
// deferred_swaps_kernel applies them to the other columns afterwards.  The L21 limb planes are double buffered (the
// bulk update of strip s still reads its planes while strip s+1 writes the next ones).
int factor_flat_lookahead(Fp& c, int64_t s0, int64_t s1, int64_t i0, int64_t jend, int64_t* r_out) {
    const Options& o = options();
    Context& cx = ctx();
    if (!cx.la_stream) {                                       // lowest priority: the bulk must never be placed before the chain
        int lo = 0, hi = 0;
        LINAC_CUDA(cudaDeviceGetStreamPriorityRange(&lo, &hi));
        LINAC_CUDA(cudaStreamCreateWithPriority(&cx.la_stream, cudaStreamNonBlocking, lo));
    }
    for (cudaEvent_t& e : cx.la_ev)
        if (!e) LINAC_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    cudaStream_t sB = cx.la_stream;
    cudaEvent_t ev_pre = cx.la_ev[0], ev_narrow = cx.la_ev[1], ev_strip = cx.la_ev[2];
    // How many SMs the look-ahead strip kernel gets, per strip.  Cost model in microseconds, fitted to sweeps of the
    // fixed-partition schedule on a B200 at config c3 (`profiles/r02_lookahead.md`): a 128-column strip kernel on G CTAs
    // takes 63.5 + 4300 (m / 1e4) / G (the chain of CTA 0 plus the in-strip updates and the L21 limb split, which spread
    // over G CTAs); the K = 128 bulk update takes 207 (m / 1e4)(n / 1e4) on the whole GPU and 1.05 + 0.62 G / (148 - G)
    // times that beside a strip kernel on G SMs (it is partly HBM-bound, so it slows less than in proportion).  The
    // partition that minimises the longer of the two is taken; option la_ctas > 0 forces a value.
    auto pick_grid = [&](int64_t m, int64_t n, double* t_la, double* t_seq) {
        const double mm = (double)m / 1e4, nn = (double)n / 1e4;
        auto t_strip = [&](int G) { return 63.5 + 4300.0 * mm / G; };
        auto t_bulk = [&](int G) { return 207.0 * mm * nn * (1.05 + 0.62 * G / (148.0 - G)); };
        int best = 32;
        double bt = 1e30;
        for (int G : {16, 24, 32, 40, 48, 56, 64, 72, 80, 96, 112}) {
            if (o.la_ctas > 0 && G != (int)o.la_ctas) continue;
            if (G >= c.coop_grid) continue;
            const double t = std::max(t_strip(G), t_bulk(G));
            if (t < bt) { bt = t; best = G; }
        }
        if (bt > 1e29) { best = (int)std::min<int64_t>(std::max<int64_t>(o.la_ctas, 4), c.coop_grid - 1); bt = std::max(t_strip(best), t_bulk(best)); }
        *t_la = bt + 14.0;                                      // + the narrow update that precedes the fork
        *t_seq = t_strip(c.coop_grid) + 207.0 * mm * nn;
        return best;
    };
    const int64_t j_first = panel_col0(c.sb0(s0));
    const int kp = (int)((c.bps * PW + 127) / 128 * 128);
    const size_t mark = c.arena->off;
    uint8_t* Bq = (uint8_t*)c.arena->take((size_t)4 * (jend - j_first) * kp, 1024);
    uint8_t* Aq[2] = {nullptr, nullptr};
    if (Bq) Aq[0] = (uint8_t*)c.arena->take((size_t)4 * (c.rows - i0) * kp, 1024);
    if (Aq[0]) Aq[1] = (uint8_t*)c.arena->take((size_t)4 * (c.rows - i0) * kp, 1024);
    if (!Aq[1]) { c.arena->off = mark; return -1; }           // not enough workspace: the caller runs the sequential sweep
    int64_t cur = i0;
    *r_out = 0;
    // strip s0 alone, on the whole GPU
    StripLaunch L;
    bool la_launched = false;                                  // was the strip in L launched as a look-ahead strip?
    int rc = launch_strip(c, s0, cur, c.s, c.coop_grid, false, true, Aq[s0 & 1], kp, &L);
    if (rc) return rc;
    rc = launch_winv(c, L, c.s, cur);
    if (rc) return rc;
    int64_t r = 0;
    rc = collect_strip(c, L, cur, &r);
    if (rc) return rc;
    for (int64_t s = s0; s < s1; ++s) {
        // here: strip s is launched and collected (r pivots from row cur), on c.s or on sB (la_launched)
        const int64_t jc = L.j1;
        if (la_launched) {
            LINAC_CUDA(cudaStreamWaitEvent(c.s, ev_strip, 0));
            const int64_t ncol_out = c.cols - (L.j1 - L.j0);
            if (ncol_out > 0 && L.nswaps > 0) {                // the host has the strip's records: no exchanges, no launch
                deferred_swaps_kernel<<<(unsigned)((ncol_out + 255) / 256), 256, 0, c.s>>>(c.A, c.ld, c.cols, L.j0, L.j1, c.d_rec,
                                                                                         c.d_pstart, (int)L.b0, (int)(L.b1 - L.b0));
                LINAC_CUDA(cudaGetLastError());
                stats().kernel_launches++;
            }
        }
        const bool last = s + 1 >= s1;
        const int64_t m2 = c.rows - (cur + r);
        const int64_t jn = last ? jc : std::min(jend, panel_col0(c.sb0(s + 2)));       // end of the next strip's columns
        bool next_launched = false;
        StripLaunch Ln;
        if (r > 0 && jend > jc) {
            const bool planes = r <= kp && (jend - jc) >= o.tc_min_mn && r >= o.tc_min_k && m2 >= o.tc_min_mn && o.gemm_path != 1 && o.tc_panel != 0;
            auto update = [&](int64_t c0, int64_t c1, int grid_limit, cudaStream_t stream, bool pdl = false) -> int {
                GemmArgs g{c.A + (cur + r) * c.ld + c0, c.ld, c.A + (cur + r) * c.ld, c.ld, c.d_pivcols + cur,
                           c.A + cur * c.ld + c0,       c.ld, m2,                      c1 - c0, r};
                if (planes) {
                    g.Bq_ready = Bq; g.kp_ready = kp; g.Aq_ready = Aq[s & 1];
                    g.bq_row0 = c0 - jc; g.bq_rows_total = jend - jc;
                    g.pdl = pdl;
                }
                g.grid_limit = grid_limit;
                return run_gemm(c, g, stream);
            };
            // look ahead only when there is bulk to hide the next strip kernel behind
            // (and only for row blocks no taller than three times their width: the cost model below was fitted on square
            // trailing blocks; on the tall flat nodes of the N = 1e5 recursion the fork measured 0.8 % slower than none)
            bool la = !last && m2 > 0 && planes && jn - jc >= o.tc_min_mn && jend - jn >= 2 * o.tc_min_mn && m2 >= 4 * o.tc_min_mn &&
                      cur + r < c.rows && m2 <= 3 * (jend - jn);
            int la_grid = 32;
            if (la) {
                double t_la = 0, t_seq = 0;
                la_grid = pick_grid(m2, jend - jn, &t_la, &t_seq);
                la = t_la < t_seq || o.la_ctas > 0;                                // not worth forking for this strip (a forced
                                                                                   // partition, option la_ctas, forks regardless)
            }
            stats().update_macs += r * r / 2 * (jend - jc);
            if (la) {
                // the whole row-block solve first (measured twice: solving only the next strip's columns before the fork and
                // the rest beside the strip kernel is SLOWER, 13.5 -> 15.3 / 16.0 ms at c3: squeezed onto the bulk's SMs the
                // solve needs two rounds of CTAs and pushes the bulk update, which then bounds the step), then the next
                // strip's columns of the update, the fork, and the bulk of the update beside the strip kernel
                const bool wsplit = L.winv && L.regular && o.trsm_split != 0;
                if (wsplit) {
                    // regular strip: the product with W is cheap and has no chain, so only the next strip's columns are
                    // solved in front of the narrow update; the rest goes to the second stream, in front of the bulk it
                    // feeds, and runs beside the narrow update instead of before it
                    LINAC_CUDA(cudaEventRecord(ev_pre, c.s));                      // exchanges of strip s applied, W written
                    rc = launch_strip_solve(c, L, cur, jc, jn - jc, Bq, kp, false, 0, jend - jc);
                    if (rc) return rc;
                    LINAC_CUDA(cudaStreamWaitEvent(sB, ev_pre, 0));
                    rc = launch_strip_solve(c, L, cur, jn, jend - jn, Bq, kp, false, jn - jc, jend - jc, sB);
                } else {
                    rc = launch_strip_solve(c, L, cur, jc, jend - jc, Bq, kp, false);
                }
                if (rc) return rc;
                // behind the W product the update is a programmatic dependent: its prologue, its A stages and its first C
                // tiles overlap the product, only its B loads wait for it
                rc = update(jc, jn, 0, c.s, wsplit && o.pdl != 0);
                if (rc) return rc;
                // the chain stays on the call's stream (the strip kernel starts the moment the narrow update ends and takes
                // its SMs first); the bulk goes to the second stream, where the cross-stream event latency does no harm
                LINAC_CUDA(cudaEventRecord(ev_narrow, c.s));
                rc = launch_strip(c, s + 1, cur + r, c.s, la_grid, true, true, Aq[(s + 1) & 1], kp, &Ln);
                if (rc) return rc;
                rc = launch_winv(c, Ln, c.s, cur + r);                              // needs the strip's own columns only
                if (rc) return rc;
                next_launched = true;
                stats().lookahead_strips++;
                LINAC_CUDA(cudaStreamWaitEvent(sB, ev_narrow, 0));
                rc = update(jn, jend, c.coop_grid - la_grid, sB, wsplit && o.pdl != 0);
                if (rc) return rc;
                LINAC_CUDA(cudaEventRecord(ev_strip, sB));                          // = "bulk of strip s done"
            } else {
                rc = launch_strip_solve(c, L, cur, jc, jend - jc, planes ? Bq : nullptr, kp, false);
                if (rc) return rc;
                if (m2 > 0) {
                    rc = update(jc, jend, 0, c.s);
                    if (rc) return rc;
                }
            }
        }
        cur += r;
        *r_out = cur - i0;
        if (last) break;
        if (cur >= c.rows) {                                   // no rows left: every remaining column of the node is free
            int64_t r_rest = 0;
            rc = factor(c, s + 1, s1, cur, &r_rest, false);
            if (rc) return rc;
            break;
        }
        if (!next_launched) {
            rc = launch_strip(c, s + 1, cur, c.s, c.coop_grid, false, true, Aq[(s + 1) & 1], kp, &Ln);
            if (rc) return rc;
            rc = launch_winv(c, Ln, c.s, cur);
            if (rc) return rc;
        }
        rc = collect_strip(c, Ln, cur, &r);
        if (rc) return rc;
        L = Ln;
        la_launched = next_launched;
    }
    c.arena->off = mark;
    return LINAC_OK;
}

// Recursive factorisation of strips [s0, s1) with active rows [i0, rows).  Fills pstart for their panels.
int factor(Fp& c, int64_t s0, int64_t s1, int64_t i0, int64_t* r_out, bool allow_flat) {
    *r_out = 0;
    if (s1 <= s0) return LINAC_OK;
    if (i0 >= c.rows) {                              // no rows left: every remaining column is free
        for (int64_t b = c.sb0(s0); b < c.sb0(s1); ++b) c.pstart[b + 1] = i0;
        std::vector<int32_t> fill((size_t)(c.sb0(s1) - c.sb0(s0)), (int32_t)i0);
        LINAC_CUDA(cudaMemcpyAsync(c.d_pstart + c.sb0(s0) + 1, fill.data(), fill.size() * 4, cudaMemcpyHostToDevice, c.s));
        LINAC_CUDA(cudaStreamSynchronize(c.s));      // `fill` is pageable and dies here
        return LINAC_OK;
    }
    if (s1 - s0 == 1) return factor_strip(c, s0, i0, r_out);
    if (allow_flat && (s1 - s0) * c.bps * PW <= options().flat_cols) {
        // Flat right-looking sweep over the node, a GROUP of flat_group strips at a time: the group is factored
        // by binary recursion confined to its own columns, then one row-block solve on the node's columns to
        // the right and ONE Schur update of everything below with K = the group's pivots (256 for two strips:
        // half as many read-modify-write passes over the trailing matrix as a per-strip update).
        const int64_t jend = std::min(c.cols, panel_col0(c.sb0(s1)));
        const int64_t grp = std::max<int64_t>(1, options().flat_group);
        if (options().lookahead != 0 && grp == 1 && options().timing != 1 && s1 - s0 >= 3 && c.bps * PW <= 256 &&
            options().gemm_path != 1 && options().tc_panel != 0 && jend - panel_col0(c.sb0(s0)) >= 1536 && c.rows - i0 >= 1536) {
            const int rc_la = factor_flat_lookahead(c, s0, s1, i0, jend, r_out);
            if (rc_la >= 0) return rc_la;                  // < 0: not enough workspace for its planes, sweep sequentially
        }
        int64_t cur = i0;
        for (int64_t s = s0; s < s1; s += grp) {
            const int64_t se = std::min(s1, s + grp);
            int64_t r = 0;
            const int64_t jc = std::min(c.cols, panel_col0(c.sb0(se)));
            int rc;
            bool solved = false;
            // the row-block solve can hand U12 to the Schur update as u8 limb planes (saves the update's own split)
            const size_t mark = c.arena->off;
            uint8_t* Bq = nullptr;
            uint8_t* Aq = nullptr;
            int kp_b = 0;
            if (se - s == 1 && cur < c.rows) {
                const int64_t ws = jc - panel_col0(c.sb0(s));
                const Options& o = options();
                if (o.gemm_path != 1 && o.tc_panel != 0 && ws <= 256 && jend - jc >= o.tc_min_mn && ws >= o.tc_min_k) {
                    kp_b = (int)((ws + 127) / 128 * 128);
                    Bq = (uint8_t*)c.arena->take((size_t)4 * (jend - jc) * kp_b, 1024);
                    if (Bq) Aq = (uint8_t*)c.arena->take((size_t)4 * (c.rows - cur) * kp_b, 1024);
                }
                rc = factor_strip(c, s, cur, &r, jc, jend - jc, Bq, kp_b, Aq);
                solved = rc == LINAC_EARLY_SOLVE_DONE;
                if (solved) rc = LINAC_OK;
            } else {
                rc = factor(c, s, se, cur, &r, false);                    // also marks columns free once rows run out
            }
            if (rc) return rc;
            if (r > 0 && jend > jc) {
                if (!solved) rc = trsm_lower(c, s, se, jc, jend);
                if (rc) return rc;
                const int64_t m2 = c.rows - (cur + r);
                if (m2 > 0) {
                    GemmArgs g{c.A + (cur + r) * c.ld + jc, c.ld, c.A + (cur + r) * c.ld, c.ld, c.d_pivcols + cur,
                               c.A + cur * c.ld + jc,       c.ld, m2,                      jend - jc, r};
                    if (solved && Bq) { g.Bq_ready = Bq; g.kp_ready = kp_b; g.Aq_ready = Aq; }
                    rc = run_gemm(c, g);
                    if (rc) return rc;
                }
            }
            c.arena->off = mark;
            cur += r;
            *r_out = cur - i0;
        }
        return LINAC_OK;
    }
    const int64_t sm = s0 + (s1 - s0) / 2;
    const int64_t jm = panel_col0(c.sb0(sm)), j1 = std::min(c.cols, panel_col0(c.sb0(s1)));
    int64_t r1 = 0, r2 = 0;
    int rc = factor(c, s0, sm, i0, &r1, allow_flat);
    if (rc) return rc;
    if (r1 > 0) {
        rc = trsm_lower(c, s0, sm, jm, j1);
        if (rc) return rc;
        const int64_t m2 = c.rows - (i0 + r1);
        if (m2 > 0) {
            GemmArgs g{c.A + (i0 + r1) * c.ld + jm, c.ld, c.A + (i0 + r1) * c.ld, c.ld, c.d_pivcols + i0,
                       c.A + i0 * c.ld + jm,        c.ld, m2,                     j1 - jm, r1};
            rc = run_gemm(c, g);
            if (rc) return rc;
        }
    }
    rc = factor(c, sm, s1, i0 + r1, &r2, allow_flat);
    *r_out = r1 + r2;
    return rc;
}

// X <- T^{-1} X on the gathered free columns F (rank x nf, ldf) for the pivots of strips [s0, s1) (S6).
// T = U[pivot rows, pivot columns] is unit upper triangular.
int trsm_upper(Fp& c, uint32_t* F, int64_t ldf, int64_t nf, int64_t s0, int64_t s1) {
    const int64_t t0 = c.sp(s0), t1 = c.sp(s1);
    if (t1 <= t0 || nf <= 0) return LINAC_OK;
    if (s1 - s0 == 1) return trsm_leaf<false>(c, s0, F + t0 * ldf, ldf, nf);
    const int64_t sh = s0 + (s1 - s0) / 2, th = c.sp(sh);
    int rc = trsm_upper(c, F, ldf, nf, sh, s1);
    if (rc) return rc;
    if (th > t0 && t1 > th) {
        // X_top -= U[top rows, bottom pivot columns] . X_bottom
        GemmArgs g{F + t0 * ldf, ldf, c.A + t0 * c.ld, c.ld, c.d_pivcols + th, F + th * ldf, ldf, th - t0, nf, t1 - th};
        rc = run_gemm(c, g);
        if (rc) return rc;
    }
    return trsm_upper(c, F, ldf, nf, s0, sh);
}

// Grid of the cooperative strip kernel: every CTA must be resident (one per SM with 1024 threads).
int strip_grid(int* grid) {
    static PerDeviceOnce once;
    const int rc = once.run([]() -> int {
        LINAC_CUDA(cudaFuncSetAttribute(strip_factor_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(StripSmem)));
        int per_sm = 0;
        LINAC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, strip_factor_kernel, SNT, sizeof(StripSmem)));
        LINAC_CUDA(cudaFuncSetAttribute(trsm_strip_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)trsm_smem_bytes(SW_MAX)));
        LINAC_CUDA(cudaFuncSetAttribute(trsm_strip_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)trsm_smem_bytes(SW_MAX)));
        LINAC_CUDA(cudaFuncSetAttribute(strip_winv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(WinvSmem)));
        LINAC_CUDA(cudaFuncSetAttribute(trsm_winv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)WTRSM_SMEM));
        if (per_sm < 1 || sm_count() < 1) return LINAC_ERR_INTERNAL;
        return LINAC_OK;
    });
    if (rc) return rc;
    *grid = sm_count();                               // one CTA per SM: more would only lengthen the grid barrier
    return LINAC_OK;
}

int64_t num_panels(int64_t cols) { return (cols + PW - 1) / PW; }

size_t meta_bytes(int64_t rows, int64_t cols) {
    const int64_t mn = std::max<int64_t>(1, std::min(rows, cols));
    const int64_t nb = num_panels(cols);
    // + the index arrays of the consumers that run behind the reduction (null space: 2 cols; solve: cols + nrhs; C.R: rank)
    return 8192 + (size_t)2 * W_A_BYTES + 1024 + (size_t)nb * (sizeof(PanelRec) + 256 + 2 * PW * PW * 4 + 4) + (size_t)mn * 4 + (size_t)cols * 4 + 10 * 256 +
           (size_t)cols * 12 + (size_t)mn * 4 + 4096;
}

// Free-column slab width for the back-elimination workspace.
int64_t backelim_slab(int64_t rows, int64_t cols) {
    (void)rows;
    return std::min<int64_t>(cols, 4096);
}

size_t workspace_bytes(int64_t rows, int64_t cols) {
    const int64_t mn = std::max<int64_t>(1, std::min(rows, cols));
    size_t b = meta_bytes(rows, cols);
    b += (size_t)mn * (size_t)backelim_slab(rows, cols) * 4 + 2 * (size_t)backelim_slab(rows, cols) * 4 + 1024;   // gathered free columns
    b += gemm_modp_tc_scratch_bytes(rows, cols, std::min<int64_t>(mn, 8192)) + 256;
    return b;
}

int validate(const uint32_t* dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p) {
    if (rows < 0 || cols < 0 || cols >= (1ll << 31) || rows >= (1ll << 31)) return LINAC_ERR_INVALID_ARG;
    if (rows > 0 && cols > 0 && (dA == nullptr || ld < cols)) return LINAC_ERR_INVALID_ARG;
    if (p < 2 || !is_prime_u64(p)) return LINAC_ERR_BAD_MODULUS;
    return LINAC_OK;
}

// The whole reduction.
int rref_impl(uint32_t* dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p, cudaStream_t s, int64_t* rank,
              int32_t* pivot_cols_out, Arena* arena) {
    linac_stats& st = stats();
    st = linac_stats{};
    int rc = validate(dA, rows, cols, ld, p);
    if (rc) return rc;
    if (!rank) return LINAC_ERR_INVALID_ARG;
    *rank = 0;
    if (rows == 0 || cols == 0) return LINAC_OK;
    // 2^31 <= p < 2^32: the CUDA-core Montgomery path of fp_wide.cu; the limb-plane tensor path and the
    // 64-bit accumulators of the strip kernels are built for p < 2^31
    rc = check_device();
    if (rc) return rc;
    rc = acquire_workspace(std::max(workspace_bytes(rows, cols), wide_workspace_u32(rows, cols)), arena);
    if (rc) return rc;
    if (p >= (1u << 31)) return rref_u32_wide(dA, rows, cols, ld, p, s, rank, pivot_cols_out, arena);

    Context& cx = ctx();
    cx.bind_device(current_device());
    if (!cx.mail) {
        LINAC_CUDA(cudaHostAlloc(&cx.mail, MAXBP * MAIL_WORDS * sizeof(unsigned long long), cudaHostAllocMapped | cudaHostAllocPortable));
        memset(cx.mail, 0, MAXBP * MAIL_WORDS * sizeof(unsigned long long));
    }
    const int slot = acquire_field_slot();
    if (slot < 0) return LINAC_ERR_INTERNAL;          // more than FIELD_SLOTS host threads inside the library at once

    Fp c;
    c.A = dA; c.rows = rows; c.cols = cols; c.ld = ld; c.f = make_modp(p); c.s = s; c.arena = arena;
    c.nb = num_panels(cols);
    c.bps = std::max<int64_t>(1, std::min<int64_t>(MAXBP, options().strip_width / PW));
    c.ns = (c.nb + c.bps - 1) / c.bps;
    rc = strip_grid(&c.coop_grid);
    if (rc) return rc;
    const int64_t mn = std::min(rows, cols);
    c.d_rec = (PanelRec*)arena->take((size_t)c.nb * sizeof(PanelRec));
    c.d_T = (uint32_t*)arena->take((size_t)c.nb * PW * PW * 4);
    c.d_E = (uint32_t*)arena->take((size_t)c.nb * PW * PW * 4);
    c.d_pivcols = (int32_t*)arena->take((size_t)mn * 4);
    int32_t* d_colinfo = (int32_t*)arena->take((size_t)cols * 4);
    c.d_pstart = (int32_t*)arena->take((size_t)(c.nb + 1) * 4);
    c.d_W = (uint8_t*)arena->take((size_t)2 * W_A_BYTES, 1024);
    if (!c.d_rec || !c.d_T || !c.d_E || !c.d_pivcols || !d_colinfo || !c.d_pstart || !c.d_W) return LINAC_ERR_WORKSPACE;
    LINAC_CUDA(cudaMemsetAsync(c.d_pstart, 0, (size_t)(c.nb + 1) * 4, s));
    c.h_mail = cx.mail;
    c.slot = slot;
    c.pivcols.assign(mn, -1);
    c.pstart.assign(c.nb + 1, 0);
    CallEvents evs;
    rc = evs.create();
    if (rc) return rc;
    c.ev0 = evs.ev0; c.ev1 = evs.ev1;
    std::vector<cudaEvent_t>& event_pool = cx.events;
    c.pool = &event_pool;
    cudaEvent_t t0 = evs.t0, t1 = evs.t1;
    LINAC_CUDA(cudaEventRecord(t0, s));

    LINAC_CUDA(cudaMemcpyToSymbolAsync(c_f, &c.f, sizeof(ModP), (size_t)slot * sizeof(ModP), cudaMemcpyHostToDevice, s));
    // S0 ingest
    {
        const bool vec = ((((uintptr_t)dA) | ((uintptr_t)ld * 4)) & 15) == 0 && cols >= 4;
        const int64_t cols4 = vec ? cols / 4 : 0;
        if (vec) {
            dim3 grid((unsigned)((cols4 + 255) / 256), (unsigned)std::min<int64_t>(rows, 4096));
            reduce_mod_p_vec4_kernel<<<grid, 256, 0, s>>>(dA, rows, cols4, ld, p);
            LINAC_CUDA(cudaGetLastError());
            st.kernel_launches++;
        }
        if (cols - 4 * cols4 > 0) {
            const int64_t rest = cols - 4 * cols4;
            dim3 grid((unsigned)((rest + 255) / 256), (unsigned)std::min<int64_t>(rows, 2048));
            reduce_mod_p_kernel<<<grid, 256, 0, s>>>(dA + 4 * cols4, rows, rest, ld, p);
            LINAC_CUDA(cudaGetLastError());
            st.kernel_launches++;
        }
    }
    // forward elimination
    int64_t r = 0;
    rc = factor(c, 0, c.ns, 0, &r, true);
    // column classification: pivot index, or the threshold row of a free column
    std::vector<int32_t> colinfo(cols);
    std::vector<int32_t> freec, freeth;
    if (rc == LINAC_OK) {
        for (int64_t b = 0; b < c.nb; ++b) {
            const int64_t j0 = panel_col0(b), j1 = std::min(cols, j0 + PW);
            for (int64_t cc = j0; cc < j1; ++cc) colinfo[cc] = -(int32_t)c.pstart[b + 1] - 1;
        }
        for (int64_t t = 0; t < r; ++t) colinfo[c.pivcols[t]] = (int32_t)t;
        for (int64_t cc = r > 0 ? c.pivcols[0] : cols; cc < cols; ++cc)   // free columns left of the first pivot are all zero
            if (colinfo[cc] < 0) { freec.push_back((int32_t)cc); freeth.push_back(-(colinfo[cc] + 1)); }
    }
    // S6 back-elimination of the free columns, a slab at a time
    if (rc == LINAC_OK && r > 0 && !freec.empty()) {
        const int64_t slab = backelim_slab(rows, cols);
        int32_t* d_free = (int32_t*)arena->take((size_t)std::max<int64_t>(1, slab) * 4);
        int32_t* d_th = (int32_t*)arena->take((size_t)std::max<int64_t>(1, slab) * 4);
        uint32_t* F = (uint32_t*)arena->take((size_t)r * (size_t)slab * 4);
        if (!d_free || !d_th || !F) rc = LINAC_ERR_WORKSPACE;
        for (size_t f0 = 0; rc == LINAC_OK && f0 < freec.size(); f0 += (size_t)slab) {
            const int64_t nf = (int64_t)std::min<size_t>((size_t)slab, freec.size() - f0);
            LINAC_CUDA(cudaMemcpyAsync(d_free, freec.data() + f0, (size_t)nf * 4, cudaMemcpyHostToDevice, s));
            LINAC_CUDA(cudaMemcpyAsync(d_th, freeth.data() + f0, (size_t)nf * 4, cudaMemcpyHostToDevice, s));
            dim3 grid((unsigned)((nf + 255) / 256), (unsigned)std::min<int64_t>(r, 1024));
            gather_cols_kernel<<<grid, 256, 0, s>>>(dA, ld, r, d_free, d_th, nf, F, nf);
            LINAC_CUDA(cudaGetLastError());
            rc = trsm_upper(c, F, nf, nf, 0, c.ns);
            if (rc) break;
            scatter_cols_kernel<<<grid, 256, 0, s>>>(dA, ld, r, d_free, nf, F, nf);
            LINAC_CUDA(cudaGetLastError());
            LINAC_CUDA(cudaStreamSynchronize(s));   // the host staging vectors are pageable memory
            st.kernel_launches += 2;
            st.host_syncs++;
        }
    }
    // S7 finalise
    if (rc == LINAC_OK) {
        LINAC_CUDA(cudaMemcpyAsync(d_colinfo, colinfo.data(), (size_t)cols * 4, cudaMemcpyHostToDevice, s));
        dim3 grid((unsigned)((cols + 255) / 256), (unsigned)std::min<int64_t>(rows, 1024));
        finalize_kernel<<<grid, 256, 0, s>>>(dA, ld, rows, cols, d_colinfo);
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
    if (e == cudaSuccess && options().timing == 2) {           // per-class device time of the production schedule
        std::vector<std::pair<float, float>> iv_strip, iv_update;      // intervals relative to the call's start
        for (const Fp::Mark& mk : c.marks) {
            float t = 0, b0 = 0, b1 = 0;
            if (cudaEventElapsedTime(&t, event_pool[mk.ev], event_pool[mk.ev + 1]) != cudaSuccess) continue;
            if (mk.cls != 2 && cudaEventElapsedTime(&b0, t0, event_pool[mk.ev]) == cudaSuccess &&
                cudaEventElapsedTime(&b1, t0, event_pool[mk.ev + 1]) == cudaSuccess)
                (mk.cls == 1 ? iv_strip : iv_update).push_back(std::make_pair(b0, b1));
            if (mk.cls == 0) {
                st.ms_update += t;
                if ((double)mk.m * mk.n * mk.k > (double)st.top_m * st.top_n * st.top_k) {
                    st.top_m = mk.m; st.top_n = mk.n; st.top_k = mk.k;
                    st.ms_update_top = t;
                }
            } else if (mk.cls == 1) st.ms_strip += t;
            else st.ms_trsm += t;
        }
        cx.marks.clear();
        for (const Fp::Mark& mk : c.marks) {
            linac_mark m{};
            m.cls = mk.cls; m.stream = mk.on == c.s ? 0 : 1; m.m = mk.m; m.n = mk.n; m.k = mk.k;
            if (cudaEventElapsedTime(&m.t0_ms, t0, event_pool[mk.ev]) != cudaSuccess ||
                cudaEventElapsedTime(&m.t1_ms, t0, event_pool[mk.ev + 1]) != cudaSuccess) continue;
            cx.marks.push_back(m);
        }
        double ov = 0;                                         // a strip kernel and an update kernel in flight together
        for (const auto& a : iv_strip)
            for (const auto& b : iv_update) ov += std::max(0.f, std::min(a.second, b.second) - std::max(a.first, b.first));
        st.ms_overlap = ov;
    }
    if (rc) return rc;
    *rank = r;
    if (pivot_cols_out) std::copy(c.pivcols.begin(), c.pivcols.begin() + r, pivot_cols_out);
    return LINAC_OK;
}

// `arena`: workspace to take the two index arrays from (the reduction's arena when called behind it).
int nullspace_from_rref_impl(const uint32_t* dR, int64_t rows, int64_t cols, int64_t ld, uint32_t p, int64_t rank,
                             const int32_t* pivot_cols, uint32_t* dK, int64_t ldk, cudaStream_t s, Arena* arena) {
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
    int32_t* dm = (int32_t*)arena->take((size_t)(cols + d) * 4);
    if (!dm) return LINAC_ERR_WORKSPACE;
    cudaError_t e = cudaMemcpyAsync(dm, colmap.data(), (size_t)cols * 4, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dm + cols, freec.data(), (size_t)d * 4, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) {
        dim3 grid((unsigned)((d + 255) / 256), (unsigned)std::min<int64_t>(cols, 4096));
        nullspace_kernel<<<grid, 256, 0, s>>>(dR, ld, cols, d, dm, dm + cols, dK, ldk, p);
        e = cudaGetLastError();
        stats().kernel_launches++;
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { set_cuda_error(e, "nullspace", __FILE__, __LINE__); return LINAC_ERR_CUDA; }
    return LINAC_OK;
}

}  // namespace
}  // namespace linac

using namespace linac;

extern "C" {

int linac_rref_u32_workspace(int64_t rows, int64_t cols, size_t* bytes) {
    if (!bytes || rows < 0 || cols < 0) return LINAC_ERR_INVALID_ARG;
    *bytes = (rows == 0 || cols == 0) ? 0 : std::max(workspace_bytes(rows, cols), wide_workspace_u32(rows, cols));
    return LINAC_OK;
}

int linac_rref_u32(uint32_t* dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p, void* stream, int64_t* rank,
                   int32_t* pivot_cols_out) {
    Arena arena;
    return rref_impl(dA, rows, cols, ld, p, (cudaStream_t)stream, rank, pivot_cols_out, &arena);
}

int linac_nullspace_u32(uint32_t* dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p, void* stream, int64_t* rank,
                        int32_t* pivot_cols_out, uint32_t* dK, int64_t ldk, int64_t k_capacity_cols, int64_t* nullity) {
    if (!nullity || k_capacity_cols < 0 || (k_capacity_cols > 0 && (!dK || ldk < k_capacity_cols)))
        return LINAC_ERR_INVALID_ARG;
    Arena arena;
    std::vector<int32_t> piv((size_t)std::max<int64_t>(1, std::min(rows, cols)));
    int64_t r = 0;
    int rc = rref_impl(dA, rows, cols, ld, p, (cudaStream_t)stream, &r, piv.data(), &arena);
    if (rc) return rc;
    if (rank) *rank = r;
    *nullity = cols - r;
    if (pivot_cols_out) std::copy(piv.begin(), piv.begin() + r, pivot_cols_out);
    if (cols - r > k_capacity_cols) return LINAC_ERR_BUFFER_TOO_SMALL;
    if (cols == 0) return LINAC_OK;
    const linac_stats keep = stats();
    rc = nullspace_from_rref_impl(dA, rows, cols, ld, p, r, piv.data(), dK, ldk, (cudaStream_t)stream, &arena);
    stats().kernel_launches = keep.kernel_launches + 1;
    return rc;
}

int linac_solve_u32(uint32_t* dM, int64_t rows, int64_t cols, int64_t nrhs, int64_t ld, uint32_t p, void* stream,
                    int64_t* rank_a, int32_t* pivot_cols_out, uint8_t* consistent, uint32_t* dX, int64_t ldx) {
    if (cols < 0 || nrhs < 0 || !rank_a || (nrhs > 0 && !consistent)) return LINAC_ERR_INVALID_ARG;
    if (cols > 0 && nrhs > 0 && (!dX || ldx < nrhs)) return LINAC_ERR_INVALID_ARG;
    const int64_t wide = cols + nrhs;
    Arena arena;
    std::vector<int32_t> piv((size_t)std::max<int64_t>(1, std::min(rows, wide)));
    int64_t r = 0;
    int rc = rref_impl(dM, rows, wide, ld, p, (cudaStream_t)stream, &r, piv.data(), &arena);
    if (rc) return rc;
    int64_t ra = 0;
    while (ra < r && piv[ra] < cols) ++ra;                     // pivot columns are ascending
    *rank_a = ra;
    if (pivot_cols_out) std::copy(piv.begin(), piv.begin() + r, pivot_cols_out);
    if (nrhs == 0) return LINAC_OK;
    if (rows == 0) {                                            // no equations: every right-hand side is empty, x = 0
        std::fill(consistent, consistent + nrhs, (uint8_t)1);
        if (cols > 0) LINAC_CUDA(cudaMemset2DAsync(dX, (size_t)ldx * 4, 0, (size_t)nrhs * 4, (size_t)cols, (cudaStream_t)stream));
        LINAC_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
        return LINAC_OK;
    }
    cudaStream_t s = (cudaStream_t)stream;
    std::vector<int32_t> colrow((size_t)std::max<int64_t>(1, cols), -1);
    for (int64_t k = 0; k < ra; ++k) colrow[piv[k]] = (int32_t)k;
    int32_t* d_colrow = (int32_t*)arena.take(colrow.size() * 4 + (size_t)nrhs + 16);
    if (!d_colrow) return LINAC_ERR_WORKSPACE;
    uint8_t* d_cons = reinterpret_cast<uint8_t*>(d_colrow + colrow.size());
    cudaError_t e = cudaMemcpyAsync(d_colrow, colrow.data(), colrow.size() * 4, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) {
        dim3 grid((unsigned)((nrhs + 127) / 128), (unsigned)std::max<int64_t>(1, std::min<int64_t>(cols, 2048)));
        solve_extract_kernel<<<grid, 128, 0, s>>>(dM, ld, cols, nrhs, ra, r, d_colrow, dX, ldx, d_cons);
        e = cudaGetLastError();
        stats().kernel_launches++;
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(consistent, d_cons, (size_t)nrhs, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { set_cuda_error(e, "linac_solve_u32", __FILE__, __LINE__); return LINAC_ERR_CUDA; }
    return LINAC_OK;
}

int linac_rank_factor_u32(const uint32_t* dA, int64_t rows, int64_t cols, int64_t lda, uint32_t p, void* stream,
                          uint32_t* dR, int64_t ldr, uint32_t* dC, int64_t ldc, int64_t* rank, int32_t* pivot_cols_out) {
    if (rows < 0 || cols < 0 || !rank) return LINAC_ERR_INVALID_ARG;
    const int64_t cap = std::min(rows, cols);
    if (rows > 0 && cols > 0 && (!dA || !dR || !dC || lda < cols || ldr < cols || ldc < cap)) return LINAC_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (rows > 0 && cols > 0) {
        int rc = check_device();
        if (rc) return rc;
        LINAC_CUDA(cudaMemcpy2DAsync(dR, (size_t)ldr * 4, dA, (size_t)lda * 4, (size_t)cols * 4, (size_t)rows,
                                     cudaMemcpyDeviceToDevice, s));
    }
    Arena arena;
    std::vector<int32_t> piv((size_t)std::max<int64_t>(1, cap));
    int64_t r = 0;
    int rc = rref_impl(dR, rows, cols, ldr, p, s, &r, piv.data(), &arena);
    if (rc) return rc;
    *rank = r;
    if (pivot_cols_out) std::copy(piv.begin(), piv.begin() + r, pivot_cols_out);
    if (r == 0) return LINAC_OK;
    int32_t* d_piv = (int32_t*)arena.take((size_t)r * 4);
    if (!d_piv) return LINAC_ERR_WORKSPACE;
    cudaError_t e = cudaMemcpyAsync(d_piv, piv.data(), (size_t)r * 4, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) {
        dim3 grid((unsigned)((r + 255) / 256), (unsigned)std::min<int64_t>(rows, 148 * 8));
        gather_columns_kernel<<<grid, 256, 0, s>>>(dA, lda, rows, r, d_piv, dC, ldc, p);
        e = cudaGetLastError();
        stats().kernel_launches++;
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { set_cuda_error(e, "linac_rank_factor_u32", __FILE__, __LINE__); return LINAC_ERR_CUDA; }
    return LINAC_OK;
}

int linac_load_matrix_u32(uint32_t* dA, int64_t n_rows, int64_t n_cols, int64_t ld, const uint32_t* dBases, int64_t n_basis,
                          int64_t ldb, const int32_t* dLindices, int64_t d, uint32_t p, void* stream) {
    if (n_rows < 0 || n_cols < 0 || n_basis < 0 || d < 0 || d > 4096) return LINAC_ERR_INVALID_ARG;
    if (p < 2 || p >= (1u << 31) || !is_prime_u32(p)) return LINAC_ERR_BAD_MODULUS;
    if (n_rows == 0 || n_cols == 0) return LINAC_OK;
    if (!dA || ld < n_cols || (d > 0 && !dLindices) || (n_basis > 0 && (!dBases || ldb < n_basis))) return LINAC_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t idx_bytes = (size_t)LM_COLS * (size_t)d * 4;
    if (idx_bytes > 160 * 1024) return LINAC_ERR_INVALID_ARG;           // d <= 160 with the tile in shared memory
    const int basis_cap = (int)std::min<int64_t>(std::max<int64_t>(n_basis, 1), (int64_t)((96 * 1024 - std::min<size_t>(idx_bytes, 64 * 1024)) / (4 * LM_ROWS)));
    const size_t smem = idx_bytes + (size_t)basis_cap * 4 * LM_ROWS;
    const ModP f = make_modp(p);
    // about eight CTAs per SM in total, each walking over many 8-row passes: the index tile is staged once per CTA
    const int64_t gx = (n_cols + LM_COLS - 1) / LM_COLS;
    const int64_t gy = std::max<int64_t>(1, std::min<int64_t>((n_rows + LM_ROWS - 1) / LM_ROWS, (148 * 8 + gx - 1) / gx));
    dim3 grid((unsigned)gx, (unsigned)gy);
    if (f.ninv) {
        LINAC_CUDA(cudaFuncSetAttribute(load_matrix_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(216 * 1024)));
        load_matrix_kernel<true><<<grid, LM_COLS, smem, s>>>(dA, n_rows, n_cols, ld, dBases, n_basis, ldb, dLindices, (int)d, basis_cap, f);
    } else {
        LINAC_CUDA(cudaFuncSetAttribute(load_matrix_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(216 * 1024)));
        load_matrix_kernel<false><<<grid, LM_COLS, smem, s>>>(dA, n_rows, n_cols, ld, dBases, n_basis, ldb, dLindices, (int)d, basis_cap, f);
    }
    LINAC_CUDA(cudaGetLastError());
    stats() = linac_stats{};
    stats().kernel_launches = 1;
    LINAC_CUDA(cudaStreamSynchronize(s));
    return LINAC_OK;
}

int linac_nullspace_from_rref_u32(const uint32_t* dR, int64_t rows, int64_t cols, int64_t ld, uint32_t p, int64_t rank,
                                  const int32_t* pivot_cols, uint32_t* dK, int64_t ldk, void* stream) {
    if (rows < 0 || cols < 0 || rank < 0 || rank > std::min(rows, cols) || (rank > 0 && !pivot_cols))
        return LINAC_ERR_INVALID_ARG;
    if (cols - rank > 0 && (!dK || ldk < cols - rank)) return LINAC_ERR_INVALID_ARG;
    if (rows > 0 && cols > 0 && (!dR || ld < cols)) return LINAC_ERR_INVALID_ARG;
    if (p < 2 || !is_prime_u64(p)) return LINAC_ERR_BAD_MODULUS;
    int rc = check_device();
    if (rc) return rc;
    Arena arena;
    rc = acquire_workspace((size_t)(2 * cols + 64) * 4, &arena);
    if (rc) return rc;
    return nullspace_from_rref_impl(dR, rows, cols, ld, p, rank, pivot_cols, dK, ldk, (cudaStream_t)stream, &arena);
}

int linac_gemm_sub_u32(uint32_t* dC, int64_t ldc, const uint32_t* dA, int64_t lda, const uint32_t* dB, int64_t ldb, int64_t M,
                       int64_t N, int64_t K, uint32_t p, int path, void* stream) {
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
    CallEvents evs;
    rc = evs.create();
    if (rc) return rc;
    cudaEvent_t e0 = evs.ev0, e1 = evs.ev1;
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
    return rc;
}

}  // extern "C"
