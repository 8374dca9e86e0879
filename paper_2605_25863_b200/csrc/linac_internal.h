// linac_internal.h -- shared host-side declarations of the library (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>
#include <vector>

#include "../../include/linac.h"
#include "modp.cuh"

namespace linac {

constexpr int PW = 32;   // base panel width (columns factored by one panel kernel)

// What the panel kernel reports for one base panel (kept on the device per panel; the host reads it
// with one small copy when it needs the pivot count).
struct PanelRec {
    int32_t r;               // pivots found in this panel (<= w)
    int32_t nswaps;          // how many of swp[] are real exchanges
    int32_t w;               // panel width
    int32_t pad;
    int32_t pc[PW];          // local pivot columns, ascending (-1 beyond r)
    int64_t swp[PW];         // LAPACK-style: at step a exchange rows (i0+a) and swp[a] (>= i0+a)
};

// Error plumbing: first failing CUDA call wins; text kept for linac_last_cuda_error().
void set_cuda_error(cudaError_t e, const char* what, const char* file, int line);
#define LINAC_CUDA(call)                                                     \
    do {                                                                     \
        cudaError_t e__ = (call);                                            \
        if (e__ != cudaSuccess) {                                            \
            ::linac::set_cuda_error(e__, #call, __FILE__, __LINE__);         \
            return LINAC_ERR_CUDA;                                           \
        }                                                                    \
    } while (0)

// Process-wide tunables (linac_set_option; set them while no call is in flight).
struct Options {
    int64_t gemm_path = 0;    // 0 = auto, 1 = CUDA-core (SIMT) only, 2 = tensor (tcgen05) where legal
    int64_t timing = 0;       // 1 = event + host sync around every launch of the UN-fused schedule (A/B of kernel classes);
                              // 2 = event pairs around every launch of the production schedule, no syncs, read at the end
    int64_t tc_min_k = 48;    // smallest K the tensor path is used for (K is zero padded to 128: a strip that found fewer than 128
                              // pivots -- free columns inside it -- must not fall to the CUDA-core kernel)
    int64_t tc_min_mn = 128;  // smallest M and N the tensor path is used for
    int64_t f64_mma = 1;      // fp64 trailing update: 1 = DMMA (FP64 tensor pipe), 0 = DFMA register tile
    int64_t f64_strip = 512;   // fp64 factorisation: flat sweep over strips of this many columns (0 = pure recursion)
    int64_t f64_panel_threads = 512, f64_panel_grid = 0;   // fp64 panel kernel: block size (256/512/1024), grid (0 = one CTA per SM)
    int64_t f64_panel_cluster = 0;    // fp64 panel: CTAs of the thread-block cluster that factors strips which fit its shared memory (0 = off)
    int64_t f64_cluster_rows = 128;   // ... up to this many rows per CTA (beyond it the per-column shared-memory traffic of one SM costs more than the grid barrier)
    int64_t f64_rref_strip = 128;     // linac_rref_f64: columns per strip (the K of the update right of the strip); 32 = every panel updates everything
    int64_t f64_panel_tags = 1;       // fp64 panel: 1 = tagged candidate records replace the per-column grid barrier, 0 = grid.sync
    int64_t f64_rhs_inv = 1;  // fp64 substitution on B: 1 = blocked with inverted diagonal blocks, 0 = recursive leaf solves
    int64_t tc_panel_deep = 1; // K <= 128 updates: one A stage and seven C-tile buffers (six tile loads in flight) instead of two and three
    int64_t tc_panel = 1;     // 1 = K <= 256 updates use the persistent A-stationary tensor kernel
    int64_t flat_cols = 16384; // nodes of at most this many columns are swept flat (right-looking), wider ones recurse
    int64_t flat_group = 1;   // strips per Schur update of the flat sweep (K = flat_group * strip_width)
    int64_t strip_width = 128; // columns factored by one cooperative strip kernel (multiple of 32, <= 256)
    int64_t lookahead = 1;    // flat sweep: 1 = factor strip s+1 on `la_ctas` SMs (second stream) while the bulk of strip s's
                              // Schur update runs on the other SMs; 0 = strictly sequential
    int64_t la_ctas = 0;      // CTAs (= SMs) of the look-ahead strip kernel; 0 = chosen per strip from a cost model
    int64_t trsm_winv = 1;    // look-ahead sweep: row-block solve of a regular strip (4 x 32 pivots) as ONE product with the strip's
                              // explicit 128 x 128 operator W (fp_trsm_inv.cuh); 0 = the panel-by-panel chain kernel everywhere
    int64_t pdl = 1;          // look-ahead sweep: the updates right behind a W solve start beside it (programmatic dependent launch)
    int64_t trsm_split = 1;   // ... and, when the update forks, only on the next strip's columns before the narrow update; the
                              // rest of the solve runs on the second stream in front of the bulk update (0 = whole solve first)
};
Options& options();

// Per-HOST-THREAD call state: the workspace handed over with linac_set_workspace, the library-owned fallback
// workspace, the statistics of the thread's last call, its mapped mailbox, its timing events and its slot in the
// constant-memory table of field descriptors.  Nothing a call mutates is shared between threads, so calls issued from
// different host threads on different streams are independent ("re-entrant across streams when each
// call has its own workspace").
struct Context {
    linac_stats stats{};
    void* user_ws = nullptr; size_t user_ws_bytes = 0;
    void* own_ws = nullptr;  size_t own_ws_bytes = 0; int own_ws_dev = -1;
    unsigned long long* mail = nullptr;       // mapped pinned host memory (strip records), allocated on first use
    unsigned long long seq = 0;               // tag of the last strip launch
    std::vector<cudaEvent_t> events;          // pool for the timing modes
    std::vector<linac_mark> marks;            // timing = 2: per-launch intervals of the thread's last F_p call
    int slot = -1;                            // index into the __constant__ ModP table of fp_strip.cuh
    cudaStream_t la_stream = nullptr;         // second stream of the look-ahead schedule (created on first use)
    cudaEvent_t la_ev[4] = {nullptr, nullptr, nullptr, nullptr};
    int res_dev = -1;                         // device the events / second stream above belong to
    void bind_device(int dev);                // drops them when the thread has moved to another device
    char cuda_error[1024] = {0};
    ~Context();
};
Context& ctx();
inline linac_stats& stats() { return ctx().stats; }
int acquire_field_slot();                      // a free slot of the constant table for this thread (kept until thread exit)
constexpr int FIELD_SLOTS = 64;

// One-time initialisation per (call site, device): function attributes are per device.
struct PerDeviceOnce {
    bool done[64] = {};
    template <class Fn> int run(Fn&& fn);
};
int current_device();
int sm_count();                                // multiprocessors of the current device (cached per device)

// Workspace arena: bump allocation inside either the caller's buffer or a library-owned one.
struct Arena {
    char* base = nullptr;
    size_t size = 0, off = 0;
    void* take(size_t bytes, size_t align = 256) {
        size_t o = (off + align - 1) / align * align;
        if (o + bytes > size) return nullptr;
        off = o + bytes;
        return base + o;
    }
};
int acquire_workspace(size_t bytes, Arena* arena);   // returns linac_status

extern std::mutex g_init_mutex;
template <class Fn> int PerDeviceOnce::run(Fn&& fn) {
    const int dev = current_device();
    if (dev < 0 || dev >= 64) return LINAC_ERR_UNSUPPORTED_DEVICE;
    std::lock_guard<std::mutex> lock(g_init_mutex);
    if (!done[dev]) {
        const int rc = fn();
        if (rc) return rc;
        done[dev] = true;
    }
    return LINAC_OK;
}

// Events of one call, destroyed on every exit path.
struct CallEvents {
    cudaEvent_t ev0 = nullptr, ev1 = nullptr, t0 = nullptr, t1 = nullptr;
    int create() {
        LINAC_CUDA(cudaEventCreate(&ev0));
        LINAC_CUDA(cudaEventCreate(&ev1));
        LINAC_CUDA(cudaEventCreate(&t0));
        LINAC_CUDA(cudaEventCreate(&t1));
        return LINAC_OK;
    }
    ~CallEvents() {
        for (cudaEvent_t e : {ev0, ev1, t0, t1}) if (e) cudaEventDestroy(e);
    }
};

ModP make_modp(uint32_t p);
bool is_prime_u32(uint32_t p);
bool is_prime_u64(uint64_t p);                         // deterministic Miller-Rabin for every p < 2^64

int check_device();                                    // LINAC_OK or UNSUPPORTED_DEVICE / CUDA

// ---- F_p GEMM  C -= Aop . B  (mod p) ------------------------------------------------------------
// C: M x N (ldc).  B: K x N (ldb).  Aop: M x K gathered from `Abase` (lda): element (m,k) is
// Abase[m*lda + kcols[k]] if kcols != nullptr (device array), else Abase[m*lda + k].
struct GemmArgs {
    uint32_t* C; int64_t ldc;
    const uint32_t* Abase; int64_t lda; const int32_t* kcols;
    const uint32_t* B; int64_t ldb;
    int64_t M, N, K;
    // Optional: the u8 limb planes of B already written by the producer of B (Bq[limb][n][kp_ready], k-major, zero
    // padded to kp_ready, a multiple of 128): the tensor path then skips its own split of B.  Only honoured by the
    // K <= 256 panel kernel; anything else ignores it and splits B itself.
    uint8_t* Bq_ready = nullptr;
    int64_t kp_ready = 0;
    uint8_t* Aq_ready = nullptr;      // same for A: Aq[limb][m][kp_ready], written by the strip kernel's tail
    // Bq_ready may describe MORE columns than this update touches (look-ahead splits one update into the next strip's
    // columns and the rest): the planes hold bq_rows_total columns (0 = N) and this update starts at column bq_row0
    int64_t bq_row0 = 0, bq_rows_total = 0;
    int grid_limit = 0;               // persistent kernels: use at most this many CTAs (0 = one per SM)
    bool pdl = false;                 // K <= 256 panel kernel with ready planes: programmatic dependent launch behind the kernel that
                                      // wrote the B planes (which must have written neither C nor the A planes)
};
int gemm_modp_simt(const GemmArgs& g, const ModP& f, cudaStream_t s);
// Tensor-core (tcgen05 int8 limb) path; returns LINAC_OK if it ran, or a negative value if the
// shape/alignment is not supported (caller falls back to the SIMT kernel).
int gemm_modp_tc(const GemmArgs& g, const ModP& f, cudaStream_t s, Arena* scratch);
size_t gemm_modp_tc_scratch_bytes(int64_t M, int64_t N, int64_t K);

size_t wide_workspace_u32(int64_t rows, int64_t cols);
// linac_rref_u32 for 2^31 <= p < 2^32 (fp_wide.cu); the caller holds the library mutex
int rref_u32_wide(uint32_t* dA, int64_t rows, int64_t cols, int64_t ld, uint32_t p, cudaStream_t s, int64_t* rank,
                  int32_t* pivot_cols_out, Arena* arena);

}  // namespace linac
