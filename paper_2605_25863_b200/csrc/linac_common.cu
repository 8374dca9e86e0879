// linac_common.cu -- library state, error plumbing, workspace, host number theory.
#include <cstring>
#include <mutex>

#include "linac_internal.h"

namespace linac {

static Options g_options;
std::mutex g_init_mutex;                       // one-time initialisations, slot table, option writes
static bool g_slot_used[FIELD_SLOTS] = {};

Context& ctx() {
    thread_local Context c;
    return c;
}

Context::~Context() {
    // the thread is leaving: give back what it owns (errors are ignored: the CUDA context may already be gone)
    if (own_ws) cudaFree(own_ws);
    if (mail) cudaFreeHost(mail);
    for (cudaEvent_t e : events) if (e) cudaEventDestroy(e);
    for (cudaEvent_t e : la_ev) if (e) cudaEventDestroy(e);
    if (la_stream) cudaStreamDestroy(la_stream);
    if (slot >= 0) {
        std::lock_guard<std::mutex> lock(g_init_mutex);
        g_slot_used[slot] = false;
    }
    cudaGetLastError();
}

void Context::bind_device(int dev) {
    if (res_dev == dev) return;
    if (res_dev >= 0) {                       // events and streams belong to the device they were created on
        int cur = -1;
        cudaGetDevice(&cur);
        cudaSetDevice(res_dev);
        for (cudaEvent_t& e : events) { if (e) cudaEventDestroy(e); e = nullptr; }
        events.clear();
        for (cudaEvent_t& e : la_ev) { if (e) cudaEventDestroy(e); e = nullptr; }
        if (la_stream) { cudaStreamDestroy(la_stream); la_stream = nullptr; }
        if (cur >= 0) cudaSetDevice(cur);
    }
    res_dev = dev;
}

int acquire_field_slot() {
    Context& c = ctx();
    if (c.slot >= 0) return c.slot;
    std::lock_guard<std::mutex> lock(g_init_mutex);
    for (int i = 0; i < FIELD_SLOTS; ++i)
        if (!g_slot_used[i]) { g_slot_used[i] = true; c.slot = i; return i; }
    return -1;                                 // more than FIELD_SLOTS threads inside the library at once
}

int current_device() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    return dev;
}

int sm_count() {
    static int sms[64] = {};
    const int dev = current_device();
    if (dev < 0 || dev >= 64) return 0;
    if (!sms[dev]) {
        int v = 0;
        cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
        sms[dev] = v;                          // benign race: every thread writes the same value
    }
    return sms[dev];
}

void set_cuda_error(cudaError_t e, const char* what, const char* file, int line) {
    snprintf(ctx().cuda_error, sizeof ctx().cuda_error, "%s (%s) at %s:%d: %s", cudaGetErrorName(e), cudaGetErrorString(e),
             file, line, what);
    cudaGetLastError();   // clear the sticky-less error so the next call starts clean
}

Options& options() { return g_options; }

int acquire_workspace(size_t bytes, Arena* arena) {
    Context& c = ctx();
    if (c.user_ws && c.user_ws_bytes >= bytes) {
        arena->base = (char*)c.user_ws;
        arena->size = c.user_ws_bytes;
        arena->off = 0;
        return LINAC_OK;
    }
    const int dev = current_device();
    if (c.own_ws_bytes < bytes || c.own_ws_dev != dev) {
        if (c.own_ws) cudaFree(c.own_ws);
        c.own_ws = nullptr;
        c.own_ws_bytes = 0;
        cudaError_t e = cudaMalloc(&c.own_ws, bytes);
        if (e != cudaSuccess) {
            set_cuda_error(e, "cudaMalloc(workspace)", __FILE__, __LINE__);
            return LINAC_ERR_WORKSPACE;
        }
        c.own_ws_bytes = bytes;
        c.own_ws_dev = dev;
    }
    arena->base = (char*)c.own_ws;
    arena->size = c.own_ws_bytes;
    arena->off = 0;
    return LINAC_OK;
}

static uint64_t mulmod_u64(uint64_t a, uint64_t b, uint64_t m) { return (unsigned __int128)a * b % m; }
static uint64_t powmod_u64(uint64_t a, uint64_t e, uint64_t m) {
    uint64_t r = 1 % m;
    a %= m;
    while (e) {
        if (e & 1) r = mulmod_u64(r, a, m);
        a = mulmod_u64(a, a, m);
        e >>= 1;
    }
    return r;
}

// Deterministic Miller-Rabin: bases {2,3,5,7} decide every n < 3,215,031,751.
bool is_prime_u32(uint32_t n) {
    if (n < 2) return false;
    for (uint32_t q : {2u, 3u, 5u, 7u, 11u, 13u}) {
        if (n == q) return true;
        if (n % q == 0) return false;
    }
    uint32_t d = n - 1;
    int s = 0;
    while ((d & 1) == 0) { d >>= 1; ++s; }
    for (uint64_t a : {2ull, 3ull, 5ull, 7ull}) {
        uint64_t x = powmod_u64(a, d, n);
        if (x == 1 || x == n - 1) continue;
        bool comp = true;
        for (int i = 1; i < s; ++i) {
            x = mulmod_u64(x, x, n);
            if (x == n - 1) { comp = false; break; }
        }
        if (comp) return false;
    }
    return true;
}

// Deterministic Miller-Rabin for every n < 2^64 (the first twelve primes as bases decide n < 3.3e24).
bool is_prime_u64(uint64_t n) {
    if (n < 2) return false;
    const uint64_t bases[] = {2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37};
    for (uint64_t q : bases) {
        if (n == q) return true;
        if (n % q == 0) return false;
    }
    uint64_t d = n - 1;
    int s = 0;
    while ((d & 1) == 0) { d >>= 1; ++s; }
    for (uint64_t a : bases) {
        uint64_t x = powmod_u64(a, d, n);
        if (x == 1 || x == n - 1) continue;
        bool comp = true;
        for (int i = 1; i < s; ++i) {
            x = mulmod_u64(x, x, n);
            if (x == n - 1) { comp = false; break; }
        }
        if (comp) return false;
    }
    return true;
}

ModP make_modp(uint32_t p) {
    ModP f;
    f.p = p;
    f.c32 = (uint32_t)((1ull << 32) % p);
    f.m64 = (uint64_t)((((unsigned __int128)1) << 64) / p);
    for (int k = 0; k < 7; ++k) f.w[k] = (uint32_t)powmod_u64(2, 8 * k, p);
    for (int k = 0; k < 7; ++k) f.wm[k] = (uint32_t)powmod_u64(2, 8 * k + 32, p);
    f.ninv = 0;
    if (p & 1) {                                   // Newton iteration for p^-1 mod 2^32, then negate
        uint32_t inv = p;                          // correct to 3 bits
        for (int i = 0; i < 5; ++i) inv *= 2u - p * inv;
        f.ninv = 0u - inv;
    }
    return f;
}

int check_device() {
    int dev = 0;
    LINAC_CUDA(cudaGetDevice(&dev));
    int major = 0;
    LINAC_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return LINAC_ERR_UNSUPPORTED_DEVICE;
    return LINAC_OK;
}

}  // namespace linac

using namespace linac;

extern "C" {

const char* linac_status_string(int status) {
    switch (status) {
        case LINAC_OK: return "ok";
        case LINAC_ERR_INVALID_ARG: return "invalid argument";
        case LINAC_ERR_BAD_MODULUS: return "modulus must be a prime in the range the entry point documents";
        case LINAC_ERR_WORKSPACE: return "workspace allocation failed";
        case LINAC_ERR_CUDA: return "CUDA error";
        case LINAC_ERR_SINGULAR: return "matrix is singular to the given tolerance";
        case LINAC_ERR_BUFFER_TOO_SMALL: return "null-space buffer has too few columns";
        case LINAC_ERR_UNSUPPORTED_DEVICE: return "current CUDA device is not compute capability 10.x";
        case LINAC_ERR_INTERNAL: return "internal consistency check failed";
        case LINAC_ERR_TOO_LARGE: return "problem exceeds the static scratch array (LINAC_STATIC_SCRATCH_BYTES) of the no-allocation entry point";
        default: return "unknown status";
    }
}

const char* linac_last_cuda_error(void) { return ctx().cuda_error; }

int linac_version(void) { return 100; }   // 0.1.0

int linac_set_workspace(void* dev_ptr, size_t bytes) {
    if ((dev_ptr == nullptr) != (bytes == 0)) return LINAC_ERR_INVALID_ARG;
    ctx().user_ws = dev_ptr;
    ctx().user_ws_bytes = bytes;
    return LINAC_OK;
}

int linac_release(void) {
    Context& c = ctx();
    if (c.own_ws) cudaFree(c.own_ws);
    c.own_ws = nullptr;
    c.own_ws_bytes = 0;
    c.own_ws_dev = -1;
    return LINAC_OK;
}

int linac_get_last_stats(linac_stats* out) {
    if (!out) return LINAC_ERR_INVALID_ARG;
    *out = ctx().stats;
    return LINAC_OK;
}

int linac_get_last_marks(linac_mark* out, int64_t capacity, int64_t* count) {
    if (!count || capacity < 0 || (capacity > 0 && !out)) return LINAC_ERR_INVALID_ARG;
    const std::vector<linac_mark>& mk = ctx().marks;
    *count = (int64_t)mk.size();
    for (int64_t i = 0; i < capacity && i < (int64_t)mk.size(); ++i) out[i] = mk[(size_t)i];
    return LINAC_OK;
}

int linac_set_option(const char* name, int64_t value) {
    if (!name) return LINAC_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_init_mutex);
    if (!strcmp(name, "gemm_path")) {
        if (value < 0 || value > 2) return LINAC_ERR_INVALID_ARG;
        g_options.gemm_path = value;
    } else if (!strcmp(name, "timing")) {
        if (value < 0 || value > 2) return LINAC_ERR_INVALID_ARG;
        g_options.timing = value;
    } else if (!strcmp(name, "tc_min_k")) {
        if (value < 32) return LINAC_ERR_INVALID_ARG;
        g_options.tc_min_k = value;
    } else if (!strcmp(name, "tc_min_mn")) {
        if (value < 128) return LINAC_ERR_INVALID_ARG;
        g_options.tc_min_mn = value;
    } else if (!strcmp(name, "f64_mma")) {
        if (value < 0 || value > 2) return LINAC_ERR_INVALID_ARG;
        g_options.f64_mma = value;
    } else if (!strcmp(name, "f64_strip")) {
        if (value < 0 || (value > 0 && value % 32 != 0)) return LINAC_ERR_INVALID_ARG;
        g_options.f64_strip = value;
    } else if (!strcmp(name, "f64_panel_threads")) {
        if (value != 256 && value != 512 && value != 1024) return LINAC_ERR_INVALID_ARG;
        g_options.f64_panel_threads = value;
    } else if (!strcmp(name, "f64_panel_grid")) {
        if (value < 0 || value > 1024) return LINAC_ERR_INVALID_ARG;
        g_options.f64_panel_grid = value;
    } else if (!strcmp(name, "f64_panel_cluster")) {
        if (value < 0 || value > 16 || (value & (value - 1))) return LINAC_ERR_INVALID_ARG;
        g_options.f64_panel_cluster = value;
    } else if (!strcmp(name, "f64_cluster_rows")) {
        if (value < 1) return LINAC_ERR_INVALID_ARG;
        g_options.f64_cluster_rows = value;
    } else if (!strcmp(name, "f64_panel_tags")) {
        if (value < 0 || value > 1) return LINAC_ERR_INVALID_ARG;
        g_options.f64_panel_tags = value;
    } else if (!strcmp(name, "f64_rref_strip")) {
        if (value < 32 || value > 128 || value % 32) return LINAC_ERR_INVALID_ARG;
        g_options.f64_rref_strip = value;
    } else if (!strcmp(name, "f64_rhs_inv")) {
        if (value < 0 || value > 1) return LINAC_ERR_INVALID_ARG;
        g_options.f64_rhs_inv = value;
    } else if (!strcmp(name, "tc_panel_deep")) {
        if (value < 0 || value > 1) return LINAC_ERR_INVALID_ARG;
        g_options.tc_panel_deep = value;
    } else if (!strcmp(name, "tc_panel")) {
        if (value < 0 || value > 1) return LINAC_ERR_INVALID_ARG;
        g_options.tc_panel = value;
    } else if (!strcmp(name, "flat_group")) {
        if (value < 1 || value > 64) return LINAC_ERR_INVALID_ARG;
        g_options.flat_group = value;
    } else if (!strcmp(name, "flat_cols")) {
        if (value < 0) return LINAC_ERR_INVALID_ARG;
        g_options.flat_cols = value;
    } else if (!strcmp(name, "lookahead")) {
        if (value < 0 || value > 1) return LINAC_ERR_INVALID_ARG;
        g_options.lookahead = value;
    } else if (!strcmp(name, "la_ctas")) {
        if (value != 0 && (value < 4 || value > 128)) return LINAC_ERR_INVALID_ARG;
        g_options.la_ctas = value;
    } else if (!strcmp(name, "trsm_winv")) {
        if (value < 0 || value > 1) return LINAC_ERR_INVALID_ARG;
        g_options.trsm_winv = value;
    } else if (!strcmp(name, "pdl")) {
        if (value < 0 || value > 1) return LINAC_ERR_INVALID_ARG;
        g_options.pdl = value;
    } else if (!strcmp(name, "trsm_split")) {
        if (value < 0 || value > 1) return LINAC_ERR_INVALID_ARG;
        g_options.trsm_split = value;
    } else if (!strcmp(name, "strip_width")) {
        if (value < 32 || value > 256 || value % 32) return LINAC_ERR_INVALID_ARG;
        g_options.strip_width = value;
    } else {
        return LINAC_ERR_INVALID_ARG;
    }
    return LINAC_OK;
}

}  // extern "C"
