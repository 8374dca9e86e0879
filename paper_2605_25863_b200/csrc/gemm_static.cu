// gemm_static.cu -- linac_gemm_sub_u32_static: C <- C - A.B (mod p) on the tensor path for callers that may not
// allocate device memory (a CUDA graph being captured, a serving loop, a harness that forbids cudaMalloc).
//
// The tensor kernels (gemm_tc.cu) need scratch for the u8 limb planes of both operands, 4 (M + N) Kc + 4096 bytes.
// Every other entry point takes it from the caller's workspace or from a buffer the library allocates; this one takes
// it from the file-scope device array below, so the call allocates nothing: no cudaMalloc / cudaFree, no events, no
// stream synchronisation -- the kernels are enqueued on `stream` and the call returns.
//
//   * LINAC_STATIC_SCRATCH_BYTES (32 MiB) is the whole budget; a larger problem is rejected with LINAC_ERR_TOO_LARGE
//     before anything is launched.  Every GPU that loads the library holds the array until the process exits.
//   * In host code the array's name is only a host-side stand-in: the device address comes from
//     cudaGetSymbolAddress, once per device with that device current, and is what the kernels are given.
//   * Every call on a device shares the one array, and it keeps the previous call's contents.  Nothing has to start
//     at zero: the limb-split pre-passes write every byte the tensor maps cover, padding included (zero padded to Kc),
//     before the MMA kernel reads it, in stream order.  Two calls that overlap on the GPU (different streams or host
//     threads, same device) RACE on the array; the caller serialises them.
#include <mutex>

#include "linac_internal.h"

namespace linac {
namespace {

constexpr size_t STATIC_SCRATCH_BYTES = (size_t)32 << 20;
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_SCRATCH_BYTES];

void* g_scratch_ptr[64];           // device address of g_static_scratch per device ordinal
PerDeviceOnce g_scratch_once;

// The array's device address on the current device (set-up, once per device).
int static_scratch(void** out) {
    const int dev = current_device();
    if (dev < 0 || dev >= 64) return LINAC_ERR_UNSUPPORTED_DEVICE;
    const int rc = g_scratch_once.run([dev]() -> int {
        void* p = nullptr;
        LINAC_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || ((uintptr_t)p & 255) != 0) return LINAC_ERR_INTERNAL;
        g_scratch_ptr[dev] = p;
        return LINAC_OK;
    });
    if (rc) return rc;
    *out = g_scratch_ptr[dev];
    return LINAC_OK;
}

}  // namespace
}  // namespace linac

using namespace linac;

extern "C" {

int linac_gemm_sub_u32_static(uint32_t* dC, int64_t ldc, const uint32_t* dA, int64_t lda, const uint32_t* dB, int64_t ldb,
                              int64_t M, int64_t N, int64_t K, uint32_t p, void* stream) {
    if (M < 0 || N < 0 || K < 0) return LINAC_ERR_INVALID_ARG;
    if (p < 2 || p >= (1u << 31) || !is_prime_u32(p)) return LINAC_ERR_BAD_MODULUS;
    if (M == 0 || N == 0 || K == 0) return LINAC_OK;
    if (!dC || !dA || !dB || ldc < N || lda < K || ldb < N) return LINAC_ERR_INVALID_ARG;
    if (M >= (1ll << 31) || N >= (1ll << 31) || K >= (1ll << 31)) return LINAC_ERR_TOO_LARGE;
    if (gemm_modp_tc_scratch_bytes(M, N, K) > STATIC_SCRATCH_BYTES) return LINAC_ERR_TOO_LARGE;
    int rc = check_device();
    if (rc) return rc;
    void* scratch = nullptr;
    rc = static_scratch(&scratch);
    if (rc) return rc;
    const ModP f = make_modp(p);
    Arena arena;
    arena.base = (char*)scratch;
    arena.size = STATIC_SCRATCH_BYTES;
    GemmArgs g{dC, ldc, dA, lda, nullptr, dB, ldb, M, N, K};
    rc = gemm_modp_tc(g, f, (cudaStream_t)stream, &arena);
    // a shape the tensor kernels do not take (nothing launched yet): the CUDA-core kernel, which needs no scratch
    if (rc < 0) rc = gemm_modp_simt(g, f, (cudaStream_t)stream);
    return rc;
}

}  // extern "C"
