// peaks.cu -- linac_measure_peak: microbenchmarks of the pipes the library's rooflines are quoted against
// ("Measure, do not assume").  MEASURED_PEAKS.json holds the HBM copy bandwidth and a bf16 GEMM rate;
// the update kernels of this library run on the int8 tensor pipe (tcgen05.mma kind::i8), the FP64 tensor pipe
// (DMMA m8n8k4) and the integer multiply-add pipe (IMAD.WIDE.U32), none of which is in that file.  Each kernel here
// keeps its operands on chip and issues nothing but the instruction under test, so the figure is the pipe's issue
// rate at the clock the run actually held (returned beside it, from %clock64 against %globaltimer).
#include <cstring>
#include <mutex>

#include "linac_internal.h"
#include "tc_ptx.cuh"

namespace linac {
namespace {
using namespace tc;

struct ClockProbe {
    unsigned long long cycles, ns;
};

__device__ __forceinline__ unsigned long long gtime() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// tcgen05.mma.cta_group::1.kind::i8, M = 128, N = NN, K = 32 per instruction: one CTA per SM, operands resident in
// shared memory (128-byte swizzled K-major tiles, arbitrary content), accumulators in TMEM.
template <int NN>
__global__ void __launch_bounds__(64, 1) peak_tc_i8_kernel(int iters, ClockProbe* probe) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sA = smem;                          // 128 rows x 128 B
    uint8_t* sB = smem + 128 * 128;              // NN rows x 128 B
    uint64_t* bar = (uint64_t*)(sB + NN * 128);
    uint32_t* holder = (uint32_t*)(bar + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // pseudo-random operand bytes: the data toggling (and with it the power draw, hence the clock a long run settles
    // at under the board's power cap) is that of real limb planes, not of constant operands
    for (int e = threadIdx.x; e < (128 + NN) * 128 / 4; e += 64) {
        uint32_t h = (uint32_t)e * 0x9E3779B9u + blockIdx.x * 0x85EBCA6Bu;
        h ^= h >> 15; h *= 0x2C1B3C6Du; h ^= h >> 12; h *= 0x297A2D39u; h ^= h >> 15;
        ((uint32_t*)smem)[e] = h;
    }
    if (warp == 0 && lane == 0) { mbar_init(bar, 1); fence_barrier_init(); }
    if (warp == 1) tmem_alloc(holder, 512);
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *holder;
    unsigned long long c0 = 0, t0 = 0;
    if (warp == 1) {
        constexpr uint32_t idesc = make_idesc_i8(NN);
        const uint64_t da = make_desc_sw128(smem_u32(sA)), db = make_desc_sw128(smem_u32(sB));
        c0 = clock64();
        t0 = gtime();
        for (int it = 0; it < iters; ++it) {
            if (elect_one()) {
                const uint32_t d = tmem_base + (uint32_t)((it & 1) * 256);
#pragma unroll
                for (int kk = 0; kk < 4; ++kk) umma_i8(d, da + (uint64_t)(kk * 2), db + (uint64_t)(kk * 2), idesc, 1u);
            }
            __syncwarp();
        }
        if (elect_one()) umma_commit(bar);
        __syncwarp();
        mbar_wait(bar, 0);
        tc_fence_after();
        if (blockIdx.x == 0 && lane == 0) { probe->cycles = clock64() - c0; probe->ns = gtime() - t0; }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) { tc_fence_after(); tmem_dealloc(tmem_base, 512); }
}

// DMMA m8n8k4: 8 warps per CTA, 8 independent accumulator pairs per warp.
__global__ void __launch_bounds__(256) peak_dmma_kernel(int iters, double* sink, ClockProbe* probe) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) c[i][0] = c[i][1] = 0.0;
    const double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
    const unsigned long long c0 = clock64(), t0 = gtime();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) { probe->cycles = clock64() - c0; probe->ns = gtime() - t0; }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    if (s == 1.2345) sink[0] = s;
}

// 32 x 32 -> 64-bit multiply with 64-bit accumulate (the CUDA-core field multiply-accumulate): 8 chains per thread.  The
// multiplier of chain i is the low word of chain i+1, so every product is new: with a loop-invariant product (the first
// version of this kernel) ptxas hoists the multiply and the loop measures 64-bit additions, 17.3 T/s.  ptxas emits each
// multiply-add as IMAD.WIDE.U32 (addend RZ) + IADD3 + IADD3.X: the wide multiply occupies the FMA pipe for two passes.
__global__ void __launch_bounds__(1024) peak_imad_wide_kernel(int iters, unsigned long long* sink, ClockProbe* probe) {
    unsigned long long acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = 0x9E3779B97F4A7C15ull * (threadIdx.x + i + 1);
    const uint32_t y = 0x85EBCA6Bu + blockIdx.x;
    const unsigned long long c0 = clock64(), t0 = gtime();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(acc[i]) : "r"((uint32_t)acc[(i + 1) & 7]), "r"(y));
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) { probe->cycles = clock64() - c0; probe->ns = gtime() - t0; }
    unsigned long long s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += acc[i];
    if (s == 0x1234567ull) sink[0] = s;
}

// STREAM-style copy / read: 16 bytes per thread and iteration, grid-stride.
__global__ void __launch_bounds__(256) peak_hbm_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, size_t n16, int mode) {
    uint4 keep = make_uint4(0, 0, 0, 0);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x) {
        const uint4 v = src[i];
        if (mode == 0) dst[i] = v;
        else { keep.x ^= v.x; keep.y ^= v.y; keep.z ^= v.z; keep.w ^= v.w; }
    }
    if (mode != 0 && (keep.x ^ keep.y ^ keep.z ^ keep.w) == 0x13579BDFu) dst[0] = keep;
}

}  // namespace
}  // namespace linac

using namespace linac;

extern "C" int linac_measure_peak(const char* what, double ms_target, void* scratch, size_t scratch_bytes, void* stream,
                                  double* value, double* sm_mhz) {
    if (!what || !value) return LINAC_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    LINAC_CUDA(cudaGetDevice(&dev));
    LINAC_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (ms_target <= 0) ms_target = 2.0;
    Arena arena;
    rc = acquire_workspace(4096, &arena);
    if (rc) return rc;
    ClockProbe* d_probe = (ClockProbe*)arena.take(sizeof(ClockProbe) + 64);
    if (!d_probe) return LINAC_ERR_WORKSPACE;
    LINAC_CUDA(cudaMemsetAsync(d_probe, 0, sizeof(ClockProbe) + 64, s));
    void* d_sink = (char*)d_probe + sizeof(ClockProbe);
    CallEvents evs;
    rc = evs.create();
    if (rc) return rc;
    cudaEvent_t e0 = evs.ev0, e1 = evs.ev1;
    float ms = 0;
    double per_iter_work = 0;      // operations (or bytes) per loop iteration over the whole grid
    const bool is_hbm = !strcmp(what, "hbm_copy") || !strcmp(what, "hbm_read");
    auto run = [&](int iters) -> cudaError_t {
        cudaEventRecord(e0, s);
        if (!strcmp(what, "tc_i8_n256")) {
            constexpr int SM = (128 + 256) * 128 + 1024 + 64;
            cudaFuncSetAttribute(peak_tc_i8_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM);
            peak_tc_i8_kernel<256><<<sms, 64, SM, s>>>(iters, d_probe);
            per_iter_work = 2.0 * 128 * 256 * 32 * 4 * sms;
        } else if (!strcmp(what, "tc_i8_n128")) {
            constexpr int SM = (128 + 128) * 128 + 1024 + 64;
            cudaFuncSetAttribute(peak_tc_i8_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM);
            peak_tc_i8_kernel<128><<<sms, 64, SM, s>>>(iters, d_probe);
            per_iter_work = 2.0 * 128 * 128 * 32 * 4 * sms;
        } else if (!strcmp(what, "dmma")) {
            peak_dmma_kernel<<<sms * 4, 256, 0, s>>>(iters, (double*)d_sink, d_probe);
            per_iter_work = 2.0 * 8 * 8 * 4 * 8 /*chains*/ * 8 /*warps*/ * sms * 4;
        } else if (!strcmp(what, "imad_wide")) {
            peak_imad_wide_kernel<<<sms * 2, 1024, 0, s>>>(iters, (unsigned long long*)d_sink, d_probe);
            per_iter_work = 8.0 * 1024 * sms * 2;
        } else {
            return cudaErrorInvalidValue;
        }
        cudaEventRecord(e1, s);
        cudaError_t e = cudaStreamSynchronize(s);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
        return e;
    };
    cudaError_t e = cudaSuccess;
    double result = 0;
    if (is_hbm) {
        const int mode = !strcmp(what, "hbm_copy") ? 0 : 1;
        const size_t half = scratch_bytes / 2 / 16;
        if (!scratch || half < (1u << 20)) return LINAC_ERR_INVALID_ARG;
        const uint4* src = (const uint4*)scratch;
        uint4* dst = (uint4*)scratch + half;
        float best = 1e30f;
        for (int rep = 0; rep < 6 && e == cudaSuccess; ++rep) {
            cudaEventRecord(e0, s);
            peak_hbm_kernel<<<sms * 16, 256, 0, s>>>(src, dst, half, mode);
            cudaEventRecord(e1, s);
            e = cudaStreamSynchronize(s);
            if (e == cudaSuccess) { cudaEventElapsedTime(&ms, e0, e1); if (rep > 0 && ms < best) best = ms; }
        }
        result = (mode == 0 ? 2.0 : 1.0) * (double)half * 16.0 / (best * 1e-3) / 1e9;         // GB/s
        if (sm_mhz) *sm_mhz = 0.0;
    } else {
        e = run(2000);                                         // calibration (also the warm-up)
        if (e == cudaSuccess && ms > 0) {
            const int iters = (int)std::max(2000.0, std::min(2.0e8, 2000.0 * ms_target / ms));
            e = run(iters);
            if (e == cudaSuccess) result = per_iter_work * iters / (ms * 1e-3) / 1e12;        // T op/s
        }
        ClockProbe h{};
        if (e == cudaSuccess) e = cudaMemcpy(&h, d_probe, sizeof h, cudaMemcpyDeviceToHost);
        if (sm_mhz) *sm_mhz = h.ns ? (double)h.cycles / (double)h.ns * 1e3 : 0.0;
    }
    if (e == cudaErrorInvalidValue) return LINAC_ERR_INVALID_ARG;
    if (e != cudaSuccess) { set_cuda_error(e, "linac_measure_peak", __FILE__, __LINE__); return LINAC_ERR_CUDA; }
    *value = result;
    return LINAC_OK;
}
