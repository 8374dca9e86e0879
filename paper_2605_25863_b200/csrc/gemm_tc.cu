// gemm_tc.cu -- S5 Schur update on the 5th-gen tensor cores:  C <- C - Aop.B  (mod p).
//
// A residue a < 2^31 is split into four 8-bit limbs a = sum_i a_i 2^(8i).  Then
//     a.b = sum_{w=0..6} 2^(8w) * S_w,   S_w = sum_{i+j=w} a_i b_j,
// and sum_k a_k b_k needs 16 u8 x u8 -> s32 products per field product: exactly what
// tcgen05.mma.kind::i8 computes (unsigned 8-bit operands, 32-bit accumulators in TMEM).
// Per output tile (128 rows x 64 columns) the seven S_w live in seven 64-column TMEM
// accumulators (448 of 512 columns).  The four limb planes of B are stacked along N (4 x 64 =
// 256 rows), so ONE 128x256x32 MMA per A-limb i adds A_i.B_j into accumulator i+j for all four j
// at once (the D operand is simply placed at column 64*i): 4 MMAs per 32-wide k step instead
// of 16, each with the N = 256 shape that keeps shared-memory operand traffic below the MMA rate.
// Overflow: S_3 collects 4 products per k, 4 * K * 255^2 < 2^31 for K <= 8256; K is chunked at
// KC <= 4096 per launch.
// Epilogue (4 warps, one TMEM lane quarter each): tcgen05.ld the seven partial sums, recombine
//     v = (S0 + S1 2^8 + S2 2^16 + S3 2^24) + ((S4 + S5 2^8 + S6 2^16) mod p) * (2^32 mod p)   < 2^63
// reduce once more (Barrett) and subtract from C.
//
// Operands reach shared memory by TMA (3-D box: 128 bytes of k x rows x 4 limb planes, 128-byte
// swizzle) from limb planes a pre-pass writes (K-major for both operands; the B planes are
// written transposed so no MN-major descriptor is needed).  Producer / MMA issuer / epilogue are
// separate warps synchronised by mbarriers; tcgen05.commit releases pipeline stages.
#include <cuda.h>

#include <algorithm>
#include <mutex>

#include "linac_internal.h"

namespace linac {
namespace {

constexpr int TM = 128;          // output tile rows  (UMMA M)
constexpr int TN = 64;           // output tile columns per limb plane
constexpr int KB = 128;          // k bytes per pipeline stage (one 128-byte swizzle row)
constexpr int STAGES = 2;
constexpr int A_STAGE = 4 * TM * KB;      // 65536
constexpr int B_STAGE = 4 * TN * KB;      // 32768
constexpr int SMEM_BYTES = STAGES * (A_STAGE + B_STAGE) + 1024 /*align*/ + 256 /*barriers*/;
constexpr int TMEM_COLS = 512;
constexpr int NTHREADS = 192;    // warp 0: TMA, warp 1: MMA + TMEM alloc, warps 2..5: epilogue
constexpr int64_t KC_MAX = 4096;

// ----------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred P1;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
        "@P1 bra DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "DONE:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void tma_load_3d(void* smem_dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(smem_dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* tm) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(tm) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t* holder_smem, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(holder_smem)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// D[tmem] (+)= A[smem desc] . B[smem desc]^T, unsigned 8-bit operands, s32 accumulate.
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
// mbarrier arrives when all previously issued tcgen05.mma of this thread have completed.
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// K-major operand tile, 128-byte swizzle: rows of 128 bytes, 8-row groups 1024 bytes apart.
__device__ __forceinline__ uint64_t make_desc_sw128(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3FFF);          // start address
    d |= (uint64_t)1 << 16;                          // leading byte offset (unused for swizzled K-major)
    d |= (uint64_t)(1024 >> 4) << 32;                // stride byte offset between 8-row groups
    d |= (uint64_t)1 << 46;                          // descriptor version (Blackwell)
    d |= (uint64_t)2 << 61;                          // SWIZZLE_128B
    return d;
}
// kind::i8 instruction descriptor: D = s32, A/B unsigned 8-bit, both K-major, M = 128.
__host__ __device__ constexpr uint32_t make_idesc_i8(int n) {
    return (2u << 4) | (0u << 7) | (0u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);
}

// ----------------------------------------------------------------------------- the GEMM kernel
__global__ void __launch_bounds__(NTHREADS, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, uint32_t* __restrict__ C,
               int64_t ldc, int64_t M, int64_t N, int kp /* padded K of this launch, multiple of KB */, ModP f) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sA = smem;                                  // [STAGES][4][TM][KB]
    uint8_t* sB = smem + STAGES * A_STAGE;               // [STAGES][4][TN][KB]
    uint64_t* bars = (uint64_t*)(smem + STAGES * (A_STAGE + B_STAGE));
    uint64_t* full = bars;                               // [STAGES]
    uint64_t* empty = bars + STAGES;                     // [STAGES]
    uint64_t* acc_full = bars + 2 * STAGES;
    uint32_t* tmem_holder = (uint32_t*)(bars + 2 * STAGES + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int m_tile = blockIdx.y, n_tile = blockIdx.x;
    const int nk = kp / KB;

    if (warp == 0 && lane == 0) {
        prefetch_tmap(&tmA);
        prefetch_tmap(&tmB);
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        mbar_init(acc_full, 1);
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_holder, TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_holder;

    if (warp == 0) {
        if (lane == 0) {
            for (int kb = 0; kb < nk; ++kb) {
                const int s = kb % STAGES;
                const uint32_t ph = (kb / STAGES) & 1;
                mbar_wait(&empty[s], ph ^ 1);
                mbar_expect_tx(&full[s], A_STAGE + B_STAGE);
                tma_load_3d(sA + s * A_STAGE, &tmA, &full[s], kb * KB, m_tile * TM, 0);
                tma_load_3d(sB + s * B_STAGE, &tmB, &full[s], kb * KB, n_tile * TN, 0);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            constexpr uint32_t idesc256 = make_idesc_i8(4 * TN);
            constexpr uint32_t idesc64 = make_idesc_i8(TN);
            for (int kb = 0; kb < nk; ++kb) {
                const int s = kb % STAGES;
                const uint32_t ph = (kb / STAGES) & 1;
                mbar_wait(&full[s], ph);
                tc_fence_after();
                const uint32_t a0 = smem_u32(sA + s * A_STAGE), b0 = smem_u32(sB + s * B_STAGE);
#pragma unroll
                for (int kk = 0; kk < KB / 32; ++kk) {
                    if (kb == 0 && kk == 0) {
                        // first k step: every accumulator is written once without accumulation
#pragma unroll
                        for (int i = 0; i < 4; ++i)
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                const uint64_t da = make_desc_sw128(a0 + i * (TM * KB));
                                const uint64_t db = make_desc_sw128(b0 + j * (TN * KB));
                                const bool first = (i == 0) || (j == 3);      // first product landing in slot i+j
                                umma_i8(tmem_base + (uint32_t)((i + j) * TN), da, db, idesc64, first ? 0u : 1u);
                            }
                    } else {
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const uint64_t da = make_desc_sw128(a0 + i * (TM * KB) + kk * 32);
                            const uint64_t db = make_desc_sw128(b0 + kk * 32);
                            umma_i8(tmem_base + (uint32_t)(i * TN), da, db, idesc256, 1u);
                        }
                    }
                }
                umma_commit(&empty[s]);            // frees this stage when the MMAs above have read it
            }
            umma_commit(acc_full);
        }
    } else {
        // epilogue warps 2..5 -> TMEM lane quarters 2,3,0,1
        const int q = warp & 3;
        mbar_wait(acc_full, 0);
        tc_fence_after();
        const int64_t m = (int64_t)m_tile * TM + q * 32 + lane;
        const int64_t n_base = (int64_t)n_tile * TN;
        uint32_t* crow = C + m * ldc + n_base;
        const bool vec_ok = ((((uintptr_t)C) | ((uintptr_t)ldc * 4)) & 15) == 0;
        const uint64_t c32 = f.c32;
#pragma unroll 1
        for (int c8 = 0; c8 < TN / 8; ++c8) {
            uint32_t S[7][8];
#pragma unroll
            for (int w = 0; w < 7; ++w) tmem_ld8(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(w * TN + c8 * 8), S[w]);
            tmem_ld_wait();
            if (m < M) {
                uint32_t cv[8];
                const int64_t n0 = n_base + c8 * 8;
                const bool full8 = n0 + 8 <= N;
                if (full8 && vec_ok) {
                    *reinterpret_cast<uint4*>(&cv[0]) = *reinterpret_cast<const uint4*>(crow + c8 * 8);
                    *reinterpret_cast<uint4*>(&cv[4]) = *reinterpret_cast<const uint4*>(crow + c8 * 8 + 4);
                } else {
#pragma unroll
                    for (int e = 0; e < 8; ++e) cv[e] = (n0 + e < N) ? crow[c8 * 8 + e] : 0u;
                }
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const uint64_t lo = (uint64_t)S[0][e] + ((uint64_t)S[1][e] << 8) + ((uint64_t)S[2][e] << 16) + ((uint64_t)S[3][e] << 24);
                    const uint64_t hi = (uint64_t)S[4][e] + ((uint64_t)S[5][e] << 8) + ((uint64_t)S[6][e] << 16);
                    const uint64_t v = lo + (uint64_t)reduce64(hi, f) * c32;
                    cv[e] = submod(cv[e], reduce64(v, f), f);
                }
                if (full8 && vec_ok) {
                    *reinterpret_cast<uint4*>(crow + c8 * 8) = *reinterpret_cast<const uint4*>(&cv[0]);
                    *reinterpret_cast<uint4*>(crow + c8 * 8 + 4) = *reinterpret_cast<const uint4*>(&cv[4]);
                } else {
#pragma unroll
                    for (int e = 0; e < 8; ++e)
                        if (n0 + e < N) crow[c8 * 8 + e] = cv[e];
                }
            }
        }
        tc_fence_before();
    }
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, TMEM_COLS);
    }
}

// ----------------------------------------------------------------------------- limb-split pre-passes
// Aq[limb][m][kp]: row m, k-major, zero padded to kp.  One thread packs 4 consecutive k.
__global__ void split_a_kernel(const uint32_t* __restrict__ Ab, int64_t lda, const int32_t* __restrict__ kcols, int64_t k0,
                               int64_t M, int64_t K /* valid k in this chunk */, int64_t kp, uint8_t* __restrict__ Aq) {
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;     // word index along k (4 k per word)
    if (w * 4 >= kp) return;
    const int64_t plane = M * kp;
    for (int64_t m = blockIdx.y; m < M; m += gridDim.y) {
        uint32_t v[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int64_t k = w * 4 + e;
            v[e] = k < K ? Ab[m * lda + (kcols ? (int64_t)kcols[k0 + k] : k0 + k)] : 0u;
        }
#pragma unroll
        for (int l = 0; l < 4; ++l) {
            const uint32_t packed = ((v[0] >> (8 * l)) & 0xFF) | (((v[1] >> (8 * l)) & 0xFF) << 8) |
                                    (((v[2] >> (8 * l)) & 0xFF) << 16) | (((v[3] >> (8 * l)) & 0xFF) << 24);
            *reinterpret_cast<uint32_t*>(Aq + l * plane + m * kp + w * 4) = packed;
        }
    }
}

// Bq[limb][n][kp] from B[k][n] (row-major): transposed through shared memory, 128 k x 32 n per block.
__global__ void __launch_bounds__(256) split_b_kernel(const uint32_t* __restrict__ B, int64_t ldb, int64_t K, int64_t N,
                                                      int64_t kp, uint8_t* __restrict__ Bq) {
    __shared__ uint32_t T[128][33];
    const int tid = threadIdx.x;
    const int64_t k_blk = (int64_t)blockIdx.x * 128, n_blk = (int64_t)blockIdx.y * 32;
    for (int i = 0; i < 16; ++i) {
        const int kk = tid / 32 + 8 * i, nn = tid % 32;
        const int64_t k = k_blk + kk, n = n_blk + nn;
        T[kk][nn] = (k < K && n < N) ? B[k * ldb + n] : 0u;
    }
    __syncthreads();
    const int64_t plane = N * kp;
    for (int i = 0; i < 16; ++i) {
        const int pair = tid / 32 + 8 * i;         // (limb, n) pair: 4 x 32
        const int l = pair / 32, nn = pair % 32;
        const int wd = tid % 32;                   // 4 k per word
        const int64_t n = n_blk + nn;
        if (n >= N) continue;
        uint32_t packed = 0;
#pragma unroll
        for (int e = 0; e < 4; ++e) packed |= ((T[4 * wd + e][nn] >> (8 * l)) & 0xFF) << (8 * e);
        *reinterpret_cast<uint32_t*>(Bq + l * plane + n * kp + k_blk + 4 * wd) = packed;
    }
}

// ----------------------------------------------------------------------------- host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    });
    return fn;
}

// 3-D map over limb planes: (k bytes, rows, 4 planes); box = (128, box_rows, 4); 128-byte swizzle.
bool make_limb_map(CUtensorMap* tm, uint8_t* base, int64_t rows, int64_t kp, int box_rows) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return false;
    cuuint64_t dims[3] = {(cuuint64_t)kp, (cuuint64_t)rows, 4};
    cuuint64_t strides[2] = {(cuuint64_t)kp, (cuuint64_t)rows * (cuuint64_t)kp};
    cuuint32_t box[3] = {(cuuint32_t)KB, (cuuint32_t)box_rows, 4};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

int64_t chunk_k(int64_t K) {
    // equal chunks of at most KC_MAX, each a multiple of KB
    const int64_t nchunks = (K + KC_MAX - 1) / KC_MAX;
    const int64_t per = (K + nchunks - 1) / nchunks;
    return (per + KB - 1) / KB * KB;
}

}  // namespace

size_t gemm_modp_tc_scratch_bytes(int64_t M, int64_t N, int64_t K) {
    const int64_t kc = chunk_k(std::max<int64_t>(K, 1));
    return (size_t)4 * (size_t)(M + N) * (size_t)kc + 4096;
}

int gemm_modp_tc(const GemmArgs& g, const ModP& f, cudaStream_t s, Arena* scratch) {
    if (g.M <= 0 || g.N <= 0 || g.K <= 0) return LINAC_OK;
    if (g.M >= (1ll << 31) || g.N >= (1ll << 31)) return -1;
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(gemm_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES) != cudaSuccess) {
            cudaGetLastError();
            return -1;
        }
        attr_set = true;
    }
    const int64_t kc = chunk_k(g.K);
    uint8_t* Aq = (uint8_t*)scratch->take((size_t)4 * g.M * kc, 1024);
    uint8_t* Bq = (uint8_t*)scratch->take((size_t)4 * g.N * kc, 1024);
    if (!Aq || !Bq) return -1;
    for (int64_t k0 = 0; k0 < g.K; k0 += kc) {
        const int64_t kv = std::min(kc, g.K - k0);
        const int64_t kp = (kv + KB - 1) / KB * KB;
        {
            dim3 grid((unsigned)((kp / 4 + 127) / 128), (unsigned)std::min<int64_t>(g.M, 16384));
            split_a_kernel<<<grid, 128, 0, s>>>(g.Abase, g.lda, g.kcols, k0, g.M, kv, kp, Aq);
            LINAC_CUDA(cudaGetLastError());
        }
        {
            dim3 grid((unsigned)(kp / 128), (unsigned)((g.N + 31) / 32));
            split_b_kernel<<<grid, 256, 0, s>>>(g.B + k0 * g.ldb, g.ldb, kv, g.N, kp, Bq);
            LINAC_CUDA(cudaGetLastError());
        }
        CUtensorMap tmA, tmB;
        if (!make_limb_map(&tmA, Aq, g.M, kp, TM) || !make_limb_map(&tmB, Bq, g.N, kp, TN)) return -1;
        dim3 grid((unsigned)((g.N + TN - 1) / TN), (unsigned)((g.M + TM - 1) / TM));
        gemm_tc_kernel<<<grid, NTHREADS, SMEM_BYTES, s>>>(tmA, tmB, g.C, g.ldc, g.M, g.N, (int)kp, f);
        LINAC_CUDA(cudaGetLastError());
        stats().kernel_launches += 3;
        stats().tc_launches++;
    }
    stats().update_macs += g.M * g.N * g.K;
    return LINAC_OK;
}

}  // namespace linac
