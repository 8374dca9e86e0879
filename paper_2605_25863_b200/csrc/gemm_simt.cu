// gemm_simt.cu -- S5 Schur update on the CUDA cores:  C <- C - Aop.B  (mod p).
//
// The arithmetic core of the paper's RowReduce kernel (row_k -= head_k * pivot_row,
// PAPER.md:245) applied for K pivots at once.  Products of two residues (< 2^62) are summed in a
// 64-bit accumulator (one IMAD.WIDE.U32 each) and the accumulator is folded back below 2^63
// every second product with x = hi*2^32 + lo == hi*(2^32 mod p) + lo; a full Barrett reduction
// happens once per output element per call.
//
// Tile: 128 x 64 outputs per CTA, 256 threads, 8 x 4 outputs per thread, K staged 16 at a time
// through shared memory (A tile stored k-major so a thread's 8 row operands are one LDS.128 x2).
#include "linac_internal.h"

namespace linac {
namespace {

constexpr int BM = 128, BN = 64, BK = 16, TM = 8, TN = 4;
constexpr int NTHREADS = (BM / TM) * (BN / TN);   // 256

__global__ void __launch_bounds__(NTHREADS, 2)
gemm_modp_simt_kernel(uint32_t* __restrict__ C, int64_t ldc, const uint32_t* __restrict__ Ab, int64_t lda,
                      const int32_t* __restrict__ kcols, const uint32_t* __restrict__ B, int64_t ldb, int64_t M,
                      int64_t N, int64_t K, ModP f) {
    __shared__ __align__(16) uint32_t As[BK][BM + 4];
    __shared__ __align__(16) uint32_t Bs[BK][BN];
    const int tid = threadIdx.x;
    const int tx = tid % (BN / TN), ty = tid / (BN / TN);
    const int64_t m0 = (int64_t)blockIdx.y * BM, n0 = (int64_t)blockIdx.x * BN;

    uint64_t acc[TM][TN];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j] = 0;

    for (int64_t k0 = 0; k0 < K; k0 += BK) {
        // stage A (gathered columns) and B
#pragma unroll
        for (int t = 0; t < BM * BK / NTHREADS; ++t) {
            const int idx = tid + t * NTHREADS;
            const int kk = idx % BK, mm = idx / BK;
            const int64_t m = m0 + mm, k = k0 + kk;
            uint32_t v = 0;
            if (m < M && k < K) v = Ab[m * lda + (kcols ? (int64_t)kcols[k] : k)];
            As[kk][mm] = v;
        }
#pragma unroll
        for (int t = 0; t < BK * BN / NTHREADS; ++t) {
            const int idx = tid + t * NTHREADS;
            const int nn = idx % BN, kk = idx / BN;
            const int64_t n = n0 + nn, k = k0 + kk;
            uint32_t v = 0;
            if (n < N && k < K) v = B[k * ldb + n];
            Bs[kk][nn] = v;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < BK; kk += 2) {
            uint32_t a0[TM], a1[TM], b0[TN], b1[TN];
            *reinterpret_cast<uint4*>(&a0[0]) = *reinterpret_cast<const uint4*>(&As[kk][ty * TM]);
            *reinterpret_cast<uint4*>(&a0[4]) = *reinterpret_cast<const uint4*>(&As[kk][ty * TM + 4]);
            *reinterpret_cast<uint4*>(&a1[0]) = *reinterpret_cast<const uint4*>(&As[kk + 1][ty * TM]);
            *reinterpret_cast<uint4*>(&a1[4]) = *reinterpret_cast<const uint4*>(&As[kk + 1][ty * TM + 4]);
            *reinterpret_cast<uint4*>(&b0[0]) = *reinterpret_cast<const uint4*>(&Bs[kk][tx * TN]);
            *reinterpret_cast<uint4*>(&b1[0]) = *reinterpret_cast<const uint4*>(&Bs[kk + 1][tx * TN]);
#pragma unroll
            for (int i = 0; i < TM; ++i)
#pragma unroll
                for (int j = 0; j < TN; ++j) {
                    uint64_t x = acc[i][j];
                    x += (uint64_t)a0[i] * b0[j];
                    x += (uint64_t)a1[i] * b1[j];
                    acc[i][j] = fold64(x, f);     // keeps x < 2^63 so two more products fit
                }
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < TM; ++i) {
        const int64_t m = m0 + ty * TM + i;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < TN; ++j) {
            const int64_t n = n0 + tx * TN + j;
            if (n >= N) continue;
            uint32_t* pc = C + m * ldc + n;
            *pc = submod(*pc, reduce64(acc[i][j], f), f);
        }
    }
}

}  // namespace

int gemm_modp_simt(const GemmArgs& g, const ModP& f, cudaStream_t s) {
    if (g.M <= 0 || g.N <= 0 || g.K <= 0) return LINAC_OK;
    // grid.y is limited to 65535: M <= 65535*128 = 8.3e6 rows is plenty for 180 GB of uint32
    dim3 grid((unsigned)((g.N + BN - 1) / BN), (unsigned)((g.M + BM - 1) / BM));
    gemm_modp_simt_kernel<<<grid, NTHREADS, 0, s>>>(g.C, g.ldc, g.Abase, g.lda, g.kcols, g.B, g.ldb, g.M, g.N, g.K, f);
    LINAC_CUDA(cudaGetLastError());
    stats().kernel_launches++;
    stats().update_macs += g.M * g.N * g.K;
    return LINAC_OK;
}

}  // namespace linac
