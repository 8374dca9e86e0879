// fp_trsm_inv.cuh -- S4 for a REGULAR strip (four full base panels, 128 pivots) as ONE dense product.
//
// trsm_strip_kernel<LOWER> walks the strip's base panels one after the other inside every CTA (X_b <- T_b X_b, then
// X_t -= L[t][b] X_b for the later panels): a dependency chain of four steps with block barriers between them, and a
// grid of one CTA per 32 columns that leaves a ragged second round on the 148 SMs.  The operator it applies is linear,
// X_final = W . X with the block lower-triangular 128 x 128 matrix
//     W[b][b] = T_b ,     W[b][c] = -T_b . sum_{c <= d < b} L[b][d] . W[d][c]     (c < b; blocks of 32 x 32)
// where L[b][d][i][k] = A[pivot row 32b+i][pivot column of pivot 32d+k] (fp_kernels.cuh storage convention).
// strip_winv_kernel builds W once per strip (sixteen CTAs, eight columns of W each, right behind the strip kernel, under
// the host's round trip) and stores it as the four u8 limb planes of a tcgen05 A operand, already in the 128-byte
// swizzled shared-memory image.  trsm_winv_kernel applies it to the row block right of the strip on the tensor cores:
// U = W . X is one 128 x 128 x n product, the same limb-plane kind::i8 formulation as the Schur update (gemm_tc.cu): a
// CTA keeps W's planes in shared memory, splits a 128 x 32 tile of X into B limb planes itself (no pre-pass over X),
// issues the sixteen 128 x 128 x 32 MMAs, recombines the seven accumulators mod p and writes the tile of U back row-major
// together with its own limb planes for the Schur update that follows.  On CUDA cores the same product is bound by the
// integer multiply pipe at about 7.7 issue cycles per 32 x 32 -> 64-bit multiply-add and warp (measured with the
// chain kernel and with a dense CUDA-core version of this product: profiles/r02_trsm_winv.md).
// PAPER.md:245-249 (the row operations of the elimination step; here applied to the pivot rows themselves).
#pragma once
#include "fp_strip.cuh"

namespace linac {

constexpr int WK = 4 * PW;           // pivots of a regular strip
constexpr int WINV_NT = 256;         // threads of strip_winv_kernel: thread (i, jj) owns row i of 8 columns of every block
constexpr int WINV_CTAS = WK / 8;
constexpr int WLS = PW + 1;          // row stride of the staged L / T blocks (four rows are read per warp and step)

struct WinvSmem {
    uint32_t Ts[4][PW][WLS];         // T_b
    uint32_t Ls[6][PW][WLS];         // L[b][d], slot b(b-1)/2 + d
    uint32_t Wc[4][PW][8];           // this CTA's eight columns of W[b][c]
    uint32_t Ys[PW][8];
};

// sum_k row[k] * col[k][jj] over one 32 x 32 block on two independent accumulators (each: two products per fold)
__device__ __forceinline__ void winv_dot(uint64_t& a0, uint64_t& a1, const uint32_t* __restrict__ row,
                                         const uint32_t (*col)[8], int jj, const ModP& f) {
#pragma unroll
    for (int k = 0; k < PW; k += 4) {
        a0 = fold64(a0 + (uint64_t)row[k] * col[k][jj] + (uint64_t)row[k + 1] * col[k + 1][jj], f);
        a1 = fold64(a1 + (uint64_t)row[k + 2] * col[k + 2][jj] + (uint64_t)row[k + 3] * col[k + 3][jj], f);
    }
}

// One CTA's share of W: column block C (compile-time, so that every loop below unrolls and the loads of a thread --
// up to 40 -- are all in flight together instead of one load-then-store after the other), columns j0..j0+7 of it.
template <int C>
__device__ __forceinline__ void winv_body(WinvSmem& sm, const uint32_t* __restrict__ A, int64_t ld, int t0, int b0, int j0,
                                          const uint32_t* __restrict__ T, int64_t jstrip, const int32_t* __restrict__ pstart,
                                          const ModP& f, uint8_t* __restrict__ Wq) {
    const int tid = threadIdx.x;
    constexpr int NQ = PW * PW / WINV_NT;                        // elements of a 32 x 32 block per thread
    const int kk = tid % PW, i0 = tid / PW;                      // element q of the thread: (row i0 + 8 q, column kk)
    // a base panel that found 32 pivots in its 32 columns has every column as a pivot column, in order: pivot 32 d + k of
    // a regular strip sits in column jstrip + 32 d + k, so no load here waits for another (the pivot-column list and the
    // pivot counts are only needed to CONFIRM that the strip is regular, below, beside these loads)
    int64_t pc[4];
#pragma unroll
    for (int d = C; d < 3; ++d) pc[d] = jstrip + PW * d + kk;
    uint32_t tv[4][NQ], lv[6][NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int ii = i0 + (WINV_NT / PW) * q;
#pragma unroll
        for (int b = C; b < 4; ++b) {
            tv[b][q] = T[(int64_t)(b0 + b) * PW * PW + ii * PW + kk];
#pragma unroll
            for (int d = C; d < b; ++d) lv[b * (b - 1) / 2 + d][q] = A[(int64_t)(t0 + PW * b + ii) * ld + pc[d]];
        }
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int ii = i0 + (WINV_NT / PW) * q;
#pragma unroll
        for (int b = C; b < 4; ++b) {
            sm.Ts[b][ii][kk] = tv[b][q];
#pragma unroll
            for (int d = C; d < b; ++d) sm.Ls[b * (b - 1) / 2 + d][ii][kk] = lv[b * (b - 1) / 2 + d][q];
        }
    }
    {
        const int p0 = pstart[b0], p1 = pstart[b0 + 1], p2 = pstart[b0 + 2], p3 = pstart[b0 + 3], p4 = pstart[b0 + 4];
        if (p0 != t0 || p1 - p0 != PW || p2 - p1 != PW || p3 - p2 != PW || p4 - p3 != PW) return;    // uniform over the CTA
    }
    __syncthreads();
    const int i = tid / 8, jj = tid % 8;
    sm.Wc[C][i][jj] = sm.Ts[C][i][j0 + jj];
    __syncthreads();
#pragma unroll
    for (int b = C + 1; b < 4; ++b) {
        uint64_t a0 = 0, a1 = 0;
#pragma unroll
        for (int d = C; d < b; ++d) winv_dot(a0, a1, sm.Ls[b * (b - 1) / 2 + d][i], sm.Wc[d], jj, f);
        sm.Ys[i][jj] = reduce64(fold64(a0, f) + fold64(a1, f), f);
        __syncthreads();
        a0 = a1 = 0;
        winv_dot(a0, a1, sm.Ts[b][i], sm.Ys, jj, f);
        const uint32_t v = reduce64(fold64(a0, f) + fold64(a1, f), f);
        sm.Wc[b][i][jj] = v ? f.p - v : 0u;
        __syncthreads();
    }
    const int k = PW * C + j0 + jj;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const int m = PW * b + i;
        const uint32_t v = b >= C ? sm.Wc[b][i][jj] : 0u;
        const int off = m * WK + (((k >> 4) ^ (m & 7)) << 4) + (k & 15);
#pragma unroll
        for (int l = 0; l < 4; ++l) Wq[l * WK * WK + off] = (uint8_t)(v >> (8 * l));
    }
}

// W for the strip whose first base panel is b0 and whose pivots start at row / pivot index t0 (= pstart[b0]), as the
// shared-memory image of a K-major tcgen05 operand: Wq[limb][m][128 bytes of k], the 16-byte pieces of a row XOR-ed
// with m % 8 (SWIZZLE_128B).  The blocks above the diagonal are written as zeros.  Exits without writing when the strip
// is not regular (the host takes the chain kernel then).
__global__ void __launch_bounds__(WINV_NT) strip_winv_kernel(const uint32_t* __restrict__ A, int64_t ld,
                                                            const int32_t* __restrict__ pstart, int b0,
                                                            const uint32_t* __restrict__ T, int t0, ModP f,
                                                            uint8_t* __restrict__ Wq) {
    extern __shared__ __align__(16) unsigned char winv_smem_raw[];
    WinvSmem& sm = *reinterpret_cast<WinvSmem*>(winv_smem_raw);
    // t0 = first pivot row of the strip, from the host (it launched the strip kernel with it); the rows t0 .. t0 + 127
    // exist (the host checks).  Whether the strip IS regular is confirmed inside winv_body, beside the loads.
    const int j0 = 8 * (blockIdx.x % 4);                         // first of this CTA's columns inside the block
    const int64_t jstrip = (int64_t)b0 * PW;
    switch (blockIdx.x / 4) {                                    // column block of W
        case 0: winv_body<0>(sm, A, ld, t0, b0, j0, T, jstrip, pstart, f, Wq); break;
        case 1: winv_body<1>(sm, A, ld, t0, b0, j0, T, jstrip, pstart, f, Wq); break;
        case 2: winv_body<2>(sm, A, ld, t0, b0, j0, T, jstrip, pstart, f, Wq); break;
        default: winv_body<3>(sm, A, ld, t0, b0, j0, T, jstrip, pstart, f, Wq); break;
    }
}

constexpr int WNT = 256;             // threads of trsm_winv_kernel: eight warps = four TMEM lane quarters x two column halves
constexpr int WTN = 32;              // columns of X per tile
constexpr int W_A_BYTES = 4 * WK * WK;           // W limb planes
constexpr int W_B_BYTES = 4 * WTN * WK;          // limb planes of one X tile, stacked along N
constexpr size_t WTRSM_SMEM = W_A_BYTES + W_B_BYTES + 1024 /*align*/ + 64 /*barriers*/;
constexpr int W_TMEM_COLS = 256;     // 7 accumulators x 32 columns

// X <- W . X on columns [0, ncols) of the WK rows at X (row stride ldx), in place; optionally also the four u8 limb
// planes of the result (Bq[limb][column][kp], k-major, kp >= WK zero padded), as trsm_strip_kernel writes them.
// Persistent: CTA b takes tiles b, b + gridDim.x, ...; two CTAs share an SM (one loads and splits its next tile while
// the other's MMAs and epilogue run).
__global__ void __launch_bounds__(WNT, 2) trsm_winv_kernel(const uint8_t* __restrict__ Wq, uint32_t* __restrict__ X,
                                                          int64_t ldx, int64_t ncols, ModP f, uint8_t* __restrict__ Bq,
                                                          int kp, int64_t bq_col0, int64_t bq_total) {
    using namespace tc;
    grid_dep_launch();                                    // an update launched as a programmatic dependent may start its prologue now
    extern __shared__ uint8_t wtrsm_smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)wtrsm_smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sA = smem;                                   // [4][WK][128]
    uint8_t* sB = smem + W_A_BYTES;                       // [4][WTN][128]
    uint64_t* bar_a = (uint64_t*)(sB + W_B_BYTES);        // W image landed
    uint64_t* bar_m = bar_a + 1;                          // the tile's MMAs have completed
    uint32_t* tmem_holder = (uint32_t*)(bar_a + 2);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ntiles = (int)((ncols + WTN - 1) / WTN);
    if ((int)blockIdx.x >= ntiles) return;

    if (tid == 0) {
        mbar_init(bar_a, 1);
        mbar_init(bar_m, 1);
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_holder, W_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_holder;
    if (tid == 0) {                                       // the W planes: four bulk copies of one limb plane each
        mbar_expect_tx(bar_a, W_A_BYTES);
        for (int l = 0; l < 4; ++l)
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(smem_u32(sA + l * WK * WK)), "l"(Wq + l * WK * WK), "r"(WK * WK), "r"(smem_u32(bar_a)) : "memory");
    }
    const bool vec = ((((uintptr_t)X) | ((uintptr_t)ldx * 4)) & 15) == 0;
    const int64_t plane = bq_total * (int64_t)kp;
    const uint64_t c32 = f.c32;
    uint32_t phase = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t n0 = (int64_t)tile * WTN;
        // ---- split the X tile into the B operand: sB[limb][n][k], lane = column n, four consecutive k per store
        {
            const int64_t c = n0 + lane;
            const bool cok = c < ncols;
            const uint32_t* src = X + c;
            const int sw = lane & 7;
            constexpr int KW = WK / (WNT / 32);                                                    // k per warp
            uint32_t v[KW];
#pragma unroll
            for (int q = 0; q < KW; ++q) v[q] = cok ? src[(int64_t)(KW * warp + q) * ldx] : 0u;     // k = KW warp + q
#pragma unroll
            for (int g = 0; g < KW / 4; ++g) {
                const int k = KW * warp + 4 * g;
                const int off = lane * WK + (((k >> 4) ^ sw) << 4) + (k & 15);
#pragma unroll
                for (int l = 0; l < 4; ++l) {
                    const uint32_t packed = ((v[4 * g] >> (8 * l)) & 0xFFu) | (((v[4 * g + 1] >> (8 * l)) & 0xFFu) << 8) |
                                            (((v[4 * g + 2] >> (8 * l)) & 0xFFu) << 16) | (((v[4 * g + 3] >> (8 * l)) & 0xFFu) << 24);
                    *reinterpret_cast<uint32_t*>(sB + l * (WTN * WK) + off) = packed;
                }
            }
        }
        fence_proxy_async();                              // generic-proxy writes -> visible to the tensor core's reads
        __syncthreads();
        // ---- the sixteen MMAs of the tile (K = 128 = four k steps of 32 bytes)
        if (tid == 0) {
            if (tile == (int)blockIdx.x) mbar_wait(bar_a, 0);
            tc_fence_after();
            const uint32_t a0 = smem_u32(sA), b0 = smem_u32(sB);
            constexpr uint32_t idesc_n = make_idesc_i8(WTN), idesc_4n = make_idesc_i8(4 * WTN);
#pragma unroll
            for (int i = 0; i < 4; ++i)                   // first k step: every accumulator is written once without accumulation
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    umma_i8(tmem_base + (uint32_t)((i + j) * WTN), make_desc_sw128(a0 + i * (WK * WK)),
                            make_desc_sw128(b0 + j * (WTN * WK)), idesc_n, (i == 0 || j == 3) ? 0u : 1u);
#pragma unroll
            for (int kk = 1; kk < WK / 32; ++kk)
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    umma_i8(tmem_base + (uint32_t)(i * WTN), make_desc_sw128(a0 + i * (WK * WK) + kk * 32),
                            make_desc_sw128(b0 + kk * 32), idesc_4n, 1u);
            umma_commit(bar_m);
        }
        mbar_wait(bar_m, phase);
        phase ^= 1;
        tc_fence_after();
        // ---- epilogue: thread = row m of U and one half of the tile's columns (a warp reaches the TMEM lanes of its
        // quarter warp % 4 only); recombine the seven limb accumulators, write U and its limb planes
        {
            const int quarter = warp & 3, half = warp >> 2;
            const int m = 32 * quarter + lane;
            uint32_t* urow = X + (int64_t)m * ldx + n0;
#pragma unroll 1
            for (int c8 = half * (WTN / 16); c8 < (half + 1) * (WTN / 16); ++c8) {
                uint32_t S[7][8];
#pragma unroll
                for (int w = 0; w < 7; ++w) tmem_ld8(tmem_base + ((uint32_t)(32 * quarter) << 16) + (uint32_t)(w * WTN + c8 * 8), S[w]);
                tmem_ld_wait();
                uint32_t u[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const uint64_t lo = (uint64_t)S[0][e] + ((uint64_t)S[1][e] << 8) + ((uint64_t)S[2][e] << 16) + ((uint64_t)S[3][e] << 24);
                    const uint64_t hi = (uint64_t)S[4][e] + ((uint64_t)S[5][e] << 8) + ((uint64_t)S[6][e] << 16);
                    u[e] = reduce64(lo + (uint64_t)reduce64(hi, f) * c32, f);
                }
                const int64_t nb = n0 + c8 * 8;
                if (vec && nb + 8 <= ncols) {
                    *reinterpret_cast<uint4*>(urow + c8 * 8) = make_uint4(u[0], u[1], u[2], u[3]);
                    *reinterpret_cast<uint4*>(urow + c8 * 8 + 4) = make_uint4(u[4], u[5], u[6], u[7]);
                } else {
#pragma unroll
                    for (int e = 0; e < 8; ++e)
                        if (nb + e < ncols) urow[c8 * 8 + e] = u[e];
                }
                if (Bq != nullptr) {
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        if (nb + e >= ncols) break;
                        uint8_t* dst = Bq + (bq_col0 + nb + e) * kp + m;
#pragma unroll
                        for (int l = 0; l < 4; ++l) dst[l * plane] = (uint8_t)(u[e] >> (8 * l));
                    }
                }
            }
        }
        tc_fence_before();
        __syncthreads();                                  // sB and the accumulators are free for the next tile
    }
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, W_TMEM_COLS);
    }
}

}  // namespace linac
