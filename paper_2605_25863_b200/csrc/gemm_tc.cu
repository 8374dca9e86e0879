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
#include <vector>

#include "linac_internal.h"
#include "tc_ptx.cuh"

namespace linac {
using namespace tc;
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
constexpr int64_t KC_MAX = 8192;     // K per launch (multiple of 128; the s32 accumulators hold K <= 8256, see the header)

// ----------------------------------------------------------------------------- the GEMM kernel
__global__ void __launch_bounds__(NTHREADS, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, uint32_t* __restrict__ C,
               int64_t ldc, int64_t M, int64_t N, int kp /* padded K of this launch, multiple of KB */, ModP f,
               int mtiles, int ntiles, int gm /* row tiles per band */) {
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
    // Tile order: bands of `gm` row tiles, row tiles fastest inside a band.  The CTAs in flight together (one wave) then
    // share gm A panels -- which stay in L2 while the band sweeps over the column tiles -- and a handful of B panels.
    // In row-major tile order a wave touched 148 different B panels (more than L2 holds at K = 4096), so every row of
    // tiles re-read all of B from DRAM: 35.7 GB of DRAM reads for a 16384^2 x 4096 product whose operands are 0.5 GB.
    int m_tile, n_tile;
    {
        const int lin = blockIdx.x, per_band = gm * ntiles;
        const int band = lin / per_band, within = lin - band * per_band;
        const int first = band * gm, gmm = min(gm, mtiles - first);
        n_tile = within / gmm;
        m_tile = first + within - n_tile * gmm;
    }
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

// ----------------------------------------------------------------------------- the small-K (panel) kernel
// K <= 256 is the Schur update behind ONE strip: every output element is read and written once per
// 128..256 field products, so the epilogue and the C traffic weigh as much as the MMAs.  This kernel is
// persistent (one CTA per SM), A-stationary (the 128-row limb planes of L21 stay in shared memory while
// the CTA sweeps a run of 32-column output tiles), and overlaps the three stages of a tile:
//   warp 0      TMA producer: A k-stages (ring of 2 x 64 KB) and B k-stages (ring of 4 x 16 KB)
//   warp 1      MMA issuer: 128x128x32 kind::i8 MMAs (four B limb planes stacked along N), two TMEM
//               accumulator buffers of 7 x 32 columns
//   warp 2      C mover (TMA loads / L2 prefetch / TMA stores of the C tiles)
//   warps 3-18  epilogue: tcgen05.ld, limb recombination sum_w S_w (2^(8w) mod p), one Barrett reduction,
//               C tile staged through shared memory by TMA in both directions (128-byte swizzle), so no
//               thread-per-row global access ever reaches the LSU.
constexpr int PN = 32;                       // output tile columns
constexpr int P_A_STAGE = 4 * TM * KB;       // 65536
constexpr int P_B_STAGE = 4 * PN * KB;       // 16384
constexpr int P_C_TILE = TM * PN * 4;        // 16384
constexpr int P_NAS = 2, P_NBS = 3, P_NCS = 3;
constexpr int P_SMEM = P_NAS * P_A_STAGE + P_NBS * P_B_STAGE + P_NCS * P_C_TILE + 1024 + 256;
static_assert(1 * P_A_STAGE + P_NBS * P_B_STAGE + 7 * P_C_TILE + 1024 + 256 == P_SMEM, "both stage configurations fill the same shared memory");
constexpr int P_EPI_WARPS = 16;              // epilogue warps: 4 TMEM lane quarters x 4 groups of 8 columns
constexpr int P_THREADS = 96 + 32 * P_EPI_WARPS;
constexpr int P_PF = 6;                      // L2 prefetch distance for C tiles
constexpr int P_ACC_COLS = 256;              // TMEM columns reserved per accumulator buffer (224 used)

struct PanelSched {
    int mtiles, ntiles, nchunks, tiles_per_chunk, nitems;
};

struct TileIter {
    int item, mt, nt, nt_end;
    bool valid;
    __device__ __forceinline__ void load_item(const PanelSched& sc) {
        valid = item < sc.nitems;
        if (!valid) return;
        mt = item / sc.nchunks;
        const int ch = item % sc.nchunks;
        nt = ch * sc.tiles_per_chunk;
        nt_end = min(sc.ntiles, nt + sc.tiles_per_chunk);
    }
    __device__ __forceinline__ void init(const PanelSched& sc) { item = blockIdx.x; load_item(sc); }
    __device__ __forceinline__ bool last_of_item() const { return nt + 1 >= nt_end; }
    __device__ __forceinline__ void next(const PanelSched& sc) {
        if (++nt >= nt_end) { item += gridDim.x; load_item(sc); }
    }
};

__device__ __forceinline__ TileIter sc_init(const PanelSched& sc) {
    TileIter it;
    it.init(sc);
    return it;
}

// NAS A stages and NCS C-tile buffers: (2, 3) serves any K <= 256; (1, 7) is the K <= 128 configuration -- one A stage is all a
// single k-stage needs, and the shared memory it frees holds four more C tiles, so the C mover keeps six tile loads in flight
// instead of two (the K = 128 update is bound by data movement: profiles/r02_experiments.md).
template <bool MONT, int NAS, int NCS>
__global__ void __launch_bounds__(P_THREADS, 1)
gemm_tc_panel_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                     const __grid_constant__ CUtensorMap tmC, int nks /* k-stages: kp / 128 */, PanelSched sc, ModP f) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sA = smem;
    uint8_t* sB = sA + NAS * P_A_STAGE;
    uint8_t* sC = sB + P_NBS * P_B_STAGE;
    uint64_t* bars = (uint64_t*)(sC + NCS * P_C_TILE);
    uint64_t* a_full = bars;                 // [2]
    uint64_t* a_empty = bars + 2;            // [2]
    uint64_t* b_full = bars + 4;             // [4]
    uint64_t* b_empty = bars + 8;            // [4]
    uint64_t* acc_full = bars + 12;          // [2]
    uint64_t* acc_empty = bars + 14;         // [2]
    uint64_t* c_full = bars + 16;            // [NCS]
    uint64_t* c_done = bars + 16 + NCS;      // [NCS]
    uint32_t* tmem_holder = (uint32_t*)(bars + 16 + 2 * NCS);
    static_assert((16 + 2 * NCS) * 8 + 4 <= 256, "the barrier block is 256 bytes");

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp == 0 && lane == 0) {
        prefetch_tmap(&tmA);
        prefetch_tmap(&tmB);
        prefetch_tmap(&tmC);
        for (int i = 0; i < 2; ++i) { mbar_init(&a_full[i], 1); mbar_init(&a_empty[i], 1); mbar_init(&acc_full[i], 1);
                                      mbar_init(&acc_empty[i], P_EPI_WARPS); }
        for (int i = 0; i < NCS; ++i) { mbar_init(&c_full[i], 1); mbar_init(&c_done[i], P_EPI_WARPS); }
        for (int i = 0; i < P_NBS; ++i) { mbar_init(&b_full[i], 1); mbar_init(&b_empty[i], 1); }
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(tmem_holder, TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_holder;

    if (warp == 0) {
        if (lane == 0) {
            uint32_t a_cnt = 0, b_cnt = 0;
            bool dep_waited = false;
            TileIter it;
            it.init(sc);
            while (it.valid) {
                for (int ks = 0; ks < nks; ++ks, ++a_cnt) {
                    const int s = a_cnt % NAS;
                    mbar_wait(&a_empty[s], ((a_cnt / NAS) & 1) ^ 1);
                    mbar_expect_tx(&a_full[s], P_A_STAGE);
                    tma_load_3d(sA + s * P_A_STAGE, &tmA, &a_full[s], ks * KB, it.mt * TM, 0);
                }
                const int item = it.item;
                // B is the only operand the kernel right before this one in the stream may have produced (the row-block
                // solve writes U12's limb planes): under a programmatic dependent launch everything above -- barriers,
                // TMEM, the A stages, the first C tiles -- has run beside that kernel, and only this waits for it
                if (!dep_waited) { grid_dep_wait(); dep_waited = true; }
                while (it.valid && it.item == item) {
                    for (int ks = 0; ks < nks; ++ks, ++b_cnt) {
                        const int s = b_cnt % P_NBS;
                        mbar_wait(&b_empty[s], ((b_cnt / P_NBS) & 1) ^ 1);
                        mbar_expect_tx(&b_full[s], P_B_STAGE);
                        tma_load_3d(sB + s * P_B_STAGE, &tmB, &b_full[s], ks * KB, it.nt * PN, 0);
                    }
                    it.next(sc);
                }
            }
        }
    } else if (warp == 1) {
        // The whole warp runs this loop with uniform control flow (so descriptors and counters live in uniform
        // registers and cost one add per MMA); one elected lane issues the tcgen05 instructions.
        constexpr uint32_t id128 = make_idesc_i8(4 * PN), id96 = make_idesc_i8(3 * PN), id32 = make_idesc_i8(PN);
        constexpr uint64_t LIMB = (uint64_t)((TM * KB) >> 4);          // descriptor step between A limb planes
        constexpr uint64_t KSTEP = 32 >> 4;                            // descriptor step of one 32-byte k slice
        uint64_t adesc[2], bdesc[P_NBS];
#pragma unroll
        for (int i = 0; i < 2; ++i) adesc[i] = make_desc_sw128(smem_u32(sA + (i % NAS) * P_A_STAGE));
#pragma unroll
        for (int i = 0; i < P_NBS; ++i) bdesc[i] = make_desc_sw128(smem_u32(sB + i * P_B_STAGE));
        uint32_t a_cnt = 0, b_cnt = 0, t_cnt = 0;
        TileIter it = sc_init(sc);
        while (it.valid) {
            const int item = it.item;
            bool first_tile = true;
            while (it.valid && it.item == item) {
                const uint32_t buf = t_cnt & 1;
                mbar_wait(&acc_empty[buf], ((t_cnt >> 1) & 1) ^ 1);
                tc_fence_after();
                const uint32_t d0 = tmem_base + buf * P_ACC_COLS;
                const bool last = it.last_of_item();
                for (int ks = 0; ks < nks; ++ks, ++b_cnt) {
                    const uint32_t ac = a_cnt + ks;
                    const int sa = ac % NAS;
                    if (first_tile) mbar_wait(&a_full[sa], (ac / NAS) & 1);
                    const int sb = b_cnt % P_NBS;
                    mbar_wait(&b_full[sb], (b_cnt / P_NBS) & 1);
                    tc_fence_after();
                    const uint64_t da = sa == 0 ? adesc[0] : adesc[1];
                    const uint64_t db = sb == 0 ? bdesc[0] : (sb == 1 ? bdesc[1] : bdesc[2]);
                    if (elect_one()) {
                        if (ks == 0) {
                            // first k step of the tile: slots 0-3 and 4-6 are overwritten, the rest accumulate
                            umma_i8(d0, da, db, id128, 0u);
                            umma_i8(d0 + 4 * PN, da + 3 * LIMB, db + ((PN * KB) >> 4), id96, 0u);
                            umma_i8(d0 + 1 * PN, da + 1 * LIMB, db, id128, 1u);
                            umma_i8(d0 + 2 * PN, da + 2 * LIMB, db, id128, 1u);
                            umma_i8(d0 + 3 * PN, da + 3 * LIMB, db, id32, 1u);
                        } else {
                            umma_i8_x4(d0, da, db, id128, PN, LIMB);
                        }
#pragma unroll
                        for (int kk = 1; kk < KB / 32; ++kk) umma_i8_x4(d0, da + kk * KSTEP, db + kk * KSTEP, id128, PN, LIMB);
                        umma_commit(&b_empty[sb]);
                        if (last) umma_commit(&a_empty[sa]);
                        if (ks == nks - 1) umma_commit(&acc_full[buf]);
                    }
                    __syncwarp();
                }
                ++t_cnt;
                first_tile = false;
                it.next(sc);
            }
            a_cnt += nks;
        }
    } else if (warp == 2) {
        // C mover: TMA loads of the C tiles NCS - 1 tiles ahead, L2 prefetch further ahead
        // (the trailing matrix is far larger than L2), TMA stores once the epilogue warps are done with a tile.
        if (lane == 0) {
            TileIter ld = sc_init(sc), pf = ld, st = ld;
            uint32_t l_cnt = 0, t_cnt = 0;
            for (int i = 0; i < P_PF + NCS - 3 && pf.valid; ++i) pf.next(sc);
            for (int i = 0; i < NCS - 1 && ld.valid; ++i, ++l_cnt) {
                mbar_expect_tx(&c_full[l_cnt % NCS], P_C_TILE);
                tma_load_2d(sC + (l_cnt % NCS) * P_C_TILE, &tmC, &c_full[l_cnt % NCS], ld.nt * PN, ld.mt * TM);
                ld.next(sc);
            }
            while (st.valid) {
                const uint32_t cb = t_cnt % NCS;
                if (pf.valid) { tma_prefetch_l2_2d(&tmC, pf.nt * PN, pf.mt * TM); pf.next(sc); }
                mbar_wait(&c_done[cb], (t_cnt / NCS) & 1);
                tma_store_2d(&tmC, sC + cb * P_C_TILE, st.nt * PN, st.mt * TM);
                tma_store_commit();
                st.next(sc);
                ++t_cnt;
                if (ld.valid) {
                    // buffer of tile t + NCS - 1 == buffer of tile t - 1, whose store was committed one iteration ago
                    tma_store_wait_read1();
                    const uint32_t lb = l_cnt % NCS;
                    mbar_expect_tx(&c_full[lb], P_C_TILE);
                    tma_load_2d(sC + lb * P_C_TILE, &tmC, &c_full[lb], ld.nt * PN, ld.mt * TM);
                    ld.next(sc);
                    ++l_cnt;
                }
            }
            tma_store_wait_all();
        }
    } else {
        const int e = warp - 3, q = warp & 3, g = e >> 2;      // TMEM lane quarter, column group of 8
        const int row = q * 32 + lane;
        uint32_t t_cnt = 0;
        TileIter it = sc_init(sc);
        while (it.valid) {
            const uint32_t buf = t_cnt & 1, ph = (t_cnt >> 1) & 1;
            const uint32_t cb = t_cnt % NCS, cph = (t_cnt / NCS) & 1;
            it.next(sc);
            mbar_wait(&acc_full[buf], ph);
            tc_fence_after();
            uint32_t S[7][8];
            const uint32_t t0 = tmem_base + ((uint32_t)(q * 32) << 16) + buf * P_ACC_COLS + g * 8;
#pragma unroll
            for (int w = 0; w < 7; ++w) tmem_ld8(t0 + w * PN, S[w]);
            tmem_ld_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&acc_empty[buf]);
            mbar_wait(&c_full[cb], cph);
            const uint32_t crow = smem_u32(sC + cb * P_C_TILE + row * 128);
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const uint32_t pc = crow + (((2 * g + j) ^ (row & 7)) << 4);
                uint32_t cv[4];
                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(cv[0]), "=r"(cv[1]), "=r"(cv[2]), "=r"(cv[3]) : "r"(pc));
#pragma unroll
                for (int x = 0; x < 4; ++x) {
                    const int el = 4 * j + x;
                    if (MONT) {
                        // sum_w S_w (2^(8w) 2^32 mod p) < 7 * 2^26 * p < 2^32 p, so one Montgomery reduction finishes
                        uint64_t v = (uint64_t)S[0][el] * f.wm[0];
#pragma unroll
                        for (int w = 1; w < 7; ++w) v += (uint64_t)S[w][el] * f.wm[w];
                        cv[x] = submod(cv[x], redc(v, f), f);
                    } else {
                        uint64_t v = (uint64_t)S[0][el] + ((uint64_t)S[1][el] << 8) + ((uint64_t)S[2][el] << 16) + ((uint64_t)S[3][el] << 24);
                        v += (uint64_t)S[4][el] * f.w[4] + (uint64_t)S[5][el] * f.w[5] + (uint64_t)S[6][el] * f.w[6];
                        cv[x] = submod(cv[x], reduce64(v, f), f);
                    }
                }
                asm volatile("st.shared.v4.u32 [%4], {%0, %1, %2, %3};" ::"r"(cv[0]), "r"(cv[1]), "r"(cv[2]), "r"(cv[3]), "r"(pc) : "memory");
            }
            fence_proxy_async();                 // the tile in shared memory is read next by the TMA store
            __syncwarp();
            if (lane == 0) mbar_arrive(&c_done[cb]);
            ++t_cnt;
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
bool make_limb_map(CUtensorMap* tm, uint8_t* base, int64_t rows, int64_t kp, int box_rows, int64_t plane_rows = 0) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return false;
    if (plane_rows <= 0) plane_rows = rows;               // rows between two limb planes (>= rows when `base` is a sub-range)
    cuuint64_t dims[3] = {(cuuint64_t)kp, (cuuint64_t)rows, 4};
    cuuint64_t strides[2] = {(cuuint64_t)kp, (cuuint64_t)plane_rows * (cuuint64_t)kp};
    cuuint32_t box[3] = {(cuuint32_t)KB, (cuuint32_t)box_rows, 4};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// 2-D map over C (uint32, row-major): box = 32 columns x 128 rows, 128-byte swizzle.
bool make_c_map(CUtensorMap* tm, uint32_t* C, int64_t ldc, int64_t M, int64_t N) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return false;
    cuuint64_t dims[2] = {(cuuint64_t)N, (cuuint64_t)M};
    cuuint64_t strides[1] = {(cuuint64_t)ldc * 4};
    cuuint32_t box[2] = {(cuuint32_t)PN, (cuuint32_t)TM};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, C, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// Work items of the panel kernel: (128-row tile, run of 32-column tiles); run length chosen so that the
// items fill a whole number of waves over the persistent grid with runs of about 24 tiles.
PanelSched make_sched(int64_t M, int64_t N, int grid) {
    PanelSched sc;
    sc.mtiles = (int)((M + TM - 1) / TM);
    sc.ntiles = (int)((N + PN - 1) / PN);
    const int64_t total = (int64_t)sc.mtiles * sc.ntiles;
    const int64_t waves = std::max<int64_t>(1, (total + (int64_t)grid * 24 - 1) / ((int64_t)grid * 24));
    int64_t nchunks = (waves * grid + sc.mtiles - 1) / sc.mtiles;
    nchunks = std::max<int64_t>(1, std::min<int64_t>(nchunks, sc.ntiles));
    sc.tiles_per_chunk = (int)((sc.ntiles + nchunks - 1) / nchunks);
    sc.nchunks = (sc.ntiles + sc.tiles_per_chunk - 1) / sc.tiles_per_chunk;
    sc.nitems = sc.mtiles * sc.nchunks;
    return sc;
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
    static PerDeviceOnce attr_once;
    if (attr_once.run([]() -> int {
            if (cudaFuncSetAttribute(gemm_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES) != cudaSuccess ||
                cudaFuncSetAttribute(gemm_tc_panel_kernel<true, 2, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SMEM) != cudaSuccess ||
                cudaFuncSetAttribute(gemm_tc_panel_kernel<false, 2, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SMEM) != cudaSuccess ||
                cudaFuncSetAttribute(gemm_tc_panel_kernel<true, 1, 7>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SMEM) != cudaSuccess ||
                cudaFuncSetAttribute(gemm_tc_panel_kernel<false, 1, 7>, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SMEM) != cudaSuccess) {
                cudaGetLastError();
                return LINAC_ERR_CUDA;
            }
            return LINAC_OK;
        }) != LINAC_OK)
        return -1;
    const bool panel_ok = g.K <= 2 * KB && options().tc_panel != 0 && ((((uintptr_t)g.C) | ((uintptr_t)g.ldc * 4)) & 15) == 0;
    if (panel_ok) {
        const bool b_ready = g.Bq_ready != nullptr && g.kp_ready >= g.K && g.kp_ready <= 2 * KB && g.kp_ready % KB == 0;
        const int64_t kp = b_ready ? g.kp_ready : (g.K + KB - 1) / KB * KB;
        const bool a_ready = b_ready && g.Aq_ready != nullptr;
        uint8_t* Aq = a_ready ? g.Aq_ready : (uint8_t*)scratch->take((size_t)4 * g.M * kp, 1024);
        uint8_t* Bq = b_ready ? g.Bq_ready : (uint8_t*)scratch->take((size_t)4 * g.N * kp, 1024);
        if (!Aq || !Bq) return -1;
        if (!a_ready) {
            dim3 grid((unsigned)((kp / 4 + 127) / 128), (unsigned)std::min<int64_t>(g.M, 16384));
            split_a_kernel<<<grid, 128, 0, s>>>(g.Abase, g.lda, g.kcols, 0, g.M, g.K, kp, Aq);
            LINAC_CUDA(cudaGetLastError());
            stats().kernel_launches++;
        }
        if (!b_ready) {
            dim3 grid((unsigned)(kp / 128), (unsigned)((g.N + 31) / 32));
            split_b_kernel<<<grid, 256, 0, s>>>(g.B, g.ldb, g.K, g.N, kp, Bq);
            LINAC_CUDA(cudaGetLastError());
            stats().kernel_launches++;
        }
        CUtensorMap tmA, tmB, tmC;
        const int64_t b_total = b_ready && g.bq_rows_total > 0 ? g.bq_rows_total : g.N;
        const int64_t b_row0 = b_ready ? g.bq_row0 : 0;
        if (!make_limb_map(&tmA, Aq, g.M, kp, TM) || !make_limb_map(&tmB, Bq + b_row0 * kp, g.N, kp, PN, b_total) ||
            !make_c_map(&tmC, g.C, g.ldc, g.M, g.N))
            return -1;
        const int grid = g.grid_limit > 0 ? std::min(g.grid_limit, sm_count()) : sm_count();
        const PanelSched sc = make_sched(g.M, g.N, grid);
        const int nks = (int)(kp / KB);
        const bool deep = nks == 1 && options().tc_panel_deep != 0;     // K <= 128: one A stage, seven C buffers
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)std::min(grid, sc.nitems));
        cfg.blockDim = dim3(P_THREADS);
        cfg.dynamicSmemBytes = P_SMEM;
        cfg.stream = s;
        // programmatic dependent launch behind the kernel that produced B (the caller vouches that this kernel wrote
        // neither A nor C): the prologue and the A / C loads overlap that kernel's tail
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = g.pdl ? 1 : 0;
        if (f.ninv && deep) LINAC_CUDA(cudaLaunchKernelEx(&cfg, gemm_tc_panel_kernel<true, 1, 7>, tmA, tmB, tmC, nks, sc, f));
        else if (f.ninv) LINAC_CUDA(cudaLaunchKernelEx(&cfg, gemm_tc_panel_kernel<true, 2, 3>, tmA, tmB, tmC, nks, sc, f));
        else if (deep) LINAC_CUDA(cudaLaunchKernelEx(&cfg, gemm_tc_panel_kernel<false, 1, 7>, tmA, tmB, tmC, nks, sc, f));
        else LINAC_CUDA(cudaLaunchKernelEx(&cfg, gemm_tc_panel_kernel<false, 2, 3>, tmA, tmB, tmC, nks, sc, f));
        LINAC_CUDA(cudaGetLastError());
        stats().kernel_launches += 1;
        stats().tc_launches++;
        stats().update_macs += g.M * g.N * g.K;
        return LINAC_OK;
    }
    const int64_t kc = chunk_k(g.K);
    uint8_t* Aq = (uint8_t*)scratch->take((size_t)4 * g.M * kc, 1024);
    uint8_t* Bq = (uint8_t*)scratch->take((size_t)4 * g.N * kc, 1024);
    if (!Aq || !Bq) return -1;
    // every chunk's tensor maps are encoded BEFORE the first launch: once a chunk has updated C there is no falling
    // back to the CUDA-core kernel over the full K (it would subtract that chunk's product twice)
    std::vector<CUtensorMap> maps;
    for (int64_t k0 = 0; k0 < g.K; k0 += kc) {
        const int64_t kp = (std::min(kc, g.K - k0) + KB - 1) / KB * KB;
        CUtensorMap tmA, tmB;
        if (!make_limb_map(&tmA, Aq, g.M, kp, TM) || !make_limb_map(&tmB, Bq, g.N, kp, TN)) return -1;
        maps.push_back(tmA);
        maps.push_back(tmB);
    }
    size_t chunk = 0;
    for (int64_t k0 = 0; k0 < g.K; k0 += kc, ++chunk) {
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
        const CUtensorMap& tmA = maps[2 * chunk];
        const CUtensorMap& tmB = maps[2 * chunk + 1];
        const int64_t mtiles = (g.M + TM - 1) / TM, ntiles = (g.N + TN - 1) / TN;
        if (mtiles * ntiles >= (1ll << 31)) return LINAC_ERR_INVALID_ARG;
        // a band's A panels (gm x 128 rows x kp x 4 planes) should take about a quarter of the 126 MB L2
        const int gm = (int)std::max<int64_t>(4, std::min<int64_t>(32, (32ll << 20) / (4 * TM * kp)));
        gemm_tc_kernel<<<(unsigned)(mtiles * ntiles), NTHREADS, SMEM_BYTES, s>>>(tmA, tmB, g.C, g.ldc, g.M, g.N, (int)kp, f, (int)mtiles,
                                                                                (int)ntiles, gm);
        LINAC_CUDA(cudaGetLastError());
        stats().kernel_launches += 3;
        stats().tc_launches++;
    }
    stats().update_macs += g.M * g.N * g.K;
    return LINAC_OK;
}

}  // namespace linac
