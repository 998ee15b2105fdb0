// a3. Prefill-phase GEMM, CTA-pair kernel (BASELINE.json config 4; ABI in include/triroof.h).
//
// Why pairs: one 128 x 256 x 16 MMA reads 4 KiB of A and 8 KiB of B from shared memory in 128 cycles (96 B/clk) while
// TMA writes the same 12 KiB per 128 cycles for the next stages — together more than the 128 B/clk a shared
// memory delivers, and the single-CTA kernel stops at 79 % tensor-pipe activity (profiles/r1a_ncu_prefill_gemm.txt).  With
// tcgen05.mma.cta_group::2 the two SMs of a TPC compute one 256 x 256 tile: each SM holds its own 128 rows of A
// and only HALF of the W tile (128 of the 256 columns), the tensor cores of both read both halves, so every SM
// stages and reads 8 KiB per MMA instead of 12.
//
// A cluster of 2 CTAs, persistent, one cluster per TPC.  Per CTA (rank r in the pair):
//   warp 0   TMA producer   A rows [256 tm + 128 r, +128) and W columns [256 tn + 128 r, +128) of each 64-wide
//                           k-block into a 6-stage ring (32 KiB per stage); the bytes of BOTH CTAs are counted
//                           on the leader's "full" barrier (cp.async.bulk.tensor ... cta_group::2)
//   warp 1   MMA issuer     leader only: four tcgen05.mma.cta_group::2.kind::f16 (M 256, N 256, K 16) per k-block;
//                           tcgen05.commit ... multicast arrives on "empty" (and, per tile, "tmem_full") in both CTAs
//   warp 2   TMEM owner     tcgen05.alloc.cta_group::2 of all 512 columns = two 128 x 256 fp32 accumulators per
//                           CTA, so the epilogue of tile t overlaps the main loop of tile t + 1
//   warps 4-7 epilogue      tcgen05.ld of the CTA's own 128 rows -> bf16 RNE -> 16-byte stores; then arrive on the
//                           LEADER's "tmem_empty" (8 arrivals: 4 warps x 2 CTAs)
// 4096 x 18944 gives 16 x 74 = 1184 pair tiles = 74 TPCs x 16: no wave quantisation.  M index fastest, as in the
// single-CTA kernel.  Ragged M / N / K: TMA zero fill, clipped stores.
#include "tri_internal.h"
#include "ptx.cuh"
#include "gemm_common.cuh"

namespace tri {

constexpr int G2_BM = 128, G2_BN = 256, G2_BK = 64;      // per CTA: 128 rows x 256 columns of C; pair: 256 x 256
constexpr int G2_BNH = G2_BN / 2;                         // W columns staged per CTA
constexpr int G2_STAGES = 6;
constexpr int G2_A_BYTES = G2_BM * G2_BK * 2;             // 16 KiB
constexpr int G2_B_BYTES = G2_BNH * G2_BK * 2;            // 16 KiB
constexpr int G2_STAGE_BYTES = G2_A_BYTES + G2_B_BYTES;
constexpr int G2_THREADS = 256;
constexpr int G2_TMEM_COLS = 512;
constexpr int G2_SMEM_BYTES = 1024 + G2_STAGES * G2_STAGE_BYTES + 256;

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(G2_THREADS, 1)
gemm_2sm_kernel(const __grid_constant__ CUtensorMap amap, const __grid_constant__ CUtensorMap wmap, const GemmParams p)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t ring = ptx::smem_u32(smem);
    const uint32_t bars = ring + G2_STAGES * G2_STAGE_BYTES;
    const uint32_t full0 = bars, empty0 = bars + 8 * G2_STAGES;
    const uint32_t tfull0 = bars + 16 * G2_STAGES, tempty0 = tfull0 + 16;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + G2_STAGES * G2_STAGE_BYTES + 16 * G2_STAGES + 32);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();
    const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;
    const int ntiles = p.tiles_m * p.tiles_n;             // pair tiles (tiles_m counts 256-row blocks)

    if (threadIdx.x == 0) {
        for (int s = 0; s < G2_STAGES; ++s) {
            ptx::mbar_init(full0 + 8 * s, 1);             // leader's copy is the one used
            ptx::mbar_init(empty0 + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            ptx::mbar_init(tfull0 + 8 * a, 1);
            ptx::mbar_init(tempty0 + 8 * a, 8);           // leader's copy: 4 epilogue warps of each CTA
        }
        ptx::fence_mbar_init();
    }
    if (warp == 2) {
        ptx::tmem_alloc_2sm(ptx::smem_u32(tmem_slot), G2_TMEM_COLS);
        ptx::tmem_relinquish_2sm();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::cluster_sync();                                   // the peer's barriers and TMEM exist before anything touches them
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===== TMA producer (both CTAs) =====
        if (ptx::elect_one()) {
            ptx::prefetch_tmap(&amap);
            ptx::prefetch_tmap(&wmap);
            const uint64_t pol_w = ptx::policy_evict_first();
            const uint64_t pol_a = ptx::policy_evict_last();
            uint32_t it = 0;
            for (int t = pair; t < ntiles; t += npairs) {
                const int tm = t % p.tiles_m, tn = t / p.tiles_m;
                const int row0 = tm * (2 * G2_BM) + (int)rank * G2_BM, col0 = tn * G2_BN + (int)rank * G2_BNH;
                for (int kb = 0; kb < p.kblocks; ++kb, ++it) {
                    const uint32_t s = it % G2_STAGES, ph = (it / G2_STAGES) & 1;
                    ptx::mbar_wait(empty0 + 8 * s, ph ^ 1);
                    const uint32_t fb = full0 + 8 * s;
                    if (rank == 0) ptx::mbar_arrive_expect_tx(fb, 2 * G2_STAGE_BYTES);
                    const uint32_t sa = ring + s * G2_STAGE_BYTES, sb = sa + G2_A_BYTES;
                    ptx::tma_load_2d_2sm(sa, &amap, kb * G2_BK, row0, fb, pol_a);
                    if (!p.b_mn_major) {
                        ptx::tma_load_2d_2sm(sb, &wmap, kb * G2_BK, col0, fb, pol_w);
                    } else {
#pragma unroll
                        for (int q = 0; q < 2; ++q)       // two 64(n) x 64(k) boxes, 8 KiB each
                            ptx::tma_load_2d_2sm(sb + q * 8192, &wmap, col0 + q * 64, kb * G2_BK, fb, pol_w);
                    }
                }
            }
        }
    } else if (warp == 1 && rank == 0) {
        // ===== MMA issuer (leader CTA) =====
        if (ptx::elect_one()) {
            const uint32_t idesc = make_idesc(2 * G2_BM, G2_BN, p.b_mn_major);
            uint32_t it = 0, tcount = 0;
            for (int t = pair; t < ntiles; t += npairs, ++tcount) {
                const uint32_t acc = tcount & 1, aph = (tcount >> 1) & 1;
                ptx::mbar_wait(tempty0 + 8 * acc, aph ^ 1);          // both epilogues have drained this accumulator
                ptx::tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * G2_BN;
                for (int kb = 0; kb < p.kblocks; ++kb, ++it) {
                    const uint32_t s = it % G2_STAGES, ph = (it / G2_STAGES) & 1;
                    ptx::mbar_wait(full0 + 8 * s, ph);
                    ptx::tc_fence_after();
                    const uint32_t sa = ring + s * G2_STAGE_BYTES, sb = sa + G2_A_BYTES;
                    const uint64_t adesc = make_sdesc(sa, 16, 1024);
                    const uint64_t bdesc = make_sdesc(sb, p.b_lbo, p.b_sbo);
#pragma unroll
                    for (int kk = 0; kk < G2_BK / 16; ++kk)
                        ptx::mma_bf16_ss_2sm(d_tmem, adesc + (uint64_t)((kk * 32) >> 4), bdesc + (uint64_t)((kk * p.b_kstep) >> 4),
                                             idesc, (kb | kk) != 0);
                    ptx::mma_commit_2sm(empty0 + 8 * s);             // stage free in both CTAs once these MMAs retire
                }
                ptx::mma_commit_2sm(tfull0 + 8 * acc);               // accumulators complete in both CTAs
            }
        }
    } else if (warp >= 4) {
        // ===== epilogue (both CTAs): own 128 rows, TMEM -> registers -> bf16 -> global =====
        const int ew = warp & 3;                                      // TMEM lanes 32*ew .. 32*ew+31
        uint32_t tcount = 0;
        for (int t = pair; t < ntiles; t += npairs, ++tcount) {
            const int tm = t % p.tiles_m, tn = t / p.tiles_m;
            const uint32_t acc = tcount & 1, aph = (tcount >> 1) & 1;
            ptx::mbar_wait(tfull0 + 8 * acc, aph);
            ptx::tc_fence_after();
            const int row = tm * (2 * G2_BM) + (int)rank * G2_BM + ew * 32 + lane;
            const bool row_ok = row < p.m;
            uint16_t *crow = p.c + (int64_t)row * p.ldc + (int64_t)tn * G2_BN;
            const int ncols = p.n - tn * G2_BN;                       // valid columns in this tile (may exceed 256)
            const uint32_t taddr = tmem_base + acc * G2_BN + ((uint32_t)(ew * 32) << 16);
#pragma unroll 1
            for (int cb = 0; cb < G2_BN / 32; ++cb) {
                uint32_t r[32];
                ptx::tmem_ld_32x32b_x32(taddr + cb * 32, r);
                ptx::tmem_ld_wait();
                if (cb == G2_BN / 32 - 1) {                           // all TMEM reads of this tile are done
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive_cluster(tempty0 + 8 * acc, 0);
                }
                if (row_ok) {
#pragma unroll
                    for (int g = 0; g < 4; ++g) {                     // 8 columns = 16 bytes per store
                        const int col = cb * 32 + g * 8;
                        uint4 v;
                        v.x = ptx::pack_bf16x2(__uint_as_float(r[g * 8 + 0]), __uint_as_float(r[g * 8 + 1]));
                        v.y = ptx::pack_bf16x2(__uint_as_float(r[g * 8 + 2]), __uint_as_float(r[g * 8 + 3]));
                        v.z = ptx::pack_bf16x2(__uint_as_float(r[g * 8 + 4]), __uint_as_float(r[g * 8 + 5]));
                        v.w = ptx::pack_bf16x2(__uint_as_float(r[g * 8 + 6]), __uint_as_float(r[g * 8 + 7]));
                        if (col + 8 <= ncols) {
                            *reinterpret_cast<uint4 *>(crow + col) = v;
                        } else if (col < ncols) {
                            const uint32_t w4[4] = {v.x, v.y, v.z, v.w};
                            for (int e = 0; e < 8 && col + e < ncols; ++e)
                                crow[col + e] = (uint16_t)(w4[e >> 1] >> ((e & 1) * 16));
                        }
                    }
                }
            }
        }
    }

    // Neither CTA may exit (or free TMEM) while the other can still read its shared memory or signal its barriers.
    ptx::tc_fence_before();
    __syncthreads();
    ptx::cluster_sync();
    if (warp == 2) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc_2sm(tmem_base, G2_TMEM_COLS);
    }
}

int launch_gemm_2sm(const CUtensorMap &amap, const CUtensorMap &wmap, const GemmParams &p, int sm_count, cudaStream_t s)
{
    static int attr_gen = -1;                     // per-device function attribute: redo after tri_init() moved to another device
    if (attr_gen != device_generation()) {
        TRI_CUDA(cudaFuncSetAttribute(gemm_2sm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, G2_SMEM_BYTES));
        attr_gen = device_generation();
    }
    const int ntiles = p.tiles_m * p.tiles_n;
    const int pairs = ntiles < sm_count / 2 ? ntiles : sm_count / 2;
    gemm_2sm_kernel<<<2 * pairs, G2_THREADS, G2_SMEM_BYTES, s>>>(amap, wmap, p);
    TRI_CUDA(cudaGetLastError());
    return TRI_OK;
}

}  // namespace tri
