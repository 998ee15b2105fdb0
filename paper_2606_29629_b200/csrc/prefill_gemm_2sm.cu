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
//   warps 4-7 epilogue      tcgen05.ld of the CTA's own 128 rows -> bf16 RNE -> swizzled shared-memory boxes -> TMA
//                           stores (32 rows x 64 columns each); arrive on the LEADER's "tmem_empty" (8 arrivals)
// 4096 x 18944 gives 16 x 74 = 1184 pair tiles = 74 TPCs x 16: no wave quantisation.  M index fastest inside row-block
// groups (tile_coords).  Ragged M / N / K: TMA zero fill on loads, TMA clipping on stores (the last n % 8 columns are
// stored from registers).
//
// Tail split (gemm_common.cuh next_work): when the tile count is not a multiple of the 74 pairs, the leftover tiles of
// the last round are cut along K into `parts` = 74 / leftover ranges, one per pair, all aligned in time like the whole
// rounds before them (so the L2 reuse of A and W panels across pairs is untouched, which a general stream-K schedule
// would lose).  Each pair writes its fp32 partial tile to a workspace slot of its own; splitk_reduce_kernel, launched
// behind this kernel with programmatic stream serialization, adds the parts in a fixed order (deterministic), rounds to
// bf16 and stores.  (Adding the partials with red.global.add.v4.f32 instead was measured: 1.2 M contended vector atomics
// on two tiles cost ~45 us.)  Down-projection 4096 x 3584 x 18944: 224 tiles = 3 rounds + 2 tiles x 37 parts of 8
// k-blocks instead of a fourth round.
#include "tri_internal.h"
#include "ptx.cuh"
#include "gemm_common.cuh"

#include <atomic>

namespace tri {

constexpr int G2_BM = 128, G2_BN = 256, G2_BK = 64;      // per CTA: 128 rows x 256 columns of C; pair: 256 x 256
constexpr int G2_BNH = G2_BN / 2;                         // W columns staged per CTA
constexpr int G2_STAGES = 6;
constexpr int G2_A_BYTES = G2_BM * G2_BK * 2;             // 16 KiB
constexpr int G2_B_BYTES = G2_BNH * G2_BK * 2;            // 16 KiB
constexpr int G2_STAGE_BYTES = G2_A_BYTES + G2_B_BYTES;
constexpr int G2_THREADS = 256;
constexpr int G2_TMEM_COLS = 512;
constexpr int G2_OUT_BYTES = 4 * 2 * 4096;                 // epilogue staging: per warp two 32-row x 64-column bf16 boxes
constexpr int G2_SMEM_BYTES = 1024 + G2_STAGES * G2_STAGE_BYTES + G2_OUT_BYTES + 256;

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(G2_THREADS, 1)
gemm_2sm_kernel(const __grid_constant__ CUtensorMap amap, const __grid_constant__ CUtensorMap wmap,
                const __grid_constant__ CUtensorMap cmap, const GemmParams p)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t ring = ptx::smem_u32(smem);
    const uint32_t outbuf = ring + G2_STAGES * G2_STAGE_BYTES;        // 1 KiB aligned: 128-byte swizzle atoms
    const uint32_t bars = outbuf + G2_OUT_BYTES;
    const uint32_t full0 = bars, empty0 = bars + 8 * G2_STAGES;
    const uint32_t tfull0 = bars + 16 * G2_STAGES, tempty0 = tfull0 + 16;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + G2_STAGES * G2_STAGE_BYTES + G2_OUT_BYTES + 16 * G2_STAGES + 32);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();
    const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;
    const int ntiles = p.tiles_m * p.tiles_n;             // pair tiles (tiles_m counts 256-row blocks)

    // Programmatic dependent launch: the next kernel of the stream (splitk_reduce_kernel when this call is split, else the next
    // call's kernel) may set itself up as SMs free up; it orders itself with griddepcontrol.wait, as this one does below.
    ptx::pdl_launch_dependents();
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
            // a W panel is read by the 16 pairs that share its tn within one wave: it must survive in L2 until the last of
            // them has passed (evict-first lets it go early: 304 MB of DRAM reads per call instead of the 165 MB of A + W);
            // measured on config 4, sustained: evict-first 1.374, evict-normal 1.371, evict-last 1.392 PFLOP/s
            const uint64_t pol_w = ptx::policy_evict_last();
            const uint64_t pol_a = ptx::policy_evict_last();
            uint32_t it = 0;
            GemmWork wk;
            ptx::pdl_wait();                                          // A may be the output of the grid before this one
            for (int i = 0; next_work(p, ntiles, pair, npairs, i, wk); ++i) {
                int tm, tn;
                tile_coords(p, wk.tile, tm, tn);
                const int row0 = tm * (2 * G2_BM) + (int)rank * G2_BM, col0 = tn * G2_BN + (int)rank * G2_BNH;
                for (int kb = wk.kb0; kb < wk.kb1; ++kb, ++it) {
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
            GemmWork wk;
            for (int i = 0; next_work(p, ntiles, pair, npairs, i, wk); ++i, ++tcount) {
                const uint32_t acc = tcount & 1, aph = (tcount >> 1) & 1;
                ptx::mbar_wait(tempty0 + 8 * acc, aph ^ 1);          // both epilogues have drained this accumulator
                ptx::tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * G2_BN;
                for (int kb = wk.kb0; kb < wk.kb1; ++kb, ++it) {
                    const uint32_t s = it % G2_STAGES, ph = (it / G2_STAGES) & 1;
                    ptx::mbar_wait(full0 + 8 * s, ph);
                    ptx::tc_fence_after();
                    const uint32_t sa = ring + s * G2_STAGE_BYTES, sb = sa + G2_A_BYTES;
                    const uint64_t adesc = make_sdesc(sa, 16, 1024);
                    const uint64_t bdesc = make_sdesc(sb, p.b_lbo, p.b_sbo);
#pragma unroll
                    for (int kk = 0; kk < G2_BK / 16; ++kk)
                        ptx::mma_bf16_ss_2sm(d_tmem, adesc + (uint64_t)((kk * 32) >> 4), bdesc + (uint64_t)((kk * p.b_kstep) >> 4),
                                             idesc, (kb > wk.kb0) | (kk != 0));
                    ptx::mma_commit_2sm(empty0 + 8 * s);             // stage free in both CTAs once these MMAs retire
                }
                ptx::mma_commit_2sm(tfull0 + 8 * acc);               // accumulators complete in both CTAs
            }
        }
    } else if (warp >= 4) {
        // ===== epilogue (both CTAs): own 128 rows, TMEM -> registers -> bf16 -> shared memory -> TMA store =====
        // A warp owns 32 rows.  Per 64-column group it packs its 32 x 64 bf16 box into one of its two 4 KiB staging
        // buffers (row = 128 bytes, 16-byte chunks XOR-swizzled by row so the 8 lanes of a quarter-warp hit 8 bank
        // groups) and one lane hands the box to TMA (cp.async.bulk.tensor store, 128-byte swizzle undone by the
        // tensor map): full 128-byte lines to L2 instead of 32 half-sector writes per store instruction, ragged
        // M / N clipped by TMA, and the warp is free again while the store drains.
        const int ew = warp & 3;                                      // TMEM lanes 32*ew .. 32*ew+31
        const uint32_t stage0 = outbuf + ew * 8192;
        uint32_t tcount = 0, sb = 0;
        if (lane == 0) ptx::prefetch_tmap(&cmap);
        ptx::pdl_wait();                                              // C / the workspace may still be in use by the grid before
        const uint64_t pol_c = ptx::policy_evict_first();
        GemmWork wk;
        for (int i = 0; next_work(p, ntiles, pair, npairs, i, wk); ++i, ++tcount) {
            int tm, tn;
            tile_coords(p, wk.tile, tm, tn);
            const uint32_t acc = tcount & 1, aph = (tcount >> 1) & 1;
            ptx::mbar_wait(tfull0 + 8 * acc, aph);
            ptx::tc_fence_after();
            const int row0 = tm * (2 * G2_BM) + (int)rank * G2_BM + ew * 32;
            const uint32_t taddr = tmem_base + acc * G2_BN + ((uint32_t)(ew * 32) << 16);
            if (wk.split >= 0) {
                // split tile: this warp's 32 x 256 slice of the pair's partial sums goes to the workspace, nothing to C
                float *slice = p.ws + ((size_t)(wk.split * p.parts + wk.part) * 8 + (size_t)rank * 4 + ew) * (32 * G2_BN);
#pragma unroll 1
                for (int blk = 0; blk < G2_BN / 32; ++blk) {
                    uint32_t r[32];
                    ptx::tmem_ld_32x32b_x32(taddr + blk * 32, r);
                    ptx::tmem_ld_wait();
                    splitk_put(slice, blk, lane, r);
                }
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_cluster(tempty0 + 8 * acc, 0);
                continue;
            }
#pragma unroll 1
            for (int g = 0; g < G2_BN / 64; ++g, sb ^= 1) {
                const uint32_t buf = stage0 + sb * 4096;
                if (lane == 0) ptx::tma_store_wait_read<1>();         // the store that last read this buffer is done with it
                __syncwarp();
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    uint32_t r[32];
                    ptx::tmem_ld_32x32b_x32(taddr + g * 64 + h * 32, r);
                    ptx::tmem_ld_wait();
                    if (g == G2_BN / 64 - 1 && h == 1) {              // all TMEM reads of this tile are done
                        ptx::tc_fence_before();
                        __syncwarp();
                        if (lane == 0) ptx::mbar_arrive_cluster(tempty0 + 8 * acc, 0);
                    }
                    {   // TMA clips a partial box only at 16-byte granularity (measured: a box cut at column 257 also zeroes
                        // columns 257..263), so the tensor map ends at n rounded down to 8 columns and the last n % 8 columns
                        // are stored from registers here
                        const int cbase = tn * G2_BN + g * 64 + h * 32, n8 = p.n & ~7, row = row0 + lane;
                        if (cbase + 32 > n8 && cbase < p.n && row < p.m) {
#pragma unroll
                            for (int j = 0; j < 32; ++j)
                                if (cbase + j >= n8 && cbase + j < p.n)
                                    p.c[(int64_t)row * p.ldc + cbase + j] = (uint16_t)(ptx::pack_bf16x2(__uint_as_float(r[j]), 0.f) & 0xffffu);
                        }
                    }
#pragma unroll
                    for (int q = 0; q < 4; ++q) {                     // 8 columns = one 16-byte chunk
                        const uint32_t v0 = ptx::pack_bf16x2(__uint_as_float(r[q * 8 + 0]), __uint_as_float(r[q * 8 + 1]));
                        const uint32_t v1 = ptx::pack_bf16x2(__uint_as_float(r[q * 8 + 2]), __uint_as_float(r[q * 8 + 3]));
                        const uint32_t v2 = ptx::pack_bf16x2(__uint_as_float(r[q * 8 + 4]), __uint_as_float(r[q * 8 + 5]));
                        const uint32_t v3 = ptx::pack_bf16x2(__uint_as_float(r[q * 8 + 6]), __uint_as_float(r[q * 8 + 7]));
                        const uint32_t dst = buf + (uint32_t)lane * 128u + (uint32_t)(((h * 4 + q) ^ (lane & 7)) << 4);
                        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(dst), "r"(v0), "r"(v1), "r"(v2), "r"(v3) : "memory");
                    }
                }
                ptx::fence_proxy_async_smem();                        // generic-proxy writes visible to the TMA engine
                __syncwarp();
                if (lane == 0) {
                    if (row0 < p.m && tn * G2_BN + g * 64 < (p.n & ~7)) ptx::tma_store_2d_hint(&cmap, buf, tn * G2_BN + g * 64, row0, pol_c);
                    // one bulk group per buffer toggle, also when nothing was stored (an empty group is legal): wait_read<1>
                    // above counts groups, and must mean "the store before the previous one" for the buffer it guards
                    ptx::tma_store_commit();
                }
            }
        }
        if (lane == 0) ptx::tma_store_wait<0>();                      // all of this warp's stores have landed
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
    CUtensorMap cmap;     // C as 64-column x 32-row boxes for the epilogue's TMA stores (out-of-range rows / columns are clipped)
    const int n8 = p.n & ~7;     // see the epilogue: the last n % 8 columns do not go through TMA
    int st = cached_tmap_2d_bf16(&cmap, p.c, (uint64_t)(n8 ? n8 : 8), (uint64_t)p.m, (uint64_t)p.ldc * 2, 64, 32, CU_TENSOR_MAP_SWIZZLE_128B);
    if (st != TRI_OK) return st;
    static std::atomic<int> attr_gen{-1};         // per-device function attribute: redo after tri_init() moved to another device
    if (attr_gen.load(std::memory_order_acquire) != device_generation()) {
        TRI_CUDA(cudaFuncSetAttribute(gemm_2sm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, G2_SMEM_BYTES));
        attr_gen.store(device_generation(), std::memory_order_release);
    }
    const int ntiles = p.tiles_m * p.tiles_n, max_pairs = sm_count / 2;
    GemmParams q = p;
    {   // rows of A kept resident: about 32 MB worth of 256-row panels, at least 4, all of them when A is small
        const double panel = 256.0 * p.k * 2.0;
        int g = (int)(32.0e6 / panel);
        g = g < 4 ? 4 : g;
        q.group_m = g < p.tiles_m ? g : p.tiles_m;
    }
    // Tail split: the leftover tiles of the last round, each cut into `parts` k-ranges (one per pair).  Worth it when the
    // time saved, (1 - 1/parts) of a tile = of kblocks k-blocks, clearly exceeds the fixed cost of writing a 256 x 256 fp32
    // partial per pair and the reduction kernel behind (a few microseconds = a few k-blocks' worth).
    const int left = ntiles % max_pairs;
    int parts = left ? max_pairs / left : 1;
    if (parts > p.kblocks / 8) parts = p.kblocks / 8;             // at least 8 k-blocks per part (4096 x 3584 x 3584: 7 parts 72 us, 37 parts 76 us, none 78 us)
    q.full_tiles = ntiles;
    q.parts = 1;
    q.ws = nullptr;
    int pairs = ntiles < max_pairs ? ntiles : max_pairs;
    if (parts >= 2 && (parts - 1) * p.kblocks >= 24 * parts) {
        q.full_tiles = ntiles - left;
        q.parts = parts;
        st = splitk_workspace(s, (size_t)left * parts * (2 * G2_BM) * G2_BN * sizeof(float), &q.ws);
        if (st != TRI_OK) return st;
        if (q.full_tiles == 0) pairs = left * parts;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2 * pairs);
    cfg.blockDim = dim3(G2_THREADS);
    cfg.dynamicSmemBytes = G2_SMEM_BYTES;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl_allowed();
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    TRI_CUDA(cudaLaunchKernelEx(&cfg, gemm_2sm_kernel, amap, wmap, cmap, q));
    if (q.parts > 1) return launch_splitk_reduce(q, 2 * G2_BM, G2_BN, true, s);
    return TRI_OK;
}

}  // namespace tri
