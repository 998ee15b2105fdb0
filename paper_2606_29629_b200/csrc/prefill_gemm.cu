// a3. Prefill-phase GEMM ("dense GEMM kernels"; BASELINE.json config 4; ABI in
// include/triroof.h):   C[m][n] = bf16_rne( sum_k A[m][k] * W[k][n] ),  fp32 accumulation in TMEM.
//
// The only tensor-core path of the library (a dense contraction).  Persistent, warp-specialised
// tcgen05 kernel, one CTA per SM:
//   warp 0   TMA producer   one elected lane: cp.async.bulk.tensor loads of the A tile (128 x 64) and the
//                           W tile (256 x 64) into a 4-stage ring (48 KiB per stage, 128-byte swizzle),
//                           completion on the stage's "full" mbarrier
//   warp 1   MMA issuer     one elected lane: per 64-wide k-block four tcgen05.mma.kind::f16
//                           (M 128, N 256, K 16) accumulating fp32 in tensor memory; tcgen05.commit
//                           releases the stage ("empty") and, after the last k-block, publishes the
//                           accumulator ("tmem_full")
//   warp 2   TMEM owner     allocates all 512 columns = two 128 x 256 fp32 accumulators, so the epilogue
//                           of tile t overlaps the main loop of tile t+1
//   warps 4-7 epilogue      tcgen05.ld (lane = row, 32 columns at a time) -> cvt.rn.bf16x2 -> 16-byte
//                           global stores; releases the accumulator ("tmem_empty")
// Tile order: tile = blockIdx.x + i * gridDim.x with the M index fastest, so the CTAs of a wave share
// W panels through L2 while A (29 MB) stays L2 resident.  4096 x 18944 gives 32 x 74 = 2368 tiles =
// 148 SMs x 16: no wave quantisation.  Ragged M / N / K: TMA zero-fills out-of-bounds reads; stores clip.
//
// W layouts: TRI_W_NK is the K-major B operand (canonical).  TRI_W_KN is the MN-major B operand: the
// W tile is loaded as four 64(n) x 64(k) boxes and described to the MMA with the MN-major descriptor.
#include "tri_internal.h"
#include "ptx.cuh"
#include "gemm_common.cuh"

#include <cstdlib>

namespace tri {

constexpr int GM_BM = 128, GM_BN = 256, GM_BK = 64;
constexpr int GM_STAGES = 4;
constexpr int GM_A_BYTES = GM_BM * GM_BK * 2;      // 16 KiB
constexpr int GM_B_BYTES = GM_BN * GM_BK * 2;      // 32 KiB
constexpr int GM_STAGE_BYTES = GM_A_BYTES + GM_B_BYTES;
constexpr int GM_THREADS = 256;
constexpr int GM_TMEM_COLS = 512;
constexpr int GM_SMEM_BYTES = 1024 + GM_STAGES * GM_STAGE_BYTES + 256;

__global__ void __launch_bounds__(GM_THREADS, 1)
gemm_kernel(const __grid_constant__ CUtensorMap amap, const __grid_constant__ CUtensorMap wmap, const GemmParams p)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t ring = ptx::smem_u32(smem);
    const uint32_t bars = ring + GM_STAGES * GM_STAGE_BYTES;
    const uint32_t full0 = bars, empty0 = bars + 8 * GM_STAGES;
    const uint32_t tfull0 = bars + 16 * GM_STAGES, tempty0 = tfull0 + 16;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + GM_STAGES * GM_STAGE_BYTES + 16 * GM_STAGES + 32);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ntiles = p.tiles_m * p.tiles_n;

    if (threadIdx.x == 0) {
        for (int s = 0; s < GM_STAGES; ++s) {
            ptx::mbar_init(full0 + 8 * s, 1);
            ptx::mbar_init(empty0 + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            ptx::mbar_init(tfull0 + 8 * a, 1);
            ptx::mbar_init(tempty0 + 8 * a, 4);      // one arrival per epilogue warp
        }
        ptx::fence_mbar_init();
    }
    if (warp == 2) {
        ptx::tmem_alloc(ptx::smem_u32(tmem_slot), GM_TMEM_COLS);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===== TMA producer =====
        if (ptx::elect_one()) {
            ptx::prefetch_tmap(&amap);
            ptx::prefetch_tmap(&wmap);
            const uint64_t pol_w = ptx::policy_evict_first();
            const uint64_t pol_a = ptx::policy_evict_last();
            uint32_t it = 0;
            for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
                const int tm = t % p.tiles_m, tn = t / p.tiles_m;
                for (int kb = 0; kb < p.kblocks; ++kb, ++it) {
                    const uint32_t s = it % GM_STAGES, ph = (it / GM_STAGES) & 1;
                    ptx::mbar_wait(empty0 + 8 * s, ph ^ 1);
                    const uint32_t fb = full0 + 8 * s;
                    ptx::mbar_arrive_expect_tx(fb, GM_STAGE_BYTES);
                    const uint32_t sa = ring + s * GM_STAGE_BYTES, sb = sa + GM_A_BYTES;
                    ptx::tma_load_2d_hint(sa, &amap, kb * GM_BK, tm * GM_BM, fb, pol_a);
                    if (!p.b_mn_major) {
                        ptx::tma_load_2d_hint(sb, &wmap, kb * GM_BK, tn * GM_BN, fb, pol_w);
                    } else {
#pragma unroll
                        for (int q = 0; q < 4; ++q)   // four 64(n) x 64(k) boxes, 8 KiB each
                            ptx::tma_load_2d_hint(sb + q * 8192, &wmap, tn * GM_BN + q * 64, kb * GM_BK, fb, pol_w);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer =====
        if (ptx::elect_one()) {
            const uint32_t idesc = make_idesc(GM_BM, GM_BN, p.b_mn_major);
            uint32_t it = 0, tcount = 0;
            for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++tcount) {
                const uint32_t acc = tcount & 1, aph = (tcount >> 1) & 1;
                ptx::mbar_wait(tempty0 + 8 * acc, aph ^ 1);          // epilogue has drained this accumulator
                ptx::tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * GM_BN;
                for (int kb = 0; kb < p.kblocks; ++kb, ++it) {
                    const uint32_t s = it % GM_STAGES, ph = (it / GM_STAGES) & 1;
                    ptx::mbar_wait(full0 + 8 * s, ph);
                    ptx::tc_fence_after();
                    const uint32_t sa = ring + s * GM_STAGE_BYTES, sb = sa + GM_A_BYTES;
                    const uint64_t adesc = make_sdesc(sa, 16, 1024);
                    const uint64_t bdesc = make_sdesc(sb, p.b_lbo, p.b_sbo);
#pragma unroll
                    for (int kk = 0; kk < GM_BK / 16; ++kk)
                        ptx::mma_bf16_ss(d_tmem, adesc + (uint64_t)((kk * 32) >> 4), bdesc + (uint64_t)((kk * p.b_kstep) >> 4),
                                         idesc, (kb | kk) != 0);
                    ptx::mma_commit(empty0 + 8 * s);                 // stage free once these MMAs retire
                }
                ptx::mma_commit(tfull0 + 8 * acc);                   // accumulator complete
            }
        }
    } else if (warp >= 4) {
        // ===== epilogue: TMEM -> registers -> bf16 -> global =====
        const int ew = warp & 3;                                      // TMEM lanes 32*ew .. 32*ew+31
        uint32_t tcount = 0;
        for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++tcount) {
            const int tm = t % p.tiles_m, tn = t / p.tiles_m;
            const uint32_t acc = tcount & 1, aph = (tcount >> 1) & 1;
            ptx::mbar_wait(tfull0 + 8 * acc, aph);
            ptx::tc_fence_after();
            const int row = tm * GM_BM + ew * 32 + lane;
            const bool row_ok = row < p.m;
            uint16_t *crow = p.c + (int64_t)row * p.ldc + (int64_t)tn * GM_BN;
            const int ncols = p.n - tn * GM_BN;                       // valid columns in this tile (may exceed 256)
            const uint32_t taddr = tmem_base + acc * GM_BN + ((uint32_t)(ew * 32) << 16);
#pragma unroll 1
            for (int cb = 0; cb < GM_BN / 32; ++cb) {
                uint32_t r[32];
                ptx::tmem_ld_32x32b_x32(taddr + cb * 32, r);
                ptx::tmem_ld_wait();
                if (cb == GM_BN / 32 - 1) {                           // all TMEM reads of this tile are done
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(tempty0 + 8 * acc);
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

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, GM_TMEM_COLS);
    }
}

static int gemm_impl(int m, int n, int k, const uint16_t *a, int64_t lda, const uint16_t *w, int64_t ldw, int w_layout,
                     uint16_t *c, int64_t ldc, void *stream)
{
    if (!a || !w || !c) return fail(TRI_ERR_INVALID_ARG, "a/w/c is NULL");
    if (m < 1 || n < 1 || k < 1) return fail(TRI_ERR_INVALID_ARG, "m = %d, n = %d, k = %d must be positive", m, n, k);
    if (w_layout != TRI_W_NK && w_layout != TRI_W_KN) return fail(TRI_ERR_INVALID_ARG, "w_layout = %d", w_layout);
    if (k % 8 != 0) return fail(TRI_ERR_UNSUPPORTED_SHAPE, "k = %d must be a multiple of 8", k);
    if (lda < k || ldc < n) return fail(TRI_ERR_INVALID_ARG, "lda = %lld < k or ldc = %lld < n", (long long)lda, (long long)ldc);
    if (ldw < (w_layout == TRI_W_NK ? k : n)) return fail(TRI_ERR_INVALID_ARG, "ldw = %lld too small", (long long)ldw);
    if (lda % 8 != 0 || ldw % 8 != 0 || ldc % 8 != 0) return fail(TRI_ERR_ALIGNMENT, "lda, ldw, ldc must be multiples of 8 elements");
    if (!aligned(a, 16) || !aligned(w, 16) || !aligned(c, 16)) return fail(TRI_ERR_ALIGNMENT, "a, w, c must be 16-byte aligned");
    {
        const uintptr_t c0 = (uintptr_t)c, c1 = c0 + ((size_t)(m - 1) * ldc + n) * 2;
        const uintptr_t a0 = (uintptr_t)a, a1 = a0 + ((size_t)(m - 1) * lda + k) * 2;
        const size_t wrows = w_layout == TRI_W_NK ? n : k, wcols = w_layout == TRI_W_NK ? k : n;
        const uintptr_t w0 = (uintptr_t)w, w1 = w0 + ((wrows - 1) * (size_t)ldw + wcols) * 2;
        if ((c0 < a1 && a0 < c1) || (c0 < w1 && w0 < c1)) return fail(TRI_ERR_INVALID_ARG, "c aliases an input");
    }
    const DeviceInfo *di = nullptr;
    int st = ensure_init(&di);
    if (st != TRI_OK) return st;

    // Default: the CTA-pair kernel (prefill_gemm_2sm.cu).  TRI_GEMM_1SM=1 (debug / A-B comparison) keeps the one-CTA kernel.
    static int one_sm = -1;
    if (one_sm < 0) { const char *e = getenv("TRI_GEMM_1SM"); one_sm = e ? atoi(e) : 0; }
    const int bn_box = one_sm ? GM_BN : GM_BN / 2;            // W columns staged per CTA
    const int rows_per_tile = one_sm ? GM_BM : 2 * GM_BM;

    CUtensorMap amap, wmap;
    st = make_tmap_2d_bf16(&amap, a, (uint64_t)k, (uint64_t)m, (uint64_t)lda * 2, GM_BK, GM_BM, CU_TENSOR_MAP_SWIZZLE_128B);
    if (st != TRI_OK) return st;
    GemmParams p;
    p.m = m; p.n = n; p.k = k;
    p.tiles_m = (m + rows_per_tile - 1) / rows_per_tile;
    p.tiles_n = (n + GM_BN - 1) / GM_BN;
    p.kblocks = (k + GM_BK - 1) / GM_BK;
    p.ldc = ldc;
    p.c = c;
    {
        static int wpol = -1;                               // debug only: TRI_GEMM_WPOL in {0, 1, 2}
        if (wpol < 0) { const char *e = getenv("TRI_GEMM_WPOL"); wpol = e ? atoi(e) : 2; }      // measured on config 4: evict-last 1.392 PFLOP/s sustained, evict-first 1.374
        p.w_policy = wpol;
    }
    if (w_layout == TRI_W_NK) {
        st = make_tmap_2d_bf16(&wmap, w, (uint64_t)k, (uint64_t)n, (uint64_t)ldw * 2, GM_BK, bn_box, CU_TENSOR_MAP_SWIZZLE_128B);
        p.b_mn_major = 0;
        p.b_lbo = 16; p.b_sbo = 1024; p.b_kstep = 32;     // 8-row groups 1024 B apart; 16 k-values = 32 B
    } else {
        st = make_tmap_2d_bf16(&wmap, w, (uint64_t)n, (uint64_t)k, (uint64_t)ldw * 2, 64, GM_BK, CU_TENSOR_MAP_SWIZZLE_128B);
        p.b_mn_major = 1;
        // MN-major, 128-byte swizzle: a 64(n) x 64(k) box is 64 k-rows of 128 B (8 KiB); 8-k groups are
        // 1024 B apart (stride), the next 64 columns of n start 8192 B later (leading); 16 k-values = 2048 B.
        p.b_lbo = 8192; p.b_sbo = 1024; p.b_kstep = 2048;
    }
    if (st != TRI_OK) return st;
    if (!one_sm) return launch_gemm_2sm(amap, wmap, p, di->sm_count, static_cast<cudaStream_t>(stream));

    static int attr_gen = -1;                     // per-device function attribute: redo after tri_init() moved to another device
    if (attr_gen != device_generation()) {
        TRI_CUDA(cudaFuncSetAttribute(gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GM_SMEM_BYTES));
        attr_gen = device_generation();
    }
    const int ntiles = p.tiles_m * p.tiles_n;
    const int grid = ntiles < di->sm_count ? ntiles : di->sm_count;
    gemm_kernel<<<grid, GM_THREADS, GM_SMEM_BYTES, static_cast<cudaStream_t>(stream)>>>(amap, wmap, p);
    TRI_CUDA(cudaGetLastError());
    return TRI_OK;
}

}  // namespace tri

extern "C" int prefill_gemm(int m, int n, int k, const uint16_t *a, int64_t lda, const uint16_t *w, int64_t ldw,
                            int w_layout, uint16_t *c, int64_t ldc, void *stream)
{
    return tri::gemm_impl(m, n, k, a, lda, w, ldw, w_layout, c, ldc, stream);
}
