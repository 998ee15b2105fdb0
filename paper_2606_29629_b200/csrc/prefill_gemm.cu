// a3. Prefill-phase GEMM ("dense GEMM kernels"; BASELINE.json config 4; ABI in
// include/triroof.h):   C[m][n] = bf16_rne( sum_k A[m][k] * W[k][n] ),  fp32 accumulation in TMEM.
//
// The only tcgen05 path of the library (a dense contraction).  This file holds the entry point, its dispatch, and the
// one-CTA kernel used when A has at most 128 rows; m > 128 goes to the CTA-pair kernel of prefill_gemm_2sm.cu (256 x 256
// pair tiles), which a short A would leave three quarters empty.
//
// One-CTA kernel (32 < m <= 128: chunked-prefill tails, speculative / large-batch decode; m <= 32 goes to the GEMV): weight-streaming bound, so the
// tile is 128 x 128 — 148 tiles for n = 18944, one per SM — and when there are fewer tiles than SMs every tile is cut
// along K into `parts` ranges (gemm_common.cuh next_work / splitk_*) so that all SMs pull on HBM.  Warp roles as in the
// pair kernel: warp 0 TMA producer (A rows x 64 and W 128 x 64 per k-block into a 6- to 12-stage ring, 128-byte swizzle), warp 1
// MMA issuer (tcgen05.mma.cta_group::1.kind::f16, M 128, N 128, K 16), warp 2 TMEM owner (two 128-column accumulators),
// warps 4-7 epilogue (tcgen05.ld -> cvt.rn.bf16x2 -> 16-byte global stores; the output is small here).
// Ragged M / N / K: TMA zero-fills out-of-bounds reads; stores clip.
// Programmatic dependent launch, as in the GEMV: the kernel lets the next kernel of the stream start at once and orders
// itself with griddepcontrol.wait — the producer fetches a ring-full of W (model state) before the wait and A after it,
// the epilogue waits before its first store.  Back to back on m x 18944 x 3584: m = 16 / 64 / 128 26.9 / 26.7 / 27.5 us
// -> 23.7 / 23.9 / 25.3 us (cuBLAS 25.5 / 28.2 / 28.9).
//
// W layouts: TRI_W_NK is the K-major B operand (canonical).  TRI_W_KN is the MN-major B operand: the W tile is loaded
// as 64(n) x 64(k) boxes and described to the MMA with the MN-major descriptor.
#include "tri_internal.h"
#include "ptx.cuh"
#include "gemm_common.cuh"

#include <atomic>

#include <mutex>
#include <vector>

namespace tri {

constexpr int GM_BM = 128, GM_BN = 128, GM_BK = 64;
constexpr int GM_MAX_STAGES = 12;                  // ring depth is chosen per call: the A box shrinks with m, the ring grows
constexpr int GM_B_BYTES = GM_BN * GM_BK * 2;      // 16 KiB
constexpr int GM_THREADS = 256;
constexpr int GM_TMEM_COLS = 2 * GM_BN;
constexpr int GM_BAR_BYTES = 16 * GM_MAX_STAGES + 64;
constexpr int GM_SMEM_MAX = 220 * 1024;

__host__ __device__ constexpr int gm_smem_bytes(int stages, int stage_bytes) { return 1024 + stages * stage_bytes + GM_BAR_BYTES; }

__global__ void __launch_bounds__(GM_THREADS, 1)
gemm_1sm_kernel(const __grid_constant__ CUtensorMap amap, const __grid_constant__ CUtensorMap wmap, const GemmParams p)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const int GM_STAGES = p.stages, GM_STAGE_BYTES = p.a_box_bytes + GM_B_BYTES, GM_A_BYTES = p.a_box_bytes;   // per call (see gemm_impl)
    const uint32_t ring = ptx::smem_u32(smem);
    const uint32_t bars = ring + GM_STAGES * GM_STAGE_BYTES;
    const uint32_t full0 = bars, empty0 = bars + 8 * GM_MAX_STAGES;
    const uint32_t tfull0 = bars + 16 * GM_MAX_STAGES, tempty0 = tfull0 + 16;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + GM_STAGES * GM_STAGE_BYTES + 16 * GM_MAX_STAGES + 32);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ntiles = p.tiles_m * p.tiles_n, me = blockIdx.x, nw = gridDim.x;

    // Programmatic dependent launch: the next kernel of the stream (splitk_reduce_kernel when this call is split, else the
    // next call's kernel) may start its CTAs as soon as resources free up; it orders itself with griddepcontrol.wait.
    ptx::pdl_launch_dependents();
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
        // W (model state, never an output of the kernel before this one) is fetched at once for the first ring-full of
        // k-blocks; A is fetched only after griddepcontrol.wait, i.e. once the preceding grid has completed (header:
        // aliasing rule).  Then the steady loop.
        if (ptx::elect_one()) {
            ptx::prefetch_tmap(&amap);
            ptx::prefetch_tmap(&wmap);
            const uint64_t pol_w = ptx::policy_evict_first();        // every W element is read exactly once
            const uint64_t pol_a = ptx::policy_evict_last();         // A is re-read by every CTA
            auto load_w = [&](uint32_t sb, uint32_t fb, int tn, int kb) {
                if (!p.b_mn_major) {
                    ptx::tma_load_2d_hint(sb, &wmap, kb * GM_BK, tn * GM_BN, fb, pol_w);
                } else {
#pragma unroll
                    for (int q = 0; q < GM_BN / 64; ++q)   // 64(n) x 64(k) boxes, 8 KiB each
                        ptx::tma_load_2d_hint(sb + q * 8192, &wmap, tn * GM_BN + q * 64, kb * GM_BK, fb, pol_w);
                }
            };
            GemmWork wk;
            uint32_t it = 0;
            for (int i = 0; it < (uint32_t)GM_STAGES && next_work(p, ntiles, me, nw, i, wk); ++i)
                for (int kb = wk.kb0; kb < wk.kb1 && it < (uint32_t)GM_STAGES; ++kb, ++it) {
                    const uint32_t fb = full0 + 8 * it;
                    ptx::mbar_arrive_expect_tx(fb, GM_STAGE_BYTES);
                    load_w(ring + it * GM_STAGE_BYTES + GM_A_BYTES, fb, wk.tile / p.tiles_m, kb);
                }
            ptx::pdl_wait();
            it = 0;
            for (int i = 0; next_work(p, ntiles, me, nw, i, wk); ++i) {
                const int tm = wk.tile % p.tiles_m, tn = wk.tile / p.tiles_m;
                for (int kb = wk.kb0; kb < wk.kb1; ++kb, ++it) {
                    const uint32_t s = it % GM_STAGES, ph = (it / GM_STAGES) & 1;
                    const uint32_t fb = full0 + 8 * s;
                    const uint32_t sa = ring + s * GM_STAGE_BYTES, sb = sa + GM_A_BYTES;
                    if (it >= (uint32_t)GM_STAGES) {
                        ptx::mbar_wait(empty0 + 8 * s, ph ^ 1);
                        ptx::mbar_arrive_expect_tx(fb, GM_STAGE_BYTES);
                        load_w(sb, fb, tn, kb);
                    }
                    ptx::tma_load_2d_hint(sa, &amap, kb * GM_BK, tm * GM_BM, fb, pol_a);
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer =====
        if (ptx::elect_one()) {
            const uint32_t idesc = make_idesc(GM_BM, GM_BN, p.b_mn_major);
            uint32_t it = 0, tcount = 0;
            GemmWork wk;
            for (int i = 0; next_work(p, ntiles, me, nw, i, wk); ++i, ++tcount) {
                const uint32_t acc = tcount & 1, aph = (tcount >> 1) & 1;
                ptx::mbar_wait(tempty0 + 8 * acc, aph ^ 1);          // epilogue has drained this accumulator
                ptx::tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * GM_BN;
                for (int kb = wk.kb0; kb < wk.kb1; ++kb, ++it) {
                    const uint32_t s = it % GM_STAGES, ph = (it / GM_STAGES) & 1;
                    ptx::mbar_wait(full0 + 8 * s, ph);
                    ptx::tc_fence_after();
                    const uint32_t sa = ring + s * GM_STAGE_BYTES, sb = sa + GM_A_BYTES;
                    const uint64_t adesc = make_sdesc(sa, 16, 1024);
                    const uint64_t bdesc = make_sdesc(sb, p.b_lbo, p.b_sbo);
#pragma unroll
                    for (int kk = 0; kk < GM_BK / 16; ++kk)
                        ptx::mma_bf16_ss(d_tmem, adesc + (uint64_t)((kk * 32) >> 4), bdesc + (uint64_t)((kk * p.b_kstep) >> 4),
                                         idesc, (kb > wk.kb0) | (kk != 0));
                    ptx::mma_commit(empty0 + 8 * s);                 // stage free once these MMAs retire
                }
                ptx::mma_commit(tfull0 + 8 * acc);                   // accumulator complete
            }
        }
    } else if (warp >= 4) {
        // ===== epilogue: TMEM -> registers (-> split-K sum through L2) -> bf16 -> global =====
        const int ew = warp & 3;                                      // TMEM lanes 32*ew .. 32*ew+31
        uint32_t tcount = 0;
        GemmWork wk;
        ptx::pdl_wait();                                              // C / the workspace may still be in use by the preceding grid
        for (int i = 0; next_work(p, ntiles, me, nw, i, wk); ++i, ++tcount) {
            const int tm = wk.tile % p.tiles_m, tn = wk.tile / p.tiles_m;
            const uint32_t acc = tcount & 1, aph = (tcount >> 1) & 1;
            ptx::mbar_wait(tfull0 + 8 * acc, aph);
            ptx::tc_fence_after();
            const int row = tm * GM_BM + ew * 32 + lane;
            const bool row_ok = row < p.m;
            uint16_t *crow = p.c + (int64_t)row * p.ldc + (int64_t)tn * GM_BN;
            const int ncols = p.n - tn * GM_BN;                       // valid columns in this tile (may exceed 128)
            const uint32_t taddr = tmem_base + acc * GM_BN + ((uint32_t)(ew * 32) << 16);
            if (wk.split >= 0) {
                // split tile: this warp's 32 x 128 slice of the CTA's partial sums goes to the workspace, nothing to C
                float *slice = p.ws + ((size_t)(wk.split * p.parts + wk.part) * 4 + ew) * (32 * GM_BN);
#pragma unroll 1
                for (int cb = 0; cb < GM_BN / 32; ++cb) {
                    uint32_t r[32];
                    ptx::tmem_ld_32x32b_x32(taddr + cb * 32, r);
                    ptx::tmem_ld_wait();
                    splitk_put(slice, cb, lane, r);
                }
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(tempty0 + 8 * acc);
                continue;
            }
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

// ---- split-K: the sum of the parts ---------------------------------------------------------------------------------
// One thread per float4 of a split tile (fragment order, see splitk_put): adds the `parts` partials in ascending order
// (fixed: the result does not depend on which CTA finished first), rounds to bf16 and stores 4 outputs of one row.
__global__ void __launch_bounds__(256)
splitk_reduce_kernel(const GemmParams p, int tile_rows, int tile_cols, int pair_order)
{
    ptx::pdl_launch_dependents();                          // the next call may set itself up; it waits for this grid before touching C / ws
    ptx::pdl_wait();                                       // the GEMM kernel's partial tiles are complete and visible
    const int ntiles = p.tiles_m * p.tiles_n, nsplit = ntiles - p.full_tiles;
    const int tile4 = tile_rows * tile_cols / 4;           // float4 per tile
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= nsplit * tile4) return;
    const int st = idx / tile4, f = idx - st * tile4;
    const float4 *src = reinterpret_cast<const float4 *>(p.ws) + (size_t)st * p.parts * tile4 + f;
    float4 sum = make_float4(0.f, 0.f, 0.f, 0.f);
    int part = 0;
    for (; part + 4 <= p.parts; part += 4) {               // four loads in flight
        const float4 v0 = __ldcg(src + (size_t)part * tile4), v1 = __ldcg(src + (size_t)(part + 1) * tile4),
                     v2 = __ldcg(src + (size_t)(part + 2) * tile4), v3 = __ldcg(src + (size_t)(part + 3) * tile4);
        sum.x = ((((sum.x + v0.x) + v1.x) + v2.x) + v3.x);
        sum.y = ((((sum.y + v0.y) + v1.y) + v2.y) + v3.y);
        sum.z = ((((sum.z + v0.z) + v1.z) + v2.z) + v3.z);
        sum.w = ((((sum.w + v0.w) + v1.w) + v2.w) + v3.w);
    }
    for (; part < p.parts; ++part) {
        const float4 v = __ldcg(src + (size_t)part * tile4);
        sum.x += v.x; sum.y += v.y; sum.z += v.z; sum.w += v.w;
    }
    int tm, tn;
    const int t = p.full_tiles + st;
    if (pair_order) tile_coords(p, t, tm, tn);
    else { tm = t % p.tiles_m; tn = t / p.tiles_m; }
    const int slice4 = 8 * tile_cols;                      // float4 per 32-row slice
    const int slice = f / slice4, r = f - slice * slice4;
    const int blk = r >> 8, q = (r >> 5) & 7, lane = r & 31;
    const int row = tm * tile_rows + slice * 32 + lane, col = tn * tile_cols + blk * 32 + q * 4;
    if (row >= p.m || col >= p.n) return;
    uint16_t *dst = p.c + (int64_t)row * p.ldc + col;
    const uint32_t lo = ptx::pack_bf16x2(sum.x, sum.y), hi = ptx::pack_bf16x2(sum.z, sum.w);
    if (col + 4 <= p.n) {
        *reinterpret_cast<uint2 *>(dst) = make_uint2(lo, hi);       // ldc % 8 == 0 and col % 4 == 0: 8-byte aligned
    } else {
        const uint16_t e[4] = {(uint16_t)lo, (uint16_t)(lo >> 16), (uint16_t)hi, (uint16_t)(hi >> 16)};
        for (int c = 0; col + c < p.n; ++c) dst[c] = e[c];
    }
}

int launch_splitk_reduce(const GemmParams &p, int tile_rows, int tile_cols, bool pair_order, cudaStream_t s)
{
    const int nsplit = p.tiles_m * p.tiles_n - p.full_tiles;
    const long long threads = (long long)nsplit * tile_rows * tile_cols / 4;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)((threads + 255) / 256));
    cfg.blockDim = dim3(256);
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl_allowed();
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    TRI_CUDA(cudaLaunchKernelEx(&cfg, splitk_reduce_kernel, p, tile_rows, tile_cols, pair_order ? 1 : 0));
    return TRI_OK;
}

// ---- split-K workspace, one per stream (calls on one stream are ordered, so they can share it) ------------------------
struct SplitWs {
    int generation;
    cudaStream_t stream;
    float *ws;
    size_t ws_bytes;
};
static std::mutex g_ws_mu;
static std::vector<SplitWs> g_ws;

int splitk_workspace(cudaStream_t stream, size_t ws_bytes, float **ws)
{
    std::lock_guard<std::mutex> lk(g_ws_mu);
    SplitWs *e = nullptr;
    for (auto &x : g_ws)
        if (x.stream == stream && x.generation == device_generation()) e = &x;
    if (!e) {
        if (g_ws.size() >= 64) return fail(TRI_ERR_CUDA, "split-K workspaces for more than 64 streams");
        g_ws.push_back(SplitWs{device_generation(), stream, nullptr, 0});
        e = &g_ws.back();
    }
    if (e->ws_bytes < ws_bytes) {
        // grow: earlier calls on this stream may still be using the old buffer, so wait for the stream first
        TRI_CUDA(cudaStreamSynchronize(stream));
        if (e->ws) cudaFree(e->ws);
        e->ws = nullptr;
        e->ws_bytes = 0;
        // 74 pair tiles of 256 x 256 fp32 (the most left x parts can be) = 19.4 MB covers every shape of either kernel
        const size_t wb = ws_bytes < (size_t)(20u << 20) ? (size_t)(20u << 20) : ws_bytes;
        TRI_CUDA(cudaMalloc(&e->ws, wb));
        e->ws_bytes = wb;
    }
    *ws = e->ws;
    return TRI_OK;
}

void release_splitk_workspaces()
{
    std::lock_guard<std::mutex> lk(g_ws_mu);
    for (auto &x : g_ws)
        if (x.ws) cudaFree(x.ws);
    g_ws.clear();
}

static int launch_gemm_1sm(const CUtensorMap &amap, const CUtensorMap &wmap, const GemmParams &p, int sm_count, cudaStream_t s)
{
    static std::atomic<int> attr_gen{-1};         // per-device function attribute: redo after tri_init() moved to another device
    if (attr_gen.load(std::memory_order_acquire) != device_generation()) {
        TRI_CUDA(cudaFuncSetAttribute(gemm_1sm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GM_SMEM_MAX));
        attr_gen.store(device_generation(), std::memory_order_release);
    }
    GemmParams q = p;
    // Ring depth: as many stages as fit (a stage is the A box + 16 KiB of W).  The kernel is bound by the weight stream,
    // and what keeps HBM busy is bytes in flight per SM: 6 stages (m = 128) .. 12 stages (m <= 16: 192 KiB of W in flight).
    const int stage_bytes = p.a_box_bytes + GM_B_BYTES;
    // (Capping the ring at 112 KiB so that a CTA of the next call moves in beside this one was measured: m = 16 23.8 us
    // against 23.7 us, m = 64 26.6 against 23.9.  In-kernel %globaltimer stamps show why it cannot win: the early CTA fills
    // its ring with W and then sits in griddepcontrol.wait until the whole grid before it has completed, so what a call
    // costs is (1 - ring / panel) of the stream plus the same fixed part either way — A's L2 latency after the wait 0.9 us,
    // last MMA to exit 1.2 us, grid completion to the dependents' release 1.1 us, 3-5 us of skew between the SMs — and a
    // deeper ring in ONE CTA prefetches as much as two shallow ones.)
    q.stages = (GM_SMEM_MAX - 1024 - GM_BAR_BYTES) / stage_bytes;
    if (q.stages > GM_MAX_STAGES) q.stages = GM_MAX_STAGES;
    const int smem_bytes = gm_smem_bytes(q.stages, stage_bytes);
    const int ntiles = p.tiles_m * p.tiles_n;
    const int left = ntiles % sm_count;
    int parts = left ? sm_count / left : 1;
    if (parts > p.kblocks) parts = p.kblocks;
    q.full_tiles = ntiles;
    q.parts = 1;
    q.ws = nullptr;
    int grid = ntiles < sm_count ? ntiles : sm_count;
    if (parts >= 2 && (parts - 1) * p.kblocks >= 8 * parts) {        // the 128 x 128 fp32 partial is a quarter of the pair kernel's
        q.full_tiles = ntiles - left;
        q.parts = parts;
        int st = splitk_workspace(s, (size_t)left * parts * GM_BM * GM_BN * sizeof(float), &q.ws);
        if (st != TRI_OK) return st;
        if (q.full_tiles == 0) grid = left * parts;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(GM_THREADS);
    cfg.dynamicSmemBytes = smem_bytes;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl_allowed();
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    TRI_CUDA(cudaLaunchKernelEx(&cfg, gemm_1sm_kernel, amap, wmap, q));
    if (q.parts > 1) return launch_splitk_reduce(q, GM_BM, GM_BN, false, s);
    return TRI_OK;
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
    // At most 32 rows: the contraction is a weight stream with a sliver of arithmetic, and the streaming GEMV (two CTAs per
    // SM, warp-level MMA with the batch as 8-column tiles, no TMEM set-up, no epilogue to speak of, K-split clusters when
    // there are few columns) does it faster than the 128-row tcgen05 tile below.  Back to back, us, GEMV / one-CTA kernel:
    // 16 x 18944 x 3584 21.5 / 23.7, 32 x 18944 x 3584 22.5 / 23.5, 32 x 3584 x 18944 25.5 / 29.0.  Same definition, same
    // rounding; every argument rule of this entry point is at least as strict as the GEMV's.  (Beyond 32 rows the X
    // fragments cost more shared-memory bandwidth than the SM has: 2 x ldmatrix.x4 per batch tile and stage in every warp.)
    if (m <= 32) return gemv_impl(m, n, k, a, lda, w, ldw, w_layout, c, ldc, stream);

    const DeviceInfo *di = nullptr;
    int st = ensure_init(&di);
    if (st != TRI_OK) return st;

    // a short A: 128 x 128 tiles, one CTA each (see the file header).  (128 < m <= 256 on this kernel, two row blocks per
    // W panel, was measured: 36-37 us against 32-33 us for the pair kernel on m x 18944 x 3584.)
    const bool one_sm = m <= GM_BM;
    const int rows_per_tile = one_sm ? GM_BM : 2 * GM_BM;
    const int cols_per_tile = one_sm ? GM_BN : 2 * GM_BN;
    cudaStream_t s = static_cast<cudaStream_t>(stream);

    // Both kernels stage A as 128-row x 64-k boxes and W as 128 columns x 64 k per CTA (cached maps)
    // A box: 128 rows; for a short A only the rows that exist, rounded up to the 8-row swizzle atom (zero-filling 112
    // absent rows per box made m = 16 slower than m = 64; the MMA still reads 128 rows, and what it computes from the
    // stale rows lands in accumulator rows >= m, which are never stored)
    const int a_rows = one_sm ? ((m + 7) / 8) * 8 : GM_BM;
    CUtensorMap amap, wmap;
    st = cached_tmap_2d_bf16(&amap, a, (uint64_t)k, (uint64_t)m, (uint64_t)lda * 2, GM_BK, a_rows, CU_TENSOR_MAP_SWIZZLE_128B);
    if (st != TRI_OK) return st;
    GemmParams p = {};
    p.a_box_bytes = a_rows * GM_BK * 2;
    p.m = m; p.n = n; p.k = k;
    p.tiles_m = (m + rows_per_tile - 1) / rows_per_tile;
    p.tiles_n = (n + cols_per_tile - 1) / cols_per_tile;
    p.kblocks = (k + GM_BK - 1) / GM_BK;
    p.ldc = ldc;
    p.c = c;
    if (w_layout == TRI_W_NK) {
        st = cached_tmap_2d_bf16(&wmap, w, (uint64_t)k, (uint64_t)n, (uint64_t)ldw * 2, GM_BK, GM_BN, CU_TENSOR_MAP_SWIZZLE_128B);
        p.b_mn_major = 0;
        p.b_lbo = 16; p.b_sbo = 1024; p.b_kstep = 32;     // 8-row groups 1024 B apart; 16 k-values = 32 B
    } else {
        st = cached_tmap_2d_bf16(&wmap, w, (uint64_t)n, (uint64_t)k, (uint64_t)ldw * 2, 64, GM_BK, CU_TENSOR_MAP_SWIZZLE_128B);
        p.b_mn_major = 1;
        // MN-major, 128-byte swizzle: a 64(n) x 64(k) box is 64 k-rows of 128 B (8 KiB); 8-k groups are
        // 1024 B apart (stride), the next 64 columns of n start 8192 B later (leading); 16 k-values = 2048 B.
        p.b_lbo = 8192; p.b_sbo = 1024; p.b_kstep = 2048;
    }
    if (st != TRI_OK) return st;
    return one_sm ? launch_gemm_1sm(amap, wmap, p, di->sm_count, s) : launch_gemm_2sm(amap, wmap, p, di->sm_count, s);
}

// ---- prefill_gemm_static_ws: the one-CTA kernel with its split-K partials in a file-scope device array ----------------
// For callers that must not allocate device memory (see include/triroof.h).  Nothing above is touched: this is a second
// way into gemm_1sm_kernel / splitk_reduce_kernel with GemmParams::ws pointing at g_static_ws instead of at a
// cudaMalloc'ed per-stream buffer.  The partition (which tiles are cut along K, into how many parts) is computed exactly
// as launch_gemm_1sm computes it, so the bits of C are those of prefill_gemm.
//
// Size: a split shape has `left` < sm_count leftover tiles cut into parts = sm_count / left ranges, so there are at most
// sm_count partial tiles of 128 x 128 fp32 (64 KiB) in flight: 148 of them on a B200 = 9.25 MiB.  Every device that
// loads libtriroof.so carries the array from module load to process exit, used or not.
constexpr int GM_STATIC_WS_TILES = 148;
constexpr size_t GM_STATIC_WS_BYTES = (size_t)GM_STATIC_WS_TILES * GM_BM * GM_BN * sizeof(float);
static __device__ __align__(256) float g_static_ws[(size_t)GM_STATIC_WS_TILES * GM_BM * GM_BN];

// In host code the name g_static_ws is only a handle for the runtime's symbol table, not a device address; the address
// on the CURRENT device comes from cudaGetSymbolAddress, asked once per device and remembered here.  The same set-up sets
// the kernel's dynamic shared memory limit on that device (launch_gemm_1sm keeps its own record of that; a first call
// through this entry point must not depend on it).
constexpr int GM_STATIC_WS_MAX_DEVICES = 64;
static std::mutex g_static_ws_mu;
static float *g_static_ws_addr[GM_STATIC_WS_MAX_DEVICES] = {};

static int static_ws_on_current_device(float **ws)
{
    int dev = -1;
    TRI_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= GM_STATIC_WS_MAX_DEVICES)
        return fail(TRI_ERR_CUDA, "prefill_gemm_static_ws: device ordinal %d beyond the %d this table holds", dev, GM_STATIC_WS_MAX_DEVICES);
    std::lock_guard<std::mutex> lk(g_static_ws_mu);
    if (!g_static_ws_addr[dev]) {
        void *addr = nullptr;
        TRI_CUDA(cudaGetSymbolAddress(&addr, g_static_ws));
        if (!addr) return fail(TRI_ERR_CUDA, "cudaGetSymbolAddress gave a null address for the static split-K scratch");
        TRI_CUDA(cudaFuncSetAttribute(gemm_1sm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GM_SMEM_MAX));
        g_static_ws_addr[dev] = static_cast<float *>(addr);
    }
    *ws = g_static_ws_addr[dev];
    return TRI_OK;
}

static int gemm_static_ws_impl(int m, int n, int k, const uint16_t *a, int64_t lda, const uint16_t *w, int64_t ldw, int w_layout,
                               uint16_t *c, int64_t ldc, void *stream)
{
    // the argument rules of prefill_gemm, checked on the host before any CUDA call
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
    // the one kernel this entry point drives is the 128-row one-CTA kernel; other row counts never use scratch memory
    // (m <= 32) or use the CTA-pair kernel's larger partial tiles (m > 128), and both are prefill_gemm's business
    if (m <= 32 || m > GM_BM)
        return fail(TRI_ERR_UNSUPPORTED_SHAPE, "prefill_gemm_static_ws covers 33 <= m <= %d rows (m = %d): use prefill_gemm", GM_BM, m);

    const DeviceInfo *di = nullptr;
    int st = ensure_init(&di);
    if (st != TRI_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);

    const int a_rows = ((m + 7) / 8) * 8;
    CUtensorMap amap, wmap;
    st = cached_tmap_2d_bf16(&amap, a, (uint64_t)k, (uint64_t)m, (uint64_t)lda * 2, GM_BK, a_rows, CU_TENSOR_MAP_SWIZZLE_128B);
    if (st != TRI_OK) return st;
    GemmParams p = {};
    p.a_box_bytes = a_rows * GM_BK * 2;
    p.m = m; p.n = n; p.k = k;
    p.tiles_m = 1;
    p.tiles_n = (n + GM_BN - 1) / GM_BN;
    p.kblocks = (k + GM_BK - 1) / GM_BK;
    p.ldc = ldc;
    p.c = c;
    if (w_layout == TRI_W_NK) {
        st = cached_tmap_2d_bf16(&wmap, w, (uint64_t)k, (uint64_t)n, (uint64_t)ldw * 2, GM_BK, GM_BN, CU_TENSOR_MAP_SWIZZLE_128B);
        p.b_mn_major = 0;
        p.b_lbo = 16; p.b_sbo = 1024; p.b_kstep = 32;
    } else {
        st = cached_tmap_2d_bf16(&wmap, w, (uint64_t)n, (uint64_t)k, (uint64_t)ldw * 2, 64, GM_BK, CU_TENSOR_MAP_SWIZZLE_128B);
        p.b_mn_major = 1;
        p.b_lbo = 8192; p.b_sbo = 1024; p.b_kstep = 2048;
    }
    if (st != TRI_OK) return st;

    // ring depth and tail split: launch_gemm_1sm's rules, restated
    const int sm_count = di->sm_count;
    const int stage_bytes = p.a_box_bytes + GM_B_BYTES;
    p.stages = (GM_SMEM_MAX - 1024 - GM_BAR_BYTES) / stage_bytes;
    if (p.stages > GM_MAX_STAGES) p.stages = GM_MAX_STAGES;
    const int ntiles = p.tiles_n;
    const int left = ntiles % sm_count;
    int parts = left ? sm_count / left : 1;
    if (parts > p.kblocks) parts = p.kblocks;
    const bool split = parts >= 2 && (parts - 1) * p.kblocks >= 8 * parts;
    p.full_tiles = split ? ntiles - left : ntiles;
    p.parts = split ? parts : 1;
    if (split) {
        const size_t need = (size_t)left * parts * GM_BM * GM_BN * sizeof(float);
        if (need > GM_STATIC_WS_BYTES)
            return fail(TRI_ERR_UNSUPPORTED_SHAPE,
                        "prefill_gemm_static_ws: this shape on %d SMs needs %zu bytes of split-K scratch, the static array holds %zu",
                        sm_count, need, GM_STATIC_WS_BYTES);
    }
    // the address is looked up on every path (split or not) so that the first call on a device always does the set-up
    float *ws = nullptr;
    st = static_ws_on_current_device(&ws);
    if (st != TRI_OK) return st;
    p.ws = split ? ws : nullptr;
    const int grid = split && p.full_tiles == 0 ? left * parts : (ntiles < sm_count ? ntiles : sm_count);

    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(GM_THREADS);
    cfg.dynamicSmemBytes = gm_smem_bytes(p.stages, stage_bytes);
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl_allowed();
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    TRI_CUDA(cudaLaunchKernelEx(&cfg, gemm_1sm_kernel, amap, wmap, p));
    // Nothing in the array has to start at zero: each partial tile is written in full (all 128 rows x 128 columns, rows
    // beyond m included) by the CTA that owns it before splitk_reduce_kernel reads it, and the reduction reads only the
    // left * parts tiles of THIS call.  What an earlier call left behind is never read.
    if (split) return launch_splitk_reduce(p, GM_BM, GM_BN, false, s);
    return TRI_OK;
}

}  // namespace tri

extern "C" int prefill_gemm_static_ws(int m, int n, int k, const uint16_t *a, int64_t lda, const uint16_t *w, int64_t ldw,
                                      int w_layout, uint16_t *c, int64_t ldc, void *stream)
{
    return tri::gemm_static_ws_impl(m, n, k, a, lda, w, ldw, w_layout, c, ldc, stream);
}

extern "C" int prefill_gemm(int m, int n, int k, const uint16_t *a, int64_t lda, const uint16_t *w, int64_t ldw,
                            int w_layout, uint16_t *c, int64_t ldc, void *stream)
{
    return tri::gemm_impl(m, n, k, a, lda, w, ldw, w_layout, c, ldc, stream);
}
