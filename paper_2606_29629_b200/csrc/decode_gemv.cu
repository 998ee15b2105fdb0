// a2. Decode-phase GEMV ("GEMV-like operators"; BASELINE.json config 3; ABI in
// include/triroof.h):   Y[m][n] = bf16_rne( sum_k X[m][k] * W[k][n] ),  m <= 16, fp32 accumulation.
//
// HBM-bound: the weight matrix is read exactly once.  CUDA-core kernel by design (the GEMM is the
// only tensor-core path): at m = 8 every weight element still costs 8 fp32 FMAs, so the FMA issue
// rate is the second budget; the mapping below keeps issue slots per weight low.
//
// TRI_W_NK kernel (W_phys[n][k], K contiguous) — one CTA per 128 output columns (18944 = 148 * 128:
// exactly one CTA per SM):
//   * thread 0 doubles as the producer: it streams the CTA's weight panel through a ring of
//     shared-memory stages with TMA (two 64(k) x 128(n) boxes per stage, 128-byte swizzle) and
//     mbarriers, always GV_STAGES - 1 stages ahead of the stage being consumed;
//   * X is converted once to fp32 and kept in shared memory as k-pairs  xs[k/2][m][2];
//   * 16 consumer warps: within a stage of 128 k-values warp w owns the 8 k-values of chunk w; lane l
//     owns columns l, l+32, l+64, l+96.  One LDS.128 per column gives 4 bf16 pairs; a pair unpacks
//     with 2 ALU ops into {w[k0], w[k1]} and feeds 8 FFMA2 (one per batch row) against the broadcast
//     X pair  ->  per 8 weights: 1 LDS + 8 ALU + 32 FFMA2, plus 16 broadcast LDS shared by 4 columns;
//   * the swizzle makes the per-column 16-byte reads bank-conflict free (rows l..l+7 hit 8 chunks);
//   * after the last stage the 16 per-warp partial sums are reduced through shared memory (the ring
//     is reused), rounded to bf16 RNE and stored.
//
// TRI_W_KN kernel (W_phys[k][n], N contiguous; secondary path): thread owns 4 adjacent columns and
// reads them with one coalesced 8-byte load per k; the 16 warps of a CTA split K; same reduction.
#include "tri_internal.h"
#include "ptx.cuh"

#include <cuda_bf16.h>

namespace tri {

constexpr int GV_M = 8;                 // batch rows per launch (padded with zeros)
constexpr int GV_COLS = 128;            // output columns per CTA
constexpr int GV_CWARPS = 16;           // consumer warps
constexpr int GV_THREADS = GV_CWARPS * 32;
constexpr int GV_STAGE_K = 128;         // k-values per stage (two TMA boxes of 64)
constexpr int GV_STAGES = 3;
constexpr int GV_BOX_BYTES = 64 * GV_COLS * 2;       // 16 KiB
constexpr int GV_STAGE_BYTES = 2 * GV_BOX_BYTES;     // 32 KiB
constexpr int GV_KMAX = 4096;

struct GemvSmemLayout {
    // offsets from the 1024-aligned base
    static constexpr int ring = 0;
    static constexpr int bars = GV_STAGES * GV_STAGE_BYTES;         // full[GV_STAGES], empty[GV_STAGES]
    static constexpr int xs = bars + 64;
    static size_t bytes(int kpad) { return 1024 + xs + (size_t)kpad * GV_M * 4; }
};

__device__ __forceinline__ float2 unpack_bf16x2(uint32_t w)
{
    return make_float2(__uint_as_float(w << 16), __uint_as_float(w & 0xffff0000u));
}

__global__ void __launch_bounds__(GV_THREADS, 1)
gemv_nk_kernel(const __grid_constant__ CUtensorMap wmap, const uint16_t *__restrict__ x, int64_t ldx,
               uint16_t *__restrict__ y, int64_t ldy, int m, int n, int k)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t ring = ptx::smem_u32(smem + GemvSmemLayout::ring);
    const uint32_t full0 = ptx::smem_u32(smem + GemvSmemLayout::bars);
    const uint32_t empty0 = full0 + 8 * GV_STAGES;
    float *xs = reinterpret_cast<float *>(smem + GemvSmemLayout::xs);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n0 = blockIdx.x * GV_COLS;
    const int nstages = (k + GV_STAGE_K - 1) / GV_STAGE_K;
    const int kpad = nstages * GV_STAGE_K;

    if (threadIdx.x == 0) {
        for (int s = 0; s < GV_STAGES; ++s) {
            ptx::mbar_init(full0 + 8 * s, 1);
            ptx::mbar_init(empty0 + 8 * s, GV_CWARPS);
        }
        ptx::fence_mbar_init();
    }
    __syncthreads();

    // ===== producer duty (thread 0): streams the CTA's weight panel; the first GV_STAGES - 1 stages
    // go out before X is converted so HBM is busy during the prologue =====
    uint64_t pol = 0;
    if (threadIdx.x == 0) {
        ptx::prefetch_tmap(&wmap);
        pol = ptx::policy_evict_first();                             // weights are read once
        for (int s = 0; s < GV_STAGES - 1 && s < nstages; ++s) {
            const uint32_t fb = full0 + 8 * s;
            ptx::mbar_arrive_expect_tx(fb, GV_STAGE_BYTES);
            ptx::tma_load_2d_hint(ring + s * GV_STAGE_BYTES, &wmap, s * GV_STAGE_K, n0, fb, pol);
            ptx::tma_load_2d_hint(ring + s * GV_STAGE_BYTES + GV_BOX_BYTES, &wmap, s * GV_STAGE_K + 64, n0, fb, pol);
        }
    }

    // ===== consumers =====
    // X -> fp32 k-pairs in shared memory: xs[(k/2)*16 + mm*2 + (k&1)], zero beyond m and beyond k.
    {
        const int cpr = kpad / 8;                                     // 16-byte chunks (8 bf16) per row
        const int units = GV_M * cpr;
#pragma unroll 4
        for (int i = threadIdx.x; i < units; i += GV_CWARPS * 32) {
            const int mm = i / cpr, c = i - mm * cpr;                 // coalesced along k within a row
            uint4 v = make_uint4(0u, 0u, 0u, 0u);
            if (mm < m && 8 * c < k) v = __ldg(reinterpret_cast<const uint4 *>(x + (int64_t)mm * ldx + 8 * c));
            float2 *dst = reinterpret_cast<float2 *>(xs + (size_t)(4 * c) * (2 * GV_M) + mm * 2);
            dst[0 * GV_M] = unpack_bf16x2(v.x);
            dst[1 * GV_M] = unpack_bf16x2(v.y);
            dst[2 * GV_M] = unpack_bf16x2(v.z);
            dst[3 * GV_M] = unpack_bf16x2(v.w);
        }
    }
    __syncthreads();

    float2 acc[4][GV_M];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int mm = 0; mm < GV_M; ++mm) acc[j][mm] = make_float2(0.f, 0.f);

    // this warp's 16-byte chunk inside a stage: box (warp / 8), chunk (warp % 8) of the 128-byte row
    const uint32_t box_off = (warp >> 3) * GV_BOX_BYTES;
    const uint32_t chunk = warp & 7;
    uint32_t woff[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t r = lane + 32 * j;
        woff[j] = box_off + r * 128 + ((chunk ^ (r & 7)) << 4);
    }

    for (int s = 0; s < nstages; ++s) {
        const int slot = s % GV_STAGES;
        if (threadIdx.x == 0 && s + GV_STAGES - 1 < nstages) {
            // refill the slot stage s-1 used (every warp released it right after its ring reads)
            const int sn = s + GV_STAGES - 1, slotn = sn % GV_STAGES;
            if (s >= 1) ptx::mbar_wait(empty0 + 8 * slotn, ((s - 1) / GV_STAGES) & 1);
            const uint32_t fb = full0 + 8 * slotn;
            ptx::mbar_arrive_expect_tx(fb, GV_STAGE_BYTES);
            ptx::tma_load_2d_hint(ring + slotn * GV_STAGE_BYTES, &wmap, sn * GV_STAGE_K, n0, fb, pol);
            ptx::tma_load_2d_hint(ring + slotn * GV_STAGE_BYTES + GV_BOX_BYTES, &wmap, sn * GV_STAGE_K + 64, n0, fb, pol);
        }
        __syncwarp();
        ptx::mbar_wait(full0 + 8 * slot, (s / GV_STAGES) & 1);
        const uint32_t base = ring + slot * GV_STAGE_BYTES;
        uint4 wv[4];
#pragma unroll
        for (int j = 0; j < 4; ++j)
            asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                         : "=r"(wv[j].x), "=r"(wv[j].y), "=r"(wv[j].z), "=r"(wv[j].w)
                         : "r"(base + woff[j]));
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(empty0 + 8 * slot);          // data is in registers: free the slot

        const float4 *xp = reinterpret_cast<const float4 *>(xs + ((size_t)(s * GV_STAGE_K + warp * 8) / 2) * (2 * GV_M));
#pragma unroll
        for (int p = 0; p < 4; ++p) {                                  // 4 k-pairs of the chunk
            float4 xq[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) xq[q] = xp[p * 4 + q];        // broadcast reads: rows 2q, 2q+1
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t word = p == 0 ? wv[j].x : p == 1 ? wv[j].y : p == 2 ? wv[j].z : wv[j].w;
                const float2 w2 = unpack_bf16x2(word);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    acc[j][2 * q] = __ffma2_rn(w2, make_float2(xq[q].x, xq[q].y), acc[j][2 * q]);
                    acc[j][2 * q + 1] = __ffma2_rn(w2, make_float2(xq[q].z, xq[q].w), acc[j][2 * q + 1]);
                }
            }
        }
    }

    // ===== cross-warp reduction through the (now idle) ring: red[warp][mm][col] =====
    __syncthreads();   // every warp is past its last ring read
    float *red = reinterpret_cast<float *>(smem + GemvSmemLayout::ring);
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int mm = 0; mm < GV_M; ++mm)
            red[(warp * GV_M + mm) * GV_COLS + 32 * j + lane] = acc[j][mm].x + acc[j][mm].y;
    __syncthreads();
    for (int o = threadIdx.x; o < GV_M * GV_COLS; o += GV_CWARPS * 32) {
        const int mm = o / GV_COLS, col = o - mm * GV_COLS;
        float sum = 0.f;
#pragma unroll
        for (int w = 0; w < GV_CWARPS; ++w) sum += red[(w * GV_M + mm) * GV_COLS + col];
        if (mm < m && n0 + col < n) y[(int64_t)mm * ldy + n0 + col] = __bfloat16_as_ushort(__float2bfloat16_rn(sum));
    }
}

// ---- TRI_W_KN: W_phys[k][n] ------------------------------------------------------------------------
constexpr int KN_WARPS = 16;
constexpr int KN_THREADS = KN_WARPS * 32;
constexpr int KN_UNROLL = 8;

__global__ void __launch_bounds__(KN_THREADS, 1)
gemv_kn_kernel(const uint16_t *__restrict__ w, int64_t ldw, const uint16_t *__restrict__ x, int64_t ldx,
               uint16_t *__restrict__ y, int64_t ldy, int m, int n, int k)
{
    extern __shared__ uint8_t smem_raw[];
    float *xs = reinterpret_cast<float *>(smem_raw);                  // xs[k][GV_M]
    float *red = xs + (size_t)k * GV_M;                               // red[warp][mm][col]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n0 = blockIdx.x * GV_COLS;
    const int c0 = n0 + lane * 4;                                     // this thread's 4 columns

    for (int i = threadIdx.x; i < k * GV_M; i += KN_THREADS) {
        const int mm = i / k, kk = i - mm * k;
        float v = 0.f;
        if (mm < m) v = __uint_as_float((uint32_t)x[(int64_t)mm * ldx + kk] << 16);
        xs[kk * GV_M + mm] = v;
    }
    __syncthreads();

    float acc[4][GV_M];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int mm = 0; mm < GV_M; ++mm) acc[j][mm] = 0.f;

    const bool full_cols = (c0 + 3 < n);
    for (int kb = warp * KN_UNROLL; kb < k; kb += KN_WARPS * KN_UNROLL) {
        uint2 wv[KN_UNROLL];
#pragma unroll
        for (int u = 0; u < KN_UNROLL; ++u) {
            const int kk = kb + u;
            wv[u] = make_uint2(0u, 0u);
            if (kk < k) {
                const uint16_t *row = w + (int64_t)kk * ldw;
                if (full_cols) {
                    wv[u] = __ldcs(reinterpret_cast<const uint2 *>(row + c0));
                } else {
                    uint32_t e[4] = {0, 0, 0, 0};
                    for (int j = 0; j < 4; ++j)
                        if (c0 + j < n) e[j] = row[c0 + j];
                    wv[u] = make_uint2(e[0] | (e[1] << 16), e[2] | (e[3] << 16));
                }
            }
        }
#pragma unroll
        for (int u = 0; u < KN_UNROLL; ++u) {
            const int kk = kb + u;
            if (kk < k) {
                const float4 xa = *reinterpret_cast<const float4 *>(xs + kk * GV_M);
                const float4 xb = *reinterpret_cast<const float4 *>(xs + kk * GV_M + 4);
                const float xv[GV_M] = {xa.x, xa.y, xa.z, xa.w, xb.x, xb.y, xb.z, xb.w};
                const float2 w01 = unpack_bf16x2(wv[u].x), w23 = unpack_bf16x2(wv[u].y);
                const float wf[4] = {w01.x, w01.y, w23.x, w23.y};
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int mm = 0; mm < GV_M; ++mm) acc[j][mm] = __fmaf_rn(wf[j], xv[mm], acc[j][mm]);
            }
        }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int mm = 0; mm < GV_M; ++mm) red[(warp * GV_M + mm) * GV_COLS + lane * 4 + j] = acc[j][mm];
    __syncthreads();
    for (int o = threadIdx.x; o < GV_M * GV_COLS; o += KN_THREADS) {
        const int mm = o / GV_COLS, col = o - mm * GV_COLS;
        float sum = 0.f;
#pragma unroll
        for (int wq = 0; wq < KN_WARPS; ++wq) sum += red[(wq * GV_M + mm) * GV_COLS + col];
        if (mm < m && n0 + col < n) y[(int64_t)mm * ldy + n0 + col] = __bfloat16_as_ushort(__float2bfloat16_rn(sum));
    }
}

static int gemv_impl(int m, int n, int k, const uint16_t *x, int64_t ldx, const uint16_t *w, int64_t ldw, int w_layout,
                     uint16_t *y, int64_t ldy, void *stream)
{
    if (!x || !w || !y) return fail(TRI_ERR_INVALID_ARG, "x/w/y is NULL");
    if (m < 1 || m > 16) return fail(TRI_ERR_INVALID_ARG, "m = %d outside [1, 16]", m);
    if (n < 1 || k < 1) return fail(TRI_ERR_INVALID_ARG, "n = %d, k = %d must be positive", n, k);
    if (w_layout != TRI_W_NK && w_layout != TRI_W_KN) return fail(TRI_ERR_INVALID_ARG, "w_layout = %d", w_layout);
    if (k % 8 != 0) return fail(TRI_ERR_UNSUPPORTED_SHAPE, "k = %d must be a multiple of 8", k);
    if (k > GV_KMAX) return fail(TRI_ERR_UNSUPPORTED_SHAPE, "k = %d exceeds %d (X must fit shared memory as fp32)", k, GV_KMAX);
    if (ldx < k || ldy < n) return fail(TRI_ERR_INVALID_ARG, "ldx = %lld < k or ldy = %lld < n", (long long)ldx, (long long)ldy);
    if (ldw < (w_layout == TRI_W_NK ? k : n)) return fail(TRI_ERR_INVALID_ARG, "ldw = %lld too small", (long long)ldw);
    if (ldx % 8 != 0 || ldw % 8 != 0) return fail(TRI_ERR_ALIGNMENT, "ldx and ldw must be multiples of 8 elements");
    if (!aligned(x, 16) || !aligned(w, 16) || !aligned(y, 2)) return fail(TRI_ERR_ALIGNMENT, "x, w must be 16-byte aligned");
    {
        const uintptr_t y0 = (uintptr_t)y, y1 = y0 + ((size_t)(m - 1) * ldy + n) * 2;
        const uintptr_t x0 = (uintptr_t)x, x1 = x0 + ((size_t)(m - 1) * ldx + k) * 2;
        const size_t wrows = w_layout == TRI_W_NK ? n : k, wcols = w_layout == TRI_W_NK ? k : n;
        const uintptr_t w0 = (uintptr_t)w, w1 = w0 + ((wrows - 1) * (size_t)ldw + wcols) * 2;
        if ((y0 < x1 && x0 < y1) || (y0 < w1 && w0 < y1)) return fail(TRI_ERR_INVALID_ARG, "y aliases an input");
    }
    const DeviceInfo *di = nullptr;
    int st = ensure_init(&di);
    if (st != TRI_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int blocks = (n + GV_COLS - 1) / GV_COLS;

    if (w_layout == TRI_W_NK) {
        CUtensorMap wmap;
        st = make_tmap_2d_bf16(&wmap, w, (uint64_t)k, (uint64_t)n, (uint64_t)ldw * 2, 64, GV_COLS, CU_TENSOR_MAP_SWIZZLE_128B);
        if (st != TRI_OK) return st;
        const int kpad = ((k + GV_STAGE_K - 1) / GV_STAGE_K) * GV_STAGE_K;
        const size_t smem = GemvSmemLayout::bytes(kpad);
        static bool attr_set = false;
        if (!attr_set) {
            TRI_CUDA(cudaFuncSetAttribute(gemv_nk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)di->smem_optin));
            attr_set = true;
        }
        if (smem > di->smem_optin) return fail(TRI_ERR_UNSUPPORTED_SHAPE, "k = %d needs %zu B of shared memory", k, smem);
        for (int r0 = 0; r0 < m; r0 += GV_M) {
            const int mr = m - r0 < GV_M ? m - r0 : GV_M;
            gemv_nk_kernel<<<blocks, GV_THREADS, smem, s>>>(wmap, x + (int64_t)r0 * ldx, ldx, y + (int64_t)r0 * ldy, ldy, mr, n, k);
            TRI_CUDA(cudaGetLastError());
        }
    } else {
        const size_t smem = ((size_t)k * GV_M + (size_t)KN_WARPS * GV_M * GV_COLS) * 4;
        static bool attr_set = false;
        if (!attr_set) {
            TRI_CUDA(cudaFuncSetAttribute(gemv_kn_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)di->smem_optin));
            attr_set = true;
        }
        if (smem > di->smem_optin) return fail(TRI_ERR_UNSUPPORTED_SHAPE, "k = %d needs %zu B of shared memory", k, smem);
        for (int r0 = 0; r0 < m; r0 += GV_M) {
            const int mr = m - r0 < GV_M ? m - r0 : GV_M;
            gemv_kn_kernel<<<blocks, KN_THREADS, smem, s>>>(w, ldw, x + (int64_t)r0 * ldx, ldx, y + (int64_t)r0 * ldy, ldy, mr, n, k);
            TRI_CUDA(cudaGetLastError());
        }
    }
    return TRI_OK;
}

}  // namespace tri

extern "C" int decode_gemv(int m, int n, int k, const uint16_t *x, int64_t ldx, const uint16_t *w, int64_t ldw,
                           int w_layout, uint16_t *y, int64_t ldy, void *stream)
{
    return tri::gemv_impl(m, n, k, x, ldx, w, ldw, w_layout, y, ldy, stream);
}
