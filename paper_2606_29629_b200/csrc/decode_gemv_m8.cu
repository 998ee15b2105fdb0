// a2, second kernel: decode GEMV for TRI_W_NK with 5..8 batch rows per launch and k <= 4096 (the config-3 shape).
//
// Why a second kernel: the FHFMA kernel of decode_gemv.cu needs one FMA-pipe slot per weight and batch row, but a
// scalar FMA with three distinct register operands fetches two registers from one of the two register-file banks
// unless one operand sits in the reuse cache, and ptxas interleaves the FMA stream so that about half of them miss
// (measured: 1.5 issue cycles per FMA; forcing the order with data or control dependencies costs as much in
// bubbles).  At m = 8 that makes the kernel FMA-issue bound at 30 us.  The packed FFMA2 reads register PAIRS (one
// register of each bank per operand) and cannot conflict, at the price of one unpack per weight and an fp32 copy of X.
//
#include "tri_internal.h"
#include "ptx.cuh"

#include <cuda_bf16.h>

namespace tri {
namespace g8 {

constexpr int GV_M = 8;                 // batch rows per launch (padded with zeros)
constexpr int GV_COLS = 128;            // output columns per CTA
constexpr int GV_CWARPS = 12;           // compute warps (3 groups of 4)
constexpr int GV_GROUPS = 3;
constexpr int GV_CTHREADS = GV_CWARPS * 32;
constexpr int GV_THREADS = (GV_CWARPS + 1) * 32;     // + producer warp
constexpr int GV_STAGE_K = 64;          // k-values per stage (one TMA box)
constexpr int GV_SLOT_BYTES = GV_STAGE_K * GV_COLS * 2;   // 16 KiB
constexpr int GV_MAX_SLOTS = 6;
constexpr int GV_XCHUNK = 72;           // floats per 8-k chunk of xs (64 used + 8 padding)
constexpr int GV_SETS = GV_CWARPS * 2;  // half-warp partial sums
constexpr int GV_SET_STRIDE = GV_M * GV_COLS + 16;   // floats; +16 keeps the two half-warps on different banks
constexpr int GV_BAR_BYTES = 128;

__device__ __forceinline__ float2 unpack_bf16x2(uint32_t w)
{
    return make_float2(__uint_as_float(w << 16), __uint_as_float(w & 0xffff0000u));
}

// Shared memory (from the 1024-aligned base): ring[nslots][16 KiB] | full[6], empty[6] | xs[nchunks][72] floats.
__host__ __device__ inline size_t gemv_smem_bytes(int nslots, int nstages)
{
    size_t main_bytes = (size_t)nslots * GV_SLOT_BYTES + GV_BAR_BYTES + (size_t)nstages * 8 * GV_XCHUNK * 4;
    size_t red_bytes = (size_t)GV_SETS * GV_SET_STRIDE * 4;
    return 1024 + (main_bytes > red_bytes ? main_bytes : red_bytes);
}

__global__ void __launch_bounds__(GV_THREADS, 1)
gemv_nk8_kernel(const __grid_constant__ CUtensorMap wmap, const uint16_t *__restrict__ x, int64_t ldx,
               uint16_t *__restrict__ y, int64_t ldy, int m, int n, int k, int nslots)
{
    extern __shared__ uint8_t smem_raw[];
    // keep the shared state space visible to the compiler: offset arithmetic on the shared window address
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *smem = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
    const uint32_t ring = smem_base;
    const uint32_t full0 = smem_base + nslots * GV_SLOT_BYTES;
    const uint32_t empty0 = full0 + 8 * GV_MAX_SLOTS;
    const uint32_t xs_addr = full0 + GV_BAR_BYTES;
    float *xs = reinterpret_cast<float *>(smem + nslots * GV_SLOT_BYTES + GV_BAR_BYTES);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n0 = blockIdx.x * GV_COLS;
    const int nstages = (k + GV_STAGE_K - 1) / GV_STAGE_K;

    // Programmatic dependent launch: let the next kernel of the stream start on SMs as they drain.  The
    // weight stream (model state, never an output of the preceding kernel) is prefetched at once; X and
    // Y are touched only after pdl_wait(), i.e. after the preceding grid has completed.
    ptx::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int s = 0; s < nslots; ++s) {
            ptx::mbar_init(full0 + 8 * s, 1);
            ptx::mbar_init(empty0 + 8 * s, 4);       // the 4 warps of the group that consumed the slot
        }
        ptx::fence_mbar_init();
    }
    __syncthreads();

    if (warp == GV_CWARPS) {
        // ===== producer warp: one lane streams the weight panel =====
        if (lane == 0) {
            ptx::prefetch_tmap(&wmap);
            const uint64_t pol = ptx::policy_evict_first();          // weights are read once
            int slot = 0;
            uint32_t par = 1;                                        // parity of the slot's previous release
            for (int s = 0; s < nstages; ++s) {
                if (s >= nslots) ptx::mbar_wait(empty0 + 8 * slot, par);
                const uint32_t fb = full0 + 8 * slot;
                ptx::mbar_arrive_expect_tx(fb, GV_SLOT_BYTES);
                ptx::tma_load_2d_hint(ring + slot * GV_SLOT_BYTES, &wmap, s * GV_STAGE_K, n0, fb, pol);
                if (++slot == nslots) { slot = 0; par ^= 1; }
            }
        }
    } else {
        // ===== compute warps =====
        // X -> fp32 in shared memory: xs[chunk * 72 + kk * 8 + mm]; zero beyond m and beyond k.
        ptx::pdl_wait();
        // A thread takes one 8-k chunk of FOUR batch rows: 4 x 16-byte loads (all issued before the first store:
        // they are L2 hits of ~1 us latency), then 8 x 16-byte stores {x[m0..m0+3][kk]} — conflict free because
        // consecutive chunks are 72 floats apart.
        {
            const int mh = threadIdx.x & 1, nchunks = nstages * 8;
            constexpr int CSTEP = GV_CTHREADS / 2, XB = 3;            // 192 chunks per pass
            for (int cb = threadIdx.x >> 1; cb < nchunks; cb += CSTEP * XB) {
                uint4 v[XB][4];
#pragma unroll
                for (int u = 0; u < XB; ++u)
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        const int c = cb + u * CSTEP, mm = mh * 4 + r;
                        v[u][r] = make_uint4(0u, 0u, 0u, 0u);
                        if (mm < m && 8 * c < k) v[u][r] = __ldg(reinterpret_cast<const uint4 *>(x + (int64_t)mm * ldx + 8 * c));
                    }
#pragma unroll
                for (int u = 0; u < XB; ++u) {
                    const int c = cb + u * CSTEP;
                    if (c < nchunks) {
                        float4 *dst = reinterpret_cast<float4 *>(xs + (size_t)c * GV_XCHUNK + mh * 4);
                        const uint32_t *w0 = &v[u][0].x, *w1 = &v[u][1].x, *w2 = &v[u][2].x, *w3 = &v[u][3].x;
#pragma unroll
                        for (int pp = 0; pp < 4; ++pp) {              // bf16 pair pp = k-values 2pp, 2pp+1
                            const float2 a = unpack_bf16x2(w0[pp]), b = unpack_bf16x2(w1[pp]), cc = unpack_bf16x2(w2[pp]),
                                         d = unpack_bf16x2(w3[pp]);
                            dst[(2 * pp) * 2] = make_float4(a.x, b.x, cc.x, d.x);        // 8 floats (2 float4) per k
                            dst[(2 * pp + 1) * 2] = make_float4(a.y, b.y, cc.y, d.y);
                        }
                    }
                }
            }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(GV_CTHREADS) : "memory");

        float2 acc[8][4];                                             // [column j][batch-row pair q]
#pragma unroll
        for (int j = 0; j < 8; ++j)
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[j][q] = make_float2(0.f, 0.f);

        const int group = warp >> 2;
        const int half = lane >> 4, i = lane & 15;
        const int chunk = 2 * (warp & 3) + half;                      // 16-byte chunk of the 128-byte weight row
        const uint32_t woff = (uint32_t)i * 128u + (uint32_t)((chunk ^ (i & 7)) << 4);

        int slot = group % nslots;
        uint32_t par = (uint32_t)(group / nslots) & 1;
        for (int s = group; s < nstages; s += GV_GROUPS) {
            ptx::mbar_wait(full0 + 8 * slot, par);
            const uint32_t base = ring + slot * GV_SLOT_BYTES + woff;
            uint4 wv[8];
#pragma unroll
            for (int j = 0; j < 8; ++j)                               // column i + 16 j is 2048 bytes further
                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                             : "=r"(wv[j].x), "=r"(wv[j].y), "=r"(wv[j].z), "=r"(wv[j].w)
                             : "r"(base + j * 2048));
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(empty0 + 8 * slot);      // weights are in registers: free the slot

            const uint32_t xa = xs_addr + (uint32_t)(s * 8 + chunk) * (GV_XCHUNK * 4);
#pragma unroll
            for (int p = 0; p < 4; ++p) {                              // k-pairs of the chunk
                float4 xv[4];                                          // x[2p][0..7], x[2p+1][0..7]
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                                 : "=f"(xv[q].x), "=f"(xv[q].y), "=f"(xv[q].z), "=f"(xv[q].w)
                                 : "r"(xa + p * 64 + q * 16));
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const uint32_t word = p == 0 ? wv[j].x : p == 1 ? wv[j].y : p == 2 ? wv[j].z : wv[j].w;
                    // PRMT / LOP3 (ALU pipe): a shift would be turned into an IMAD on the FMA pipe, which is the busy one
                    const float w0 = __uint_as_float(__byte_perm(word, 0u, 0x1044)), w1 = __uint_as_float(word & 0xffff0000u);
                    const float2 w0b = make_float2(w0, w0), w1b = make_float2(w1, w1);
                    acc[j][0] = __ffma2_rn(w0b, make_float2(xv[0].x, xv[0].y), acc[j][0]);
                    acc[j][1] = __ffma2_rn(w0b, make_float2(xv[0].z, xv[0].w), acc[j][1]);
                    acc[j][2] = __ffma2_rn(w0b, make_float2(xv[1].x, xv[1].y), acc[j][2]);
                    acc[j][3] = __ffma2_rn(w0b, make_float2(xv[1].z, xv[1].w), acc[j][3]);
                    acc[j][0] = __ffma2_rn(w1b, make_float2(xv[2].x, xv[2].y), acc[j][0]);
                    acc[j][1] = __ffma2_rn(w1b, make_float2(xv[2].z, xv[2].w), acc[j][1]);
                    acc[j][2] = __ffma2_rn(w1b, make_float2(xv[3].x, xv[3].y), acc[j][2]);
                    acc[j][3] = __ffma2_rn(w1b, make_float2(xv[3].z, xv[3].w), acc[j][3]);
                }
            }
#pragma unroll
            for (int t = 0; t < GV_GROUPS; ++t)                        // advance GV_GROUPS stages round the ring
                if (++slot == nslots) { slot = 0; par ^= 1; }
        }

        // ===== cross-warp reduction through shared memory (ring, barriers and xs are dead now) =====
        asm volatile("bar.sync 1, %0;" ::"n"(GV_CTHREADS) : "memory");
        // red[set][(j * 4 + q) * 32 + i * 2 + e] holds the partial sum of column i + 16 j, batch row 2 q + e.
        float2 *red = reinterpret_cast<float2 *>(smem);
        float2 *mine = red + (size_t)(warp * 2 + half) * (GV_SET_STRIDE / 2) + i;
#pragma unroll
        for (int j = 0; j < 8; ++j)
#pragma unroll
            for (int q = 0; q < 4; ++q) mine[(j * 4 + q) * 16] = acc[j][q];
        asm volatile("bar.sync 1, %0;" ::"n"(GV_CTHREADS) : "memory");
        for (int o = threadIdx.x; o < GV_M * GV_COLS / 2; o += GV_CTHREADS) {
            float2 sum = make_float2(0.f, 0.f);
#pragma unroll
            for (int t = 0; t < GV_SETS; ++t) {
                const float2 v = red[t * (GV_SET_STRIDE / 2) + o];
                sum.x += v.x;
                sum.y += v.y;
            }
            const int ii = o & 15, q = (o >> 4) & 3, j = o >> 6, col = n0 + ii + 16 * j;
            if (col < n) {
                if (2 * q < m) y[(int64_t)(2 * q) * ldy + col] = __bfloat16_as_ushort(__float2bfloat16_rn(sum.x));
                if (2 * q + 1 < m) y[(int64_t)(2 * q + 1) * ldy + col] = __bfloat16_as_ushort(__float2bfloat16_rn(sum.y));
            }
        }
    }
}

}  // namespace g8

// Enqueues the kernel above for up to 8 rows (x, y already offset to the first of them).  Returns a TRI_* status.
int launch_gemv_nk8(int mr, int n, int k, const uint16_t *x, int64_t ldx, const uint16_t *w, int64_t ldw, uint16_t *y,
                    int64_t ldy, const DeviceInfo *di, cudaStream_t s)
{
    using namespace g8;
    CUtensorMap wmap;
    int st = make_tmap_2d_bf16(&wmap, w, (uint64_t)k, (uint64_t)n, (uint64_t)ldw * 2, GV_STAGE_K, GV_COLS, CU_TENSOR_MAP_SWIZZLE_128B);
    if (st != TRI_OK) return st;
    const int nstages = (k + GV_STAGE_K - 1) / GV_STAGE_K;
    int nslots = GV_MAX_SLOTS < nstages ? GV_MAX_SLOTS : nstages;       // deepest ring that fits beside xs
    while (nslots > 2 && gemv_smem_bytes(nslots, nstages) > di->smem_optin) --nslots;
    const size_t smem = gemv_smem_bytes(nslots, nstages);
    if (smem > di->smem_optin) return fail(TRI_ERR_UNSUPPORTED_SHAPE, "k = %d needs %zu B of shared memory", k, smem);
    static int attr_gen = -1;                     // per-device function attribute: redo after tri_init() moved to another device
    if (attr_gen != device_generation()) {
        TRI_CUDA(cudaFuncSetAttribute(gemv_nk8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)di->smem_optin));
        attr_gen = device_generation();
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((n + GV_COLS - 1) / GV_COLS);
    cfg.blockDim = dim3(GV_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    TRI_CUDA(cudaLaunchKernelEx(&cfg, gemv_nk8_kernel, wmap, x, ldx, y, ldy, mr, n, k, nslots));
    return TRI_OK;
}

}  // namespace tri
