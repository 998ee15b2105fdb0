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
constexpr int GV_W_BYTES = GV_STAGE_K * GV_COLS * 2;      // 16 KiB of weights per stage
constexpr int GV_X_BYTES = GV_STAGE_K * GV_M * 2;         // 1 KiB: the stage's slice of X, bf16 [8 rows][64 k]
constexpr int GV_SLOT_BYTES = GV_W_BYTES + GV_X_BYTES;
constexpr int GV_MAX_SLOTS = 8;
constexpr int GV_XCHUNK = 72;           // floats per half-warp scratch buffer: x[8 k][8 rows] fp32 (64 used + 8 padding against bank conflicts)
constexpr int GV_SETS = GV_CWARPS * 2;  // half-warp partial sums
constexpr int GV_SET_STRIDE = GV_M * GV_COLS + 16;   // floats; +16 keeps the two half-warps on different banks
constexpr int GV_BAR_BYTES = 128;

__device__ __forceinline__ float2 unpack_bf16x2(uint32_t w)
{
    return make_float2(__uint_as_float(w << 16), __uint_as_float(w & 0xffff0000u));
}

// Shared memory (from the 1024-aligned base): ring[nslots][17 KiB] | full[8], empty[8] | scratch[24 half-warps][2][72] floats.
__host__ __device__ inline size_t gemv_smem_bytes(int nslots)
{
    size_t main_bytes = (size_t)nslots * GV_SLOT_BYTES + GV_BAR_BYTES + (size_t)GV_SETS * 2 * GV_XCHUNK * 4;
    size_t red_bytes = (size_t)GV_SETS * GV_SET_STRIDE * 4;
    return 1024 + (main_bytes > red_bytes ? main_bytes : red_bytes);
}

__global__ void __launch_bounds__(GV_THREADS, 1)
gemv_nk8_kernel(const __grid_constant__ CUtensorMap wmap, const __grid_constant__ CUtensorMap xmap,
                uint16_t *__restrict__ y, int64_t ldy, int m, int n, int k, int nslots)
{
    extern __shared__ uint8_t smem_raw[];
    // keep the shared state space visible to the compiler: offset arithmetic on the shared window address
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *smem = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
    const uint32_t ring = smem_base;
    const uint32_t full0 = smem_base + nslots * GV_SLOT_BYTES;
    const uint32_t empty0 = full0 + 8 * GV_MAX_SLOTS;
    const uint32_t xs_addr = full0 + GV_BAR_BYTES;            // per half-warp fp32 scratch for the stage's X chunk

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
        // ===== producer warp: one lane streams the weight panel and the matching slices of X =====
        if (lane == 0) {
            ptx::prefetch_tmap(&wmap);
            ptx::prefetch_tmap(&xmap);
            const uint64_t pol_w = ptx::policy_evict_first();        // weights are read once
            const uint64_t pol_x = ptx::policy_evict_last();         // X is re-read by every CTA
            const int npre = nstages < nslots ? nstages : nslots;
            for (int s = 0; s < npre; ++s) {                         // weights first: they do not depend on the preceding kernel
                ptx::mbar_arrive_expect_tx(full0 + 8 * s, GV_SLOT_BYTES);
                ptx::tma_load_2d_hint(ring + s * GV_SLOT_BYTES, &wmap, s * GV_STAGE_K, n0, full0 + 8 * s, pol_w);
            }
            ptx::pdl_wait();
            for (int s = 0; s < npre; ++s)
                ptx::tma_load_2d_hint(ring + s * GV_SLOT_BYTES + GV_W_BYTES, &xmap, s * GV_STAGE_K, 0, full0 + 8 * s, pol_x);
            int slot = 0;
            uint32_t par = 0;                                        // parity of the slot's first release
            for (int s = npre; s < nstages; ++s) {
                ptx::mbar_wait(empty0 + 8 * slot, par);
                const uint32_t fb = full0 + 8 * slot, dst = ring + slot * GV_SLOT_BYTES;
                ptx::mbar_arrive_expect_tx(fb, GV_SLOT_BYTES);
                ptx::tma_load_2d_hint(dst, &wmap, s * GV_STAGE_K, n0, fb, pol_w);
                ptx::tma_load_2d_hint(dst + GV_W_BYTES, &xmap, s * GV_STAGE_K, 0, fb, pol_x);
                if (++slot == nslots) { slot = 0; par ^= 1; }
            }
        }
    } else {
        // ===== compute warps =====
        float2 acc[8][4];                                             // [column j][batch-row pair q]
#pragma unroll
        for (int j = 0; j < 8; ++j)
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[j][q] = make_float2(0.f, 0.f);

        const int group = warp >> 2;
        const int half = lane >> 4, i = lane & 15;
        const int chunk = 2 * (warp & 3) + half;                      // 16-byte chunk of the 128-byte weight row
        const uint32_t woff = (uint32_t)i * 128u + (uint32_t)((chunk ^ (i & 7)) << 4);
        const int kp = i >> 2, mq = i & 3;                            // conversion role of the lane inside its half-warp
        const uint32_t xraw_off = GV_W_BYTES + (uint32_t)(2 * mq) * 128u + (uint32_t)chunk * 16u + (uint32_t)kp * 4u;
        const uint32_t xs_half = xs_addr + (uint32_t)(warp * 2 + half) * (2 * GV_XCHUNK * 4);   // two buffers of 72 floats
        const uint32_t xs_st = xs_half + (uint32_t)(2 * kp) * 32u + (uint32_t)mq * 8u;   // x[2 kp][2 mq]; x[2 kp + 1][..] is 32 B on

        // The half-warp's X chunk of a stage: rows 2 mq, 2 mq + 1, k-pair kp (bf16 pairs, as TMA left them), widened
        // to fp32 into scratch buffer `buf` as x[kk][row].  Called for the group's NEXT stage: before the FMAs of the
        // current one if that stage has already landed (the load -> store -> load chain is then off the critical
        // path), after them otherwise (never waiting ahead of the FMAs keeps the whole ring depth for HBM latency).
        auto convert_x = [&](int sl, uint32_t buf) {
            uint32_t xr0, xr1;
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(xr0) : "r"(ring + sl * GV_SLOT_BYTES + xraw_off));
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(xr1) : "r"(ring + sl * GV_SLOT_BYTES + xraw_off + 128));
            const float2 r0 = unpack_bf16x2(xr0), r1 = unpack_bf16x2(xr1);
            const uint32_t dst = xs_st + buf * (GV_XCHUNK * 4);
            asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(dst), "f"(r0.x), "f"(r1.x) : "memory");
            asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(dst + 32), "f"(r0.y), "f"(r1.y) : "memory");
        };

        int slot = group % nslots;
        uint32_t par = (uint32_t)(group / nslots) & 1;
        if (group < nstages) {
            ptx::mbar_wait(full0 + 8 * slot, par);
            convert_x(slot, 0);
        }
        __syncwarp();
        uint32_t it = 0;
        for (int s = group; s < nstages; s += GV_GROUPS, ++it) {
            const int cur = slot;                                     // full: waited for when its X was converted
            const uint32_t base = ring + cur * GV_SLOT_BYTES + woff;
            uint4 wv[8];
#pragma unroll
            for (int j = 0; j < 8; ++j)                               // column i + 16 j is 2048 bytes further
                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                             : "=r"(wv[j].x), "=r"(wv[j].y), "=r"(wv[j].z), "=r"(wv[j].w)
                             : "r"(base + j * 2048));
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(empty0 + 8 * cur);       // the stage's words are in registers: free the slot
#pragma unroll
            for (int t = 0; t < GV_GROUPS; ++t)                        // advance GV_GROUPS stages round the ring
                if (++slot == nslots) { slot = 0; par ^= 1; }
            const bool more = s + GV_GROUPS < nstages;
            const bool early = more && __all_sync(0xffffffffu, ptx::mbar_try_wait(full0 + 8 * slot, par));
            if (early) convert_x(slot, (it + 1) & 1);

            const uint32_t xa = xs_half + (it & 1) * (GV_XCHUNK * 4);
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
            if (more && !early) {
                ptx::mbar_wait(full0 + 8 * slot, par);
                convert_x(slot, (it + 1) & 1);
            }
            __syncwarp();                                             // scratch: next buffer written, this one read by all lanes
        }

        // ===== cross-warp reduction through shared memory (ring, barriers and scratch are dead now) =====
        asm volatile("bar.sync 1, %0;" ::"n"(GV_CTHREADS) : "memory");
        // red[set][(j * 4 + q) * 32 + i * 2 + e] holds the partial sum of column i + 16 j, batch row 2 q + e.
        float2 *red = reinterpret_cast<float2 *>(smem);
        float2 *mine = red + (size_t)(warp * 2 + half) * (GV_SET_STRIDE / 2) + i;
#pragma unroll
        for (int j = 0; j < 8; ++j)
#pragma unroll
            for (int q = 0; q < 4; ++q) mine[(j * 4 + q) * 16] = acc[j][q];
        asm volatile("bar.sync 1, %0;" ::"n"(GV_CTHREADS) : "memory");
        ptx::pdl_wait();                                              // Y may still be read by the preceding kernel
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
                    int64_t ldy, const DeviceInfo *, cudaStream_t s)
{
    using namespace g8;
    CUtensorMap wmap, xmap;
    int st = make_tmap_2d_bf16(&wmap, w, (uint64_t)k, (uint64_t)n, (uint64_t)ldw * 2, GV_STAGE_K, GV_COLS, CU_TENSOR_MAP_SWIZZLE_128B);
    if (st != TRI_OK) return st;
    // X rows 0 .. mr - 1; the 8-row box is zero-filled beyond them and beyond k
    st = make_tmap_2d_bf16(&xmap, x, (uint64_t)k, (uint64_t)mr, (uint64_t)ldx * 2, GV_STAGE_K, GV_M, CU_TENSOR_MAP_SWIZZLE_NONE);
    if (st != TRI_OK) return st;
    const int nslots = GV_MAX_SLOTS;
    const size_t smem = gemv_smem_bytes(nslots);
    static bool attr_set = false;
    if (!attr_set) {
        TRI_CUDA(cudaFuncSetAttribute(gemv_nk8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
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
    TRI_CUDA(cudaLaunchKernelEx(&cfg, gemv_nk8_kernel, wmap, xmap, y, ldy, mr, n, k, nslots));
    return TRI_OK;
}

}  // namespace tri
