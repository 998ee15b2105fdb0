// a2. Decode-phase GEMV ("GEMV-like operators"; BASELINE.json config 3; ABI in
// include/triroof.h):   Y[m][n] = bf16_rne( sum_k X[m][k] * W[k][n] ),  m <= 16, fp32 accumulation.
//
// HBM-bound: the weight matrix is read exactly once.  CUDA-core kernel by design (the GEMM is the
// only tensor-core path).  The arithmetic is the sm_100 mixed-precision FMA  fma.rn.f32.bf16
// (SASS FHFMA.BF16): d = a * b + c with a, b bf16 taken from either half of a 32-bit register and c, d
// fp32, one rounding — bit-identical to fmaf on the widened inputs, at the full FP32 rate (measured:
// 125 of 128 lanes/clk/SM) and with no unpack instruction at all.  So the packed bf16 words of W and X
// go from shared memory straight into the FMA, and a weight costs m FMA-pipe slots.
//
// What limits it (measured, B200): the register file has two banks (even / odd register numbers) and each delivers
// one new register per cycle; an operand held over from the previous instruction (.reuse) is free.  A scalar FMA
// with three distinct operands therefore issues every 2 cycles unless one operand is reused, and ptxas interleaves
// the FMA stream so that about half of them miss (1.5 cycles per FMA; forcing the order through data or control
// dependencies cost as much in bubbles).  For m <= 4 the kernel stays HBM-bound (21.7 us at m = 1, 22.8 us at m = 4 on
// the config-3 shape with the 8-slot ring; 20.1 / 21.2 us = 103 % / 98 % of the measured copy peak with 10 slots); at m = 5..8 it is
// FMA-issue bound (39 us NK, 29 us KN as first written; 28.3 / 27.8 us with X transposed to row pairs, see below),
// so TRI_W_NK with 5..8 rows and k <= 4096 goes to the packed-FFMA2 kernel of decode_gemv_m8.cu (24.8 us), whose
// 64-bit operands read one register of each bank and cannot conflict.
//
// One kernel, both layouts.  A CTA owns 64 output columns; 4 compute warps + 1 producer warp (160
// threads), TWO CTAs per SM (18944 = 296 * 64: one wave on 148 SMs), so the prologue, the reduction
// and the tail of one CTA are covered by its neighbour and, with programmatic dependent launch, by the
// first CTAs of the next call.
//   * producer warp (one lane): per 64-k stage one TMA box of W (64 x 64 bf16 = 8 KiB, 128-byte
//     swizzle, L2 evict-first) and one of X (64 k x 8 rows = 1 KiB; rows >= m and k >= K arrive as
//     zeros) into a ring of 9 KiB slots; full / empty mbarriers.  X rides in the ring, so there is no
//     prologue, no limit on K, and nothing but the ring in shared memory.
//   * compute warps, TRI_W_NK (slot row = column n, 128 B = 64 k): half-warp h of warp w owns the
//     8-k chunk 2w + h of the stage, lane i of it the columns i, i+16, i+32, i+48: four LDS.128 of
//     W (the swizzle puts the 8 lanes of a quarter-warp on 8 different 16-byte bank groups), eight
//     broadcast LDS.128 of X (row mm, same chunk), 4 x 8 x 8 = 256 FMAs.
//   * compute warps, TRI_W_KN (slot row = k, 128 B = 64 columns n): lane (c = lane & 7, q = lane >> 3)
//     of warp w owns the 8 columns of chunk c and the k-rows 16w + 4q .. + 3: four LDS.128 of W (a
//     quarter-warp reads one whole row), eight broadcast LDS.64 of X, 8 x 4 x 8 = 256 FMAs.
//   * 8-row kernels: each (half-)warp first transposes its slice of X to row PAIRS per k (2 LDS.32, 2 PRMT, 2 STS.32 per
//     lane and stage), so that one X word holds rows (2q, 2q+1) at one k.  Two (NK) or four (KN) independent FMAs then
//     use the same two registers, which is the operand pattern that needs no register-file read (tri_probe_fma_issue
//     pattern 0) and the one ptxas keeps together; statically 1.17 instead of 1.4-1.6 issue cycles per FMA;
//   * the W registers of stage s + 1 are loaded before the FMAs of stage s, and a slot is released as
//     soon as its words are in registers.
//   * after the last stage the partial sums (8 sets for NK, 16 for KN) are added through shared
//     memory (the ring is dead by then), rounded to bf16 RNE and stored.
#include "tri_internal.h"
#include "ptx.cuh"

#include <cuda_bf16.h>
#include <cstdlib>

namespace tri {

constexpr int GV_M = 8;                  // batch rows per launch (the X box is always 8 rows; missing rows are zeros)
constexpr int GV_COLS = 64;              // output columns per CTA
constexpr int GV_CWARPS = 4;             // compute warps
constexpr int GV_CTHREADS = GV_CWARPS * 32;
constexpr int GV_THREADS = GV_CTHREADS + 32;          // + producer warp
constexpr int GV_STAGE_K = 64;           // k-values per stage
constexpr int GV_W_BYTES = GV_STAGE_K * GV_COLS * 2;  // 8 KiB
constexpr int GV_X_BYTES = GV_STAGE_K * GV_M * 2;     // 1 KiB
constexpr int GV_SLOT_BYTES = GV_W_BYTES + GV_X_BYTES;
constexpr int GV_MAX_SLOTS = 12;
#ifndef GV_XT_ENABLED
#define GV_XT_ENABLED 1      // 8-row kernels read X transposed to row pairs (0: A/B comparison only)
#endif
constexpr int GV_BAR_BYTES = 2 * 8 * GV_MAX_SLOTS + 8 * 128;   // full[], empty[], per-half-warp transposition scratch
constexpr int GV_RED_STRIDE = GV_M * GV_COLS + 16;    // floats per partial-sum set; +16 keeps the two half-warps on different banks

__host__ __device__ constexpr size_t gemv_smem_bytes(int nslots)
{
    return 1024 + (size_t)nslots * GV_SLOT_BYTES + GV_BAR_BYTES;
}

// acc + w.half * x.half: the sm_100 mixed-precision FMA (SASS FHFMA.BF16; the half selects become operand modifiers of
// the 32-bit registers, so no unpack instruction is issued).  WH / XH pick the low (0) or high (1) bf16 of the words.
#define TRI_FMA_BF16(WSEL, XSEL)                                                                                      \
    asm("{\n\t.reg .b16 wl, wh, xl, xh;\n\tmov.b32 {wl, wh}, %1;\n\tmov.b32 {xl, xh}, %2;\n\t"                      \
        "fma.rn.f32.bf16 %0, " WSEL ", " XSEL ", %3;\n\t}" : "=f"(d) : "r"(w), "r"(x), "f"(acc))
template <int WH, int XH>
__device__ __forceinline__ float fma_bf16(uint32_t w, uint32_t x, float acc)
{
    float d;
    if constexpr (WH == 0 && XH == 0) TRI_FMA_BF16("wl", "xl");
    else if constexpr (WH == 1 && XH == 1) TRI_FMA_BF16("wh", "xh");
    else if constexpr (WH == 0 && XH == 1) TRI_FMA_BF16("wl", "xh");
    else TRI_FMA_BF16("wh", "xl");
    return d;
}
#undef TRI_FMA_BF16
__device__ __forceinline__ void lds128(uint32_t (&r)[4], uint32_t addr)
{
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void lds64(uint32_t (&r)[2], uint32_t addr)
{
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "r"(addr));
}

// MR: batch rows computed (1, 2, 4 or 8 >= m).  KN: W_phys[k][n] (slot row = k) instead of W_phys[n][k] (slot row = n).
template <int MR, bool KN>
__global__ void __launch_bounds__(GV_THREADS, 2)
gemv_kernel(const __grid_constant__ CUtensorMap wmap, const __grid_constant__ CUtensorMap xmap, uint16_t *__restrict__ y,
            int64_t ldy, int m, int n, int k, int nslots)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;     // 128-byte swizzle atoms are 1 KiB
    float *red = reinterpret_cast<float *>(smem_raw + (smem_base - ptx::smem_u32(smem_raw)));
    const uint32_t ring = smem_base;
    const uint32_t full0 = smem_base + nslots * GV_SLOT_BYTES;
    const uint32_t empty0 = full0 + 8 * GV_MAX_SLOTS;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n0 = blockIdx.x * GV_COLS;
    const int nstages = (k + GV_STAGE_K - 1) / GV_STAGE_K;

    // Programmatic dependent launch: the next kernel of the stream may start its CTAs as SM resources free up.
    // W (model state, never an output of the preceding kernel) is fetched at once; X is fetched and Y is written
    // only after pdl_wait(), i.e. after the preceding grid has completed (aliasing rule in include/triroof.h).
    ptx::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int s = 0; s < nslots; ++s) {
            ptx::mbar_init(full0 + 8 * s, 1);
            ptx::mbar_init(empty0 + 8 * s, GV_CWARPS);
        }
        ptx::fence_mbar_init();
    }
    __syncthreads();

    if (warp == GV_CWARPS) {
        // ===== producer warp: one lane streams the CTA's weight panel and the matching X slices =====
        if (lane == 0) {
            ptx::prefetch_tmap(&wmap);
            ptx::prefetch_tmap(&xmap);
            const uint64_t pol_w = ptx::policy_evict_first();          // weights are read once
            const uint64_t pol_x = ptx::policy_evict_last();           // X is re-read by every CTA
            const int npre = nstages < nslots ? nstages : nslots;
            for (int s = 0; s < npre; ++s) {
                const uint32_t fb = full0 + 8 * s;
                ptx::mbar_arrive_expect_tx(fb, GV_SLOT_BYTES);
                if (KN) ptx::tma_load_2d_hint(ring + s * GV_SLOT_BYTES, &wmap, n0, s * GV_STAGE_K, fb, pol_w);
                else ptx::tma_load_2d_hint(ring + s * GV_SLOT_BYTES, &wmap, s * GV_STAGE_K, n0, fb, pol_w);
            }
            ptx::pdl_wait();
            for (int s = 0; s < npre; ++s)
                ptx::tma_load_2d_hint(ring + s * GV_SLOT_BYTES + GV_W_BYTES, &xmap, s * GV_STAGE_K, 0, full0 + 8 * s, pol_x);
            int slot = 0;
            uint32_t par = 0;                                          // parity of the slot's first release
            for (int s = npre; s < nstages; ++s) {
                ptx::mbar_wait(empty0 + 8 * slot, par);
                const uint32_t fb = full0 + 8 * slot, dst = ring + slot * GV_SLOT_BYTES;
                ptx::mbar_arrive_expect_tx(fb, GV_SLOT_BYTES);
                if (KN) ptx::tma_load_2d_hint(dst, &wmap, n0, s * GV_STAGE_K, fb, pol_w);
                else ptx::tma_load_2d_hint(dst, &wmap, s * GV_STAGE_K, n0, fb, pol_w);
                ptx::tma_load_2d_hint(dst + GV_W_BYTES, &xmap, s * GV_STAGE_K, 0, fb, pol_x);
                if (++slot == nslots) { slot = 0; par ^= 1; }
            }
        }
        return;
    }

    // ===== compute warps =====
    constexpr int NCOL = KN ? 8 : 4;                                  // columns per lane
    float acc[NCOL][MR];
#pragma unroll
    for (int j = 0; j < NCOL; ++j)
#pragma unroll
        for (int mm = 0; mm < MR; ++mm) acc[j][mm] = 0.f;

    // NK: half-warp -> 8-k chunk, lane i -> columns i + 16 j.   KN: lane -> (chunk c of 8 columns, k-rows 16 w + 4 q + t).
    const int i16 = lane & 15, chunk = 2 * warp + (lane >> 4);
    const int c8 = lane & 7, q4 = lane >> 3, krow = 16 * warp + 4 * q4;
    uint32_t woff[4], xoff;
    if (KN) {
#pragma unroll
        for (int t = 0; t < 4; ++t) woff[t] = (uint32_t)(krow + t) * 128u + (uint32_t)((c8 ^ ((krow + t) & 7)) << 4);
        xoff = GV_W_BYTES + (uint32_t)krow * 2u;
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) woff[j] = (uint32_t)(i16 + 16 * j) * 128u + (uint32_t)((chunk ^ (i16 & 7)) << 4);
        xoff = GV_W_BYTES + (uint32_t)chunk * 16u;
    }

    const uint32_t xt_scratch = empty0 + 8 * GV_MAX_SLOTS + (uint32_t)(warp * 2 + (lane >> 4)) * 128u;   // per half-warp, 8 k x 16 B
    const uint32_t xt_warp = empty0 + 8 * GV_MAX_SLOTS + (uint32_t)warp * 256u;                       // KN: per warp, 16 k x 16 B
    uint32_t wv[2][4][4];
    int slot = 0;
    uint32_t par = 0;
    ptx::mbar_wait(full0, 0);
#pragma unroll
    for (int j = 0; j < 4; ++j) lds128(wv[0][j], ring + woff[j]);

    auto stage = [&](auto cur_tag, int s) {
        constexpr int CUR = decltype(cur_tag)::value, NXT = CUR ^ 1;
        const uint32_t base = ring + slot * GV_SLOT_BYTES;
        [[maybe_unused]] uint32_t xv[MR][KN ? 2 : 4];
        constexpr bool XT = GV_XT_ENABLED && MR == 8;                 // X transposed to row pairs per k (see below)
        [[maybe_unused]] uint32_t xq[XT ? 8 : 1][4];
        if constexpr (XT && !KN) {
            // lane (kp, rq) of the half-warp: rows 2rq, 2rq+1 at k-pair kp of the chunk -> words (row pair at k), (row pair at k+1)
            const int kp = i16 >> 2, rq = i16 & 3;
            uint32_t a, b;
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(a) : "r"(base + xoff + (2 * rq) * 128 + kp * 4));
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(b) : "r"(base + xoff + (2 * rq + 1) * 128 + kp * 4));
            const uint32_t sc = xt_scratch + (uint32_t)(2 * kp) * 16u + (uint32_t)rq * 4u;
            asm volatile("st.shared.u32 [%0], %1;" ::"r"(sc), "r"(__byte_perm(a, b, 0x5410)) : "memory");
            asm volatile("st.shared.u32 [%0], %1;" ::"r"(sc + 16), "r"(__byte_perm(a, b, 0x7632)) : "memory");
            __syncwarp();
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) lds128(xq[kk], xt_scratch + kk * 16);
        } else if constexpr (XT && KN) {
            // the warp's 16 k-rows: lane (kp = lane >> 2, rq = lane & 3) transposes rows 2rq, 2rq+1 at k-pair kp; then every
            // lane reads the row-pair words of its own 4 k-rows
            const int kp = lane >> 2, rq = lane & 3;
            uint32_t a, b;
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(a) : "r"(base + GV_W_BYTES + (2 * rq) * 128 + (16 * warp + 2 * kp) * 2));
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(b) : "r"(base + GV_W_BYTES + (2 * rq + 1) * 128 + (16 * warp + 2 * kp) * 2));
            const uint32_t sw = xt_warp + (uint32_t)(2 * kp) * 16u + (uint32_t)rq * 4u;
            asm volatile("st.shared.u32 [%0], %1;" ::"r"(sw), "r"(__byte_perm(a, b, 0x5410)) : "memory");
            asm volatile("st.shared.u32 [%0], %1;" ::"r"(sw + 16), "r"(__byte_perm(a, b, 0x7632)) : "memory");
            __syncwarp();
#pragma unroll
            for (int t = 0; t < 4; ++t) lds128(xq[t], xt_warp + (uint32_t)(4 * q4 + t) * 16u);
        } else {
#pragma unroll
            for (int mm = 0; mm < MR; ++mm) {
                if constexpr (KN) lds64(xv[mm], base + xoff + mm * 128);
                else lds128(xv[mm], base + xoff + mm * 128);
            }
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(empty0 + 8 * slot);          // this stage's words are in registers: free the slot
        if (++slot == nslots) { slot = 0; par ^= 1; }
        if (s + 1 < nstages) {
            ptx::mbar_wait(full0 + 8 * slot, par);
            const uint32_t nb = ring + slot * GV_SLOT_BYTES;
#pragma unroll
            for (int j = 0; j < 4; ++j) lds128(wv[NXT][j], nb + woff[j]);
        }
        if constexpr (KN && XT) {
#pragma unroll
            for (int t = 0; t < 4; ++t)                               // k-row of the lane
#pragma unroll
                for (int u = 0; u < 4; ++u)                           // word u = columns 2u, 2u + 1 of the chunk
#pragma unroll
                    for (int q = 0; q < 4; ++q) {                     // rows 2q, 2q + 1: four FMAs on the same two words
                        acc[2 * u][2 * q] = fma_bf16<0, 0>(wv[CUR][t][u], xq[t][q], acc[2 * u][2 * q]);
                        acc[2 * u][2 * q + 1] = fma_bf16<0, 1>(wv[CUR][t][u], xq[t][q], acc[2 * u][2 * q + 1]);
                        acc[2 * u + 1][2 * q] = fma_bf16<1, 0>(wv[CUR][t][u], xq[t][q], acc[2 * u + 1][2 * q]);
                        acc[2 * u + 1][2 * q + 1] = fma_bf16<1, 1>(wv[CUR][t][u], xq[t][q], acc[2 * u + 1][2 * q + 1]);
                    }
        } else if constexpr (KN) {
#pragma unroll
            for (int t = 0; t < 4; ++t)                               // k-row of the lane: x word t >> 1, half t & 1
#pragma unroll
                for (int u = 0; u < 4; ++u)                           // word u = columns 2u, 2u + 1 of the chunk
#pragma unroll
                    for (int mm = 0; mm < MR; ++mm) {
                        if (t & 1) {
                            acc[2 * u][mm] = fma_bf16<0, 1>(wv[CUR][t][u], xv[mm][t >> 1], acc[2 * u][mm]);
                            acc[2 * u + 1][mm] = fma_bf16<1, 1>(wv[CUR][t][u], xv[mm][t >> 1], acc[2 * u + 1][mm]);
                        } else {
                            acc[2 * u][mm] = fma_bf16<0, 0>(wv[CUR][t][u], xv[mm][t >> 1], acc[2 * u][mm]);
                            acc[2 * u + 1][mm] = fma_bf16<1, 0>(wv[CUR][t][u], xv[mm][t >> 1], acc[2 * u + 1][mm]);
                        }
                    }
        } else if constexpr (XT) {
#pragma unroll
            for (int p = 0; p < 4; ++p)
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int e = 0; e < 2; ++e)
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            if (e == 0) {
                                acc[j][2 * q] = fma_bf16<0, 0>(wv[CUR][j][p], xq[2 * p][q], acc[j][2 * q]);
                                acc[j][2 * q + 1] = fma_bf16<0, 1>(wv[CUR][j][p], xq[2 * p][q], acc[j][2 * q + 1]);
                            } else {
                                acc[j][2 * q] = fma_bf16<1, 0>(wv[CUR][j][p], xq[2 * p + 1][q], acc[j][2 * q]);
                                acc[j][2 * q + 1] = fma_bf16<1, 1>(wv[CUR][j][p], xq[2 * p + 1][q], acc[j][2 * q + 1]);
                            }
                        }
        } else {
#pragma unroll
            for (int p = 0; p < 4; ++p)                               // word p = k-values 2p, 2p + 1 of the chunk
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int mm = 0; mm < MR; ++mm) {
                        acc[j][mm] = fma_bf16<0, 0>(wv[CUR][j][p], xv[mm][p], acc[j][mm]);
                        acc[j][mm] = fma_bf16<1, 1>(wv[CUR][j][p], xv[mm][p], acc[j][mm]);
                    }
        }
    };
    for (int s = 0; s < nstages; s += 2) {
        stage(std::integral_constant<int, 0>{}, s);
        if (s + 1 < nstages) stage(std::integral_constant<int, 1>{}, s + 1);
    }

    // ===== add the partial sums through shared memory (every TMA write has landed and been read: the ring is dead) =====
    constexpr int NSETS = KN ? 16 : 8;
    asm volatile("bar.sync 1, %0;" ::"n"(GV_CTHREADS) : "memory");
    if constexpr (KN) {
        float *mine = red + (size_t)(warp * 4 + q4) * GV_RED_STRIDE + 8 * c8;
#pragma unroll
        for (int mm = 0; mm < MR; ++mm) {
            *reinterpret_cast<float4 *>(mine + mm * GV_COLS) = make_float4(acc[0][mm], acc[1][mm], acc[2][mm], acc[3][mm]);
            *reinterpret_cast<float4 *>(mine + mm * GV_COLS + 4) = make_float4(acc[4][mm], acc[5][mm], acc[6][mm], acc[7][mm]);
        }
    } else {
        float *mine = red + (size_t)(warp * 2 + (lane >> 4)) * GV_RED_STRIDE + i16;
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int mm = 0; mm < MR; ++mm) mine[mm * GV_COLS + 16 * j] = acc[j][mm];
    }
    asm volatile("bar.sync 1, %0;" ::"n"(GV_CTHREADS) : "memory");
    ptx::pdl_wait();                                                  // Y may be read by the preceding kernel
    const int mm = threadIdx.x >> 4, col = (threadIdx.x & 15) * 4;    // 128 threads x 4 outputs = 8 rows x 64 columns
    if (mm < m && mm < MR && n0 + col < n) {
        float4 sum = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int t = 0; t < NSETS; ++t) {
            const float4 v = *reinterpret_cast<const float4 *>(red + (size_t)t * GV_RED_STRIDE + mm * GV_COLS + col);
            sum.x += v.x; sum.y += v.y; sum.z += v.z; sum.w += v.w;
        }
        uint16_t *dst = y + (int64_t)mm * ldy + n0 + col;
        const uint32_t lo = ptx::pack_bf16x2(sum.x, sum.y), hi = ptx::pack_bf16x2(sum.z, sum.w);
        if (n0 + col + 4 <= n && (reinterpret_cast<uintptr_t>(dst) & 7) == 0) {
            *reinterpret_cast<uint2 *>(dst) = make_uint2(lo, hi);
        } else {
            const uint16_t e[4] = {(uint16_t)lo, (uint16_t)(lo >> 16), (uint16_t)hi, (uint16_t)(hi >> 16)};
            for (int c = 0; c < 4 && n0 + col + c < n; ++c) dst[c] = e[c];
        }
    }
}

template <int MR, bool KN>
static cudaError_t launch_gemv(const CUtensorMap &wmap, const CUtensorMap &xmap, uint16_t *y, int64_t ldy, int m, int n, int k,
                               int nslots, size_t smem, int blocks, cudaStream_t s)
{
    static int attr_gen = -1;                     // per-device function attribute: redo after tri_init() moved to another device
    if (attr_gen != device_generation()) {
        cudaError_t e = cudaFuncSetAttribute(gemv_kernel<MR, KN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gemv_smem_bytes(GV_MAX_SLOTS));
        if (e != cudaSuccess) return e;
        attr_gen = device_generation();
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(blocks);
    cfg.blockDim = dim3(GV_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, gemv_kernel<MR, KN>, wmap, xmap, y, ldy, m, n, k, nslots);
}

template <bool KN>
static cudaError_t launch_gemv_rows(int mr, const CUtensorMap &wmap, const CUtensorMap &xmap, uint16_t *y, int64_t ldy, int n, int k,
                                    int nslots, size_t smem, int blocks, cudaStream_t s)
{
    if (mr <= 1) return launch_gemv<1, KN>(wmap, xmap, y, ldy, mr, n, k, nslots, smem, blocks, s);
    if (mr <= 2) return launch_gemv<2, KN>(wmap, xmap, y, ldy, mr, n, k, nslots, smem, blocks, s);
    if (mr <= 4) return launch_gemv<4, KN>(wmap, xmap, y, ldy, mr, n, k, nslots, smem, blocks, s);
    return launch_gemv<8, KN>(wmap, xmap, y, ldy, mr, n, k, nslots, smem, blocks, s);
}

static int gemv_impl(int m, int n, int k, const uint16_t *x, int64_t ldx, const uint16_t *w, int64_t ldw, int w_layout,
                     uint16_t *y, int64_t ldy, void *stream)
{
    if (!x || !w || !y) return fail(TRI_ERR_INVALID_ARG, "x/w/y is NULL");
    if (m < 1 || m > 16) return fail(TRI_ERR_INVALID_ARG, "m = %d outside [1, 16]", m);
    if (n < 1 || k < 1) return fail(TRI_ERR_INVALID_ARG, "n = %d, k = %d must be positive", n, k);
    if (w_layout != TRI_W_NK && w_layout != TRI_W_KN) return fail(TRI_ERR_INVALID_ARG, "w_layout = %d", w_layout);
    if (k % 8 != 0) return fail(TRI_ERR_UNSUPPORTED_SHAPE, "k = %d must be a multiple of 8", k);
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
    const bool kn = w_layout == TRI_W_KN;

    CUtensorMap wmap;
    if (kn) st = make_tmap_2d_bf16(&wmap, w, (uint64_t)n, (uint64_t)k, (uint64_t)ldw * 2, GV_COLS, GV_STAGE_K, CU_TENSOR_MAP_SWIZZLE_128B);
    else st = make_tmap_2d_bf16(&wmap, w, (uint64_t)k, (uint64_t)n, (uint64_t)ldw * 2, GV_STAGE_K, GV_COLS, CU_TENSOR_MAP_SWIZZLE_128B);
    if (st != TRI_OK) return st;

    // Ring depth: 10 slots of 9 KiB per CTA (160 KiB of weights in flight per SM with two CTAs resident).  Measured on the
    // config-3 shape: 8 -> 10 slots takes m = 1 from 21.6 to 20.1 us, m = 4 from 22.9 to 21.2, m = 8 (NK) from 36.6 to 28.3.
    // Ten slots also fill the SM with two CTAs, so that no CTA of the NEXT call (programmatic dependent launch) moves in
    // early and spins on its barriers in the issue slots of the running ones; 12 is no better.  KN with 5..8 rows likes 8.
    // The partial-sum sets reuse the ring, so it is never smaller than they are.  TRI_GEMV_SLOTS is a debug override.
    static int slots_cfg = -1;
    if (slots_cfg < 0) {
        const char *e = getenv("TRI_GEMV_SLOTS");
        slots_cfg = e ? atoi(e) : 0;
        if (slots_cfg < 4 || slots_cfg > GV_MAX_SLOTS) slots_cfg = 0;
    }
    const int nslots = slots_cfg ? slots_cfg : (kn && m > 4 ? 8 : 10);
    static int force_fhfma = -1;                                     // debug only: TRI_GEMV_FHFMA=1 keeps every shape on this kernel
    if (force_fhfma < 0) {
        const char *e = getenv("TRI_GEMV_FHFMA");
        force_fhfma = e ? atoi(e) : 0;
    }
    const size_t smem = gemv_smem_bytes(nslots);
    static_assert((size_t)4 * GV_SLOT_BYTES >= (size_t)16 * GV_RED_STRIDE * 4, "the partial sums must fit the smallest ring");

    for (int r0 = 0; r0 < m; r0 += GV_M) {
        const int mr = m - r0 < GV_M ? m - r0 : GV_M;
        if (!kn && mr > 4 && k <= GEMV_NK8_KMAX && !force_fhfma) {       // FFMA2 kernel: see decode_gemv_m8.cu for why
            st = launch_gemv_nk8(mr, n, k, x + (int64_t)r0 * ldx, ldx, w, ldw, y + (int64_t)r0 * ldy, ldy, di, s);
            if (st != TRI_OK) return st;
            continue;
        }
        CUtensorMap xmap;            // X rows r0 .. r0 + mr - 1; the 8-row box is zero-filled beyond them and beyond k
        st = make_tmap_2d_bf16(&xmap, x + (int64_t)r0 * ldx, (uint64_t)k, (uint64_t)mr, (uint64_t)ldx * 2, GV_STAGE_K, GV_M,
                               CU_TENSOR_MAP_SWIZZLE_NONE);
        if (st != TRI_OK) return st;
        cudaError_t e = kn ? launch_gemv_rows<true>(mr, wmap, xmap, y + (int64_t)r0 * ldy, ldy, n, k, nslots, smem, blocks, s)
                           : launch_gemv_rows<false>(mr, wmap, xmap, y + (int64_t)r0 * ldy, ldy, n, k, nslots, smem, blocks, s);
        if (e != cudaSuccess) return fail(TRI_ERR_CUDA, "decode_gemv launch: %s", cudaGetErrorString(e));
    }
    return TRI_OK;
}

}  // namespace tri

extern "C" int decode_gemv(int m, int n, int k, const uint16_t *x, int64_t ldx, const uint16_t *w, int64_t ldw,
                           int w_layout, uint16_t *y, int64_t ldy, void *stream)
{
    return tri::gemv_impl(m, n, k, x, ldx, w, ldw, w_layout, y, ldy, stream);
}
