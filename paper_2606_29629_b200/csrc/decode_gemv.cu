// a2. Decode-phase GEMV ("GEMV-like operators"; BASELINE.json config 3; ABI in
// include/triroof.h):   Y[m][n] = bf16_rne( sum_k X[m][k] * W[k][n] ),  m <= 32 here (decode_gemv's ABI: m <= 16), fp32 accumulation.
//
// HBM-bound: the weight matrix is read exactly once, whatever m is.  One skeleton, both layouts: a CTA owns 64 output
// columns; 4 compute warps + 1 producer warp (160 threads), TWO CTAs per SM (18944 = 296 * 64: one wave on 148 SMs),
// so the prologue and the tail of one CTA are covered by its neighbour and, with programmatic dependent launch, by
// the first CTAs of the next call.
//   * producer warp (one lane): per 64-k stage one TMA box of W (64 x 64 bf16 = 8 KiB, 128-byte swizzle, L2
//     evict-first) and one of X (64 k x 8 or 16 rows; rows >= m and k >= K arrive as zeros) into a ring of ten
//     slots; full / empty mbarriers.  X rides in the ring, so there is no prologue, no limit on K, and nothing but
//     the ring in shared memory.
//
//   * few columns (N / 64 < 148 CTAs, e.g. the down-projection 18944 -> 3584: 56 column blocks): the launch is a grid of
//     CTA CLUSTERS along K — cluster rank r streams stages [r S'/S, (r+1) S'/S) of the same 64 columns, writes its fp32
//     partial sums into its own (by then dead) ring, and after a cluster barrier rank 0 adds the S partials in rank order
//     through distributed shared memory (ld.shared::cluster) and stores.  No workspace, no second kernel, fixed order.
//
// Two arithmetic paths behind it:
//
// (1) m <= 4: CUDA cores, the sm_100 mixed-precision FMA  fma.rn.f32.bf16  (SASS FHFMA.BF16): d = a * b + c with a, b
//     bf16 taken from either half of a 32-bit register and c, d fp32, one rounding — bit-identical to fmaf on the
//     widened inputs, at the full FP32 rate and with no unpack instruction.  A weight costs m FMA-pipe slots;
//     measured on the config-3 shape: 20.1 us at m = 1, 21.2 us at m = 4 (103 % / 98 % of the measured copy peak).
//       - TRI_W_NK (slot row = column n, 128 B = 64 k): half-warp h of warp w owns the 8-k chunk 2w + h of the stage,
//         lane i of it the columns i, i+16, i+32, i+48: four LDS.128 of W, m broadcast LDS.128 of X, 4 x 8 x m FMAs;
//         8 partial sums per output are added through shared memory at the end.
//       - TRI_W_KN (slot row = k, 128 B = 64 columns n): lane (c = lane & 7, q = lane >> 3) of warp w owns the 8
//         columns of chunk c and the k-rows 16w + 4q .. + 3; 16 partial sums per output.
//
// (2) 5 <= m <= 32: the warp-level tensor-core instruction  mma.sync.m16n8k16 (bf16 in, fp32 accumulate; SASS HMMA)
//     with the WEIGHT tile as the 16-row operand and the batch as n = 8 (one tile for m <= 8, two for m <= 16, four for
//     m <= 32 — the last only through prefill_gemm, decode_gemv's ABI stops at 16): zero padding waste at m = 8, and W is
//     still read once at m = 32.  Why not CUDA cores here (DESIGN.md §5.2 has the
//     numbers): m FMAs per weight are 14.6 us of FMA-pipe time at m = 8 and 1965 MHz (17 us at the ~1.7 GHz the part
//     holds under its power cap) inside a 20.8 us HBM budget, and 29 us at m = 16 — the round-1 FFMA2 / FHFMA kernels
//     stopped at 24.8 us back to back and 26.9 us inside the bench step (0.77 of the roofline) with the FMA pipe 60 %
//     busy and no other unit saturated.  SURVEY.md §7.3-B names this instruction as the escape hatch; the stream, the
//     ring and the accounting are unchanged, only the inner product moved.  Warp w owns the 16 columns 16w .. 16w+15
//     of the CTA over ALL k (no cross-warp reduction): per 64-k stage four ldmatrix.x4 of W (conflict-free on the
//     128-byte swizzle; .trans for TRI_W_KN), two ldmatrix.x4 of X per batch tile, four mma per batch tile, alternating
//     between two accumulator sets.
#include "tri_internal.h"
#include "ptx.cuh"

#include <atomic>

#include <cuda_bf16.h>

namespace tri {

constexpr int GV_COLS = 64;              // output columns per CTA
constexpr int GV_CWARPS = 4;             // compute warps
constexpr int GV_CTHREADS = GV_CWARPS * 32;
constexpr int GV_THREADS = GV_CTHREADS + 32;          // + producer warp
constexpr int GV_STAGE_K = 64;           // k-values per stage
constexpr int GV_W_BYTES = GV_STAGE_K * GV_COLS * 2;  // 8 KiB
constexpr int GV_XROW_BYTES = GV_STAGE_K * 2;         // 128 B: one batch row of a stage
constexpr int GV_MAX_SLOTS = 10;
constexpr int GV_MAX_ROWS = 32;          // rows the kernels take (decode_gemv's ABI stops at 16; prefill_gemm hands over up to 32)
constexpr int GV_BAR_BYTES = 2 * 8 * GV_MAX_SLOTS;    // full[], empty[]
constexpr int GV_RED_STRIDE = 4 * GV_COLS + 16;       // FHFMA path: floats per partial-sum set; +16 keeps the two half-warps on different banks

// X rows per slot: 8 for the FHFMA path and one batch tile of the MMA path, 16 for two tiles.
__host__ __device__ constexpr int gemv_slot_bytes(int xrows) { return GV_W_BYTES + xrows * GV_XROW_BYTES; }
__host__ __device__ constexpr size_t gemv_smem_bytes(int nslots, int xrows)
{
    return 1024 + (size_t)nslots * gemv_slot_bytes(xrows) + GV_BAR_BYTES;
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
// Four 8 x 8 bf16 matrices, row addresses from lanes 8j .. 8j+7; thread (g = lane / 4, t = lane % 4) gets elements
// (g, 2t), (g, 2t+1) of matrix j in r[j] — (2t, g), (2t+1, g) with TRANS.
template <bool TRANS>
__device__ __forceinline__ void ldmatrix_x4(uint32_t (&r)[4], uint32_t addr)
{
    if constexpr (TRANS)
        asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
    else
        asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
// D (16 x 8, fp32) += A (16 x 16, row) * B (16 x 8, col), bf16 inputs: the warp-level tensor-core MMA.
__device__ __forceinline__ void mma_16816(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

struct GemvBars {
    uint32_t ring, full0, empty0;
};

// Carves the dynamic shared memory (1 KiB aligned: 128-byte swizzle atoms), initialises the barriers and lets the next
// kernel of the stream start its CTAs as SM resources free up (programmatic dependent launch).
template <int SLOT_BYTES>
__device__ __forceinline__ GemvBars gemv_setup(uint8_t *smem_raw, int nslots, uint8_t **aligned)
{
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    *aligned = smem_raw + (base - ptx::smem_u32(smem_raw));
    GemvBars b;
    b.ring = base;
    b.full0 = base + nslots * SLOT_BYTES;
    b.empty0 = b.full0 + 8 * GV_MAX_SLOTS;
    ptx::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int s = 0; s < nslots; ++s) {
            ptx::mbar_init(b.full0 + 8 * s, 1);
            ptx::mbar_init(b.empty0 + 8 * s, GV_CWARPS);
        }
        ptx::fence_mbar_init();
    }
    __syncthreads();
    return b;
}

// Producer (one lane): streams the CTA's weight panel and the matching X slices through the ring.  W (model state,
// never an output of the preceding kernel) is fetched at once; X is fetched only after pdl_wait(), i.e. after the
// preceding grid has completed (aliasing rule in include/triroof.h).
// Stages [s0, s0 + nstages) of the K range belong to this CTA (the whole range unless the launch is a K-split cluster).
template <int SLOT_BYTES, bool KN>
__device__ __forceinline__ void gemv_producer(const GemvBars &b, const CUtensorMap *wmap, const CUtensorMap *xmap, int n0,
                                              int s0, int nstages, int nslots)
{
    ptx::prefetch_tmap(wmap);
    ptx::prefetch_tmap(xmap);
    const uint64_t pol_w = ptx::policy_evict_first();          // weights are read once
    const uint64_t pol_x = ptx::policy_evict_last();           // X is re-read by every CTA
    const int npre = nstages < nslots ? nstages : nslots;
    for (int s = 0; s < npre; ++s) {
        const uint32_t fb = b.full0 + 8 * s;
        ptx::mbar_arrive_expect_tx(fb, SLOT_BYTES);
        if (KN) ptx::tma_load_2d_hint(b.ring + s * SLOT_BYTES, wmap, n0, (s0 + s) * GV_STAGE_K, fb, pol_w);
        else ptx::tma_load_2d_hint(b.ring + s * SLOT_BYTES, wmap, (s0 + s) * GV_STAGE_K, n0, fb, pol_w);
    }
    ptx::pdl_wait();
    for (int s = 0; s < npre; ++s)
        ptx::tma_load_2d_hint(b.ring + s * SLOT_BYTES + GV_W_BYTES, xmap, (s0 + s) * GV_STAGE_K, 0, b.full0 + 8 * s, pol_x);
    int slot = 0;
    uint32_t par = 0;                                          // parity of the slot's first release
    for (int s = npre; s < nstages; ++s) {
        ptx::mbar_wait(b.empty0 + 8 * slot, par);
        const uint32_t fb = b.full0 + 8 * slot, dst = b.ring + slot * SLOT_BYTES;
        ptx::mbar_arrive_expect_tx(fb, SLOT_BYTES);
        if (KN) ptx::tma_load_2d_hint(dst, wmap, n0, (s0 + s) * GV_STAGE_K, fb, pol_w);
        else ptx::tma_load_2d_hint(dst, wmap, (s0 + s) * GV_STAGE_K, n0, fb, pol_w);
        ptx::tma_load_2d_hint(dst + GV_W_BYTES, xmap, (s0 + s) * GV_STAGE_K, 0, fb, pol_x);
        if (++slot == nslots) { slot = 0; par ^= 1; }
    }
}

// K-split clusters: this CTA's share of the stages and of the column blocks.
struct GemvSplit {
    uint32_t rank, nranks;     // position in the cluster along K (0, 1 when the launch has no clusters)
    int n0, s0, nstages;
};
__device__ __forceinline__ GemvSplit gemv_split(int k)
{
    GemvSplit g;
    g.rank = ptx::cluster_ctarank();
    g.nranks = ptx::cluster_nctarank();
    g.n0 = (int)(blockIdx.x / g.nranks) * GV_COLS;
    const int total = (k + GV_STAGE_K - 1) / GV_STAGE_K;
    g.s0 = (int)((int64_t)g.rank * total / g.nranks);
    g.nstages = (int)((int64_t)(g.rank + 1) * total / g.nranks) - g.s0;
    return g;
}
constexpr uint32_t GV_PART_OFFSET = 20480;      // partial sums of a K-split rank, inside its ring (beyond the FHFMA path's 17 KiB of sets)
// Rank 0 adds the partials of ranks 1 .. nranks - 1 (written at `part` + 16 * tid * VEC in each rank's own ring) to `v`, in
// rank order.  Every thread of every CTA of the cluster calls this (two cluster barriers).
template <int VEC>
__device__ __forceinline__ void gemv_cluster_reduce(const GemvSplit &g, uint32_t part, bool compute_thread, float4 (&v)[VEC])
{
    if (compute_thread && g.rank != 0) {
#pragma unroll
        for (int i = 0; i < VEC; ++i)
            asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(part + 16 * (threadIdx.x * VEC + i)), "f"(v[i].x), "f"(v[i].y),
                         "f"(v[i].z), "f"(v[i].w) : "memory");
    }
    ptx::cluster_sync();                                              // partials are written (release / acquire at cluster scope)
    if (compute_thread && g.rank == 0) {
        for (uint32_t r = 1; r < g.nranks; ++r)
#pragma unroll
            for (int i = 0; i < VEC; ++i) {
                const float4 o = ptx::ld_shared_cluster_f4(part + 16 * (threadIdx.x * VEC + i), r);
                v[i].x += o.x; v[i].y += o.y; v[i].z += o.z; v[i].w += o.w;
            }
    }
    ptx::cluster_sync();                                              // nobody leaves while rank 0 reads its shared memory
}

// ---------------------------------------------------------------------------------------------------------------------
// (1) CUDA-core path.  MR: batch rows computed (1, 2 or 4 >= m).  KN: W_phys[k][n] (slot row = k) instead of W_phys[n][k].
// ---------------------------------------------------------------------------------------------------------------------
template <int MR, bool KN>
__global__ void __launch_bounds__(GV_THREADS, 2)
gemv_kernel(const __grid_constant__ CUtensorMap wmap, const __grid_constant__ CUtensorMap xmap, uint16_t *__restrict__ y,
            int64_t ldy, int m, int n, int k, int nslots)
{
    constexpr int SLOT = gemv_slot_bytes(8);
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem;
    const GemvBars b = gemv_setup<SLOT>(smem_raw, nslots, &smem);
    float *red = reinterpret_cast<float *>(smem);
    const uint32_t ring = b.ring, full0 = b.full0, empty0 = b.empty0;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const GemvSplit g = gemv_split(k);
    const int n0 = g.n0, nstages = g.nstages;

    if (warp == GV_CWARPS) {
        if (lane == 0) gemv_producer<SLOT, KN>(b, &wmap, &xmap, n0, g.s0, nstages, nslots);
        if (g.nranks > 1) {
            __syncwarp();
            float4 none[1];
            gemv_cluster_reduce<1>(g, 0, false, none);
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

    uint32_t wv[2][4][4];
    int slot = 0;
    uint32_t par = 0;
    ptx::mbar_wait(full0, 0);
#pragma unroll
    for (int j = 0; j < 4; ++j) lds128(wv[0][j], ring + woff[j]);

    auto stage = [&](auto cur_tag, int s) {
        constexpr int CUR = decltype(cur_tag)::value, NXT = CUR ^ 1;
        const uint32_t base = ring + slot * SLOT;
        uint32_t xv[MR][KN ? 2 : 4];
#pragma unroll
        for (int mm = 0; mm < MR; ++mm) {
            if constexpr (KN) lds64(xv[mm], base + xoff + mm * 128);
            else lds128(xv[mm], base + xoff + mm * 128);
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(empty0 + 8 * slot);          // this stage's words are in registers: free the slot
        if (++slot == nslots) { slot = 0; par ^= 1; }
        if (s + 1 < nstages) {
            ptx::mbar_wait(full0 + 8 * slot, par);
            const uint32_t nb = ring + slot * SLOT;
#pragma unroll
            for (int j = 0; j < 4; ++j) lds128(wv[NXT][j], nb + woff[j]);
        }
        if constexpr (KN) {
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
    const int mm = threadIdx.x >> 4, col = (threadIdx.x & 15) * 4;    // 16 threads x 4 outputs per row of 64 columns
    const bool valid = mm < m && mm < MR && n0 + col < n;
    float4 tot[1] = {make_float4(0.f, 0.f, 0.f, 0.f)};
    if (valid) {
#pragma unroll
        for (int t = 0; t < NSETS; ++t) {
            const float4 v = *reinterpret_cast<const float4 *>(red + (size_t)t * GV_RED_STRIDE + mm * GV_COLS + col);
            tot[0].x += v.x; tot[0].y += v.y; tot[0].z += v.z; tot[0].w += v.w;
        }
    }
    if (g.nranks > 1) {                                               // K-split cluster: rank 0 collects the other ranks' sums
        gemv_cluster_reduce<1>(g, ring + GV_PART_OFFSET, true, tot);
        if (g.rank != 0) return;
    }
    ptx::pdl_wait();                                                  // Y may be read by the preceding kernel
    if (valid) {
        const float4 sum = tot[0];
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

// ---------------------------------------------------------------------------------------------------------------------
// (2) Warp-MMA path, 5 <= m <= 32.  NT: batch tiles of 8 rows (1, 2 or 4).
// Fragment layouts (PTX ISA, mma.m16n8k16, g = lane / 4, t = lane % 4): A regs = (row g | g+8) x (k 2t,2t+1 | +8);
// B regs = (k 2t,2t+1 | +8) x (column g); D regs = (row g | g+8) x (columns 2t, 2t+1).  Here "row" is the output
// column n of the GEMV (W tile) and "column" is the batch row.
// ---------------------------------------------------------------------------------------------------------------------
template <int NT, bool KN>
__global__ void __launch_bounds__(GV_THREADS, 2)
gemv_mma_kernel(const __grid_constant__ CUtensorMap wmap, const __grid_constant__ CUtensorMap xmap, uint16_t *__restrict__ y,
                int64_t ldy, int m, int n, int k, int nslots)
{
    constexpr int SLOT = gemv_slot_bytes(8 * NT);
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem;
    const GemvBars b = gemv_setup<SLOT>(smem_raw, nslots, &smem);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const GemvSplit g = gemv_split(k);
    const int n0 = g.n0, nstages = g.nstages;

    if (warp == GV_CWARPS) {
        if (lane == 0) gemv_producer<SLOT, KN>(b, &wmap, &xmap, n0, g.s0, nstages, nslots);
        if (g.nranks > 1) {
            __syncwarp();
            float4 none[NT];
            gemv_cluster_reduce<NT>(g, 0, false, none);
        }
        return;
    }

    // ldmatrix row addresses of this lane inside a slot, for k-step 0 (k-step ks adds a_step * ks, XOR-free: see below).
    // NK: slot row = column (128 B = 64 k, 16-byte chunk c stored at c ^ (row & 7)).  Matrix j = lane >> 3:
    //     rows 16w + (j & 1) * 8 + (lane & 7), chunk 2 ks + (j >> 1)  ->  a0..a3 in order.
    // KN: slot row = k (128 B = 64 columns).  Matrix j: k-rows 16 ks + (j >> 1) * 8 + (lane & 7), chunk 2w + (j & 1),
    //     read transposed; (krow & 7) = lane & 7 for every ks, so the swizzled chunk is a constant.
    const int j4 = lane >> 3, r8 = lane & 7;
    uint32_t a_off;
    if (KN) a_off = (uint32_t)((j4 >> 1) * 8 + r8) * 128u + (uint32_t)(((2 * warp + (j4 & 1)) ^ r8) << 4);
    else a_off = (uint32_t)(16 * warp + (j4 & 1) * 8 + r8) * 128u;
    // X: slot row = batch row (128 B = 64 k, 128-byte swizzle).  One ldmatrix.x4 = chunks 4 kp + j of rows 0..7: the B
    // fragments (b0, b1) of k-steps 2 kp and 2 kp + 1.
    const uint32_t x_off = GV_W_BYTES + (uint32_t)r8 * 128u;

    float acc[2][NT][4];
#pragma unroll
    for (int e = 0; e < 2; ++e)
#pragma unroll
        for (int t = 0; t < NT; ++t)
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[e][t][c] = 0.f;

    int slot = 0;
    uint32_t par = 0;
    for (int s = 0; s < nstages; ++s) {
        ptx::mbar_wait(b.full0 + 8 * slot, par);
        const uint32_t base = b.ring + slot * SLOT;
        uint32_t af[4][4], bf[NT][2][4];
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
            if constexpr (KN) ldmatrix_x4<true>(af[ks], base + a_off + ks * 2048);
            else ldmatrix_x4<false>(af[ks], base + a_off + (uint32_t)(((2 * ks + (j4 >> 1)) ^ r8) << 4));
        }
#pragma unroll
        for (int t = 0; t < NT; ++t)
#pragma unroll
            for (int kp = 0; kp < 2; ++kp) ldmatrix_x4<false>(bf[t][kp], base + x_off + t * 1024 + (uint32_t)(((4 * kp + j4) ^ r8) << 4));
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(b.empty0 + 8 * slot);        // this stage's fragments are in registers: free the slot
        if (++slot == nslots) { slot = 0; par ^= 1; }
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
#pragma unroll
            for (int t = 0; t < NT; ++t) mma_16816(acc[ks & 1][t], af[ks], bf[t][ks >> 1][2 * (ks & 1)], bf[t][ks >> 1][2 * (ks & 1) + 1]);
    }

    float4 tot[NT];
#pragma unroll
    for (int t = 0; t < NT; ++t)
        tot[t] = make_float4(acc[0][t][0] + acc[1][t][0], acc[0][t][1] + acc[1][t][1], acc[0][t][2] + acc[1][t][2], acc[0][t][3] + acc[1][t][3]);
    if (g.nranks > 1) {                                               // K-split cluster: rank 0 collects the other ranks' sums
        asm volatile("bar.sync 1, %0;" ::"n"(GV_CTHREADS) : "memory");   // every warp of this CTA is done with the ring
        gemv_cluster_reduce<NT>(g, b.ring + GV_PART_OFFSET, true, tot);
        if (g.rank != 0) return;
    }
    ptx::pdl_wait();                                                  // Y may be read by the preceding kernel
    const int gq = lane >> 2, t4 = lane & 3;
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        const float d[4] = {tot[t].x, tot[t].y, tot[t].z, tot[t].w};
#pragma unroll
        for (int h = 0; h < 2; ++h) {                                 // D rows g, g + 8 = output columns
            const int col = n0 + 16 * warp + gq + 8 * h;
#pragma unroll
            for (int e = 0; e < 2; ++e) {                             // D columns 2t, 2t + 1 = batch rows
                const int row = 8 * t + 2 * t4 + e;
                if (col < n && row < m) y[(int64_t)row * ldy + col] = __bfloat16_as_ushort(__float2bfloat16_rn(d[2 * h + e]));
            }
        }
    }
}

// ksplit > 1: a grid of CTA clusters of that size along K (see the file header).
template <typename Kernel>
static cudaError_t launch_gemv(Kernel kernel, std::atomic<int> *attr_gen, int xrows, const CUtensorMap &wmap, const CUtensorMap &xmap, uint16_t *y,
                               int64_t ldy, int m, int n, int k, int nslots, int blocks, int ksplit, cudaStream_t s)
{
    if (attr_gen->load(std::memory_order_acquire) != device_generation()) {   // per-device function attribute: redo after tri_init() moved to
                                                                              // another device (two threads may both do it: same value, idempotent)
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gemv_smem_bytes(9, 32));   // the largest configuration (>= GV_MAX_SLOTS slots of 16 rows)
        if (e != cudaSuccess) return e;
        attr_gen->store(device_generation(), std::memory_order_release);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(blocks * ksplit);
    cfg.blockDim = dim3(GV_THREADS);
    cfg.dynamicSmemBytes = gemv_smem_bytes(nslots, xrows);
    cfg.stream = s;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl_allowed();
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = ksplit;
    attr[1].val.clusterDim.y = 1;
    attr[1].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = ksplit > 1 ? 2 : 1;
    return cudaLaunchKernelEx(&cfg, kernel, wmap, xmap, y, ldy, m, n, k, nslots);
}

// Row-count dispatch.  One static generation counter per instantiation (function attributes are per device).
template <bool KN>
static cudaError_t launch_gemv_rows(int m, const CUtensorMap &wmap, const CUtensorMap &xmap, uint16_t *y, int64_t ldy, int n, int k,
                                    int nslots, int blocks, int ksplit, cudaStream_t s)
{
    static std::atomic<int> gen[6] = {{-1}, {-1}, {-1}, {-1}, {-1}, {-1}};
    if (m <= 1) return launch_gemv(gemv_kernel<1, KN>, &gen[0], 8, wmap, xmap, y, ldy, m, n, k, nslots, blocks, ksplit, s);
    if (m <= 2) return launch_gemv(gemv_kernel<2, KN>, &gen[1], 8, wmap, xmap, y, ldy, m, n, k, nslots, blocks, ksplit, s);
    if (m <= 4) return launch_gemv(gemv_kernel<4, KN>, &gen[2], 8, wmap, xmap, y, ldy, m, n, k, nslots, blocks, ksplit, s);
    if (m <= 8) return launch_gemv(gemv_mma_kernel<1, KN>, &gen[3], 8, wmap, xmap, y, ldy, m, n, k, nslots, blocks, ksplit, s);
    if (m <= 16) return launch_gemv(gemv_mma_kernel<2, KN>, &gen[4], 16, wmap, xmap, y, ldy, m, n, k, nslots, blocks, ksplit, s);
    return launch_gemv(gemv_mma_kernel<4, KN>, &gen[5], 32, wmap, xmap, y, ldy, m, n, k, nslots, blocks, ksplit, s);
}

int gemv_impl(int m, int n, int k, const uint16_t *x, int64_t ldx, const uint16_t *w, int64_t ldw, int w_layout,
                     uint16_t *y, int64_t ldy, void *stream)
{
    if (!x || !w || !y) return fail(TRI_ERR_INVALID_ARG, "x/w/y is NULL");
    if (m < 1 || m > GV_MAX_ROWS) return fail(TRI_ERR_INVALID_ARG, "m = %d outside [1, %d]", m, GV_MAX_ROWS);
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

    // Tensor maps (cached: re-encoding two maps costs more host time than the launch).  W: 64 x 64 boxes, 128-byte
    // swizzle.  X: rows beyond m and k-values beyond k arrive as zeros; the MMA path reads it with ldmatrix, so its box
    // is swizzled like W's; the FHFMA path reads plain rows.
    CUtensorMap wmap, xmap;
    if (kn) st = cached_tmap_2d_bf16(&wmap, w, (uint64_t)n, (uint64_t)k, (uint64_t)ldw * 2, GV_COLS, GV_STAGE_K, CU_TENSOR_MAP_SWIZZLE_128B);
    else st = cached_tmap_2d_bf16(&wmap, w, (uint64_t)k, (uint64_t)n, (uint64_t)ldw * 2, GV_STAGE_K, GV_COLS, CU_TENSOR_MAP_SWIZZLE_128B);
    if (st != TRI_OK) return st;
    const int xrows = m <= 8 ? 8 : m <= 16 ? 16 : 32;
    st = cached_tmap_2d_bf16(&xmap, x, (uint64_t)k, (uint64_t)m, (uint64_t)ldx * 2, GV_STAGE_K, xrows,
                             m <= 4 ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_128B);
    if (st != TRI_OK) return st;

    // Ring depth: 10 slots of 9-10 KiB per CTA (160 KiB of weights in flight per SM with two CTAs resident).  Measured on
    // the config-3 shape with the FHFMA path: 8 -> 10 slots takes m = 1 from 21.6 to 20.1 us, m = 4 from 22.9 to 21.2.  Ten
    // slots also fill the SM with two CTAs, so that no CTA of the NEXT call (programmatic dependent launch) moves in early
    // and spins on its barriers in the issue slots of the running ones.  The FHFMA path's partial-sum sets reuse the ring.
    const int nslots = m <= 16 ? GV_MAX_SLOTS : 9;         // 32 rows of X per slot: nine slots of 12 KiB keep two CTAs on an SM
    static_assert((size_t)GV_MAX_SLOTS * gemv_slot_bytes(8) >= GV_PART_OFFSET + 4096 && GV_PART_OFFSET >= (size_t)16 * GV_RED_STRIDE * 4,
                  "the partial sums must fit the ring");
    static_assert(gemv_smem_bytes(9, 32) >= gemv_smem_bytes(GV_MAX_SLOTS, 16) && 2 * (gemv_smem_bytes(9, 32) + 1024) <= 228 * 1024, "two CTAs per SM");
    static_assert((size_t)9 * gemv_slot_bytes(32) >= GV_PART_OFFSET + 4 * 2048, "the partial sums of four batch tiles must fit the ring");

    // Fewer column blocks than two per SM: clusters of 2 or 4 along K, as long as a rank keeps at least 24 stages (a CTA's
    // fixed cost is worth ~10 stages).  Measured on 8 x 3584 x 18944 (56 column blocks): 1 / 2 / 3 / 4 / 5 / 6 / 8 ranks ->
    // 39.6 / 25.8 / 22.4 / 21.6 / 27.4 / 26.6 / 24.1 us (sizes that do not pack the GPCs evenly run in two waves); on
    // 8 x 4608 x 3584 (56 stages in all): 9.0 / 8.7 / 8.2 / 11.0 us for 1 / 2 / 3 / 4.
    const int total_stages = (k + GV_STAGE_K - 1) / GV_STAGE_K;
    const int room = (2 * di->sm_count) / blocks;
    int ksplit = room >= 4 ? 4 : room >= 2 ? 2 : 1;
    while (ksplit > 1 && total_stages / ksplit < 24) ksplit /= 2;

    cudaError_t e = kn ? launch_gemv_rows<true>(m, wmap, xmap, y, ldy, n, k, nslots, blocks, ksplit, s)
                       : launch_gemv_rows<false>(m, wmap, xmap, y, ldy, n, k, nslots, blocks, ksplit, s);
    if (e != cudaSuccess) return fail(TRI_ERR_CUDA, "decode_gemv launch: %s", cudaGetErrorString(e));
    return TRI_OK;
}

}  // namespace tri

extern "C" int decode_gemv(int m, int n, int k, const uint16_t *x, int64_t ldx, const uint16_t *w, int64_t ldw,
                           int w_layout, uint16_t *y, int64_t ldy, void *stream)
{
    if (m > 16) return tri::fail(TRI_ERR_INVALID_ARG, "m = %d outside [1, 16]", m);     // the ABI's decode batch (include/triroof.h)
    return tri::gemv_impl(m, n, k, x, ldx, w, ldw, w_layout, y, ldy, stream);
}
