// Shared by the two prefill-GEMM kernels (prefill_gemm.cu: one CTA per tile; prefill_gemm_2sm.cu: CTA pairs):
// tcgen05 instruction / shared-memory descriptors and the kernel parameter block.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>

namespace tri {

// Instruction descriptor (PTX ISA, tcgen05.mma kind::f16): D = f32 (bits 4-5 = 1), A = B = bf16
// (bits 7-9, 10-12 = 1), A K-major (bit 15 = 0), B major in bit 16, N >> 3 in bits 17-22, M >> 4 in 24-28.
__host__ __device__ constexpr uint32_t make_idesc(int mdim, int ndim, int b_mn_major)
{
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(ndim >> 3) << 17) |
           ((uint32_t)(mdim >> 4) << 24);
}

// Shared-memory matrix descriptor: start address >> 4 (bits 0-13), leading byte offset >> 4 (16-29),
// stride byte offset >> 4 (32-45), descriptor version 1 (bits 46-47), swizzle mode 2 = 128 B (61-63).
__device__ __forceinline__ uint64_t make_sdesc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(sbo_bytes >> 4) << 32) |
           (1ull << 46) | (2ull << 61);
}

struct GemmParams {
    int m, n, k;
    int tiles_m, tiles_n, kblocks;
    int64_t ldc;
    uint16_t *c;
    int b_mn_major;          // 0: W is [n][k] (K-major);  1: W is [k][n] (MN-major)
    uint32_t b_lbo, b_sbo;   // descriptor strides of the B operand
    uint32_t b_kstep;        // byte advance of the B start address per UMMA_K = 16
    int group_m;             // CTA-pair kernel: row blocks per tile group (see tile_coords)
    // Tail split (see next_work): tiles [0, full_tiles) are computed whole, one per work unit; each of the remaining
    // tiles is cut along K into `parts` work units whose fp32 partial tiles go to `ws` and are summed, in a fixed
    // order, by splitk_reduce_kernel.
    int full_tiles, parts;
    int a_box_bytes;         // bytes of one A box (one-CTA kernel: the box holds only the rows that exist)
    int stages;              // one-CTA kernel: ring depth
    float *ws;               // fp32 workspace: [split tile][part][warp slice][fragment order]
};

// One unit of a CTA's (or CTA pair's) work list: k-blocks [kb0, kb1) of tile `tile`; split >= 0 numbers the split tile
// and `part` its k-range.
struct GemmWork {
    int tile, kb0, kb1, split, part;
};

// The i-th unit of worker `w` out of `nw` (a CTA, or a CTA pair).  Whole tiles first, round robin (unit i of worker w is
// tile w + i * nw, so the workers of a round share W panels and A stays L2 resident); then ONE round in which the
// ntiles - full_tiles leftover tiles are each cut into `parts` k-ranges, one per worker, so that the tail of a shape
// whose tile count is not a multiple of the worker count costs 1 / parts of a tile time instead of a whole one.
// full_tiles is a multiple of nw (or equals ntiles when nothing is split).  (Taking the k-range first, or between whole
// tiles at a position that depends on w, was measured on the down-projection and is 1 % slower: it shifts the workers
// against each other and the panels they share stay in L2 for less of the time.)
__device__ __forceinline__ bool next_work(const GemmParams &p, int ntiles, int w, int nw, int i, GemmWork &out)
{
    const int t = w + i * nw;
    if (t < p.full_tiles) {
        out = GemmWork{t, 0, p.kblocks, -1, 0};
        return true;
    }
    const int u = t - p.full_tiles;
    if (u >= (ntiles - p.full_tiles) * p.parts) return false;
    const int st = u / p.parts, part = u - st * p.parts;
    out = GemmWork{p.full_tiles + st, (int)((int64_t)part * p.kblocks / p.parts), (int)((int64_t)(part + 1) * p.kblocks / p.parts), st, part};
    return true;
}

// ---- split-K: a warp's slice (32 rows, one per lane) of a partial tile goes to the workspace ------------------------------
// Layout of a slice: float4 index (blk * 8 + q) * 32 + lane holds columns 32 blk + 4 q .. + 3 of the lane's row, so every
// store instruction of the warp writes 512 contiguous bytes.  Slices of a tile follow each other in row order, parts of
// a tile follow each other, so partial `part` of split tile `st` starts at float ((st * parts + part) * rows * cols).
// splitk_reduce_kernel (prefill_gemm.cu) is the only reader.
__device__ __forceinline__ void splitk_put(float *slice, int blk, int lane, const uint32_t (&r)[32])
{
    float4 *dst = reinterpret_cast<float4 *>(slice) + (size_t)blk * 256 + lane;
#pragma unroll
    for (int q = 0; q < 8; ++q)
        __stcg(dst + q * 32, make_float4(__uint_as_float(r[4 * q]), __uint_as_float(r[4 * q + 1]), __uint_as_float(r[4 * q + 2]),
                                         __uint_as_float(r[4 * q + 3])));
}

// Split-K workspace of `stream` (allocated on first use and kept; calls on one stream are ordered, so they share it).
int splitk_workspace(cudaStream_t stream, size_t ws_bytes, float **ws);
// Enqueues the reduction of the split tiles of `p` (tile_rows x tile_cols each; pair_order: tile index -> coordinates as
// in the CTA-pair kernel) behind the GEMM kernel, with programmatic stream serialization.
int launch_splitk_reduce(const GemmParams &p, int tile_rows, int tile_cols, bool pair_order, cudaStream_t s);

// Tile order of the CTA-pair kernel: M index fastest inside groups of p.group_m row blocks, groups one after the other.
// A group's A panels (group_m x 256 rows x K) stay L2-resident while the W panels stream past once per group; group_m =
// all row blocks when A fits (config 4: 29 MB), smaller for tall A so that the resident set stays near 32 MB.
__device__ __forceinline__ void tile_coords(const GemmParams &p, int t, int &tm, int &tn)
{
    const int per_group = p.group_m * p.tiles_n, grp = t / per_group, r = t - grp * per_group;
    const int m0 = grp * p.group_m, gm = (p.tiles_m - m0 < p.group_m) ? p.tiles_m - m0 : p.group_m;
    tm = m0 + r % gm;
    tn = r / gm;
}

// prefill_gemm_2sm.cu: enqueue the CTA-pair kernel.  Returns a TRI_* status.
int launch_gemm_2sm(const CUtensorMap &amap, const CUtensorMap &wmap, const GemmParams &p, int sm_count, cudaStream_t s);

}  // namespace tri
