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
    int w_policy;            // L2 policy of the W loads: 0 evict-first, 1 evict-normal, 2 evict-last
};

// prefill_gemm_2sm.cu: enqueue the CTA-pair kernel.  Returns a TRI_* status.
int launch_gemm_2sm(const CUtensorMap &amap, const CUtensorMap &wmap, const GemmParams &p, int sm_count, cudaStream_t s);

}  // namespace tri
