// a1. A.I.-parameterised FMA-chain streaming kernel (the roofline microbenchmark; PAPER.md lines 92,
// 205; BASELINE.json configs 1-2; ABI in include/triroof.h).
//
//   out[i] = chain_k(in[i]),  chain: y <- fmaf(a, y, b) repeated k times, fp32 RN, fused.
//
// Layout: a tile is FMA_THREADS * VEC float4 (coalesced: float4 j of thread t sits at tile + j*FMA_THREADS + t).
// Every thread carries VEC*4 independent chains (VEC*2 packed FFMA2 chains), which hides the FFMA
// latency at the compute end; at the memory end all VEC 128-bit loads are issued before the first
// FMA.  The k loop is a runtime loop (k is arbitrary, not a power of two) unrolled by 8 with a
// remainder loop.  __ffma2_rn is, per component, __fmaf_rn (crt/sm_100_rt.h), so packing two chains
// in one instruction does not change a bit; no fast-math, no FTZ.
#include "tri_internal.h"

#include <cmath>
#include <cstdlib>

namespace tri {


__device__ __forceinline__ float4 ld_stream(const float4 *p)
{
    float4 v;
    asm volatile("ld.global.cs.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_stream(float4 *p, const float4 &v)
{
    asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

template <int NPAIR>
__device__ __forceinline__ void chain_steps(float2 (&y)[NPAIR], unsigned k, float a, float b)
{
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
    unsigned s = k;
#pragma unroll 1
    for (; s >= 8; s -= 8) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int j = 0; j < NPAIR; ++j) y[j] = __ffma2_rn(a2, y[j], b2);
    }
#pragma unroll 1
    for (; s > 0; --s) {
#pragma unroll
        for (int j = 0; j < NPAIR; ++j) y[j] = __ffma2_rn(a2, y[j], b2);
    }
}

// n4 = number of whole float4 groups; `tail` (< 4) scalars follow them and are done by block 0.
template <int VEC, int FMA_THREADS>
__global__ void __launch_bounds__(FMA_THREADS)
fma_chain_kernel(const float *__restrict__ in, float *__restrict__ out, size_t n4, unsigned tail, unsigned k, float a, float b)
{
    const float4 *in4 = reinterpret_cast<const float4 *>(in);
    float4 *out4 = reinterpret_cast<float4 *>(out);
    const size_t tile = (size_t)blockIdx.x * (FMA_THREADS * VEC);
    const size_t base = tile + threadIdx.x;

    if (tile + (size_t)FMA_THREADS * VEC <= n4) {           // full tile: no predicates
        float2 y[VEC * 2];
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
            float4 v = ld_stream(in4 + base + (size_t)j * FMA_THREADS);
            y[2 * j] = make_float2(v.x, v.y);
            y[2 * j + 1] = make_float2(v.z, v.w);
        }
        chain_steps<VEC * 2>(y, k, a, b);
#pragma unroll
        for (int j = 0; j < VEC; ++j)
            st_stream(out4 + base + (size_t)j * FMA_THREADS, make_float4(y[2 * j].x, y[2 * j].y, y[2 * j + 1].x, y[2 * j + 1].y));
    } else {                                                 // ragged last tile
#pragma unroll 1
        for (int j = 0; j < VEC; ++j) {
            size_t idx = base + (size_t)j * FMA_THREADS;
            if (idx < n4) {
                float4 v = in4[idx];
                float2 y[2] = {make_float2(v.x, v.y), make_float2(v.z, v.w)};
                chain_steps<2>(y, k, a, b);
                out4[idx] = make_float4(y[0].x, y[0].y, y[1].x, y[1].y);
            }
        }
    }
    if (blockIdx.x == 0 && threadIdx.x < tail) {            // scalar tail (n % 4 elements)
        size_t i = n4 * 4 + threadIdx.x;
        float y = in[i];
#pragma unroll 1
        for (unsigned s = 0; s < k; ++s) y = __fmaf_rn(a, y, b);
        out[i] = y;
    }
}

template <int VEC, int FMA_THREADS>
static cudaError_t launch(const float *in, float *out, size_t n, unsigned k, float a, float b, cudaStream_t s)
{
    size_t n4 = n / 4;
    unsigned tail = (unsigned)(n % 4);
    size_t per = (size_t)FMA_THREADS * VEC;
    size_t blocks = (n4 + per - 1) / per;
    if (blocks == 0) blocks = 1;   // tail only
    fma_chain_kernel<VEC, FMA_THREADS><<<(unsigned)blocks, FMA_THREADS, 0, s>>>(in, out, n4, tail, k, a, b);
    return cudaGetLastError();
}

static int run(unsigned k, float a, float b, size_t n, const float *in, float *out, void *stream)
{
    if (k < 1 || k > (1u << 20)) return fail(TRI_ERR_INVALID_ARG, "k = %u outside [1, 2^20]", k);
    if (n == 0) return TRI_OK;
    if (!in || !out) return fail(TRI_ERR_INVALID_ARG, "in/out is NULL");
    if (!aligned(in, 16) || !aligned(out, 16)) return fail(TRI_ERR_ALIGNMENT, "in/out must be 16-byte aligned");
    if (n > ((size_t)1 << 40)) return fail(TRI_ERR_UNSUPPORTED_SHAPE, "n = %zu exceeds 2^40", n);
    if (in != out) {
        uintptr_t i0 = (uintptr_t)in, o0 = (uintptr_t)out, bytes = n * sizeof(float);
        if (i0 < o0 + bytes && o0 < i0 + bytes) return fail(TRI_ERR_INVALID_ARG, "in and out overlap partially");
    }
    int st = ensure_init(nullptr);
    if (st != TRI_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    // float4 loads in flight per thread (= 4 x VEC chains), chosen by measurement on B200 (N = 2^28) in BOTH regimes the
    // bench reports: a single launch at the boost clock, and a seconds-long loop, where the 1000 W cap pulls the clock to
    // ~1.5 GHz and moves the ridge down to k ~ 36.  Fraction of min(A.I. x HBM, ALU at the recorded clock), burst / sustained:
    //   k = 16: VEC 2 1.04 / 1.07, VEC 4 1.03 / 1.04          k = 24: VEC 2 1.06 / 0.97, VEC 4 1.04 / 1.04
    //   k = 28: VEC 4 1.03 / 0.98, VEC 8 1.03 / 1.03          k = 32: VEC 4 1.04 / 0.93, VEC 8 1.03 / 0.995
    //   k = 40: VEC 4 0.95 / 0.88, VEC 8 1.04 / 0.95          k = 64: VEC 4 - / 0.94,  VEC 8 0.965 / 0.97
    // More chains per thread mean fewer address / loop instructions per element: under the cap the kernel then draws less
    // power per byte, and at k = 32 it is faster at 1462 MHz (VEC 8) than at 1545 MHz (VEC 4).  The far compute-bound end is
    // indifferent (VEC 2: 0.998); VEC 16 is no better anywhere.
    const int vec = k <= 16 ? 2 : k <= 24 ? 4 : k < 2048 ? 8 : 2;
    // Block size: 256 threads; 128 for the compute-leaning VEC 8 range (k >= 48), where a launch is a few dozen waves of long
    // blocks and the last, partly filled wave costs one block's duration: halving the block halves it (sustained, fraction of
    // the roofline at the recorded clock: k = 64 0.969 -> 0.975, k = 128 0.981 -> 0.984, k = 256 0.987 -> 0.990; at k = 32
    // the smaller block is slower in a burst, 1.01 against 1.03).  256-bit accesses (ld / st.global.v8.f32, SASS LDG.E.256)
    // were measured at k <= 32 and change nothing: 6.83-6.90 TB/s either way, the stream is HBM-bound.
    cudaError_t e;
    switch (vec) {
        case 2: e = launch<2, 256>(in, out, n, k, a, b, s); break;
        case 8: e = k >= 48 ? launch<8, 128>(in, out, n, k, a, b, s) : launch<8, 256>(in, out, n, k, a, b, s); break;
        default: e = launch<4, 256>(in, out, n, k, a, b, s); break;
    }
    if (e != cudaSuccess) return fail(TRI_ERR_CUDA, "fma_chain launch: %s", cudaGetErrorString(e));
    return TRI_OK;
}

}  // namespace tri

extern "C" {

int roofline_run_k(unsigned k, float a, float b, size_t n, const float *in, float *out, void *stream)
{
    return tri::run(k, a, b, n, in, out, stream);
}

int roofline_run(double ai, size_t n, const float *in, float *out, void *stream)
{
    if (!(ai > 0.0) || !std::isfinite(ai)) return tri::fail(TRI_ERR_INVALID_ARG, "ai must be a positive finite number");
    double k4 = 4.0 * ai, kr = std::nearbyint(k4);
    if (std::fabs(k4 - kr) >= 1e-9 || kr < 1.0 || kr > 1048576.0)
        return tri::fail(TRI_ERR_INVALID_ARG, "k = 4*ai = %.12g is not an integer in [1, 2^20]", k4);
    return tri::run((unsigned)kr, 0.9990234375f, 0.0009765625f, n, in, out, stream);
}

}  // extern "C"
