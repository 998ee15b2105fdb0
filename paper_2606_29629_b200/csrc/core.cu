// Library core: status strings, thread-local error detail, device initialisation, the tensor-map
// encoder hook and the in-kernel SM clock probe.  include/triroof.h documents the ABI.
#include "tri_internal.h"

#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>

namespace tri {

static thread_local char g_err[512] = "";

int fail(int status, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return status;
}

static std::mutex g_mu;
static DeviceInfo g_info;
static bool g_ready = false;
static std::atomic<int> g_generation{0};
static unsigned long long *g_clock_scratch = nullptr;

static int init_locked(int device)
{
    if (g_ready && g_info.device == device) return TRI_OK;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || count == 0) {
        cudaGetLastError();
        return fail(TRI_ERR_CUDA, "no CUDA device: %s", e == cudaSuccess ? "device count is 0" : cudaGetErrorString(e));
    }
    if (device < 0 || device >= count) return fail(TRI_ERR_INVALID_ARG, "device %d out of range [0, %d)", device, count);
    TRI_CUDA(cudaSetDevice(device));
    DeviceInfo di;
    di.device = device;
    int v = 0;
    TRI_CUDA(cudaDeviceGetAttribute(&di.cc_major, cudaDevAttrComputeCapabilityMajor, device));
    TRI_CUDA(cudaDeviceGetAttribute(&di.cc_minor, cudaDevAttrComputeCapabilityMinor, device));
    if (di.cc_major != 10)
        return fail(TRI_ERR_ARCH, "device %d is compute capability %d.%d; this library is sm_100a only", device,
                    di.cc_major, di.cc_minor);
    TRI_CUDA(cudaDeviceGetAttribute(&di.sm_count, cudaDevAttrMultiProcessorCount, device));
    TRI_CUDA(cudaDeviceGetAttribute(&v, cudaDevAttrL2CacheSize, device));
    di.l2_bytes = (size_t)v;
    TRI_CUDA(cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, device));
    di.smem_optin = (size_t)v;
    g_info = di;
    g_ready = true;
    ++g_generation;
    return TRI_OK;
}

int device_generation() { return g_generation.load(std::memory_order_acquire); }

int pdl_allowed()
{
    static const int v = [] {
        const char *e = getenv("TRI_PDL");
        return (e && e[0] == '0' && e[1] == 0) ? 0 : 1;
    }();
    return v;
}

int ensure_init(const DeviceInfo **info)
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_ready) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return fail(TRI_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
        }
        int st = init_locked(dev);
        if (st != TRI_OK) return st;
    }
    if (info) *info = &g_info;
    return TRI_OK;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_tmap_2d_bf16(CUtensorMap *map, const void *base, uint64_t inner, uint64_t outer, uint64_t pitch_bytes,
                      uint32_t box_inner, uint32_t box_outer, CUtensorMapSwizzle swz)
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        TRI_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q));
        if (!p || q != cudaDriverEntryPointSuccess) return fail(TRI_ERR_CUDA, "cuTensorMapEncodeTiled not available");
        fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    cuuint64_t dims[2] = {inner, outer};
    cuuint64_t strides[1] = {pitch_bytes};
    cuuint32_t box[2] = {box_inner, box_outer};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS)
        return fail(TRI_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d (dims %llu x %llu, pitch %llu, box %u x %u)",
                    (int)r, (unsigned long long)inner, (unsigned long long)outer, (unsigned long long)pitch_bytes,
                    box_inner, box_outer);
    return TRI_OK;
}

// Direct-mapped cache of encoded maps.  cuTensorMapEncodeTiled costs about a microsecond per map, a 20 us decode_gemv
// needs two and a prefill_gemm three; serving loops call with the same buffers every step.
struct TmapKey {
    const void *base;
    uint64_t inner, outer, pitch;
    uint32_t box_inner, box_outer;
    int swz;
    bool operator==(const TmapKey &o) const
    {
        return base == o.base && inner == o.inner && outer == o.outer && pitch == o.pitch && box_inner == o.box_inner &&
               box_outer == o.box_outer && swz == o.swz;
    }
};
struct TmapEntry {
    bool valid = false;
    TmapKey key;
    CUtensorMap map;
};
constexpr int TMAP_CACHE_SIZE = 256;
static TmapEntry g_tmaps[TMAP_CACHE_SIZE];
static std::mutex g_tmap_mu;

int cached_tmap_2d_bf16(CUtensorMap *map, const void *base, uint64_t inner, uint64_t outer, uint64_t pitch_bytes,
                        uint32_t box_inner, uint32_t box_outer, CUtensorMapSwizzle swz)
{
    const TmapKey key{base, inner, outer, pitch_bytes, box_inner, box_outer, (int)swz};
    uint64_t h = (uint64_t)(uintptr_t)base * 0x9E3779B97F4A7C15ull;
    h ^= (inner * 0xBF58476D1CE4E5B9ull) ^ (outer * 0x94D049BB133111EBull) ^ (pitch_bytes << 17) ^ ((uint64_t)box_inner << 40) ^
         ((uint64_t)box_outer << 48) ^ ((uint64_t)swz << 56);
    TmapEntry &e = g_tmaps[(h ^ (h >> 29)) % TMAP_CACHE_SIZE];
    {
        std::lock_guard<std::mutex> lk(g_tmap_mu);
        if (e.valid && e.key == key) {
            *map = e.map;
            return TRI_OK;
        }
    }
    int st = make_tmap_2d_bf16(map, base, inner, outer, pitch_bytes, box_inner, box_outer, swz);
    if (st != TRI_OK) return st;
    std::lock_guard<std::mutex> lk(g_tmap_mu);
    e.key = key;
    e.map = *map;
    e.valid = true;
    return TRI_OK;
}

// One block, one thread: spins until `spin_ns` of %globaltimer have passed and reports both clocks.
__global__ void sm_clock_probe(unsigned long long spin_ns, unsigned long long *out)
{
    unsigned long long t0, t1, c0, c1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    c0 = clock64();
    do {
        // a dependent FMA chain keeps the SM busy so the probe reads a loaded, not an idle, clock
        float y = (float)(c0 & 1);
#pragma unroll 1
        for (int i = 0; i < 256; ++i) y = __fmaf_rn(0.999f, y, 0.001f);
        if (y == 123.f) out[2] = 1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
    } while (t1 - t0 < spin_ns);
    c1 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
    out[0] = c1 - c0;
    out[1] = t1 - t0;
}

}  // namespace tri

extern "C" {

const char *tri_status_string(int status)
{
    switch (status) {
        case TRI_OK: return "ok";
        case TRI_ERR_INVALID_ARG: return "invalid argument";
        case TRI_ERR_UNSUPPORTED_SHAPE: return "unsupported shape";
        case TRI_ERR_ALIGNMENT: return "misaligned pointer or leading dimension";
        case TRI_ERR_CUDA: return "CUDA error";
        case TRI_ERR_ARCH: return "device is not compute capability 10.x (sm_100a required)";
        case TRI_ERR_NVML_UNAVAILABLE: return "NVML unavailable";
        case TRI_ERR_NO_PERMISSION: return "no permission";
        case TRI_ERR_BUFFER_TOO_SMALL: return "buffer too small";
        default: return "unknown status";
    }
}

const char *tri_last_error(void) { return tri::g_err; }

int tri_init(int device)
{
    std::lock_guard<std::mutex> lk(tri::g_mu);
    return tri::init_locked(device);
}

int tri_sm_count(void) { return tri::g_ready ? tri::g_info.sm_count : 0; }
size_t tri_l2_bytes(void) { return tri::g_ready ? tri::g_info.l2_bytes : 0; }

int tri_sm_clock_mhz(unsigned spin_us, double *mhz, void *stream)
{
    if (!mhz) return tri::fail(TRI_ERR_INVALID_ARG, "mhz is NULL");
    if (spin_us == 0 || spin_us > 1000000u) return tri::fail(TRI_ERR_INVALID_ARG, "spin_us must be in [1, 1e6]");
    int st = tri::ensure_init(nullptr);
    if (st != TRI_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    {
        std::lock_guard<std::mutex> lk(tri::g_mu);
        if (!tri::g_clock_scratch) TRI_CUDA(cudaMalloc(&tri::g_clock_scratch, 64));
    }
    tri::sm_clock_probe<<<1, 1, 0, s>>>((unsigned long long)spin_us * 1000ull, tri::g_clock_scratch);
    TRI_CUDA(cudaGetLastError());
    unsigned long long h[2] = {0, 0};
    TRI_CUDA(cudaMemcpyAsync(h, tri::g_clock_scratch, sizeof(h), cudaMemcpyDeviceToHost, s));
    TRI_CUDA(cudaStreamSynchronize(s));
    if (h[1] == 0) return tri::fail(TRI_ERR_CUDA, "clock probe measured zero nanoseconds");
    *mhz = (double)h[0] / (double)h[1] * 1000.0;
    return TRI_OK;
}

}  // extern "C"

namespace tri {
void release_clock_scratch()
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (g_clock_scratch) {
        cudaFree(g_clock_scratch);
        g_clock_scratch = nullptr;
    }
    g_ready = false;
}
}  // namespace tri
