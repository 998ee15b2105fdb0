// Internal helpers shared by the library's translation units (not part of the ABI).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstddef>
#include <cstdint>
#include "../../include/triroof.h"

namespace tri {

struct DeviceInfo {
    int device = -1;
    int sm_count = 0;
    size_t l2_bytes = 0;
    int cc_major = 0, cc_minor = 0;
    size_t smem_optin = 0;
};

// Sets the calling thread's detail text and returns `status` (so call sites can `return fail(...)`).
int fail(int status, const char *fmt, ...) __attribute__((format(printf, 2, 3)));

// Incremented every time the library (re)initialises on a device; kernels cache per-device function attributes against it.
int device_generation();

// Lazily initialises on the current device; returns TRI_OK or an error status.
int ensure_init(const DeviceInfo **info);

// cuTensorMapEncodeTiled resolved through cudaGetDriverEntryPoint (no -lcuda link dependency).
// 2-D bf16 tensor: dims {inner, outer} elements, row pitch in bytes, box {box_inner, box_outer}.
int make_tmap_2d_bf16(CUtensorMap *map, const void *base, uint64_t inner, uint64_t outer,
                      uint64_t pitch_bytes, uint32_t box_inner, uint32_t box_outer, CUtensorMapSwizzle swz);

// The same through a small cache keyed on every argument (a tensor map depends on nothing else, so an entry can never
// be stale): a decode_gemv / prefill_gemm call on buffers it has seen before encodes nothing.  Copies the map out.
int cached_tmap_2d_bf16(CUtensorMap *map, const void *base, uint64_t inner, uint64_t outer,
                        uint64_t pitch_bytes, uint32_t box_inner, uint32_t box_outer, CUtensorMapSwizzle swz);

// decode_gemv.cu: the streaming GEMV (1 <= m <= 32 = GV_MAX_ROWS) behind decode_gemv(), whose ABI stops at 16 rows;
// prefill_gemm() hands it an A of at most 32 rows.
int gemv_impl(int m, int n, int k, const uint16_t *x, int64_t ldx, const uint16_t *w, int64_t ldw, int w_layout,
              uint16_t *y, int64_t ldy, void *stream);

// Launch attribute value for programmatic stream serialization: 1, or 0 when the environment has TRI_PDL=0 (read once).
// With 0 every kernel of the library starts only after the kernel before it on the stream has completed and flushed,
// so W may be produced by that kernel (include/triroof.h, decode_gemv); the griddepcontrol instructions become no-ops.
int pdl_allowed();

inline bool aligned(const void *p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }

}  // namespace tri

#define TRI_CUDA(call)                                                                         \
    do {                                                                                       \
        cudaError_t e__ = (call);                                                              \
        if (e__ != cudaSuccess)                                                                \
            return tri::fail(TRI_ERR_CUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e__),   \
                             __FILE__, __LINE__);                                              \
    } while (0)
