/* triroof.h — C ABI of the B200-native (sm_100a) roofline microbenchmark and the two serving-phase
 * kernels it stands in for, after "Energy-Efficient Multimodal Inference Serving with Tri-serve"
 * (arxiv 2606.29629; text in PAPER.md).
 *
 * What the paper defines (citations are PAPER.md line numbers):
 *   - a frequency-locked roofline microbenchmark: "a synthetic roofline kernel" swept across
 *     arithmetic intensity (A.I., FLOP per byte) while throughput, power and core clock are
 *     recorded (P:37-42 contribution 2, Sec. II-C.1, Sec. IV-A.3, Fig. 3 caption P:72);
 *   - the two serving phases it stands in for: prefill = "dense GEMM kernels" with high A.I.,
 *     decode = "GEMV-like operators" with low A.I. (P:90 Observation 2);
 *   - per-phase SM clock / power observation and actuation through NVML,
 *     nvmlDeviceSetGpuLockedClocks.
 * BASELINE.json (north_star, configs 1-5) fixes the concrete operations; DESIGN.md lists every
 * reading taken where the paper is silent.
 *
 * Conventions for every entry point:
 *   - extern "C", returns an int status (TRI_OK == 0); no exception crosses the ABI;
 *     tri_last_error() gives the detail text of the calling thread's last failure.
 *   - "device pointer" = CUDA device memory of the current device, owned by the caller; the
 *     library allocates no device memory per call (one lazily created 64-byte scratch excepted,
 *     see tri_sm_clock_mhz) and never frees or retains caller buffers.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream). Compute calls
 *     validate their arguments on the host BEFORE any CUDA call, enqueue their kernel(s) on
 *     `stream` and return; asynchronous faults surface at the caller's next synchronisation.
 *   - CUDA graphs: the compute calls (roofline_run, decode_gemv, prefill_gemm) enqueue kernels only, so a sequence of
 *     them can be captured in a CUDA graph once each distinct call has run once on the capture stream (a prefill_gemm
 *     shape that is split along k allocates that stream's fp32 workspace on first use, which capture does not allow);
 *     replays give the bits of the eager calls (tested).  A graph captured from a split shape holds the ADDRESS of
 *     that stream's workspace in its kernel parameters: it must not be replayed after tri_shutdown() (which frees the
 *     workspaces, also when it leaves NVML loaded because a trace is running) nor after a later, larger split shape on
 *     the same stream has made the workspace grow (free + allocate; shapes up to 20 MB of partials - every shape with
 *     n, m as in configs 3-4 - never grow it).  Re-capture after either.
 *   - Threads: the compute calls, the trace calls and the f3 host functions may be called from several host threads at
 *     once (internal caches are locked, per-kernel set-up is idempotent and atomic); ordering on the GPU is the caller's
 *     business, through `stream`.  tri_init() on another device and tri_shutdown() must not run while another thread is
 *     inside the library.  prefill_gemm_static_ws has its own, stricter rule (one scratch array per device).
 *   - There is no CPU fallback: a device that is not compute capability 10.x yields TRI_ERR_ARCH.
 *   - bf16 values are passed as raw uint16_t bit patterns.
 */
#ifndef TRIROOF_H_
#define TRIROOF_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    TRI_OK = 0,
    TRI_ERR_INVALID_ARG = 1,       /* null pointer, non-positive size, ai not a multiple of 1/4, partial overlap */
    TRI_ERR_UNSUPPORTED_SHAPE = 2, /* shape outside what the kernels cover (no silent fallback) */
    TRI_ERR_ALIGNMENT = 3,         /* pointer or leading dimension not aligned as stated below */
    TRI_ERR_CUDA = 4,              /* a CUDA runtime / driver call failed; see tri_last_error() */
    TRI_ERR_ARCH = 5,              /* device is not compute capability 10.x */
    TRI_ERR_NVML_UNAVAILABLE = 6,  /* libnvidia-ml.so.1 could not be loaded or initialised */
    TRI_ERR_NO_PERMISSION = 7,     /* NVML refused a clock lock (a normal outcome in containers) */
    TRI_ERR_BUFFER_TOO_SMALL = 8   /* sample / summary capacity exhausted; output truncated */
};

/* Physical layout of the weight operand W (logical shape W[k][n], value at (k, n) independent of layout). */
enum {
    TRI_W_NK = 0, /* W_phys[n * ldw + k], K contiguous, ldw >= k   (nn.Linear storage; the reported path) */
    TRI_W_KN = 1  /* W_phys[k * ldw + n], N contiguous, ldw >= n   ("[3584 x 18944]" as BASELINE.json writes it) */
};

/* Static string for a status code (never NULL). */
const char *tri_status_string(int status);
/* Thread-local detail of the calling thread's most recent failure ("" if none). Valid until that
 * thread's next failing call. */
const char *tri_last_error(void);

/* Selects `device` (cudaSetDevice), checks it is cc 10.x, caches SM count / L2 size.
 * Idempotent; the compute calls call it lazily with the current device. */
int tri_init(int device);
/* Resets clocks this process locked through tri_lock_clocks, releases NVML and the scratch buffer. */
void tri_shutdown(void);
/* Cached device facts (0 before a successful tri_init). */
int tri_sm_count(void);
size_t tri_l2_bytes(void);

/* ------------------------------------------------------------------------------------------------
 * a1. A.I.-parameterised FMA-chain streaming kernel — the roofline microbenchmark
 *     ("synthetic roofline kernel"; BASELINE.json configs 1-2).
 *
 *     for i in [0, n):  y = in[i];  repeat k times: y = fmaf(a, y, b);  out[i] = y
 *
 * fp32, IEEE round-to-nearest-even, fused (one rounding per step), steps in this order; the result
 * is bit-exact against the CPU definition.  Per element: 4 B read + 4 B written and 2k FLOP, so
 * A.I. = 2k/8 = k/4 FLOP/B.
 *
 * roofline_run:   ai in FLOP/byte; k = 4*ai must be an integer in [1, 2^20] (|4ai - round(4ai)| <
 *                 1e-9) else TRI_ERR_INVALID_ARG.  Uses a = 0.9990234375, b = 0.0009765625
 *                 (BASELINE.json config 1).
 * roofline_run_k: explicit k in [1, 2^20] and explicit a, b.
 * n:   number of elements, any value >= 0 (n == 0 enqueues nothing and returns TRI_OK).
 * in:  device pointer, n floats, 16-byte aligned.   out: device pointer, n floats, 16-byte aligned.
 *      in == out is allowed (each element is read, then written, by the same thread); any other
 *      overlap of [in, in+n) and [out, out+n) is TRI_ERR_INVALID_ARG.
 * Asynchronous: one kernel on `stream`.
 */
int roofline_run(double ai, size_t n, const float *in, float *out, void *stream);
int roofline_run_k(unsigned k, float a, float b, size_t n, const float *in, float *out, void *stream);

/* ------------------------------------------------------------------------------------------------
 * a2. Decode-phase GEMV ("GEMV-like operators", memory-bound; BASELINE.json config 3).
 *
 *     Y[i][j] = bf16_rne( sum_k float(X[i][k]) * float(W[k][j]) ),  fp32 accumulation (any order)
 *
 * m: rows of X, 1 <= m <= 16 (the decode batch).  n: columns of W, >= 1.  k: inner size, >= 8,
 * k % 8 == 0.  x: device, bf16 X[i * ldx + kk], ldx >= k, ldx % 8 == 0.
 * w: device, bf16, layout w_layout (TRI_W_NK: ldw >= k; TRI_W_KN: ldw >= n), ldw % 8 == 0.
 * y: device, bf16 Y[i * ldy + j], ldy >= n.  x, w 16-byte aligned; y 2-byte aligned (any ldy).
 * Outputs must not alias inputs.  Asynchronous: one kernel on `stream`, whatever m is (W is read once).
 * The kernel is launched with programmatic stream serialization: it prefetches W (model state) while
 * the kernel before it on `stream` drains, and reads X / writes Y only after that kernel has completed.
 * W must therefore not be written by the kernel that immediately precedes the call on `stream`, whatever its origin
 * (a decode_gemv / prefill_gemm of this library, or a caller's dequantisation, weight update or cache append): under
 * programmatic serialization a predecessor's writes are guaranteed visible only after griddepcontrol.wait, and W is
 * fetched before it.  Any earlier producer of W is ordered as usual.  A caller that does produce W right before the
 * call puts any other kernel in between, or runs the process with the environment variable TRI_PDL=0 (read once, at the
 * first launch): every kernel of the library is then launched without the attribute and starts only after its
 * predecessor has completed (tested; costs the overlap, about 1-2 us per call).
 */
int decode_gemv(int m, int n, int k, const uint16_t *x, int64_t ldx, const uint16_t *w, int64_t ldw,
                int w_layout, uint16_t *y, int64_t ldy, void *stream);

/* ------------------------------------------------------------------------------------------------
 * a3. Prefill-phase GEMM ("dense GEMM kernels", compute-bound; BASELINE.json config 4).
 *
 *     C[i][j] = bf16_rne( sum_k float(A[i][k]) * float(W[k][j]) ),  fp32 accumulation in tensor
 *     memory (tcgen05.mma kind::f16), operands staged by TMA.
 *
 * m, n >= 1; k >= 8, k % 8 == 0.  a: device bf16 A[i * lda + kk], lda >= k, lda % 8 == 0.
 * w: as in decode_gemv.  c: device bf16 C[i * ldc + j], ldc >= n, ldc % 8 == 0.
 * a, w, c 16-byte aligned.  Ragged m, n, k tiles are handled inside (TMA zero fill, clipped stores).
 * Outputs must not alias inputs.  Asynchronous: one kernel on `stream` (two when the shape is split along k: the
 * second adds the fp32 partial tiles in a fixed order).
 * m <= 32 is computed by decode_gemv's streaming kernels (same definition and rounding).
 * The kernels are launched with programmatic stream serialization, like decode_gemv: a call sets itself up while the
 * kernel before it on `stream` drains and, for m <= 128, prefetches W (model state) meanwhile; it reads A / writes C
 * only after that kernel has completed.  The rule on W stated for decode_gemv holds here for every m (m <= 32 runs
 * decode_gemv's kernels): W must not be written by the kernel immediately preceding the call on `stream`; TRI_PDL=0
 * lifts it.
 */
int prefill_gemm(int m, int n, int k, const uint16_t *a, int64_t lda, const uint16_t *w, int64_t ldw,
                 int w_layout, uint16_t *c, int64_t ldc, void *stream);

/* a3, for callers that cannot allocate.  prefill_gemm keeps the fp32 partial tiles of a shape that is split along k in
 * a per-stream workspace which it cudaMalloc's on first use (and re-allocates when a larger shape arrives).  Some
 * callers cannot live with that: a serving loop inside a memory pool that owns all of HBM and treats any cudaMalloc
 * outside it as an error (or runs with so little left that one fails); code running while another stream of the process
 * is being captured into a CUDA graph, when an allocation aborts the capture; a real-time or latency-bounded thread, for
 * which cudaMalloc's device-wide synchronisation and unbounded duration are not acceptable; a sandboxed plug-in whose
 * host forbids the allocator.  prefill_gemm_static_ws is the same contraction, same definition, same kernels and the same
 * bits of C as prefill_gemm, for 33 <= m <= 128 (the one-CTA kernel: the short-A / chunked-prefill-tail case), with the
 * partial tiles in an array that is part of the library image instead:
 *   - the array is static device memory of 148 partial tiles x 128 x 128 fp32 = 9 699 328 bytes (9.25 MiB), 256-byte
 *     aligned.  Every GPU on which the process loads this library holds those bytes until the process exits, whether
 *     this entry point is ever called or not.  That is the price of the entry point and the reason the size is modest.
 *   - the call allocates nothing and frees nothing, on the device or through a library routine that would; the caller
 *     passes a, w, c as for prefill_gemm and owns them.
 *   - limits: m outside [33, 128] is TRI_ERR_UNSUPPORTED_SHAPE (fewer rows never need scratch, more rows use the
 *     CTA-pair kernel: call prefill_gemm); so is a shape whose partial tiles exceed the array, which the message
 *     spells out in bytes (the need is at most one tile per SM, so it cannot happen on a 148-SM B200 and can on a
 *     device with more SMs).  Every other argument rule and error is prefill_gemm's.
 *   - first call on a device: it looks up the array's address on the current device (cudaGetSymbolAddress) and raises
 *     the kernel's shared-memory limit there, once; later calls on that device reuse both.  Make that first call,
 *     with the device current, before any stream capture begins.
 *   - ONE array serves every call, stream and thread of the process on that device.  Calls on one stream are ordered
 *     and may follow each other freely; two calls that can run on the GPU at the same time (different streams, say)
 *     write the same bytes and give wrong results without any error: serialise them,
 *     or use prefill_gemm, whose workspaces are per stream.  The array keeps whatever the last call left in it;
 *     nothing needs clearing, because every partial tile is written in full before it is read.
 * Asynchronous: one kernel on `stream`, two when the shape is split along k, launched like prefill_gemm's (the W rule
 * above applies). */
int prefill_gemm_static_ws(int m, int n, int k, const uint16_t *a, int64_t lda, const uint16_t *w, int64_t ldw,
                           int w_layout, uint16_t *c, int64_t ldc, void *stream);

/* ------------------------------------------------------------------------------------------------
 * a4. Phase trace (Fig. 1 bottom, Fig. 4a, P:124 NVML, P:126 event-anchored phase
 *     boundaries; BASELINE.json config 5).  All buffers here are HOST memory owned by the caller.
 */
typedef struct {
    double t_s;                 /* CLOCK_MONOTONIC seconds since phase_trace_start */
    int32_t phase;              /* tag current when the sample was taken */
    uint32_t sm_mhz, mem_mhz;   /* nvmlDeviceGetClockInfo(SM / MEM) */
    uint32_t temp_c;            /* GPU temperature */
    float power_w;              /* nvmlDeviceGetPowerUsage / 1000 */
    uint32_t read_us;           /* how long this sample's NVML queries took (t_s is taken after them): the age bound of the
                                 * values, and where a blocked NVML call shows up in the record */
    uint64_t energy_mj;         /* nvmlDeviceGetTotalEnergyConsumption (0 if unsupported); inside a trace polled by a thread
                                 * of its own about every 100 ms and carried forward in between (the query takes 4-13 ms
                                 * on B200, more than the 10 ms sampling period) */
    uint64_t clk_event_reasons; /* nvmlDeviceGetCurrentClocksEventReasons bitmask */
} tri_sample;

typedef struct {
    int32_t phase;              /* TRI_PHASE_* */
    int32_t expected_samples;   /* floor((t_end_s - t_begin_s) / period): what n_samples would be at the requested cadence */
    double t_begin_s, t_end_s;  /* host clock, same origin as tri_sample.t_s */
    double gpu_ms;              /* cudaEvent time between the phase's first and last kernel (0 for idle) */
    uint64_t launches;          /* kernel launches completed in the phase */
    double flop, bytes, tokens; /* algorithmic work done (tokens: m per call) */
    double energy_j, mean_power_w, j_per_flop, j_per_byte, j_per_token;
    float sm_mhz_mean, sm_mhz_first10, sm_mhz_last10; /* clock over the phase / over the samples stamped inside the first, last
                                 * 10 % of [t_begin_s, t_end_s] (spans of time; 0 when that span holds no sample) */
    float temp_c_max;
    uint32_t n_samples;         /* samples stamped inside [t_begin_s, t_end_s] */
    uint32_t max_gap_us;        /* longest stretch of the phase without a sample, its two edges included */
} tri_phase_summary;

enum { TRI_PHASE_IDLE = 0, TRI_PHASE_PREFILL = 1, TRI_PHASE_DECODE = 2, TRI_PHASE_ROOFLINE = 3 };

/* Low-level sampler: a host thread polls NVML every period_us (>= 1000) into buf[0..cap), tagging
 * each sample with the current phase.  *handle receives an opaque pointer.  When cap is reached
 * sampling stops silently and phase_trace_stop returns TRI_ERR_BUFFER_TOO_SMALL (data kept).
 * Cadence: the period is a request, not a guarantee.  NVML queries are quick on an idle or memory-bound GPU (tens of
 * microseconds) but were seen to take tens of milliseconds each while the prefill GEMM saturates the part, and the
 * first query after an idle spell to block for over a second; phase_trace_start therefore issues every query once
 * before it takes the time origin, a late sampler does not burst to catch up, and each sample records its own
 * read_us, so that gaps are visible in the data (tri_phase_summary.max_gap_us, expected_samples) instead of assumed
 * away. */
int phase_trace_start(int device, unsigned period_us, tri_sample *buf, size_t cap, void **handle);
int phase_trace_mark(void *handle, int phase); /* atomic tag switch; any thread */
int phase_trace_stop(void *handle, size_t *n_samples); /* joins the sampler thread, frees the handle */

/* Caller-owned DEVICE buffers and shapes for the two phase kernels. */
typedef struct {
    int pm, pn, pk;             /* prefill GEMM shape (config 4: 4096, 18944, 3584) */
    const uint16_t *pa;         /* A [pm][pk] bf16, lda = pk */
    const uint16_t *pw;         /* W, layout w_layout, ld = pk (NK) or pn (KN) */
    uint16_t *pc;               /* C [pm][pn] bf16, ldc = pn */
    int dm, dn, dk;             /* decode GEMV shape (config 3: 8, 18944, 3584) */
    const uint16_t *dx;         /* X [dm][dk] */
    const uint16_t *const *dw_ring; /* HOST array of dw_count device pointers: rotating weight copies */
    int dw_count;               /* >= 1; rotate so the stream stays HBM-resident, not L2-resident */
    uint16_t *dy;               /* Y [dm][dn] */
    int w_layout;
    void *stream;
} tri_trace_workload;

/* Config-5 driver (blocking; runs on the calling host thread): repeats
 * [prefill GEMM for prefill_s | decode GEMV for decode_s | idle for idle_s] until total_s has
 * elapsed, sampling NVML every period_ms.  Kernels are launched back to back with a bounded queue
 * depth; the idle phase launches nothing and blocks the host thread (stands in for the sem_wait
 * dependency stall).  samples[0..cap) / summaries[0..scap) are filled; the counts
 * are returned through n_samples / n_summaries. */
int phase_trace(const tri_trace_workload *wl, double total_s, double prefill_s, double decode_s,
                double idle_s, unsigned period_ms, tri_sample *samples, size_t cap, size_t *n_samples,
                tri_phase_summary *summaries, size_t scap, size_t *n_summaries);

/* NVML actuation primitive of the paper.  TRI_ERR_NO_PERMISSION is a normal outcome. */
int tri_lock_clocks(int device, unsigned sm_mhz, unsigned mem_mhz); /* mem_mhz == 0: leave memory clock */
int tri_reset_clocks(int device);

/* One NVML reading outside a trace (phase = -1). */
int tri_nvml_sample(int device, tri_sample *out);

/* SM clock seen from inside the GPU: a one-block kernel spins for about spin_us microseconds and
 * returns delta(clock64) / delta(globaltimer ns) * 1000 in *mhz.  Blocking (synchronises stream). */
int tri_sm_clock_mhz(unsigned spin_us, double *mhz, void *stream);

/* ------------------------------------------------------------------------------------------------
 * f3. A.I.-aware frequency selection (section III-C): the throughput and power
 *     models the sweep data feed, and the Eq. 6 solver.  HOST functions: no GPU, no NVML; every pointer
 *     is host memory owned by the caller.  Clocks in MHz, throughput in any one unit (TFLOP/s here),
 *     A.I. in FLOP/byte, beta in throughput per unit A.I. (bandwidth), eta in throughput per MHz.
 */
typedef struct {
    double eta;             /* peak throughput per MHz: compute roof = eta * f            (Eq. 1)          */
    double beta;            /* memory coefficient:      memory roof  = beta * ai          (Eq. 1)          */
    double omega, gamma;    /* saturation term ai / (ai + omega * f^gamma) of Eq. 4; omega = 0 is Eq. 1     */
    double p_tdp;           /* power cap of Eq. 2 (W)                                                       */
    int32_t n_f;            /* number of supported clocks                                                   */
    const double *f_mhz;    /* n_f clocks, strictly ascending (the discrete levels the solver searches)     */
    const double *p_idle_w; /* P_idle(f) at those clocks                                                    */
    const double *p_dyn_w;  /* P_dyn(f)  at those clocks                                                    */
} tri_model;

/* Eq. 4: min(eta f ai / (ai + omega f^gamma), beta ai).  NaN if an argument is not positive / finite. */
double tri_model_theta(const tri_model *m, double ai, double f_mhz);
/* Eq. 3: min(eta f / (beta ai), beta ai / (eta f)), in (0, 1]. */
double tri_model_phi(const tri_model *m, double ai, double f_mhz);
/* Eq. 2 at the i-th supported clock: min(P_idle[i] + P_dyn[i] * phi(ai, f[i]), P_tdp).  NaN if i is out of range. */
double tri_model_power(const tri_model *m, double ai, int32_t i);
/* Eq. 5: duration-weighted A.I. of a phase, sum(d_i ai_i) / sum(d_i); NaN if n == 0 or sum(d) <= 0. */
double tri_phase_ai(const double *d, const double *ai, size_t n);
/* The premise of the Eq. 6 solver, checked ONCE per (model, phase A.I.) — O(n_f): the clock table is positive and
 * strictly ascending, the power tables non-negative, p_tdp positive, and at this A.I. theta(ai, f) and the modelled
 * power are non-decreasing along the table ("monotone frequency levels").  TRI_ERR_INVALID_ARG otherwise. */
int tri_model_validate(const tri_model *m, double ai);
/* Eq. 6: among the supported clocks f <= f_limit_mhz with theta(ai, f) >= (1 - eps) * theta(ai, f_max)
 * (f_max = the highest supported clock), the one of least modelled power; ties go to the HIGHEST such clock
 * ("the highest frequency that achieves this lower power").  Solved as the paper does — "a low-overhead solver ...
 * for every decode period", P:186-188 — by three binary searches over the discrete levels: O(log n_f) model
 * evaluations, no scan of the tables.  Exact on a model that passed tri_model_validate(m, ai); on one that would not,
 * the result is still an index <= the highest clock <= f_limit_mhz, but need not be the optimum.
 * TRI_ERR_INVALID_ARG if a pointer is NULL, n_f < 1, ai / f_limit_mhz is not positive, eps is outside [0, 1), or no
 * clock <= f_limit_mhz exists.  If no clock meets the throughput constraint the highest clock <= f_limit_mhz is
 * returned (best effort, *feasible = 0).  Outputs: index into f_mhz, and flag. */
int tri_solve_clock(const tri_model *m, double ai, double f_limit_mhz, double eps, int32_t *index, int32_t *feasible);
/* Fit of Eq. 4 to n measured points (ai_i, f_i, theta_i) at a caller-chosen gamma: beta = mean of theta / ai over
 * the points with ai <= ai_mem (memory branch); on the compute branch f / theta = 1 / eta + (omega / eta) * f^gamma / ai
 * is a straight line, so eta and omega come from the ordinary least-squares line of f / theta against f^gamma / ai over
 * the points with ai >= ai_cmp (omega is clamped at 0).  Writes m->eta, m->beta, m->omega, m->gamma only.
 * TRI_ERR_INVALID_ARG if the memory set is empty, the compute set has fewer than 2 distinct abscissae, or a value
 * is not positive and finite. */
int tri_fit_theta(const double *ai, const double *f_mhz, const double *theta, size_t n, double ai_mem, double ai_cmp,
                  double gamma, tri_model *m);
/* Fit of Eq. 2 at ONE clock: among the n measured points (ai_i, f_i, p_i) those with |f_i - f_sel_mhz| <= f_tol_mhz and
 * p_i < p_cap_w (not limited by the cap) give P_idle(f_sel) and P_dyn(f_sel) as intercept and slope of the ordinary
 * least-squares line of p against phi(ai_i, f_i) (Eq. 3 with m->eta, m->beta).  TRI_ERR_INVALID_ARG with fewer than 2
 * distinct abscissae or non-finite input.  *n_used (optional) returns how many points qualified. */
int tri_fit_power(const double *ai, const double *f_mhz, const double *p_w, size_t n, const tri_model *m, double f_sel_mhz,
                  double f_tol_mhz, double p_cap_w, double *p_idle_w, double *p_dyn_w, size_t *n_used);

/* ------------------------------------------------------------------------------------------------
 * f2 / f4. The two event-driven clock policies of the paper as HOST functions that only COMPUTE the schedule: nothing is
 *     actuated here, the caller (which may hold the right to call tri_lock_clocks; tenants of a shared pool do not) applies
 *     it.  A step with auto_boost = 1 means "release the lock" (tri_reset_clocks); otherwise lock SM (and, if mem_mhz > 0,
 *     memory) to the given clocks.  duration_s = 0 means "until the next event".
 */
typedef struct {
    double sm_mhz, mem_mhz;
    double duration_s;
    int32_t auto_boost;
    int32_t reserved;
} tri_clock_step;

/* Thermal-headroom-aware pace-and-race for a high-A.I. phase (section III-D).  sustained_mhz[0..n): the
 * SM clock each A.I. point holds in steady state (`characterise thermal` measures them).  f_mhz[0..n_f): the supported clock
 * levels, strictly ascending.  Pace clock = "the highest frequency that can run sustainably across all A.I." = the highest
 * level that exceeds no entry of sustained_mhz; out[0] = pace at that clock for pace_fraction * prefill_s, out[1] = race on
 * auto-boost for the rest (the paper: pace_fraction = 0.10).  TRI_ERR_INVALID_ARG on NULL, n == 0, n_f < 1, levels not
 * ascending, a non-positive / non-finite value, pace_fraction outside [0, 1], or when even the lowest level exceeds some
 * sustained clock (no level is sustainable everywhere). */
int tri_policy_pace_race(const double *sustained_mhz, size_t n, const double *f_mhz, int32_t n_f, double prefill_s,
                         double pace_fraction, tri_clock_step out[2]);
/* Dependency-stall-aware idle clocks (section III-B): entering != 0 is the sem_wait() entry - lock
 * SM / memory to idle_sm_mhz / idle_mem_mhz, where a value <= 0 selects the paper's 210 / 810 MHz (the lowest P8 state);
 * entering == 0 is the exit - restore auto-boost.  TRI_ERR_INVALID_ARG on NULL or a non-finite clock. */
int tri_policy_stall(int entering, double idle_sm_mhz, double idle_mem_mhz, tri_clock_step *out);

#ifdef __cplusplus
}
#endif
#endif /* TRIROOF_H_ */
