// a4. Phase trace (BASELINE.json config 5; ABI in include/triroof.h).
// A host sampler thread polls NVML (SM / memory clock, temperature, power, cumulative energy,
// clocks-event reasons) every period into a caller-owned buffer, tagging each sample with the phase
// current at that instant; phase_trace() is the config-5 driver that alternates the prefill GEMM, the
// decode GEMV and an idle gap and reduces the samples to per-phase summaries.
#include "nvml_dyn.h"
#include "tri_internal.h"

#include <time.h>
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>
#include <thread>
#include <vector>

namespace tri {

static double now_s()
{
    timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return (double)ts.tv_sec + 1e-9 * (double)ts.tv_nsec;
}

static void sleep_until(double t_abs)
{
    timespec ts;
    ts.tv_sec = (time_t)t_abs;
    ts.tv_nsec = (long)((t_abs - (double)ts.tv_sec) * 1e9);
    while (clock_nanosleep(CLOCK_MONOTONIC, TIMER_ABSTIME, &ts, nullptr) != 0) {
    }
}

struct Tracer {
    const nvml::Api *api = nullptr;
    nvml::Device dev = nullptr;
    tri_sample *buf = nullptr;
    size_t cap = 0;
    std::atomic<size_t> n{0};
    std::atomic<int> phase{TRI_PHASE_IDLE};
    std::atomic<bool> stop{false};
    bool overflow = false;
    unsigned period_us = 10000;
    double t0 = 0.0;
    std::atomic<uint64_t> energy_mj{0};
    std::mutex energy_mu;                 // one energy query at a time: the poller below and the driver's phase-edge reads
    std::thread th, eth;

    uint64_t read_energy(uint64_t fallback)
    {
        unsigned long long e = 0;
        std::lock_guard<std::mutex> lk(energy_mu);
        if (api->total_energy && api->total_energy(dev, &e) == nvml::SUCCESS) return e;
        return fallback;
    }

    // The energy counter is the one slow NVML query (4-13 ms on B200, more while the driver is busy launching): it is polled
    // by a thread of its own about every 100 ms and the sampler copies the last value, so that the clock / temperature /
    // power samples keep the requested period whatever that query costs.
    void run_energy()
    {
        const double step = period_us >= 100000 ? 1e-6 * period_us : 0.1;
        double next = now_s();
        while (!stop.load(std::memory_order_acquire)) {
            energy_mj.store(read_energy(energy_mj.load(std::memory_order_relaxed)), std::memory_order_release);
            next += step;
            const double t = now_s();
            if (next < t) next = t;
            // sleep in slices of at most 20 ms so that stop() is not held up by a whole step
            while (!stop.load(std::memory_order_acquire) && now_s() < next) sleep_until(std::min(next, now_s() + 0.02));
        }
    }

    void run()
    {
        double next = t0;
        while (!stop.load(std::memory_order_acquire)) {
            size_t i = n.load(std::memory_order_relaxed);
            if (i >= cap) {
                overflow = true;
                break;
            }
            tri_sample s;
            memset(&s, 0, sizeof(s));
            const double t_before = now_s();
            nvml::read_sample(api, dev, &s, false);
            s.energy_mj = energy_mj.load(std::memory_order_acquire);
            const double t_after = now_s();
            s.t_s = t_after - t0;                      // stamped after the reads: the values are at most read_us old
            s.read_us = (uint32_t)std::min((t_after - t_before) * 1e6, 4.0e9);   // a blocked NVML call shows in the record
            s.phase = phase.load(std::memory_order_acquire);
            buf[i] = s;
            n.store(i + 1, std::memory_order_release);
            next += 1e-6 * period_us;
            double t = now_s();
            if (next < t) next = t;                    // NVML was slower than the period: do not burst
            sleep_until(next);
        }
    }
};

// Reduces samples[0..ns) in [t_begin, t_end] into the clock / temperature / cadence fields of *out.
// First / last 10 % are spans of TIME, not of whatever samples there are: a window that lost its opening samples to a
// slow NVML call reports 0 for sm_mhz_first10 instead of passing off its middle as its start (Fig. 4a, PAPER.md line 104,
// is exactly that number).  max_gap_us counts the window's edges too: begin to first sample, last sample to end.
static void reduce_window(const tri_sample *samples, size_t ns, double period_s, tri_phase_summary *out)
{
    const double tb = out->t_begin_s, te = out->t_end_s, dur = te - tb;
    out->expected_samples = period_s > 0 && dur > 0 ? (int32_t)std::min(std::floor(dur / period_s), 2.0e9) : 0;
    double sum = 0.0, tmax = 0.0, f = 0.0, l = 0.0, prev = tb, gap = 0.0;
    uint32_t n = 0, nf = 0, nl = 0;
    for (size_t i = 0; i < ns; ++i) {
        const tri_sample &s = samples[i];
        if (s.t_s < tb || s.t_s > te) continue;
        ++n;
        sum += s.sm_mhz;
        if (s.temp_c > tmax) tmax = s.temp_c;
        if (s.t_s - prev > gap) gap = s.t_s - prev;
        prev = s.t_s;
        if (s.t_s <= tb + 0.1 * dur) { f += s.sm_mhz; ++nf; }
        if (s.t_s >= te - 0.1 * dur) { l += s.sm_mhz; ++nl; }
    }
    if (te - prev > gap) gap = te - prev;
    out->max_gap_us = (uint32_t)std::min(gap * 1e6, 4.0e9);
    out->n_samples = n;
    if (n == 0) return;
    out->sm_mhz_mean = (float)(sum / (double)n);
    out->temp_c_max = (float)tmax;
    out->sm_mhz_first10 = nf ? (float)(f / (double)nf) : 0.f;
    out->sm_mhz_last10 = nl ? (float)(l / (double)nl) : 0.f;
}

}  // namespace tri

extern "C" {
int phase_trace_start(int device, unsigned period_us, tri_sample *buf, size_t cap, void **handle)
{
    if (!buf || !handle || cap == 0) return tri::fail(TRI_ERR_INVALID_ARG, "buf/handle is NULL or cap is 0");
    if (period_us < 1000) return tri::fail(TRI_ERR_INVALID_ARG, "period_us = %u below 1000", period_us);
    const tri::nvml::Api *a = tri::nvml::api();
    if (!a) return TRI_ERR_NVML_UNAVAILABLE;
    tri::nvml::Device h = tri::nvml::device_handle(device);
    if (!h) return TRI_ERR_NVML_UNAVAILABLE;
    tri::Tracer *t = new (std::nothrow) tri::Tracer();
    if (!t) return tri::fail(TRI_ERR_INVALID_ARG, "out of host memory");
    t->api = a;
    t->dev = h;
    t->buf = buf;
    t->cap = cap;
    t->period_us = period_us;
    tri::nvml::tracer_enter();                    // tri_shutdown() keeps NVML loaded while this sampler runs
    {
        // Every query once, BEFORE the time origin: the first NVML call after an idle spell can block for a long time (1.25 s
        // seen on a fresh B200 lease after 1 s of idle), and that cost belongs to set-up, not to the trace.  The energy
        // value read here is what the first samples carry.
        tri_sample warm;
        memset(&warm, 0, sizeof(warm));
        tri::nvml::read_sample(a, h, &warm, false);
        t->energy_mj.store(t->read_energy(0));
    }
    t->t0 = tri::now_s();
    t->th = std::thread([t] { t->run(); });
    t->eth = std::thread([t] { t->run_energy(); });
    *handle = t;
    return TRI_OK;
}

int phase_trace_mark(void *handle, int phase)
{
    if (!handle) return tri::fail(TRI_ERR_INVALID_ARG, "handle is NULL");
    static_cast<tri::Tracer *>(handle)->phase.store(phase, std::memory_order_release);
    return TRI_OK;
}

int phase_trace_stop(void *handle, size_t *n_samples)
{
    if (!handle) return tri::fail(TRI_ERR_INVALID_ARG, "handle is NULL");
    tri::Tracer *t = static_cast<tri::Tracer *>(handle);
    t->stop.store(true, std::memory_order_release);
    if (t->th.joinable()) t->th.join();
    if (t->eth.joinable()) t->eth.join();
    tri::nvml::tracer_leave();
    if (n_samples) *n_samples = t->n.load();
    bool ovf = t->overflow;
    delete t;
    if (ovf) return tri::fail(TRI_ERR_BUFFER_TOO_SMALL, "sample buffer full; trace truncated");
    return TRI_OK;
}

int phase_trace(const tri_trace_workload *wl, double total_s, double prefill_s, double decode_s, double idle_s,
                unsigned period_ms, tri_sample *samples, size_t cap, size_t *n_samples, tri_phase_summary *summaries,
                size_t scap, size_t *n_summaries)
{
    using namespace tri;
    if (!wl || !samples || !summaries || !n_samples || !n_summaries) return fail(TRI_ERR_INVALID_ARG, "NULL argument");
    if (!(total_s > 0) || prefill_s < 0 || decode_s < 0 || idle_s < 0 || prefill_s + decode_s + idle_s <= 0)
        return fail(TRI_ERR_INVALID_ARG, "durations must be non-negative with a positive cycle and total");
    if (period_ms < 1) return fail(TRI_ERR_INVALID_ARG, "period_ms must be >= 1");
    if (prefill_s > 0 && (!wl->pa || !wl->pw || !wl->pc)) return fail(TRI_ERR_INVALID_ARG, "prefill buffers are NULL");
    if (decode_s > 0 && (!wl->dx || !wl->dw_ring || wl->dw_count < 1 || !wl->dy))
        return fail(TRI_ERR_INVALID_ARG, "decode buffers are NULL or dw_count < 1");
    *n_samples = 0;
    *n_summaries = 0;
    const DeviceInfo *di = nullptr;
    int st = ensure_init(&di);
    if (st != TRI_OK) return st;
    const nvml::Api *a = nvml::api();
    if (!a) return TRI_ERR_NVML_UNAVAILABLE;
    nvml::Device h = nvml::device_handle(di->device);
    if (!h) return TRI_ERR_NVML_UNAVAILABLE;

    cudaStream_t s = static_cast<cudaStream_t>(wl->stream);
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};      // e0, e1 (timed), ring[0..1] (queue depth)
    auto destroy_events = [&ev] {
        for (cudaEvent_t &e : ev)
            if (e) {
                cudaEventDestroy(e);
                e = nullptr;
            }
    };
    for (int i = 0; i < 4; ++i) {
        cudaError_t ce = i < 2 ? cudaEventCreate(&ev[i]) : cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming);
        if (ce != cudaSuccess) {
            destroy_events();
            return fail(TRI_ERR_CUDA, "cudaEventCreate: %s", cudaGetErrorString(ce));
        }
    }
    cudaEvent_t e0 = ev[0], e1 = ev[1], ring[2] = {ev[2], ev[3]};

    void *handle = nullptr;
    st = phase_trace_start(di->device, period_ms * 1000u, samples, cap, &handle);
    if (st != TRI_OK) {
        destroy_events();
        return st;
    }
    Tracer *tr = static_cast<Tracer *>(handle);
    const double t0 = tr->t0;
    // The first phase begins once the sampler has delivered a sample (normally a fraction of a period; bounded at 2 s), so
    // that the opening of the first window - the Fig. 4a number - is never lost to a slow first read.
    for (const double tw = now_s(); tr->n.load(std::memory_order_acquire) == 0 && now_s() - tw < 2.0;) sleep_until(now_s() + 0.001);

    const int lda = wl->pk, ldc = wl->pn, ldx = wl->dk, ldy = wl->dn;
    const int p_ldw = wl->w_layout == TRI_W_NK ? wl->pk : wl->pn;
    const int d_ldw = wl->w_layout == TRI_W_NK ? wl->dk : wl->dn;
    const double p_flop = 2.0 * wl->pm * (double)wl->pn * wl->pk;
    const double p_bytes = 2.0 * ((double)wl->pm * wl->pk + (double)wl->pk * wl->pn + (double)wl->pm * wl->pn);
    const double d_flop = 2.0 * wl->dm * (double)wl->dn * wl->dk;
    const double d_bytes = 2.0 * ((double)wl->dm * wl->dk + (double)wl->dk * wl->dn + (double)wl->dm * wl->dn);

    int status = TRI_OK;
    size_t nsum = 0;
    uint64_t dcalls = 0;
    bool truncated = false;
    const int phases[3] = {TRI_PHASE_PREFILL, TRI_PHASE_DECODE, TRI_PHASE_IDLE};
    const double durs[3] = {prefill_s, decode_s, idle_s};
    while (status == TRI_OK && now_s() - t0 < total_s) {
        for (int pi = 0; pi < 3 && status == TRI_OK; ++pi) {
            if (durs[pi] <= 0) continue;
            double remaining = total_s - (now_s() - t0);
            if (remaining <= 0) break;
            const double dur = durs[pi] < remaining ? durs[pi] : remaining;
            const int ph = phases[pi];
            tri_phase_summary sm;
            memset(&sm, 0, sizeof(sm));
            sm.phase = ph;
            phase_trace_mark(handle, ph);
            const uint64_t en0 = tr->read_energy(0);
            const double tb = now_s();
            sm.t_begin_s = tb - t0;
            if (ph == TRI_PHASE_IDLE) {
                sleep_until(tb + dur);                  // no kernels queued, context alive, host thread blocked
            } else {
                const unsigned depth = ph == TRI_PHASE_PREFILL ? 4u : 64u;   // launches per queue-bounding event
                cudaError_t ce = cudaEventRecord(e0, s);
                if (ce != cudaSuccess) status = fail(TRI_ERR_CUDA, "cudaEventRecord: %s", cudaGetErrorString(ce));
                uint64_t launches = 0;
                unsigned slot = 0;
                bool have[2] = {false, false};
                while (status == TRI_OK && now_s() - tb < dur) {
                    for (unsigned q = 0; q < depth; ++q) {
                        if (ph == TRI_PHASE_PREFILL)
                            status = prefill_gemm(wl->pm, wl->pn, wl->pk, wl->pa, lda, wl->pw, p_ldw, wl->w_layout, wl->pc, ldc, s);
                        else
                            status = decode_gemv(wl->dm, wl->dn, wl->dk, wl->dx, ldx, wl->dw_ring[dcalls++ % wl->dw_count], d_ldw,
                                                 wl->w_layout, wl->dy, ldy, s);
                        if (status != TRI_OK) break;
                        ++launches;
                    }
                    if (status != TRI_OK) break;
                    ce = cudaEventRecord(ring[slot], s);
                    if (ce != cudaSuccess) {
                        status = fail(TRI_ERR_CUDA, "cudaEventRecord: %s", cudaGetErrorString(ce));
                        break;
                    }
                    have[slot] = true;
                    slot ^= 1;
                    if (have[slot]) cudaEventSynchronize(ring[slot]);   // at most 2 * depth launches in flight
                }
                ce = cudaEventRecord(e1, s);
                if (ce == cudaSuccess) ce = cudaEventSynchronize(e1);
                if (ce != cudaSuccess && status == TRI_OK) status = fail(TRI_ERR_CUDA, "phase end: %s", cudaGetErrorString(ce));
                float ms = 0.f;
                if (status == TRI_OK) cudaEventElapsedTime(&ms, e0, e1);
                sm.gpu_ms = ms;
                sm.launches = launches;
                const double per_flop = ph == TRI_PHASE_PREFILL ? p_flop : d_flop;
                const double per_bytes = ph == TRI_PHASE_PREFILL ? p_bytes : d_bytes;
                sm.flop = per_flop * (double)launches;
                sm.bytes = per_bytes * (double)launches;
                sm.tokens = (double)(ph == TRI_PHASE_PREFILL ? wl->pm : wl->dm) * (double)launches;
            }
            const double te = now_s();
            const uint64_t en1 = tr->read_energy(0);
            sm.t_end_s = te - t0;
            sm.energy_j = en1 >= en0 ? 1e-3 * (double)(en1 - en0) : 0.0;
            if (nsum < scap) summaries[nsum++] = sm;
            else truncated = true;
        }
    }
    phase_trace_mark(handle, TRI_PHASE_IDLE);
    size_t ns = 0;
    int st2 = phase_trace_stop(handle, &ns);
    *n_samples = ns;
    for (size_t i = 0; i < nsum; ++i) {
        tri_phase_summary *q = &summaries[i];
        reduce_window(samples, ns, 1e-3 * period_ms, q);
        const double dt = q->t_end_s - q->t_begin_s;
        if (q->energy_j <= 0.0 && q->n_samples > 0) {          // no energy counter: integrate the power samples
            double pw = 0.0;
            uint32_t c = 0;
            for (size_t j = 0; j < ns; ++j)
                if (samples[j].t_s >= q->t_begin_s && samples[j].t_s <= q->t_end_s) { pw += samples[j].power_w; ++c; }
            q->energy_j = c ? pw / c * dt : 0.0;
        }
        q->mean_power_w = dt > 0 ? q->energy_j / dt : 0.0;
        q->j_per_flop = q->flop > 0 ? q->energy_j / q->flop : 0.0;
        q->j_per_byte = q->bytes > 0 ? q->energy_j / q->bytes : 0.0;
        q->j_per_token = q->tokens > 0 ? q->energy_j / q->tokens : 0.0;
    }
    *n_summaries = nsum;
    destroy_events();
    if (status != TRI_OK) return status;
    if (st2 != TRI_OK) return st2;
    if (truncated) return fail(TRI_ERR_BUFFER_TOO_SMALL, "summary buffer full; later phases dropped");
    return TRI_OK;
}

}  // extern "C"
