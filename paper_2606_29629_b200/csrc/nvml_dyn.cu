// Run-time NVML binding, clock-lock helpers and single-sample read (include/triroof.h: a4 helpers).
#include "nvml_dyn.h"

#include <time.h>
#include "tri_internal.h"

#include <dlfcn.h>
#include <cstring>
#include <mutex>

namespace tri {
namespace nvml {

static std::mutex g_mu;
static void *g_lib = nullptr;
static Api g_api;
static bool g_tried = false;
static Device g_locked_handle[64] = {nullptr};   // by CUDA ordinal: the NVML handle the lock was taken through (ordinals differ
                                                    // from NVML indices under CUDA_VISIBLE_DEVICES, so unload() must not re-derive it)
static int g_active_tracers = 0;                    // sampler threads using g_api; unload() waits for none

template <typename F>
static bool sym(F &f, const char *name, const char *alt = nullptr)
{
    void *p = dlsym(g_lib, name);
    if (!p && alt) p = dlsym(g_lib, alt);
    f = reinterpret_cast<F>(p);
    return p != nullptr;
}

const Api *api()
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (g_api.ok) return &g_api;
    if (g_tried) {
        fail(TRI_ERR_NVML_UNAVAILABLE, "NVML unavailable (earlier load attempt failed)");
        return nullptr;
    }
    g_tried = true;
    g_lib = dlopen("libnvidia-ml.so.1", RTLD_NOW | RTLD_LOCAL);
    if (!g_lib) {
        fail(TRI_ERR_NVML_UNAVAILABLE, "dlopen(libnvidia-ml.so.1): %s", dlerror());
        return nullptr;
    }
    Api a;
    bool ok = sym(a.init, "nvmlInit_v2", "nvmlInit") && sym(a.shutdown, "nvmlShutdown") &&
              sym(a.error_string, "nvmlErrorString") && sym(a.device_by_index, "nvmlDeviceGetHandleByIndex_v2", "nvmlDeviceGetHandleByIndex") &&
              sym(a.clock_info, "nvmlDeviceGetClockInfo") && sym(a.temperature, "nvmlDeviceGetTemperature") &&
              sym(a.power_usage, "nvmlDeviceGetPowerUsage");
    sym(a.device_by_pci, "nvmlDeviceGetHandleByPciBusId_v2", "nvmlDeviceGetHandleByPciBusId");
    sym(a.total_energy, "nvmlDeviceGetTotalEnergyConsumption");
    sym(a.clock_reasons, "nvmlDeviceGetCurrentClocksEventReasons", "nvmlDeviceGetCurrentClocksThrottleReasons");
    sym(a.set_gpu_locked, "nvmlDeviceSetGpuLockedClocks");
    sym(a.reset_gpu_locked, "nvmlDeviceResetGpuLockedClocks");
    sym(a.set_mem_locked, "nvmlDeviceSetMemoryLockedClocks");
    sym(a.reset_mem_locked, "nvmlDeviceResetMemoryLockedClocks");
    if (!ok) {
        fail(TRI_ERR_NVML_UNAVAILABLE, "libnvidia-ml.so.1 lacks a required symbol");
        dlclose(g_lib);
        g_lib = nullptr;
        return nullptr;
    }
    int r = a.init();
    if (r != SUCCESS) {
        fail(TRI_ERR_NVML_UNAVAILABLE, "nvmlInit: %s", a.error_string ? a.error_string(r) : "error");
        dlclose(g_lib);
        g_lib = nullptr;
        return nullptr;
    }
    a.ok = true;
    g_api = a;
    return &g_api;
}

Device device_handle(int device)
{
    const Api *a = api();
    if (!a) return nullptr;
    Device h = nullptr;
    char bus[64] = "";
    if (a->device_by_pci && cudaDeviceGetPCIBusId(bus, sizeof(bus), device) == cudaSuccess &&
        a->device_by_pci(bus, &h) == SUCCESS)
        return h;
    cudaGetLastError();
    int r = a->device_by_index((unsigned)device, &h);
    if (r != SUCCESS) {
        fail(TRI_ERR_NVML_UNAVAILABLE, "nvmlDeviceGetHandleByIndex(%d): %s", device, a->error_string(r));
        return nullptr;
    }
    return h;
}

void tracer_enter()
{
    std::lock_guard<std::mutex> lk(g_mu);
    ++g_active_tracers;
}

void tracer_leave()
{
    std::lock_guard<std::mutex> lk(g_mu);
    --g_active_tracers;
}

bool unload()
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (g_active_tracers > 0) return false;       // a sampler thread is inside NVML: keep the library mapped
    if (g_api.ok) {
        for (int d = 0; d < 64; ++d)
            if (g_locked_handle[d]) {
                if (g_api.reset_gpu_locked) g_api.reset_gpu_locked(g_locked_handle[d]);
                if (g_api.reset_mem_locked) g_api.reset_mem_locked(g_locked_handle[d]);
                g_locked_handle[d] = nullptr;
            }
        g_api.shutdown();
        g_api = Api();
    }
    if (g_lib) {
        dlclose(g_lib);
        g_lib = nullptr;
    }
    g_tried = false;
    return true;
}

int read_sample(const Api *a, Device h, tri_sample *s, bool with_energy)
{
    unsigned v = 0;
    unsigned long long e = 0;
    s->sm_mhz = (a->clock_info(h, CLOCK_SM, &v) == SUCCESS) ? v : 0;
    s->mem_mhz = (a->clock_info(h, CLOCK_MEM, &v) == SUCCESS) ? v : 0;
    s->temp_c = (a->temperature(h, TEMPERATURE_GPU, &v) == SUCCESS) ? v : 0;
    s->power_w = (a->power_usage(h, &v) == SUCCESS) ? (float)v * 1e-3f : 0.f;
    if (with_energy) s->energy_mj = (a->total_energy && a->total_energy(h, &e) == SUCCESS) ? e : 0;
    s->clk_event_reasons = (a->clock_reasons && a->clock_reasons(h, &e) == SUCCESS) ? e : 0;
    return TRI_OK;
}

}  // namespace nvml
void release_clock_scratch();
void release_splitk_workspaces();
}  // namespace tri

extern "C" {

int tri_nvml_sample(int device, tri_sample *out)
{
    if (!out) return tri::fail(TRI_ERR_INVALID_ARG, "out is NULL");
    const tri::nvml::Api *a = tri::nvml::api();
    if (!a) return TRI_ERR_NVML_UNAVAILABLE;
    tri::nvml::Device h = tri::nvml::device_handle(device);
    if (!h) return TRI_ERR_NVML_UNAVAILABLE;
    memset(out, 0, sizeof(*out));
    out->phase = -1;
    timespec t0, t1;
    clock_gettime(CLOCK_MONOTONIC, &t0);
    int st = tri::nvml::read_sample(a, h, out);
    clock_gettime(CLOCK_MONOTONIC, &t1);
    const double us = 1e6 * (double)(t1.tv_sec - t0.tv_sec) + 1e-3 * (double)(t1.tv_nsec - t0.tv_nsec);
    out->read_us = us < 4.0e9 ? (uint32_t)us : 4000000000u;      // the energy query included here (4-13 ms on B200)
    return st;
}

int tri_lock_clocks(int device, unsigned sm_mhz, unsigned mem_mhz)
{
    if (device < 0 || device >= 64 || sm_mhz == 0) return tri::fail(TRI_ERR_INVALID_ARG, "device/sm_mhz invalid");
    const tri::nvml::Api *a = tri::nvml::api();
    if (!a) return TRI_ERR_NVML_UNAVAILABLE;
    tri::nvml::Device h = tri::nvml::device_handle(device);
    if (!h) return TRI_ERR_NVML_UNAVAILABLE;
    if (!a->set_gpu_locked) return tri::fail(TRI_ERR_NVML_UNAVAILABLE, "nvmlDeviceSetGpuLockedClocks not exported");
    int r = a->set_gpu_locked(h, sm_mhz, sm_mhz);
    if (r == tri::nvml::ERROR_NO_PERMISSION) return tri::fail(TRI_ERR_NO_PERMISSION, "nvmlDeviceSetGpuLockedClocks: %s", a->error_string(r));
    if (r != tri::nvml::SUCCESS) return tri::fail(TRI_ERR_NVML_UNAVAILABLE, "nvmlDeviceSetGpuLockedClocks: %s", a->error_string(r));
    tri::nvml::g_locked_handle[device] = h;
    if (mem_mhz && a->set_mem_locked) {
        r = a->set_mem_locked(h, mem_mhz, mem_mhz);
        if (r == tri::nvml::ERROR_NO_PERMISSION) return tri::fail(TRI_ERR_NO_PERMISSION, "nvmlDeviceSetMemoryLockedClocks: %s", a->error_string(r));
        if (r != tri::nvml::SUCCESS) return tri::fail(TRI_ERR_NVML_UNAVAILABLE, "nvmlDeviceSetMemoryLockedClocks: %s", a->error_string(r));
    }
    return TRI_OK;
}

int tri_reset_clocks(int device)
{
    if (device < 0 || device >= 64) return tri::fail(TRI_ERR_INVALID_ARG, "device invalid");
    const tri::nvml::Api *a = tri::nvml::api();
    if (!a) return TRI_ERR_NVML_UNAVAILABLE;
    tri::nvml::Device h = tri::nvml::device_handle(device);
    if (!h) return TRI_ERR_NVML_UNAVAILABLE;
    int r = a->reset_gpu_locked ? a->reset_gpu_locked(h) : tri::nvml::ERROR_NOT_SUPPORTED;
    if (a->reset_mem_locked) a->reset_mem_locked(h);
    tri::nvml::g_locked_handle[device] = nullptr;
    if (r == tri::nvml::ERROR_NO_PERMISSION) return tri::fail(TRI_ERR_NO_PERMISSION, "nvmlDeviceResetGpuLockedClocks: %s", a->error_string(r));
    if (r != tri::nvml::SUCCESS) return tri::fail(TRI_ERR_NVML_UNAVAILABLE, "nvmlDeviceResetGpuLockedClocks: %s", a->error_string(r));
    return TRI_OK;
}

void tri_shutdown(void)
{
    // With a phase trace still running NVML stays loaded (its sampler thread is inside it) and clocks this process locked
    // stay locked until the trace has been stopped and tri_shutdown() is called again.
    tri::nvml::unload();
    tri::release_splitk_workspaces();
    tri::release_clock_scratch();
}

}  // extern "C"
