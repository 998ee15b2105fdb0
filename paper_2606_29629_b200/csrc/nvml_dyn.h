// NVML resolved at run time with dlopen("libnvidia-ml.so.1") — the build box has only the stub and the
// compute calls must keep working where NVML is absent (include/triroof.h, TRI_ERR_NVML_UNAVAILABLE).
// Only the handful of entry points the phase tracer and the clock-lock helpers use.
#pragma once
#include <cstdint>
#include "../../include/triroof.h"

namespace tri {
namespace nvml {

typedef struct nvmlDevice_st *Device;
enum { SUCCESS = 0, ERROR_NOT_SUPPORTED = 3, ERROR_NO_PERMISSION = 4 };
enum { CLOCK_SM = 1, CLOCK_MEM = 2 };
enum { TEMPERATURE_GPU = 0 };

struct Api {
    bool ok = false;
    int (*init)(void) = nullptr;
    int (*shutdown)(void) = nullptr;
    const char *(*error_string)(int) = nullptr;
    int (*device_by_index)(unsigned, Device *) = nullptr;
    int (*device_by_pci)(const char *, Device *) = nullptr;
    int (*clock_info)(Device, int, unsigned *) = nullptr;
    int (*temperature)(Device, int, unsigned *) = nullptr;
    int (*power_usage)(Device, unsigned *) = nullptr;
    int (*total_energy)(Device, unsigned long long *) = nullptr;
    int (*clock_reasons)(Device, unsigned long long *) = nullptr;
    int (*set_gpu_locked)(Device, unsigned, unsigned) = nullptr;
    int (*reset_gpu_locked)(Device) = nullptr;
    int (*set_mem_locked)(Device, unsigned, unsigned) = nullptr;
    int (*reset_mem_locked)(Device) = nullptr;
};

// Loads and initialises NVML once per process; returns nullptr (with tri::fail text set) if unavailable.
const Api *api();
// NVML handle of CUDA device `device` (matched through its PCI bus id); nullptr on failure.
Device device_handle(int device);
// Resets clocks locked through tri_lock_clocks (by the handle they were locked through) and unloads NVML; false (and
// nothing done) while a sampler thread is registered.
bool unload();
void tracer_enter();
void tracer_leave();
// Fills the NVML fields of *s (t_s and phase are left to the caller).
// with_energy = false skips nvmlDeviceGetTotalEnergyConsumption (measured on B200: 4 ms idle, 10-13 ms under load, against
// microseconds for the other queries) and leaves s->energy_mj untouched.
int read_sample(const Api *a, Device h, tri_sample *s, bool with_energy = true);

}  // namespace nvml
}  // namespace tri
