"""paper_2606_29629_b200 — thin Python binding of libtriroof.so (include/triroof.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of csrc/.  PyTorch is
used by callers for device memory and streams; this module accepts torch tensors (or raw integer
device pointers) and passes pointers / sizes through ctypes.  There is no CPU fallback: if the library
cannot be built or loaded, importing `lib()` raises.

Functions mirror the C ABI by name: roofline_run, roofline_run_k, decode_gemv, prefill_gemm,
phase_trace, phase_trace_start / mark / stop, tri_lock_clocks, tri_reset_clocks, tri_nvml_sample,
tri_sm_clock_mhz, tri_init, tri_shutdown.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import (POINTER, Structure, byref, c_char_p, c_double, c_float, c_int, c_int32, c_int64, c_size_t,
                    c_uint, c_uint16, c_uint32, c_uint64, c_void_p)

TRI_OK = 0
TRI_ERR_INVALID_ARG = 1
TRI_ERR_UNSUPPORTED_SHAPE = 2
TRI_ERR_ALIGNMENT = 3
TRI_ERR_CUDA = 4
TRI_ERR_ARCH = 5
TRI_ERR_NVML_UNAVAILABLE = 6
TRI_ERR_NO_PERMISSION = 7
TRI_ERR_BUFFER_TOO_SMALL = 8

TRI_W_NK = 0
TRI_W_KN = 1

TRI_PHASE_IDLE, TRI_PHASE_PREFILL, TRI_PHASE_DECODE, TRI_PHASE_ROOFLINE = 0, 1, 2, 3
PHASE_NAMES = {0: "idle", 1: "prefill", 2: "decode", 3: "roofline"}

A_DEFAULT = 0.9990234375
B_DEFAULT = 0.0009765625

# Every symbol include/triroof.h declares (tests check the library exports each one).
EXPORTS = ["tri_status_string", "tri_last_error", "tri_init", "tri_shutdown", "tri_sm_count", "tri_l2_bytes",
           "roofline_run", "roofline_run_k", "decode_gemv", "prefill_gemm", "phase_trace_start", "phase_trace_mark",
           "phase_trace_stop", "phase_trace", "tri_lock_clocks", "tri_reset_clocks", "tri_nvml_sample",
           "tri_sm_clock_mhz", "tri_model_theta", "tri_model_phi", "tri_model_power", "tri_phase_ai", "tri_model_validate", "tri_solve_clock",
           "tri_fit_theta", "tri_fit_power", "prefill_gemm_static_ws",
           "tri_policy_pace_race", "tri_policy_stall"]


class TriError(RuntimeError):
    def __init__(self, status: int, name: str, detail: str):
        self.status = status
        super().__init__(f"{name}: status {status} ({detail})")


class tri_model(Structure):
    """include/triroof.h tri_model (f3: PAPER.md Eq. 1-4 parameters + the P_idle / P_dyn tables on the clock list)."""
    _fields_ = [("eta", c_double), ("beta", c_double), ("omega", c_double), ("gamma", c_double), ("p_tdp", c_double),
                ("n_f", c_int32), ("f_mhz", POINTER(c_double)), ("p_idle_w", POINTER(c_double)), ("p_dyn_w", POINTER(c_double))]


class tri_clock_step(Structure):
    """include/triroof.h tri_clock_step: one step of a clock schedule (auto_boost = 1: release the lock)."""
    _fields_ = [("sm_mhz", c_double), ("mem_mhz", c_double), ("duration_s", c_double), ("auto_boost", c_int32), ("reserved", c_int32)]


class tri_sample(Structure):
    _fields_ = [("t_s", c_double), ("phase", c_int32), ("sm_mhz", c_uint32), ("mem_mhz", c_uint32),
                ("temp_c", c_uint32), ("power_w", c_float), ("read_us", c_uint32), ("energy_mj", c_uint64), ("clk_event_reasons", c_uint64)]


class tri_phase_summary(Structure):
    _fields_ = [("phase", c_int32), ("expected_samples", c_int32), ("t_begin_s", c_double), ("t_end_s", c_double),
                ("gpu_ms", c_double), ("launches", c_uint64), ("flop", c_double), ("bytes", c_double),
                ("tokens", c_double), ("energy_j", c_double), ("mean_power_w", c_double), ("j_per_flop", c_double),
                ("j_per_byte", c_double), ("j_per_token", c_double), ("sm_mhz_mean", c_float),
                ("sm_mhz_first10", c_float), ("sm_mhz_last10", c_float), ("temp_c_max", c_float),
                ("n_samples", c_uint32), ("max_gap_us", c_uint32)]


class tri_trace_workload(Structure):
    _fields_ = [("pm", c_int), ("pn", c_int), ("pk", c_int), ("pa", c_void_p), ("pw", c_void_p), ("pc", c_void_p),
                ("dm", c_int), ("dn", c_int), ("dk", c_int), ("dx", c_void_p), ("dw_ring", POINTER(c_void_p)),
                ("dw_count", c_int), ("dy", c_void_p), ("w_layout", c_int), ("stream", c_void_p)]


_lib = None


def library_path() -> str:
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "libtriroof.so")


def lib():
    """Loads (building first if the .so is missing or stale) libtriroof.so.  Raises if that fails."""
    global _lib
    if _lib is not None:
        return _lib
    from .build import build
    path = build()
    L = ctypes.CDLL(path)
    L.tri_status_string.argtypes = [c_int]
    L.tri_status_string.restype = c_char_p
    L.tri_last_error.argtypes = []
    L.tri_last_error.restype = c_char_p
    L.tri_init.argtypes = [c_int]
    L.tri_shutdown.argtypes = []
    L.tri_shutdown.restype = None
    L.tri_sm_count.argtypes = []
    L.tri_l2_bytes.argtypes = []
    L.tri_l2_bytes.restype = c_size_t
    L.roofline_run.argtypes = [c_double, c_size_t, c_void_p, c_void_p, c_void_p]
    L.roofline_run_k.argtypes = [c_uint, c_float, c_float, c_size_t, c_void_p, c_void_p, c_void_p]
    gemm_args = [c_int, c_int, c_int, c_void_p, c_int64, c_void_p, c_int64, c_int, c_void_p, c_int64, c_void_p]
    L.decode_gemv.argtypes = gemm_args
    L.prefill_gemm.argtypes = gemm_args
    L.prefill_gemm_static_ws.argtypes = gemm_args
    L.phase_trace_start.argtypes = [c_int, c_uint, POINTER(tri_sample), c_size_t, POINTER(c_void_p)]
    L.phase_trace_mark.argtypes = [c_void_p, c_int]
    L.phase_trace_stop.argtypes = [c_void_p, POINTER(c_size_t)]
    L.phase_trace.argtypes = [POINTER(tri_trace_workload), c_double, c_double, c_double, c_double, c_uint,
                              POINTER(tri_sample), c_size_t, POINTER(c_size_t), POINTER(tri_phase_summary), c_size_t,
                              POINTER(c_size_t)]
    L.tri_lock_clocks.argtypes = [c_int, c_uint, c_uint]
    L.tri_reset_clocks.argtypes = [c_int]
    L.tri_nvml_sample.argtypes = [c_int, POINTER(tri_sample)]
    L.tri_sm_clock_mhz.argtypes = [c_uint, POINTER(c_double), c_void_p]
    L.tri_fit_power.argtypes = [POINTER(c_double), POINTER(c_double), POINTER(c_double), c_size_t, POINTER(tri_model), c_double, c_double,
                                c_double, POINTER(c_double), POINTER(c_double), POINTER(c_size_t)]
    for name in ("tri_model_theta", "tri_model_phi"):
        getattr(L, name).argtypes = [POINTER(tri_model), c_double, c_double]
        getattr(L, name).restype = c_double
    L.tri_model_power.argtypes = [POINTER(tri_model), c_double, c_int32]
    L.tri_model_power.restype = c_double
    L.tri_phase_ai.argtypes = [POINTER(c_double), POINTER(c_double), c_size_t]
    L.tri_phase_ai.restype = c_double
    L.tri_model_validate.argtypes = [POINTER(tri_model), c_double]
    L.tri_solve_clock.argtypes = [POINTER(tri_model), c_double, c_double, c_double, POINTER(c_int32), POINTER(c_int32)]
    L.tri_fit_theta.argtypes = [POINTER(c_double), POINTER(c_double), POINTER(c_double), c_size_t, c_double, c_double, c_double,
                                POINTER(tri_model)]
    L.tri_policy_pace_race.argtypes = [POINTER(c_double), c_size_t, POINTER(c_double), c_int32, c_double, c_double, POINTER(tri_clock_step)]
    L.tri_policy_stall.argtypes = [c_int, c_double, c_double, POINTER(tri_clock_step)]
    for name in EXPORTS:
        if getattr(L, name).restype is None and name not in ("tri_shutdown",):
            getattr(L, name).restype = c_int
    _lib = L
    return L


def status_string(status: int) -> str:
    return lib().tri_status_string(status).decode()


def last_error() -> str:
    return lib().tri_last_error().decode()


def _check(status: int, name: str) -> None:
    if status != TRI_OK:
        raise TriError(status, name, f"{status_string(status)}: {last_error()}")


def _ptr(t) -> int:
    """Device (or host) address of a torch tensor / numpy array / int."""
    if t is None:
        return 0
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    if hasattr(t, "ctypes"):
        return t.ctypes.data
    raise TypeError(f"cannot take the address of {type(t)}")


def _stream(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def tri_init(device: int = 0) -> None:
    _check(lib().tri_init(device), "tri_init")


def tri_shutdown() -> None:
    lib().tri_shutdown()


def sm_count() -> int:
    return lib().tri_sm_count()


def l2_bytes() -> int:
    return lib().tri_l2_bytes()


def roofline_run(ai: float, n: int, inp, out, stream=None) -> None:
    """out[i] = chain_{4*ai}(inp[i]) with the config-1 constants; asynchronous on `stream`."""
    _check(lib().roofline_run(float(ai), int(n), _ptr(inp), _ptr(out), _stream(stream)), "roofline_run")


def roofline_run_k(k: int, a: float, b: float, n: int, inp, out, stream=None) -> None:
    _check(lib().roofline_run_k(int(k), float(a), float(b), int(n), _ptr(inp), _ptr(out), _stream(stream)),
           "roofline_run_k")


def decode_gemv(m, n, k, x, ldx, w, ldw, w_layout, y, ldy, stream=None) -> None:
    _check(lib().decode_gemv(m, n, k, _ptr(x), ldx, _ptr(w), ldw, w_layout, _ptr(y), ldy, _stream(stream)),
           "decode_gemv")


def prefill_gemm(m, n, k, a, lda, w, ldw, w_layout, c, ldc, stream=None) -> None:
    _check(lib().prefill_gemm(m, n, k, _ptr(a), lda, _ptr(w), ldw, w_layout, _ptr(c), ldc, _stream(stream)),
           "prefill_gemm")


def prefill_gemm_static_ws(m, n, k, a, lda, w, ldw, w_layout, c, ldc, stream=None) -> None:
    """prefill_gemm for 33 <= m <= 128 that allocates no device memory: the split-K partial tiles live in a 9.25 MiB
    static device array of the library (include/triroof.h: one array per device, shared by every call; calls that
    overlap on the GPU race; first call on a device before any stream capture)."""
    _check(lib().prefill_gemm_static_ws(m, n, k, _ptr(a), lda, _ptr(w), ldw, w_layout, _ptr(c), ldc, _stream(stream)),
           "prefill_gemm_static_ws")


def tri_sm_clock_mhz(spin_us: int = 2000, stream=None) -> float:
    v = c_double(0.0)
    _check(lib().tri_sm_clock_mhz(int(spin_us), byref(v), _stream(stream)), "tri_sm_clock_mhz")
    return v.value


def _sample_dict(s: tri_sample) -> dict:
    return {"t_s": s.t_s, "phase": s.phase, "sm_mhz": s.sm_mhz, "mem_mhz": s.mem_mhz, "temp_c": s.temp_c,
            "power_w": s.power_w, "read_us": s.read_us, "energy_mj": s.energy_mj, "clk_event_reasons": s.clk_event_reasons}


def tri_nvml_sample(device: int = 0) -> dict:
    s = tri_sample()
    _check(lib().tri_nvml_sample(device, byref(s)), "tri_nvml_sample")
    return _sample_dict(s)


def tri_lock_clocks(device: int, sm_mhz: int, mem_mhz: int = 0) -> int:
    """Returns the status (TRI_ERR_NO_PERMISSION is a normal outcome); raises only on invalid arguments."""
    st = lib().tri_lock_clocks(device, sm_mhz, mem_mhz)
    if st == TRI_ERR_INVALID_ARG:
        _check(st, "tri_lock_clocks")
    return st


def tri_reset_clocks(device: int) -> int:
    return lib().tri_reset_clocks(device)


class PhaseTracer:
    """phase_trace_start / mark / stop around caller-launched work."""

    def __init__(self, device: int = 0, period_us: int = 10000, capacity: int = 65536):
        self._buf = (tri_sample * capacity)()
        self._cap = capacity
        self._handle = c_void_p()
        self._device, self._period = device, period_us
        self.samples: list = []

    def start(self, phase: int = TRI_PHASE_IDLE):
        _check(lib().phase_trace_start(self._device, self._period, self._buf, self._cap, byref(self._handle)),
               "phase_trace_start")
        self.mark(phase)
        return self

    def mark(self, phase: int) -> None:
        _check(lib().phase_trace_mark(self._handle, phase), "phase_trace_mark")

    def stop(self) -> list:
        n = c_size_t(0)
        st = lib().phase_trace_stop(self._handle, byref(n))
        self._handle = c_void_p()
        self.samples = [_sample_dict(self._buf[i]) for i in range(n.value)]
        if st not in (TRI_OK, TRI_ERR_BUFFER_TOO_SMALL):
            _check(st, "phase_trace_stop")
        return self.samples


def phase_trace(pm, pn, pk, pa, pw, pc, dm, dn, dk, dx, dw_list, dy, w_layout=TRI_W_NK, total_s=60.0, prefill_s=2.0,
                decode_s=2.0, idle_s=1.0, period_ms=10, stream=None):
    """Config-5 driver.  Returns (samples, summaries) as lists of dicts."""
    cap = int(total_s * 1000 / period_ms) + 1024
    scap = int(3 * (total_s / max(prefill_s + decode_s + idle_s, 1e-9) + 2)) + 8
    sbuf = (tri_sample * cap)()
    pbuf = (tri_phase_summary * scap)()
    ring = (c_void_p * len(dw_list))(*[_ptr(w) for w in dw_list])
    wl = tri_trace_workload(pm, pn, pk, _ptr(pa), _ptr(pw), _ptr(pc), dm, dn, dk, _ptr(dx),
                            ctypes.cast(ring, POINTER(c_void_p)), len(dw_list), _ptr(dy), w_layout, _stream(stream))
    ns, np_ = c_size_t(0), c_size_t(0)
    st = lib().phase_trace(byref(wl), total_s, prefill_s, decode_s, idle_s, period_ms, sbuf, cap, byref(ns), pbuf, scap,
                           byref(np_))
    _check(st, "phase_trace")
    samples = [_sample_dict(sbuf[i]) for i in range(ns.value)]
    summaries = []
    for i in range(np_.value):
        q = pbuf[i]
        d = {name: getattr(q, name) for name, _ in tri_phase_summary._fields_ if not name.startswith("reserved")}
        d["phase_name"] = PHASE_NAMES.get(q.phase, str(q.phase))
        summaries.append(d)
    return samples, summaries


# ---- f3: A.I.-aware frequency selection (host functions; argument marshalling only) ----------------------------
class Model:
    """Owns the ctypes arrays behind a tri_model."""

    def __init__(self, eta, beta, omega=0.0, gamma=0.0, p_tdp=1000.0, f_mhz=(), p_idle_w=(), p_dyn_w=()):
        n = len(f_mhz)
        self._validated = set()
        self._f = (c_double * n)(*f_mhz)
        self._pi = (c_double * n)(*p_idle_w)
        self._pd = (c_double * n)(*p_dyn_w)
        self.c = tri_model(eta, beta, omega, gamma, p_tdp, n, ctypes.cast(self._f, POINTER(c_double)),
                           ctypes.cast(self._pi, POINTER(c_double)), ctypes.cast(self._pd, POINTER(c_double)))

    def theta(self, ai, f_mhz):
        return lib().tri_model_theta(byref(self.c), ai, f_mhz)

    def phi(self, ai, f_mhz):
        return lib().tri_model_phi(byref(self.c), ai, f_mhz)

    def power(self, ai, i):
        return lib().tri_model_power(byref(self.c), ai, i)

    def validate(self, ai):
        """The premise of solve_clock at this A.I. (tables well formed, theta and power monotone in f); raises TriError."""
        _check(lib().tri_model_validate(byref(self.c), ai), "tri_model_validate")

    def solve_clock(self, ai, f_limit_mhz, eps, check=True):
        """Eq. 6 -> (index into f_mhz, feasible).  check=True runs tri_model_validate the first time this Model sees this
        A.I. (O(n_f), remembered: the tables of a Model do not change) and raises TriError on tables the binary search is
        not exact on; check=False is the bare O(log n_f) C call for callers that validated themselves."""
        if check and ai not in self._validated:
            self.validate(ai)
            self._validated.add(ai)
        idx, feas = c_int32(-1), c_int32(0)
        _check(lib().tri_solve_clock(byref(self.c), ai, f_limit_mhz, eps, byref(idx), byref(feas)), "tri_solve_clock")
        return idx.value, bool(feas.value)


def tri_phase_ai(durations, ais) -> float:
    n = len(durations)
    return lib().tri_phase_ai((c_double * n)(*durations), (c_double * n)(*ais), n)


def tri_fit_theta(ai, f_mhz, theta, ai_mem, ai_cmp, gamma=0.0):
    """Eq. 4 fit -> dict(eta, beta, omega, gamma)."""
    n = len(ai)
    m = tri_model()
    _check(lib().tri_fit_theta((c_double * n)(*ai), (c_double * n)(*f_mhz), (c_double * n)(*theta), n, ai_mem, ai_cmp, gamma,
                               byref(m)), "tri_fit_theta")
    return {"eta": m.eta, "beta": m.beta, "omega": m.omega, "gamma": m.gamma}


def tri_fit_power(ai, f_mhz, p_w, eta, beta, f_sel_mhz, f_tol_mhz, p_cap_w):
    """Eq. 2 at one clock -> dict(p_idle_w, p_dyn_w, n_used)."""
    n = len(ai)
    m = Model(eta, beta)
    pi, pd, used = c_double(0.0), c_double(0.0), c_size_t(0)
    _check(lib().tri_fit_power((c_double * n)(*ai), (c_double * n)(*f_mhz), (c_double * n)(*p_w), n, byref(m.c), f_sel_mhz, f_tol_mhz,
                               p_cap_w, byref(pi), byref(pd), byref(used)), "tri_fit_power")
    return {"p_idle_w": pi.value, "p_dyn_w": pd.value, "n_used": used.value}


def _step_dict(st: tri_clock_step) -> dict:
    return {"sm_mhz": st.sm_mhz, "mem_mhz": st.mem_mhz, "duration_s": st.duration_s, "auto_boost": bool(st.auto_boost)}


def tri_policy_pace_race(sustained_mhz, f_mhz, prefill_s: float, pace_fraction: float = 0.10) -> list:
    """P:192 pace-and-race -> [pace step, race step] (dicts); computes the schedule only, actuates nothing."""
    n, nf = len(sustained_mhz), len(f_mhz)
    out = (tri_clock_step * 2)()
    _check(lib().tri_policy_pace_race((c_double * n)(*sustained_mhz), n, (c_double * nf)(*f_mhz), nf, prefill_s, pace_fraction, out),
           "tri_policy_pace_race")
    return [_step_dict(out[0]), _step_dict(out[1])]


def tri_policy_stall(entering: bool, idle_sm_mhz: float = 0.0, idle_mem_mhz: float = 0.0) -> dict:
    """P:130-132 stall-aware idle clocks -> one step (dict); computes only."""
    out = tri_clock_step()
    _check(lib().tri_policy_stall(int(bool(entering)), idle_sm_mhz, idle_mem_mhz, byref(out)), "tri_policy_stall")
    return _step_dict(out)


# the C names of the row-f3 entry points, on a Model
def tri_model_theta(model: Model, ai: float, f_mhz: float) -> float:
    return model.theta(ai, f_mhz)


def tri_model_phi(model: Model, ai: float, f_mhz: float) -> float:
    return model.phi(ai, f_mhz)


def tri_model_power(model: Model, ai: float, i: int) -> float:
    return model.power(ai, i)


def tri_model_validate(model: Model, ai: float) -> None:
    model.validate(ai)


def tri_solve_clock(model: Model, ai: float, f_limit_mhz: float, eps: float, check: bool = True):
    return model.solve_clock(ai, f_limit_mhz, eps, check)


# the remaining C names, as thin aliases of the wrappers above
tri_status_string = status_string
tri_last_error = last_error
tri_sm_count = sm_count
tri_l2_bytes = l2_bytes


def phase_trace_start(device: int = 0, period_us: int = 10000, capacity: int = 65536, phase: int = TRI_PHASE_IDLE) -> PhaseTracer:
    return PhaseTracer(device, period_us, capacity).start(phase)


def phase_trace_mark(tracer: PhaseTracer, phase: int) -> None:
    tracer.mark(phase)


def phase_trace_stop(tracer: PhaseTracer) -> list:
    return tracer.stop()
