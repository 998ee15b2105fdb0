"""bench.py — one "step" = one pass of the whole hot path over one batch of synthetic input:

    13 launches of the FMA-chain roofline kernel (BASELINE.json config 2: N = 2^28 fp32, k = 2^0 .. 2^12,
    A.I. = k/4 = 0.25 .. 1024 FLOP/B)  +  1 prefill GEMM (config 4)  +  8 decode GEMVs over 8 rotating weight copies
    (config 3), with the NVML phase tracer sampling clock / power / energy alongside.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

stdout carries exactly ONE compact JSON line (< 3 KB): `value` is the aggregate
algorithmic TFLOP/s of the step (fp32-FMA and bf16-tensor FLOP blended by the workload's own mix), `fracs` / `min_frac`
are the fractions of roofline per A.I. point — the metric BASELINE.json names — and `roofline`, `cpu_baseline`, `e2e`
the objects of the bench contract.  The full per-point detail (GB/s, TFLOP/s, clock, temperature, power, J/op, model
fit) goes to gpurun_out/bench_points.json and, one JSON line per point, to stderr.
`--impl reference` times the CPU oracle, as it stands, on a bounded sample of the same step.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "achieved GB/s or TFLOP/s and % of roofline per A.I. point on 1 B200; J/op"
N_FMA = 1 << 28
KS = [1 << i for i in range(13)]
GEMV_SHAPE = (8, 18944, 3584)         # m, n, k
GEMM_SHAPE = (4096, 18944, 3584)
GEMV_COPIES = 8
PAPER_KS = [4, 100, 200, 400, 800]      # the paper's own A.I. set {1, 25, 50, 100, 200} FLOP/B
RIDGE_KS = [24, 40, 48, 96]             # between the powers of two around the ridge (A.I. 6 .. 24), where the sweep is weakest
# Thinker-shaped GEMMs beside config 4: label -> (m, n, k)
GEMM_SHAPES = {"down_proj": (4096, 3584, 18944), "qkv": (4096, 4608, 3584), "o_proj": (4096, 3584, 3584),
               "up_m512": (512, 18944, 3584), "up_m256": (256, 18944, 3584), "up_m128": (128, 18944, 3584), "up_m64": (64, 18944, 3584),
               "up_m16": (16, 18944, 3584), "down_m64": (64, 3584, 18944)}
# Decode-size GEMVs of one Thinker layer ("GEMV-like operators"): label -> (m, n, k)
GEMV_SHAPES = {"qkv_m8": (8, 4608, 3584), "o_proj_m8": (8, 3584, 3584), "up_m8": (8, 18944, 3584), "down_m8": (8, 3584, 18944),
               "up_m1": (1, 18944, 3584)}
DECODE_LAYER = ["qkv_m8", "o_proj_m8", "up_m8", "down_m8"]     # the GEMVs of one layer at decode batch 8, back to back
NOMINAL_HBM_GBS = 8000.0               # BASELINE.json north_star "roughly 8 TB/s" (context; `frac` uses the measured peaks)
NOMINAL_BF16_TFLOPS = 2250.0           # dense bf16, nominal
FP32_LANES_PER_SM = 128                # FP32 FMA lanes per SM (4 SMSPs x 32); DESIGN.md "ALU peak"
REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
           0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
           0x100: "display_clock_setting"}


def fma_flop(k, n=N_FMA):
    return 2.0 * k * n


def gemm_flop(shape):
    m, n, k = shape
    return 2.0 * m * n * k


def gemm_bytes(shape):
    m, n, k = shape
    return 2.0 * (m * k + k * n + m * n)


STEP_FLOP = sum(fma_flop(k) for k in KS) + GEMV_COPIES * gemm_flop(GEMV_SHAPE) + gemm_flop(GEMM_SHAPE)
STEP_BYTES = len(KS) * 8.0 * N_FMA + GEMV_COPIES * gemm_bytes(GEMV_SHAPE) + gemm_bytes(GEMM_SHAPE)


def load_peaks():
    """Measured denominators (driver-written MEASURED_PEAKS.json), else the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0,
            "source": "fallback"}


# The ncu --set full captures the DRAM traffic figures come from, by name (not "the newest by sort order"): re-capture
# a kernel -> commit the new summary and change its line here.
NCU_CAPTURES = {"fma_chain": "profiles/r2b_ncu_fma_chain.txt", "decode_gemv": "profiles/r2b_ncu_decode_gemv.txt",
                "prefill_gemm": "profiles/r2b_ncu_prefill_gemm.txt"}


def ncu_traffic_bytes(kernel, column):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch, read from the committed text summary of that kernel's
    ncu --set full capture (NCU_CAPTURES) - a stored figure of an earlier run of the same kernel, not measured in this
    run (`traffic_source` on the line says which file); None when there is no summary."""
    import re
    files = [os.path.join(ROOT, NCU_CAPTURES[kernel])] if os.path.exists(os.path.join(ROOT, NCU_CAPTURES.get(kernel, "-"))) else []
    if not files:
        return None
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    total = 0.0
    for name in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
        m = re.search(r"^%s \[(\w+)\]: (.*)$" % re.escape(name), open(files[-1]).read(), re.M)
        if not m:
            return None
        total += float(m.group(2).split("|")[column].strip().replace(",", "")) * scale[m.group(1)]
    return total


# ----------------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline of our arm; the whole of --impl reference)
# ----------------------------------------------------------------------------------------------------------
class OracleSample:
    """A bounded sample of the step for the CPU oracle: 2^18 elements per A.I. point, the full config-3 GEMV once,
    8 rows of the config-4 GEMM.  Throughput in the step's unit (algorithmic TFLOP/s)."""
    N_FMA_S = 1 << 18
    GEMM_ROWS = 8

    def __init__(self):
        import oracle
        from synth_inputs import normal_bf16, uniform_pm1
        self.oracle = oracle
        self.x = uniform_pm1(1, self.N_FMA_S)
        m, n, k = GEMV_SHAPE
        self.gx = normal_bf16(2, (m, k), 1.0, stream=0)
        self.gw = np.ascontiguousarray(normal_bf16(2, (k, n), 0.02, stream=1).T)
        self.ga = normal_bf16(3, (self.GEMM_ROWS, k), 1.0, stream=0)
        self.flop = (sum(fma_flop(kk, self.N_FMA_S) for kk in KS) + gemm_flop(GEMV_SHAPE)
                     + gemm_flop((self.GEMM_ROWS, n, k)))
        self.desc = f"per step: 2^18 of 2^28 elements per k (13 k); 1 of 8 GEMVs; {self.GEMM_ROWS} of 4096 GEMM rows"

    def step(self):
        t0 = time.perf_counter()
        for k in KS:
            self.oracle.fma_chain(self.x, k)
        self.oracle.gemm_rows(self.gx, self.gw, w_layout=self.oracle.W_NK)
        self.oracle.gemm_rows(self.ga, self.gw, w_layout=self.oracle.W_NK)
        return time.perf_counter() - t0


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    s = OracleSample()
    for _ in range(args.warmup):
        s.step()
    times = [s.step() for _ in range(args.steps)]
    tot = sum(times)
    value = s.flop * args.steps / tot / 1e12
    cores = s.oracle.num_threads()
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
           "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32 chain; bf16 in / f32 acc",
           "data": "synthetic", "config": workload_config(args.gpus),
           "cpu_baseline": {"value": value, "unit": "TFLOP/s", "cores": cores, "kind": "oracle", "sample": s.desc},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0,
                   "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def workload_config(n_gpus):
    return {"workload": "configs[1] FMA-chain A.I. sweep N=2^28 k=2^0..2^12 + configs[2] GEMV 8x3584x18944 x 8 W copies "
                        "+ configs[3] GEMM 4096x3584x18944; W layout NK",
            "parallelism": f"replicas x{n_gpus} (no collective)",
            "l2": "inputs larger than L2 (2 GiB stream; 8 x 136 MB rotating W; 320 MB GEMM operands)"}


# ----------------------------------------------------------------------------------------------------------
# GPU arm
# ----------------------------------------------------------------------------------------------------------
def max_over_ranks(ms, dist, device):
    """Device time of the slowest rank (the replicas share nothing, so the job is as slow as its slowest GPU)."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(flop_per_step, steps, world, ms):
    """Aggregate TFLOP/s of `world` independent replicas that each ran `steps` steps in `ms` (max over ranks)."""
    return flop_per_step * steps * world / (ms * 1e-3) / 1e12


class GpuStep:
    """Device buffers (seeded synthetic, generated on the device with the bit-identical integer generator for the
    fp32 stream) and the launch sequence of one step.  Every launch goes through the C ABI binding."""

    def __init__(self, torch, tri):
        from synth_inputs import normal_bf16_torch, uniform_pm1_torch
        self.torch, self.tri = torch, tri
        dev = "cuda"
        self.x = uniform_pm1_torch(1, N_FMA, device=dev)
        self.y = torch.empty_like(self.x)
        m, n, k = GEMV_SHAPE
        self.gx = normal_bf16_torch(2, (m, k), 1.0, dev, stream=0)
        # copy 0 is the configured matrix (R6: value(k, n) = gen(seed 2, stream 1, k * N + n), stored [n][k]) — the
        # one the parity test checks; the other seven rotate distinct weights past L2 and are drawn in storage order
        self.gw = [normal_bf16_torch(2, (k, n), 0.02, dev, stream=1).t().contiguous()]
        self.gw += [normal_bf16_torch(2, (n, k), 0.02, dev, stream=1 + r) for r in range(1, GEMV_COPIES)]
        self.gy = torch.empty((m, n), dtype=torch.bfloat16, device=dev)
        pm, pn, pk = GEMM_SHAPE
        self.pa = normal_bf16_torch(3, (pm, pk), 1.0, dev, stream=0)
        self.pw = normal_bf16_torch(3, (pn, pk), 0.02, dev, stream=1)
        self.pc = torch.empty((pm, pn), dtype=torch.bfloat16, device=dev)
        self.launches_per_step = len(KS) + GEMV_COPIES + 1
        self.names = [f"fma_k{k}" for k in KS] + ["gemv"] + ["gemm"]

    def run(self, events=None, io=None):
        """Enqueues one step on torch's current stream.  events: optional list collecting (name, start, end).
        io: optional dict of per-step input / output buffers (x, y, gx, gy, pa, pc) replacing the resident ones."""
        torch, tri = self.torch, self.tri
        b = io or {"x": self.x, "y": self.y, "gx": self.gx, "gy": self.gy, "pa": self.pa, "pc": self.pc}

        def timed(name, fn):
            if events is None:
                fn()
                return
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            events.append((name, a, b))

        for k in KS:
            timed(f"fma_k{k}", lambda k=k: tri.roofline_run(k / 4.0, N_FMA, b["x"], b["y"]))
        # prefill before decode, the order of the serving phases (BASELINE.json config 5).  It is also the
        # cheaper order: the compute-bound GEMM absorbs the write-back of the dirty L2 lines the FMA sweep leaves behind at no
        # cost, where the memory-bound GEMVs would pay for it (22.0 against 23.2 us per GEMV)
        pm, pn, pk = GEMM_SHAPE
        timed("gemm", lambda: tri.prefill_gemm(pm, pn, pk, b["pa"], pk, self.pw, pk, tri.TRI_W_NK, b["pc"], pn))
        m, n, k = GEMV_SHAPE

        def gemvs():
            for w in self.gw:
                tri.decode_gemv(m, n, k, b["gx"], k, w, k, tri.TRI_W_NK, b["gy"], n)
        timed("gemv", gemvs)


def summarise_clocks(samples, peaks):
    busy = [s for s in samples if s["sm_mhz"] > 0]
    if not busy:
        return {"sm_mhz": None, "sm_max_mhz": peaks["sm_max_mhz"], "reasons": [], "source": "nvml unavailable"}
    bits = 0
    for s in busy:
        bits |= int(s["clk_event_reasons"])
    reasons = [name for bit, name in REASONS.items() if bits & bit and name != "gpu_idle"]
    return {"sm_mhz": statistics.median(s["sm_mhz"] for s in busy), "sm_max_mhz": peaks["sm_max_mhz"],
            "reasons": reasons, "temp_c_max": max(s["temp_c"] for s in busy),
            "power_w_mean": sum(s["power_w"] for s in busy) / len(busy), "samples": len(busy), "source": "nvml"}


def characterise(torch, tri, step, local, seconds, peaks, sms, est_ms):
    """Per-point sustained pass (outside the timed region): every A.I. point, the paper's own A.I. series and the two
    phase kernels are looped for `seconds` each while the library's NVML sampler runs; returns, per point, the device
    time per launch, the SM clock / temperature / power seen during that window and the energy per FLOP and per byte
    (NVML energy counter read at both ends) — BASELINE.json north_star "SM clock, temperature and joules per op per phase"."""
    m, n, k = GEMV_SHAPE
    pm, pn, pk = GEMM_SHAPE

    def gemvs():
        for w in step.gw:
            tri.decode_gemv(m, n, k, step.gx, k, w, k, tri.TRI_W_NK, step.gy, n)

    specs = [(f"fma_k{kk}", "sweep", kk, (lambda kk=kk: tri.roofline_run(kk / 4.0, N_FMA, step.x, step.y)), 1, fma_flop(kk), 8.0 * N_FMA)
             for kk in KS]
    specs += [(f"paper_ai{kk / 4:g}", "paper_ai", kk, (lambda kk=kk: tri.roofline_run(kk / 4.0, N_FMA, step.x, step.y)), 1,
               fma_flop(kk), 8.0 * N_FMA) for kk in PAPER_KS]
    specs += [(f"ridge_k{kk}", "ridge", kk, (lambda kk=kk: tri.roofline_run(kk / 4.0, N_FMA, step.x, step.y)), 1,
               fma_flop(kk), 8.0 * N_FMA) for kk in RIDGE_KS]
    specs.append(("gemv", "phase", None, gemvs, GEMV_COPIES, gemm_flop(GEMV_SHAPE), gemm_bytes(GEMV_SHAPE)))
    specs.append(("gemm", "phase", None,
                  lambda: tri.prefill_gemm(pm, pn, pk, step.pa, pk, step.pw, pk, tri.TRI_W_NK, step.pc, pn), 1,
                  gemm_flop(GEMM_SHAPE), gemm_bytes(GEMM_SHAPE)))
    try:
        tracer = tri.PhaseTracer(local, period_us=10000, capacity=1 << 17).start(tri.TRI_PHASE_IDLE)
    except tri.TriError:
        return {}
    out, windows = {}, []
    side = torch.cuda.Stream()
    for idx, (name, series, kk, fn, per_call, flop, nbytes) in enumerate(specs):
        est = est_ms.get(name) or (fma_flop(kk) / (0.9 * sms * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6) * 1e3 + 0.33)
        batch = max(1, int(20.0 / (est * per_call)))                  # about 20 ms of work per host round trip
        torch.cuda.synchronize()
        tracer.mark(100 + idx)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0 = tri.tri_nvml_sample(local)["energy_mj"]
        t0 = time.perf_counter()
        a.record()
        calls = 0
        clk_in_kernel = None
        while time.perf_counter() - t0 < seconds:
            for _ in range(batch):
                fn()
            calls += batch * per_call
            if clk_in_kernel is None and time.perf_counter() - t0 >= 0.5 * seconds:
                # the SM clock seen from inside the GPU, per point and UNDER this point's load - the one-block
                # clock64 / globaltimer probe runs on a side stream beside the batch just enqueued (blocks ~2 ms)
                try:
                    clk_in_kernel = tri.tri_sm_clock_mhz(2000, stream=side)
                except tri.TriError:
                    clk_in_kernel = 0.0
            torch.cuda.synchronize()
        b.record()
        torch.cuda.synchronize()
        e1 = tri.tri_nvml_sample(local)["energy_mj"]
        windows.append((name, series, kk, 100 + idx, a.elapsed_time(b), calls, flop, nbytes, (e1 - e0) * 1e-3, clk_in_kernel))
    samples = tracer.stop()
    for name, series, kk, tag, ms, calls, flop, nbytes, joule, clk_in_kernel in windows:
        ss = [x for x in samples if x["phase"] == tag and x["sm_mhz"] > 0]
        bits = 0
        for x in ss:
            bits |= int(x["clk_event_reasons"])
        per_ms = ms / calls
        out[name] = {"series": series, "k": kk, "ms_sustained": per_ms, "launches": calls, "window_s": ms * 1e-3,
                     "gbs_sustained": nbytes / per_ms / 1e6, "tflops_sustained": flop / per_ms / 1e9,
                     "sm_mhz": statistics.median(x["sm_mhz"] for x in ss) if ss else None,
                     "sm_mhz_in_kernel": clk_in_kernel or None,
                     "mem_mhz": statistics.median(x["mem_mhz"] for x in ss) if ss else None,
                     "temp_c_max": max(x["temp_c"] for x in ss) if ss else None,
                     "power_w_mean": sum(x["power_w"] for x in ss) / len(ss) if ss else None,
                     "reasons": [nm for bit, nm in REASONS.items() if bits & bit and nm != "gpu_idle"],
                     "j_per_flop": joule / (flop * calls) if joule > 0 else None,
                     "j_per_byte": joule / (nbytes * calls) if joule > 0 else None,
                     "j_per_call": joule / calls if joule > 0 else None, "nvml_samples": len(ss)}
    return out


def time_gemm_pair(torch, tri, m, n, k, group=8):
    """Device time per call (ms) of prefill_gemm and of torch.matmul (cuBLAS, context) on one m x n x k shape.  Weights
    rotate over enough copies to exceed L2 (a model's next use of a matrix comes after all its other weights); calls are
    timed in groups of `group` between one CUDA-event pair, median of 9 groups — an event pair around every single call
    measures the host's launch rate, not the kernel, once a call is shorter than ~40 us — after a short rest, so that a
    point does not inherit the power-capped clock of the one before it."""
    copies = max(2, min(8, int(300e6 / (2.0 * n * k)) + 1))
    a = torch.randn(m, k, device="cuda").bfloat16()
    ws = [(torch.randn(n, k, device="cuda") * 0.02).bfloat16() for _ in range(copies)]
    c = torch.empty(m, n, device="cuda", dtype=torch.bfloat16)

    def med(fn):
        torch.cuda.synchronize()
        time.sleep(0.2)
        for i in range(2 * group):
            fn(ws[i % copies])
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(9)]
        for x, y in ev:
            x.record()
            for i in range(group):
                fn(ws[i % copies])
            y.record()
        torch.cuda.synchronize()
        return sorted(x.elapsed_time(y) for x, y in ev)[4] / group

    ours = med(lambda w: tri.prefill_gemm(m, n, k, a, k, w, k, tri.TRI_W_NK, c, n))
    lib = med(lambda w: torch.matmul(a, w.T, out=c))
    del a, ws, c
    return ours, lib


def gemm_point(series, m, n, k, ours, lib, peaks, **extra):
    flop, nbytes = 2.0 * m * n * k, 2.0 * (m * k + n * k + m * n)
    ai = flop / nbytes
    roof = min(peaks["bf16_tflops"], ai * peaks["hbm_gbs"] / 1e3)
    return dict({"kernel": "prefill_gemm", "series": series, "m": m, "n": n, "k": k, "ai": ai, "ms": ours, "tflops": flop / ours / 1e9,
                 "gbs": nbytes / ours / 1e6, "roofline_tflops": roof, "frac": flop / ours / 1e9 / roof,
                 "bound": "tensor" if roof == peaks["bf16_tflops"] else "hbm", "timing": "groups of 8 calls, rotating W copies",
                 "cublas_ms": lib, "cublas_tflops": flop / lib / 1e9}, **extra)


def controller_preview(tri, fit, pf, peaks, fma_pts, points, eps=0.05):
    """Row f3 end to end on this run's own data (Eq. 5 and Eq. 6): the phase A.I. of
    Eq. 5 from the measured kernel durations, and the clock Eq. 6 selects (the library's binary search, tri_solve_clock) on
    the fitted throughput model, per A.I. point, with f_limit = the auto-boost clock this run recorded at that point.
    P_idle(f) and P_dyn(f) exist on this pool only at the boost ceiling (no locked-clock columns), so the power tables are
    that one fitted pair scaled LINEARLY in f — an assumption, stated in the output; Eq. 6's answer depends on them only
    through their monotonicity (the paper's own premise, line 186), i.e. it is the lowest clock that keeps the throughput
    within eps.  Nothing is actuated: clock locking is not used on this pool (R17)."""
    fmax = peaks["sm_max_mhz"]
    clocks = [float(f) for f in range(1005, int(fmax) + 1, 15)]       # a 15 MHz grid up to the boost ceiling, the step NVML reports on B200
    if clocks[-1] != fmax:
        clocks.append(fmax)
    mdl = tri.Model(fit["eta"], fit["beta"], fit["omega"], fit["gamma"], p_tdp=1000.0, f_mhz=clocks,
                    p_idle_w=[pf["p_idle_w"] * f / fmax for f in clocks], p_dyn_w=[pf["p_dyn_w"] * f / fmax for f in clocks])
    rows = []
    for pt in fma_pts:
        f_limit = float(pt["sustained"]["sm_mhz"])
        try:
            mdl.validate(pt["ai"])
            idx, feasible = mdl.solve_clock(pt["ai"], f_limit, eps)
            rows.append({"ai": pt["ai"], "f_autoboost_mhz": f_limit, "f_selected_mhz": clocks[idx], "feasible": feasible,
                         "theta_ratio": mdl.theta(pt["ai"], clocks[idx]) / mdl.theta(pt["ai"], fmax),
                         "p_model_ratio": mdl.power(pt["ai"], idx) / mdl.power(pt["ai"], len(clocks) - 1)})
        except tri.TriError as e:
            rows.append({"ai": pt["ai"], "error": str(e)})
    # Eq. 5 over the kernels of the timed step: the whole FMA sweep as one "phase", and the decode phase (8 GEMVs)
    sweep = [pt for pt in points if pt["kernel"] == "fma_chain"]
    gemv = next(pt for pt in points if pt["kernel"] == "decode_gemv")
    ai_sweep = tri.tri_phase_ai([pt["ms"] for pt in sweep], [pt["ai"] for pt in sweep])
    ai_decode = tri.tri_phase_ai([gemv["ms"]] * GEMV_COPIES, [gemv["ai"]] * GEMV_COPIES)
    dec = {}
    try:                                                               # the decode phase on the CUDA-core throughput model
        idx, feasible = mdl.solve_clock(ai_decode, float((gemv.get("sustained") or {}).get("sm_mhz") or fmax), eps)
        dec = {"f_selected_mhz": clocks[idx], "feasible": feasible, "f_autoboost_mhz": (gemv.get("sustained") or {}).get("sm_mhz")}
    except tri.TriError as e:
        dec = {"error": str(e)}
    return {"eps": eps, "clock_grid_mhz": [clocks[0], clocks[-1], 15], "eq5_phase_ai": {"fma_sweep": ai_sweep, "decode": ai_decode},
            "eq6_decode_phase": dec, "eq6_per_point": rows,
            "assumption": "P_idle(f), P_dyn(f) = the boost-ceiling fit scaled linearly in f (no locked-clock data on this pool); "
                          "Eq. 6 then returns the lowest clock within eps of the throughput at f_max; nothing is actuated"}


def gemm_ai_series(torch, tri, peaks):
    """Row f4 (next): the paper's own microbenchmark form — a matmul whose A.I. is varied — on the
    tensor-core path: C[8192 x 8192] = A[8192 x K] W[K x 8192], bf16, K swept; A.I. = 2 m n K / (2 (m K + K n + m n)).
    Roofline: min(measured cuBLAS burst, A.I. x measured HBM copy rate).  The low-K points only write C: a write-only
    stream reaches 3.6-3.9 TB/s on this part (torch fill), not the copy rate, so their `frac` has a ceiling
    near 0.75.  torch.matmul (cuBLAS) on the same operands is timed beside it as context."""
    m = n = 8192
    out = []
    for k in (16, 64, 256, 1024, 4096):
        ours, lib = time_gemm_pair(torch, tri, m, n, k)
        out.append(gemm_point("matmul-based A.I. sweep (PAPER.md line 92), 8192 x 8192 x K", m, n, k, ours, lib, peaks))
    return out


def gemm_shape_series(torch, tri, peaks):
    """Row f4: the other Thinker-shaped GEMMs (down-projection, fused QKV, output projection, short A), each with its
    roofline min(measured cuBLAS burst, A.I. x measured HBM) and torch.matmul (cuBLAS) on the same operands as context."""
    out = []
    for label, (m, n, k) in GEMM_SHAPES.items():
        ours, lib = time_gemm_pair(torch, tri, m, n, k)
        out.append(gemm_point("Thinker-shaped GEMMs (SURVEY 8(f).4)", m, n, k, ours, lib, peaks, label=label))
    return out


def gemv_shape_series(torch, tri, peaks, group=16):
    """Row f4: the decode-size matrices a real decode step is mostly made of, each against the HBM roofline (bytes of X, W
    and Y over the measured copy rate), timed like time_gemm_pair (groups of calls between one event pair, weights rotating
    over more copies than L2 holds); and the four GEMVs of one layer back to back as one unit ("decode_layer_m8"), whose
    roofline is the sum of their bytes."""
    out = []

    def med(fn, calls_per_group):
        torch.cuda.synchronize()
        time.sleep(0.2)
        for i in range(2 * calls_per_group):
            fn(i)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(9)]
        for x, y in ev:
            x.record()
            for i in range(calls_per_group):
                fn(i)
            y.record()
        torch.cuda.synchronize()
        return sorted(x.elapsed_time(y) for x, y in ev)[4] / calls_per_group

    bufs = {}
    for label, (m, n, k) in GEMV_SHAPES.items():
        copies = max(2, min(8, int(300e6 / (2.0 * n * k)) + 1))
        bufs[label] = (torch.randn(m, k, device="cuda").bfloat16(), [(torch.randn(n, k, device="cuda") * 0.02).bfloat16() for _ in range(copies)],
                       torch.empty(m, n, device="cuda", dtype=torch.bfloat16))

    def call(label, i):
        m, n, k = GEMV_SHAPES[label]
        x, ws, y = bufs[label]
        tri.decode_gemv(m, n, k, x, k, ws[i % len(ws)], k, tri.TRI_W_NK, y, n)

    for label, (m, n, k) in GEMV_SHAPES.items():
        ms = med(lambda i: call(label, i), group)
        nbytes = gemm_bytes((m, n, k))
        out.append({"kernel": "decode_gemv", "series": "decode-size GEMVs (SURVEY 8(f).4)", "label": label, "m": m, "n": n, "k": k,
                    "bytes": nbytes, "ms": ms, "gbs": nbytes / ms / 1e6, "frac": nbytes / ms / 1e6 / peaks["hbm_gbs"], "bound": "hbm",
                    "timing": f"groups of {group} calls, rotating W copies"})

    def layer(i):
        for label in DECODE_LAYER:
            call(label, i)
    ms = med(layer, 8)
    nbytes = sum(gemm_bytes(GEMV_SHAPES[l]) for l in DECODE_LAYER)
    out.append({"kernel": "decode_gemv", "series": "decode-size GEMVs (SURVEY 8(f).4)", "label": "decode_layer_m8", "m": 8, "n": 0, "k": 0,
                "bytes": nbytes, "ms": ms, "gbs": nbytes / ms / 1e6, "frac": nbytes / ms / 1e6 / peaks["hbm_gbs"], "bound": "hbm",
                "timing": "qkv, o_proj, up, down back to back = one unit; groups of 8 units, rotating W copies"})
    bufs.clear()
    return out


UNIT = "TFLOP/s (algorithmic, whole step: fp32 FMA + bf16 tensor)"
DETAIL_FILE = os.path.join("gpurun_out", "bench_points.json")
COMPACT_KEYS = ["impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline", "min_frac", "min_frac_kernel"]


def point_key(pt):
    if pt["kernel"] == "fma_chain":
        return f"fma_k{pt['k']}"
    return {"decode_gemv": "gemv", "prefill_gemm": "gemm"}[pt["kernel"]]


def sig(x, digits=4):
    return None if x is None else float(f"{x:.{digits}g}")


def compact_line(full):
    """The ONE line of stdout: the bench contract's keys, plus the metric BASELINE.json names in compact form —
    `fracs` = fraction of roofline per A.I. point (burst, per-launch CUDA-event medians of the timed steps) and
    `sustained` = per point, in the order of `fracs`, [fraction of the roofline at the recorded clock, SM MHz, W, pJ/FLOP] from the looped pass
    (the ridge and paper-A.I. extra series are in the detail file only).
    Everything bulky (`points`, `extra_points`, `model_fit`) stays in the detail file.  Kept near 2 KB: the round-1
    line was 20 KB and the driver, which reads the last 3000 bytes of stdout, could not parse it."""
    out = {k: full[k] for k in COMPACT_KEYS if k in full}
    pts = full.get("points") or []
    out["fracs"] = {point_key(p): round(p["frac"], 3) for p in pts}
    def short(x, digits):                                             # 640.0 -> 640 on the line
        x = sig(x, digits)
        return int(x) if x is not None and x >= 100 else x
    sus = []
    for p in pts:
        c = p.get("sustained")
        if c and p.get("frac_sustained_at_clock") is not None:
            pj = c.get("j_per_flop")
            sus.append([round(p["frac_sustained_at_clock"], 2), int(c.get("sm_mhz") or 0), int(c.get("power_w_mean") or 0),
                        short(pj * 1e12 if pj else None, 2)])
    if len(sus) == len(pts) and sus:
        out["sustained"] = sus
        out["sustained_cols"] = "order of fracs: frac at clock, SM MHz, W, pJ/FLOP"
    # the extra FMA series of the sustained pass (between the powers of two around the ridge; the paper's own A.I. set):
    # fraction of the roofline at the recorded clock, keyed by k
    xs = [q for q in (full.get("extra_points") or []) if q.get("kernel") == "fma_chain" and q.get("frac_sustained_at_clock") is not None]
    for key, tag in (("ridge", "ridge"), ("paper_ai", "paper A.I.")):
        sel = {f"k{q['k']}": round(q["frac_sustained_at_clock"], 2) for q in xs if str(q.get("series", "")).startswith(tag)}
        if sel:
            out[key] = sel
    gm = [q for q in (full.get("extra_points") or []) if q.get("kernel") == "prefill_gemm" and q.get("label")]
    if gm:
        out["gemm_shapes"] = {q["label"]: round(q["frac"], 3) for q in gm}
    gv = [q for q in (full.get("extra_points") or []) if q.get("kernel") == "decode_gemv" and q.get("label")]
    if gv:
        out["gemv_shapes"] = {q["label"]: round(q["frac"], 3) for q in gv}
    cp = ((full.get("model_fit") or {}).get("controller_preview") or {}).get("eq6_decode_phase") or {}
    if cp.get("f_selected_mhz"):                                       # Eq. 6 on the fitted model, decode phase: [selected, auto-boost] MHz
        out["eq6_decode_mhz"] = [int(cp["f_selected_mhz"]), int(cp.get("f_autoboost_mhz") or 0)]
    if full.get("energy"):
        out["j_per_flop"] = sig(full["energy"].get("j_per_flop"), 3)
    out["detail"] = DETAIL_FILE

    def rounded(x):                                                   # 5 significant digits are plenty on the line; the file has them all
        if isinstance(x, float):
            return sig(x, 5)
        if isinstance(x, dict):
            return {k: rounded(v) for k, v in x.items()}
        if isinstance(x, list):
            return [rounded(v) for v in x]
        return x
    out = rounded(out)
    line = json.dumps(out, separators=(",", ":"))
    for key in ("sustained_cols", "paper_ai", "ridge", "eq6_decode_mhz", "gemv_shapes", "gemm_shapes", "sustained"):   # optional keys, least needed first
        if len(line) <= 2800:
            break
        out.pop(key, None)                                             # the driver reads the last 3000 bytes of stdout: never outgrow them
        line = json.dumps(out, separators=(",", ":"))
    return line


def emit(full):
    """Detail first (file + one JSON line per point on stderr), then the single compact line on stdout."""
    try:
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        with open(os.path.join(ROOT, DETAIL_FILE), "w") as f:
            json.dump(full, f, indent=1)
    except OSError as e:
        print(f"bench.py: could not write {DETAIL_FILE}: {e}", file=sys.stderr)
    for p in (full.get("points") or []) + (full.get("extra_points") or []):
        print(json.dumps(p), file=sys.stderr)
    if full.get("model_fit"):
        print(json.dumps({"model_fit": full["model_fit"]}), file=sys.stderr)
    sys.stderr.flush()
    print(compact_line(full), flush=True)


def run_ours(args):
    import torch
    import paper_2606_29629_b200 as tri          # raises if the CUDA library cannot be built / loaded: no fallback

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    tri.tri_init(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    peaks = load_peaks()
    step = GpuStep(torch, tri)
    sms = tri.sm_count()

    for _ in range(max(args.warmup, 3)):
        step.run()
    barrier()

    # ---- device-resident timing: K steps, per-launch CUDA events on the launching (current) stream ----
    tracer = None
    try:
        tracer = tri.PhaseTracer(local, period_us=10000, capacity=1 << 16).start(tri.TRI_PHASE_ROOFLINE)
    except tri.TriError:
        tracer = None
    events = []
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0 = tri.tri_nvml_sample(local)["energy_mj"] if tracer else 0
    t_begin.record()
    for _ in range(args.steps):
        step.run(events)
    t_end.record()
    barrier()
    e1 = tri.tri_nvml_sample(local)["energy_mj"] if tracer else 0
    samples = tracer.stop() if tracer else []
    total_ms = t_begin.elapsed_time(t_end)
    total_ms = max_over_ranks(total_ms, dist, "cuda")
    clk_probe = tri.tri_sm_clock_mhz(2000)

    per = {}
    for name, a, b in events:
        per.setdefault(name, []).append(a.elapsed_time(b))
    clocks = summarise_clocks(samples, peaks)
    f_obs = clocks["sm_mhz"] or peaks["sm_max_mhz"]
    alu_peak = sms * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12     # TFLOP/s at the max SM clock
    points = []
    for k in KS:
        ms = statistics.median(per[f"fma_k{k}"])
        gbs, tf = 8.0 * N_FMA / ms / 1e6, fma_flop(k) / ms / 1e9
        roof = min(alu_peak, k / 4.0 * peaks["hbm_gbs"] / 1e3)
        points.append({"kernel": "fma_chain", "k": k, "ai": k / 4.0, "ms": ms, "gbs": gbs, "tflops": tf,
                       "bound": "hbm" if k / 4.0 * peaks["hbm_gbs"] / 1e3 < alu_peak else "alu",
                       "roofline_tflops": roof, "frac": tf / roof, "ms_min": min(per[f"fma_k{k}"]),
                       "frac_vs_nominal": tf / min(alu_peak, k / 4.0 * NOMINAL_HBM_GBS / 1e3), "algorithmic_bytes": 8.0 * N_FMA,
                       "traffic": ncu_traffic_bytes("fma_chain", column=KS.index(k))})
    ms = statistics.median(per["gemv"]) / GEMV_COPIES
    gv_gbs = gemm_bytes(GEMV_SHAPE) / ms / 1e6
    points.append({"kernel": "decode_gemv", "ai": gemm_flop(GEMV_SHAPE) / gemm_bytes(GEMV_SHAPE), "ms": ms, "gbs": gv_gbs,
                   "tflops": gemm_flop(GEMV_SHAPE) / ms / 1e9, "bound": "hbm", "roofline_gbs": peaks["hbm_gbs"],
                   "frac": gv_gbs / peaks["hbm_gbs"], "ms_min": min(per["gemv"]) / GEMV_COPIES,
                   "frac_vs_nominal": gv_gbs / NOMINAL_HBM_GBS, "algorithmic_bytes": gemm_bytes(GEMV_SHAPE),
                   "traffic": ncu_traffic_bytes("decode_gemv", column=0)})
    ms = statistics.median(per["gemm"])
    gm_tf = gemm_flop(GEMM_SHAPE) / ms / 1e9
    points.append({"kernel": "prefill_gemm", "ai": gemm_flop(GEMM_SHAPE) / gemm_bytes(GEMM_SHAPE), "ms": ms,
                   "gbs": gemm_bytes(GEMM_SHAPE) / ms / 1e6, "tflops": gm_tf, "bound": "tensor",
                   "roofline_tflops": peaks["bf16_tflops"], "frac": gm_tf / peaks["bf16_tflops"], "ms_min": min(per["gemm"]),
                   "frac_vs_nominal": gm_tf / NOMINAL_BF16_TFLOPS, "algorithmic_bytes": gemm_bytes(GEMM_SHAPE),
                   "traffic": ncu_traffic_bytes("prefill_gemm", column=0)})

    # the paper takes a kernel's A.I. from Nsight Compute: FLOP over the DRAM bytes ncu counted for the launch
    for pt in points:
        if pt.get("traffic"):
            flop = fma_flop(pt["k"]) if pt["kernel"] == "fma_chain" else gemm_flop(GEMV_SHAPE if pt["kernel"] == "decode_gemv" else GEMM_SHAPE)
            pt["ai_from_ncu_traffic"] = flop / pt["traffic"]

    # ---- per-point sustained pass: clock, temperature, power, J/op per A.I. point and per phase kernel ----
    extra_points, model_fit = [], None
    if args.char_seconds > 0 and world == 1:
        est = {f"fma_k{k}": statistics.median(per[f"fma_k{k}"]) for k in KS}
        est["gemv"] = statistics.median(per["gemv"]) / GEMV_COPIES
        est["gemm"] = statistics.median(per["gemm"])
        ch = characterise(torch, tri, step, local, args.char_seconds, peaks, sms, est)

        def at_clock(pt, c):
            """Roofline fraction of the sustained rate against the roofline AT THE RECORDED SM CLOCK (BASELINE.json
            north_star): HBM points are clock-independent, ALU points scale with the clock seen in the window; the
            tensor point is held against the measured sustained cuBLAS rate (power-capped clock, MEASURED_PEAKS.json)."""
            if not c:
                return
            pt["sustained"] = c
            alu_at_clock = sms * FP32_LANES_PER_SM * 2 * (c["sm_mhz"] or peaks["sm_max_mhz"]) * 1e6 / 1e12
            if pt["bound"] == "tensor":
                roof = peaks["bf16_tflops_sustained"]
            else:                                                      # CUDA-core kernels: min(A.I. x HBM, FP32 ALUs at the clock seen)
                roof = min(pt["ai"] * peaks["hbm_gbs"] / 1e3, alu_at_clock)
            pt["roofline_tflops_at_clock"] = roof
            pt["frac_sustained_at_clock"] = c["tflops_sustained"] / roof

        for pt in points:
            key = f"fma_k{pt['k']}" if pt["kernel"] == "fma_chain" else ("gemv" if pt["kernel"] == "decode_gemv" else "gemm")
            at_clock(pt, ch.get(key))
        for kk, key, series in ([(kk, f"paper_ai{kk / 4:g}", "paper A.I. set {1,25,50,100,200} (PAPER.md line 92)") for kk in PAPER_KS] +
                                [(kk, f"ridge_k{kk}", "ridge: between the powers of two, A.I. 6 .. 24") for kk in RIDGE_KS]):
            c = ch.get(key)                                            # the paper's x-axis (Fig. 3) and the ridge, labelled extra series
            if c:
                hb = kk / 4.0 * peaks["hbm_gbs"] / 1e3
                pt = {"kernel": "fma_chain", "series": series, "k": kk, "ai": kk / 4.0, "bound": "hbm" if hb < alu_peak else "alu"}
                at_clock(pt, c)
                extra_points.append(pt)
        # row f3 on the measured sweep: Eq. 4 fitted to (A.I., recorded clock, sustained TFLOP/s) of the 13 sweep points plus
        # the ridge and paper-A.I. series with the library's own tri_fit_theta.  gamma is not identified by a least-squares
        # line, so it is scanned: the clock varies only between ~1.55 and 1.97 GHz across an auto-boost sweep (no locked-clock
        # columns on this pool), which is what limits how well it can be told apart; the model's residuals are reported per point
        fma_pts = [pt for pt in points + extra_points if pt["kernel"] == "fma_chain" and pt.get("sustained") and pt["sustained"].get("sm_mhz")]
        fma_pts.sort(key=lambda pt: pt["ai"])
        sw = [(pt["ai"], pt["sustained"]["sm_mhz"], pt["sustained"]["tflops_sustained"]) for pt in fma_pts]
        if len(sw) >= 6:
            try:
                best = None
                scan = {}
                for gamma in (0.0, 0.5, 1.0, 1.5, 2.0):
                    fit = tri.tri_fit_theta([x[0] for x in sw], [x[1] for x in sw], [x[2] for x in sw], ai_mem=4.0, ai_cmp=24.0, gamma=gamma)
                    mdl = tri.Model(fit["eta"], fit["beta"], fit["omega"], fit["gamma"])
                    res = [mdl.theta(a, f) / t - 1.0 for a, f, t in sw]
                    rms = (sum(r * r for r in res) / len(res)) ** 0.5
                    scan[f"{gamma:g}"] = round(rms, 5)
                    if best is None or rms < best[0]:
                        best = (rms, fit, res)
                rms, fit, res = best
                model_fit = dict(fit, unit="TFLOP/s per MHz (eta), TB/s (beta), FLOP/B per MHz^gamma (omega)",
                                 eta_nominal=sms * FP32_LANES_PER_SM * 2 / 1e6, beta_measured_copy=peaks["hbm_gbs"] / 1e3,
                                 rms_rel_residual_by_gamma=scan, max_abs_rel_residual=max(abs(r) for r in res),
                                 ai=[x[0] for x in sw], rel_residuals=[round(r, 4) for r in res],
                                 source="PAPER.md Eq. 4 via tri_fit_theta on the sustained sweep + ridge + paper-A.I. points "
                                        "(memory set A.I. <= 4, compute set A.I. >= 24), gamma scanned")
                # Eq. 2 at the one clock this box shows below the cap (the boost ceiling): P_idle(f), P_dyn(f) from the
                # compute-bound points that ran there
                allp = [(pt["ai"], pt["sustained"]["sm_mhz"], pt["sustained"]["power_w_mean"]) for pt in fma_pts
                        if pt["sustained"].get("power_w_mean")]
                try:
                    pf = tri.tri_fit_power([x[0] for x in allp], [x[1] for x in allp], [x[2] for x in allp], fit["eta"], fit["beta"],
                                           peaks["sm_max_mhz"], 2.0, 950.0)
                    model_fit["power_at_max_clock"] = dict(pf, f_mhz=peaks["sm_max_mhz"],
                                                           source="PAPER.md Eq. 2-3 via tri_fit_power on the points at the boost ceiling, below the power cap")
                    model_fit["controller_preview"] = controller_preview(tri, fit, pf, peaks, fma_pts, points)
                    # Row f2, second half, as a preview: the pace-and-race schedule for one config-4 prefill call from
                    # the sustained clocks this run recorded per A.I. point and phase kernel, on the 15 MHz clock grid.  About
                    # 1 s per point is not the paper's 240 s steady state (`characterise thermal` is), and nothing is actuated.
                    sus = [pt["sustained"]["sm_mhz"] for pt in fma_pts + [q for q in points if q["kernel"] != "fma_chain"]
                           if (pt.get("sustained") or {}).get("sm_mhz")]
                    grid = [float(f) for f in range(1005, int(peaks["sm_max_mhz"]) + 1, 15)]
                    gemm_pt = next(q for q in points if q["kernel"] == "prefill_gemm")
                    steps = tri.tri_policy_pace_race(sus, grid, gemm_pt["ms"] * 1e-3, 0.10)
                    model_fit["pace_race_preview"] = {"pace_mhz": steps[0]["sm_mhz"], "pace_s": steps[0]["duration_s"], "race_s": steps[1]["duration_s"],
                                                      "sustained_mhz_min": min(sus), "points": len(sus), "actuated": False,
                                                      "stall_idle_clocks_mhz": [tri.tri_policy_stall(True)["sm_mhz"], tri.tri_policy_stall(True)["mem_mhz"]],
                                                      "source": "PAPER.md section III-D line 192 via tri_policy_pace_race; III-B lines 130-132 via tri_policy_stall"}
                except tri.TriError as e:
                    model_fit["power_at_max_clock"] = {"error": str(e)}
            except tri.TriError as e:
                model_fit = {"error": str(e)}
        extra_points += gemm_ai_series(torch, tri, peaks)
        extra_points += gemm_shape_series(torch, tri, peaks)
        extra_points += gemv_shape_series(torch, tri, peaks)

    # dominant kernel of the step: the FMA-chain kernel at k = 4096 (about half of the step time), ALU-bound
    dom = points[len(KS) - 1]
    traffic = ncu_traffic_bytes("fma_chain", column=len(KS) - 1)
    roofline = {"kernel": "fma_chain_kernel (k=4096 launch)", "bound": "alu", "achieved": dom["tflops"], "peak": alu_peak,
                "unit": "TFLOP/s", "frac": dom["tflops"] / alu_peak, "traffic": traffic,
                "traffic_source": NCU_CAPTURES["fma_chain"] + " (stored ncu capture)" if traffic else None,
                "share_of_step": dom["ms"] * args.steps / total_ms,
                "peak_source": f"derived {sms} SMs x {FP32_LANES_PER_SM} x 2 x {peaks['sm_max_mhz']:.0f} MHz; fracs vs {peaks['source']} "
                               f"{peaks['hbm_gbs']:.0f} GB/s, {peaks['bf16_tflops']:.0f} TF/s"}

    # ---- end to end: host buffers in, host buffers out, copies inside the timed region ----
    e2e = run_e2e(torch, tri, step, args, barrier, dist)

    value = whole_job_value(STEP_FLOP, args.steps, world, total_ms)
    energy_j = (e1 - e0) * 1e-3 if e1 > e0 else None
    full = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32 chain; bf16 in / f32 acc",
            "data": "synthetic", "config": workload_config(world), "clocks": dict(clocks, sm_mhz_in_kernel_probe=clk_probe),
            "e2e": e2e, "gpu_launches": step.launches_per_step * args.steps, "roofline": roofline, "points": points,
            "extra_points": extra_points, "model_fit": model_fit, "min_frac": min(p["frac"] for p in points),
            "min_frac_kernel": point_key(min(points, key=lambda p: p["frac"])),
            "energy": {"j_per_step": energy_j / args.steps if energy_j else None,
                       "j_per_flop": energy_j / (STEP_FLOP * args.steps) if energy_j else None,
                       "j_per_byte": energy_j / (STEP_BYTES * args.steps) if energy_j else None},
            "peaks": peaks,
            "paper_context": "Tri-serve reports -22.1 % J/output-token on 3x RTX 6000 Ada (Qwen2.5-Omni-7B, vLLM-Omni); "
                             "no throughput number is published for this path (BASELINE.md)"}
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            s = OracleSample()
            s.step()
            reps, t = 0, 0.0
            while t < 10.0 and reps < 50:
                t += s.step()
                reps += 1
            full["cpu_baseline"] = {"value": s.flop * reps / t / 1e12, "unit": "TFLOP/s", "cores": s.oracle.num_threads(),
                                    "kind": "oracle", "sample": s.desc + f"; {reps} repetitions, {t:.1f} s"}
        emit(full)
    if dist is not None:
        dist.destroy_process_group()


def run_e2e(torch, tri, step, args, barrier, dist):
    """Same step through the public API with HOST buffers: every step copies its inputs (FMA stream, GEMV X, GEMM A —
    weights are resident model state) from pinned host memory and reads its results (last sweep output, Y, C) back,
    all inside the timed region.  The three legs run on three streams over two sets of device buffers, so the H2D copy
    of step i + 1 and the D2H copy of step i - 1 overlap the kernels of step i (PCIe is full duplex); the events make
    every step's kernels wait for that step's inputs and every read-back wait for that step's kernels."""
    hx = torch.empty(N_FMA, dtype=torch.float32, pin_memory=True)
    hx.copy_(step.x)
    hy = torch.empty(N_FMA, dtype=torch.float32, pin_memory=True)
    hgx = step.gx.cpu().pin_memory()
    hpa = step.pa.cpu().pin_memory()
    hgy = torch.empty(step.gy.shape, dtype=torch.bfloat16, pin_memory=True)
    hpc = torch.empty(step.pc.shape, dtype=torch.bfloat16, pin_memory=True)
    h2d = hx.numel() * 4 + hgx.numel() * 2 + hpa.numel() * 2
    d2h = hy.numel() * 4 + hgy.numel() * 2 + hpc.numel() * 2
    sets = [{"x": step.x, "y": step.y, "gx": step.gx, "gy": step.gy, "pa": step.pa, "pc": step.pc}]
    sets.append({k: torch.empty_like(v) for k, v in sets[0].items()})
    s_in, s_run, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()

    def pipeline(n):
        ev_in, ev_run, ev_out = [], [], []
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for i in range(n):
            b = sets[i % 2]
            with torch.cuda.stream(s_in):
                if i == 0:
                    t0.record()
                if i >= 2:
                    s_in.wait_event(ev_run[i - 2])                    # the kernels that read this input set are done
                b["x"].copy_(hx, non_blocking=True)
                b["gx"].copy_(hgx, non_blocking=True)
                b["pa"].copy_(hpa, non_blocking=True)
                e = torch.cuda.Event()
                e.record()
                ev_in.append(e)
            with torch.cuda.stream(s_run):
                s_run.wait_event(ev_in[i])
                if i >= 2:
                    s_run.wait_event(ev_out[i - 2])                   # the previous results in this output set are read back
                step.run(io=b)
                e = torch.cuda.Event()
                e.record()
                ev_run.append(e)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_run[i])
                hy.copy_(b["y"], non_blocking=True)
                hgy.copy_(b["gy"], non_blocking=True)
                hpc.copy_(b["pc"], non_blocking=True)
                e = torch.cuda.Event()
                e.record()
                ev_out.append(e)
                if i == n - 1:
                    t1.record()
        torch.cuda.synchronize()
        return t0.elapsed_time(t1)

    pipeline(2)
    barrier()
    n = max(1, min(args.steps, 16))                                    # the fill (first H2D) and drain (last D2H) are inside the timed region
    ms = pipeline(n)
    barrier()
    # The read-back is the last step's result: what crossed PCIe equals what that step left on the device - a strided
    # sample of the FMA output, ALL of the GEMV's Y and 8 rows spread over the GEMM's C.  (The results themselves are held
    # to the oracle by tests/ and smoke(); bench.py's GPU arm may not execute oracle/ outside the cpu_baseline leg.)
    last = sets[(n - 1) % 2]
    rows = torch.linspace(0, hpc.shape[0] - 1, 8).long()
    ok = bool(torch.equal(hy[:: N_FMA // 4096], last["y"][:: N_FMA // 4096].cpu()) and torch.equal(hgy, last["gy"].cpu())
              and torch.equal(hpc[rows], last["pc"][rows.to(last["pc"].device)].cpu())
              and bool(torch.isfinite(hgy.float()).all()) and bool(torch.isfinite(hpc[rows].float()).all()))
    ms = max_over_ranks(ms, dist, "cuda")
    world = dist.get_world_size() if dist is not None else 1
    return {"value": whole_job_value(STEP_FLOP, n, world, ms), "unit": UNIT,
            "ms_per_step": ms / n, "steps": n, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
            "overlap": "H2D(i+1)|kernels(i)|D2H(i-1)", "readback_checked": ok}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)     # 20 timed reps per A.I. point (BASELINE.json config 2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--char-seconds", type=float, default=1.0,
                    help="seconds of sustained looping per A.I. point for clock / temperature / J-per-op (0 = skip)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
