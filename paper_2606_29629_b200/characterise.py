"""Long-running characterisation runs on one B200 (the paper's Fig. 1-bottom / Fig. 4 experiments on this library's kernels).

    python -m paper_2606_29629_b200.characterise trace   [--seconds 60] [--out FILE.json]
    python -m paper_2606_29629_b200.characterise thermal [--seconds 240] [--points k1,k16,k64,k4096,gemv,gemm] [--out FILE.json]

trace    BASELINE.json config 5: 60 s of [prefill GEMM 2 s | decode GEMV 2 s | idle 1 s] through the library's
         phase_trace() driver (NVML every 10 ms, tagged by phase); prints the per-phase-kind aggregates and the clock
         decay inside the prefill phases (Fig. 4a).
thermal  PAPER.md lines 106-110 (Fig. 4b / 4c): every chosen A.I. point is looped for `seconds`; throughput (CUDA events
         per ~50 ms batch), SM clock, temperature and power (NVML every 100 ms) are reduced to 1 s bins.

Everything runs through the C ABI binding; synthetic seeded inputs (synth_inputs).  Output: one JSON document (to
--out or stdout) and a short table on stderr.  Clocks are never locked (reading R17).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

N_FMA = 1 << 28
GEMV_SHAPE = (8, 18944, 3584)          # m, n, k   (BASELINE.json config 3)
GEMM_SHAPE = (4096, 18944, 3584)       # config 4
GEMV_COPIES = 8


def _buffers(torch, seed, want_fma=True):
    from synth_inputs import normal_bf16_torch, uniform_pm1_torch
    dev = "cuda"
    b = {}
    if want_fma:
        b["x"] = uniform_pm1_torch(1, N_FMA, device=dev)
        b["y"] = torch.empty_like(b["x"])
    m, n, k = GEMV_SHAPE
    b["gx"] = normal_bf16_torch(seed, (m, k), 1.0, dev, stream=0)
    b["gw"] = [normal_bf16_torch(seed, (n, k), 0.02, dev, stream=1 + r) for r in range(GEMV_COPIES)]
    b["gy"] = torch.empty((m, n), dtype=torch.bfloat16, device=dev)
    pm, pn, pk = GEMM_SHAPE
    b["pa"] = normal_bf16_torch(seed, (pm, pk), 1.0, dev, stream=20)
    b["pw"] = normal_bf16_torch(seed, (pn, pk), 0.02, dev, stream=21)
    b["pc"] = torch.empty((pm, pn), dtype=torch.bfloat16, device=dev)
    return b


def run_trace(args):
    import torch
    import paper_2606_29629_b200 as tri
    torch.cuda.set_device(0)
    tri.tri_init(0)
    b = _buffers(torch, 4, want_fma=False)
    (pm, pn, pk), (dm, dn, dk) = GEMM_SHAPE, GEMV_SHAPE
    samples, summ = tri.phase_trace(pm, pn, pk, b["pa"], b["pw"], b["pc"], dm, dn, dk, b["gx"], b["gw"], b["gy"], tri.TRI_W_NK,
                                    total_s=args.seconds, prefill_s=2.0, decode_s=2.0, idle_s=1.0, period_ms=10)
    kinds = {}
    for s in summ:
        kinds.setdefault(s["phase_name"], []).append(s)
    agg = {}
    for name, ss in kinds.items():
        def mean(key):
            v = [x[key] for x in ss if x.get(key) is not None]
            return sum(v) / len(v) if v else None
        agg[name] = {"instances": len(ss), "launches": sum(x["launches"] for x in ss),
                     "sm_mhz_mean": mean("sm_mhz_mean"), "sm_mhz_first10": mean("sm_mhz_first10"),
                     "sm_mhz_last10": mean("sm_mhz_last10"), "temp_c_max": max(x["temp_c_max"] for x in ss),
                     "mean_power_w": mean("mean_power_w"), "energy_j": sum(x["energy_j"] for x in ss),
                     "j_per_flop": mean("j_per_flop") if name != "idle" else None,
                     "j_per_byte": mean("j_per_byte") if name != "idle" else None,
                     "j_per_token": mean("j_per_token") if name != "idle" else None,
                     "tflops": (sum(x["flop"] for x in ss) / sum(x["gpu_ms"] for x in ss) / 1e9) if name != "idle" else None,
                     "gbs": (sum(x["bytes"] for x in ss) / sum(x["gpu_ms"] for x in ss) / 1e6) if name != "idle" else None}
    # cadence of the sampler, from the record itself: per phase kind the samples against the nominal count, the longest gap,
    # and the distribution of how long one sample's NVML queries took (tri_sample.read_us)
    def pct(v, q):
        return v[min(len(v) - 1, int(q * len(v)))] if v else None
    cadence = {"first_sample_t_s": samples[0]["t_s"] if samples else None}
    for name, ss in kinds.items():
        code = ss[0]["phase"]
        rd = sorted(x["read_us"] for x in samples if x["phase"] == code)
        cadence[name] = {"n_samples": sum(x["n_samples"] for x in ss), "expected_samples": sum(x["expected_samples"] for x in ss),
                         "max_gap_ms": max(x["max_gap_us"] for x in ss) / 1e3,
                         "read_us_p50": pct(rd, 0.50), "read_us_p95": pct(rd, 0.95), "read_us_p99": pct(rd, 0.99), "read_us_max": rd[-1] if rd else None}
    doc = {"experiment": "config 5 phase trace", "seconds": args.seconds, "period_ms": 10, "n_samples": len(samples),
           "aggregate": agg, "cadence": cadence, "phases": summ,
           "samples": [[round(s["t_s"], 3), s["phase"], s["sm_mhz"], s["temp_c"], round(s["power_w"], 1), s["read_us"]] for s in samples],
           "samples_columns": ["t_s", "phase", "sm_mhz", "temp_c", "power_w", "read_us"]}
    sys.stderr.write(f"first sample at {cadence['first_sample_t_s'] * 1e3:.2f} ms\n")
    for name in kinds:
        c = cadence[name]
        sys.stderr.write(f"{name:8s} samples {c['n_samples']} of {c['expected_samples']} nominal, longest gap {c['max_gap_ms']:.1f} ms, "
                         f"NVML read p50 / p95 / p99 / max {c['read_us_p50']} / {c['read_us_p95']} / {c['read_us_p99']} / {c['read_us_max']} us\n")
    for name, a in agg.items():
        sys.stderr.write(f"{name:8s} x{a['instances']:2d}  clock mean {a['sm_mhz_mean'] or 0:6.0f} MHz (first 10 % {a['sm_mhz_first10'] or 0:6.0f}, "
                         f"last 10 % {a['sm_mhz_last10'] or 0:6.0f})  Tmax {a['temp_c_max']:.0f} C  P {a['mean_power_w'] or 0:5.0f} W"
                         + (f"  {a['tflops']:8.1f} TFLOP/s  {a['gbs']:7.0f} GB/s  {a['j_per_flop'] * 1e12:7.2f} pJ/FLOP  {a['j_per_token'] * 1e3:8.3f} mJ/token"
                            if a["tflops"] else "") + "\n")
    return doc


def run_thermal(args):
    import torch
    import paper_2606_29629_b200 as tri
    torch.cuda.set_device(0)
    tri.tri_init(0)
    names = [p.strip() for p in args.points.split(",") if p.strip()]
    b = _buffers(torch, 2, want_fma=any(p.startswith("k") for p in names))
    (pm, pn, pk), (dm, dn, dk) = GEMM_SHAPE, GEMV_SHAPE

    def spec(name):
        """-> (callable enqueueing `calls` launches, calls, FLOP per call, bytes per call, A.I.)"""
        if name == "gemm":
            fl, by = 2.0 * pm * pn * pk, 2.0 * (pm * pk + pk * pn + pm * pn)
            return (lambda: tri.prefill_gemm(pm, pn, pk, b["pa"], pk, b["pw"], pk, tri.TRI_W_NK, b["pc"], pn)), 1, fl, by, fl / by
        if name == "gemv":
            fl, by = 2.0 * dm * dn * dk, 2.0 * (dm * dk + dk * dn + dm * dn)

            def f():
                for w in b["gw"]:
                    tri.decode_gemv(dm, dn, dk, b["gx"], dk, w, dk, tri.TRI_W_NK, b["gy"], dn)
            return f, GEMV_COPIES, fl, by, fl / by
        k = int(name[1:])
        return (lambda: tri.roofline_run(k / 4.0, N_FMA, b["x"], b["y"])), 1, 2.0 * k * N_FMA, 8.0 * N_FMA, k / 4.0

    doc = {"experiment": "thermal steady state (PAPER.md lines 106-110)", "seconds_per_point": args.seconds, "points": []}
    for name in names:
        fn, per_call, flop, nbytes, ai = spec(name)
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        fn()
        torch.cuda.synchronize()
        est = max(time.perf_counter() - t0, 1e-5)
        batch = max(1, int(0.05 / est))                                   # about 50 ms of work per batch
        tracer = tri.PhaseTracer(0, period_us=100000, capacity=int(args.seconds * 12) + 256).start(tri.TRI_PHASE_ROOFLINE)
        e0 = tri.tri_nvml_sample(0)["energy_mj"]
        batches = []                                                      # (host time at end, device ms, calls)
        start = time.perf_counter()
        pending = []
        while time.perf_counter() - start < args.seconds:
            a, c = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(batch):
                fn()
            c.record()
            pending.append((a, c))
            if len(pending) >= 2:                                         # keep one batch queued behind the running one
                pa_, pc_ = pending.pop(0)
                pc_.synchronize()
                batches.append((time.perf_counter() - start, pa_.elapsed_time(pc_), batch * per_call))
        for pa_, pc_ in pending:
            pc_.synchronize()
            batches.append((time.perf_counter() - start, pa_.elapsed_time(pc_), batch * per_call))
        e1 = tri.tri_nvml_sample(0)["energy_mj"]
        samples = tracer.stop()
        nbin = int(args.seconds)
        series = []
        for sec in range(nbin):
            bb = [x for x in batches if sec <= x[0] < sec + 1]
            ss = [x for x in samples if sec <= x["t_s"] < sec + 1 and x["sm_mhz"] > 0]
            if not bb or not ss:
                continue
            ms, calls = sum(x[1] for x in bb), sum(x[2] for x in bb)
            series.append([sec, round(flop * calls / ms / 1e9, 3), round(nbytes * calls / ms / 1e6, 1),
                           statistics.median(x["sm_mhz"] for x in ss), max(x["temp_c"] for x in ss),
                           round(sum(x["power_w"] for x in ss) / len(ss), 1)])

        def window(lo, hi, col):
            v = [r[col] for r in series if lo <= r[0] < hi]
            return sum(v) / len(v) if v else None

        bits = 0
        for x in samples:
            bits |= int(x["clk_event_reasons"])
        tot_calls = sum(x[2] for x in batches)
        w = max(10, nbin // 24)
        pt = {"point": name, "ai": ai, "calls": tot_calls, "series_columns": ["t_s", "tflops", "gbs", "sm_mhz", "temp_c", "power_w"],
              "series": series, "clk_event_reasons": bits,
              "tflops_first": window(0, w, 1), "tflops_last": window(nbin - w, nbin, 1),
              "sm_mhz_first": window(0, w, 3), "sm_mhz_last": window(nbin - w, nbin, 3),
              "temp_c_first": window(0, w, 4), "temp_c_last": window(nbin - w, nbin, 4),
              "power_w_first": window(0, w, 5), "power_w_last": window(nbin - w, nbin, 5),
              "window_s": w, "j_per_flop": (e1 - e0) * 1e-3 / (flop * tot_calls) if e1 > e0 else None}
        doc["points"].append(pt)
        f = lambda v, fmt: format(v, fmt) if v is not None else "   n/a"
        sys.stderr.write(f"{name:6s} A.I. {ai:8.2f}: TFLOP/s {f(pt['tflops_first'], '8.2f')} -> {f(pt['tflops_last'], '8.2f')}   clock "
                         f"{f(pt['sm_mhz_first'], '6.0f')} -> {f(pt['sm_mhz_last'], '6.0f')} MHz   T {f(pt['temp_c_first'], '4.1f')} -> "
                         f"{f(pt['temp_c_last'], '4.1f')} C   P {f(pt['power_w_first'], '5.0f')} -> {f(pt['power_w_last'], '5.0f')} W   "
                         f"{f((pt['j_per_flop'] or 0) * 1e12, '7.2f')} pJ/FLOP  reasons 0x{bits:x}\n")
        time.sleep(args.cooldown)                                          # let the die cool before the next point
    return doc


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    sub = ap.add_subparsers(dest="cmd", required=True)
    t = sub.add_parser("trace")
    t.add_argument("--seconds", type=float, default=60.0)
    t.add_argument("--out", default=None)
    h = sub.add_parser("thermal")
    h.add_argument("--seconds", type=float, default=240.0)
    h.add_argument("--cooldown", type=float, default=20.0)
    h.add_argument("--points", default="k1,k16,k32,k64,k256,k4096,gemv,gemm")
    h.add_argument("--out", default=None)
    args = ap.parse_args()
    doc = run_trace(args) if args.cmd == "trace" else run_thermal(args)
    text = json.dumps(doc)
    if args.out:
        with open(args.out, "w") as fh:
            fh.write(text + "\n")
    else:
        print(text)


if __name__ == "__main__":
    main()
