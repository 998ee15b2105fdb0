"""bench.py's output contract: stdout ends with ONE compact JSON line that the driver can parse (round 1's 20 KB line
could not be: BENCH_r01.json "parsed": null).  The formatter is exercised on a full-sized mock of the GPU arm's result
and the reference arm is run for real (CPU oracle)."""
import json
import os
import subprocess
import sys

import bench

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

REQUIRED = ["metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
            "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline", "min_frac", "fracs"]


def mock_full():
    """What run_ours() hands to emit(): every point of the sweep with its sustained record, the extra series (paper A.I.
    set, ridge points, matmul-based series, second GEMM shapes) and the model fit — the bulk that must NOT be on the line."""
    sus = {"series": "sweep", "k": 1, "ms_sustained": 0.3161, "launches": 1590, "window_s": 0.5026, "gbs_sustained": 6793.812,
           "tflops_sustained": 1.698, "sm_mhz": 1965.0, "mem_mhz": 3996.0, "temp_c_max": 48, "power_w_mean": 812.123,
           "reasons": ["sw_power_cap"], "j_per_flop": 1.2345e-11, "j_per_byte": 1.1e-10, "j_per_call": 0.25, "nvml_samples": 50}
    pts = [{"kernel": "fma_chain", "k": k, "ai": k / 4, "ms": 0.3161234, "gbs": 6793.812345, "tflops": 1.698453, "bound": "hbm",
            "roofline_tflops": 1.635775, "frac": 1.0383112, "ms_min": 0.3142, "frac_vs_nominal": 0.8492, "sustained": dict(sus),
            "roofline_tflops_at_clock": 1.6357, "frac_sustained_at_clock": 1.0381234} for k in bench.KS]
    pts.append({"kernel": "decode_gemv", "ai": 7.98, "ms": 0.0215, "gbs": 6332.6, "tflops": 50.5, "bound": "hbm", "roofline_gbs": 6543.1,
                "frac": 0.9678, "ms_min": 0.0209, "frac_vs_nominal": 0.79, "sustained": dict(sus), "frac_sustained_at_clock": 0.95})
    pts.append({"kernel": "prefill_gemm", "ai": 1736.0, "ms": 0.3312, "gbs": 967.0, "tflops": 1679.3, "bound": "tensor",
                "roofline_tflops": 1664.6, "frac": 1.0088, "ms_min": 0.3301, "frac_vs_nominal": 0.746, "sustained": dict(sus),
                "frac_sustained_at_clock": 0.99})
    extra = [dict(pts[i % 13], series="paper A.I. set {1,25,50,100,200} (PAPER.md line 92)") for i in range(12)]
    extra += [{"kernel": "prefill_gemm", "label": lab, "frac": 0.93, "ms": 0.33, "tflops": 1500.0, "cublas_ms": 0.4}
              for lab in ("down_proj", "qkv", "o_proj", "m512", "m64", "m16")]
    return {"metric": bench.METRIC, "value": 80.1234567, "unit": bench.UNIT, "n_gpus": 1, "steps": 20, "warmup": 5,
            "ms_per_step": 61.4567891, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 chain; bf16 in / f32 acc", "data": "synthetic", "config": bench.workload_config(1),
            "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": ["sw_power_cap"], "temp_c_max": 55, "power_w_mean": 812.2,
                       "samples": 123, "source": "nvml", "sm_mhz_in_kernel_probe": 1964.9},
            "e2e": {"value": 77.3, "unit": bench.UNIT, "ms_per_step": 69.6, "steps": 16, "h2d_bytes_per_step": 1103233024,
                    "d2h_bytes_per_step": 1229234176, "overlap": "H2D(i+1) | kernels(i) | D2H(i-1)", "readback_checked": True},
            "gpu_launches": 440,
            "roofline": {"kernel": "fma_chain_kernel (k=4096 launch)", "bound": "alu", "achieved": 74.2, "peak": 74.45, "unit": "TFLOP/s",
                         "frac": 0.997, "traffic": 2.1e9, "share_of_step": 0.48,
                         "peak_source": "derived 148 SMs x 128 lanes x 2 x 1965 MHz; fracs: measured 6543.1 GB/s, 1664.6 TFLOP/s"},
            "points": pts, "extra_points": extra, "model_fit": {"rel_residuals": [0.001] * 13, "eta": 0.0377, "beta": 6.87},
            "min_frac": 0.9678, "energy": {"j_per_step": 50.0, "j_per_flop": 1.0e-11, "j_per_byte": 1.7e-9},
            "peaks": {"hbm_gbs": 6543.1},
            "cpu_baseline": {"value": 0.0156, "unit": "TFLOP/s", "cores": 16, "kind": "oracle",
                             "sample": "per step: 2^18 of 2^28 elements per k (13 k); 1 of 8 GEMVs; 8 of 4096 GEMM rows; 24 repetitions, 10.1 s"}}


def test_compact_line_is_small_and_round_trips():
    full = mock_full()
    assert len(json.dumps(full)) > 15000, "the mock must be as bulky as the real result"
    line = bench.compact_line(full)
    assert "\n" not in line and len(line) < 2600, len(line)
    d = json.loads(line)
    for k in REQUIRED:
        assert k in d, k
    assert d["value"] > 0 and d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    assert set(d["roofline"]) >= {"bound", "achieved", "peak", "unit", "frac", "traffic"}
    assert set(d["cpu_baseline"]) >= {"value", "unit", "cores", "kind", "sample"}
    assert len(d["fracs"]) == len(bench.KS) + 2 and abs(d["min_frac"] - min(d["fracs"].values())) < 1e-3
    assert "points" not in d and "extra_points" not in d and "model_fit" not in d


def test_emit_prints_exactly_one_stdout_line(tmp_path, capsys, monkeypatch):
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    bench.emit(mock_full())
    cap = capsys.readouterr()
    lines = [l for l in cap.out.splitlines() if l.strip()]
    assert len(lines) == 1 and json.loads(lines[0])["min_frac"] > 0
    detail = json.load(open(tmp_path / bench.DETAIL_FILE))
    assert len(detail["points"]) == len(bench.KS) + 2 and detail["model_fit"]
    assert all(json.loads(l) for l in cap.err.splitlines() if l.startswith("{"))


def test_reference_arm_last_line_parses():
    r = subprocess.run([sys.executable, "bench.py", "--impl", "reference", "--steps", "1", "--warmup", "0"], cwd=ROOT,
                       capture_output=True, text=True, timeout=600, env=dict(os.environ, OMP_NUM_THREADS="4"))
    assert r.returncode == 0, r.stderr[-2000:]
    last = r.stdout.strip().splitlines()[-1]
    assert len(last) < 3000
    d = json.loads(last)
    assert d["impl"] == "reference" and d["value"] > 0 and d["unit"] == bench.UNIT and d["metric"] == bench.METRIC
    assert d["config"] == bench.workload_config(1)


def test_controller_preview_on_a_synthetic_sweep():
    """bench.controller_preview (row f3 end to end: Eq. 5 + Eq. 6 on the fitted model) on points generated from a planted Eq. 4
    model: memory-bound points get a clock well below the boost ceiling with the throughput within eps, compute-bound points
    keep (1 - eps) of f_max, and Eq. 5 of equal-A.I. kernels is that A.I."""
    import paper_2606_29629_b200 as tri
    eta, beta, omega, gamma, fmax = 0.0377, 6.87, 0.7, 0.0, 1965.0
    peaks = {"sm_max_mhz": fmax}

    def theta(ai, f):
        return min(eta * f * ai / (ai + omega), beta * ai)
    pts = [{"kernel": "fma_chain", "k": k, "ai": k / 4.0, "ms": 2.0 * k * bench.N_FMA / theta(k / 4.0, fmax) / 1e9,
            "sustained": {"sm_mhz": 1600.0 if k == 32 else fmax, "tflops_sustained": theta(k / 4.0, fmax)}} for k in bench.KS]
    gemv = {"kernel": "decode_gemv", "ai": 7.98, "ms": 0.0215, "sustained": {"sm_mhz": 1650.0}}
    out = bench.controller_preview(tri, {"eta": eta, "beta": beta, "omega": omega, "gamma": gamma}, {"p_idle_w": 500.0, "p_dyn_w": 900.0},
                                   peaks, pts, pts + [gemv])
    assert abs(out["eq5_phase_ai"]["decode"] - 7.98) < 1e-12
    total = sum(p["ms"] for p in pts)
    assert abs(out["eq5_phase_ai"]["fma_sweep"] - sum(p["ms"] * p["ai"] for p in pts) / total) < 1e-9
    rows = {r["ai"]: r for r in out["eq6_per_point"]}
    assert len(rows) == len(bench.KS) and all("error" not in r for r in rows.values())
    for ai, r in rows.items():
        assert r["f_selected_mhz"] <= r["f_autoboost_mhz"] + 1e-9
        if r["feasible"]:
            assert r["theta_ratio"] >= 0.95 - 1e-12
    assert rows[0.25]["f_selected_mhz"] == 1005.0 and rows[0.25]["feasible"]          # far memory-bound: the lowest clock suffices
    assert rows[1024.0]["f_selected_mhz"] >= 0.95 * fmax - 15 and rows[1024.0]["feasible"]   # compute-bound: theta ~ f
    assert rows[1024.0]["p_model_ratio"] < 1.0 < 1.0 + rows[0.25]["p_model_ratio"]
    assert not rows[8.0]["feasible"] or rows[8.0]["f_selected_mhz"] <= 1600.0        # f_limit = the auto-boost clock of that point
    d = out["eq6_decode_phase"]
    assert d["feasible"] and 1005.0 <= d["f_selected_mhz"] <= 1650.0
    json.dumps(out)


def test_compact_line_sheds_optional_keys_rather_than_outgrow_the_tail():
    full = mock_full()
    full["config"]["workload"] = full["config"]["workload"] + " " + "x" * 600          # something made the line longer than planned
    line = bench.compact_line(full)
    d = json.loads(line)
    assert len(line) <= 2800 and "sustained_cols" not in d
    for k in REQUIRED:
        assert k in d, k
