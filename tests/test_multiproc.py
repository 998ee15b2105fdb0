"""The N > 1 path of bench.py on CPU: world_size 2, gloo.  The hot path shards with no collective (DESIGN.md §7:
replicas only), so what is multi-rank is host logic: barrier, max-over-ranks time, whole-job aggregate, and the
reference arm running on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(script_args, nproc=2, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port())] + script_args
    env = dict(os.environ, OMP_NUM_THREADS="2")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def _json_lines(text):
    return [json.loads(l) for l in text.splitlines() if l.startswith("{")]


def test_max_over_ranks_and_whole_job_value_world2():
    r = _torchrun([os.path.join("tests", "gloo_worker.py")])
    assert r.returncode == 0, r.stderr[-2000:]
    out = _json_lines(r.stdout)
    assert len(out) == 1
    import bench
    assert out[0]["world"] == 2 and out[0]["ms"] == 20.0                      # the slower rank's time
    assert abs(out[0]["value"] - bench.STEP_FLOP * 4 * 2 / 20e-3 / 1e12) < 1e-9 * out[0]["value"]


def test_reference_arm_runs_on_rank0_only():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"])
    assert r.returncode == 0, r.stderr[-2000:]
    out = _json_lines(r.stdout)
    assert len(out) == 1, "exactly one JSON line, from rank 0"
    d = out[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
