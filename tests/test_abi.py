"""CPU-side checks of the C-ABI library (no compute call reaches a GPU here): it builds, loads, exports
every symbol include/triroof.h declares, and rejects bad arguments BEFORE any CUDA call
(include/triroof.h "Conventions")."""
import ctypes
import os
import re

import pytest

import paper_2606_29629_b200 as tri

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_loads():
    L = tri.lib()
    assert os.path.exists(tri.library_path())
    assert L.tri_status_string(0).decode() == "ok"
    assert "unknown" in L.tri_status_string(12345).decode()


def test_every_declared_symbol_is_exported():
    header = open(os.path.join(ROOT, "include", "triroof.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b([a-z_0-9]+)\s*\([^;{]*\)\s*;", header))
    declared -= {"defined"}
    assert declared == set(tri.EXPORTS), declared ^ set(tri.EXPORTS)
    L = tri.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_struct_sizes_match_header_layout():
    # tri_sample: f64, i32, 4 x u32 (one of them float), 2 x u64, naturally aligned -> 48 bytes
    assert ctypes.sizeof(tri.tri_sample) == 48
    assert ctypes.sizeof(tri.tri_phase_summary) == 128


@pytest.mark.parametrize("ai", [0.3, 0.0, -1.0, float("nan"), float("inf"), 0.26, 262144.25, 1e9])
def test_roofline_run_rejects_bad_ai(ai):
    L = tri.lib()
    assert L.roofline_run(ai, 16, 1024, 4096, 0) == tri.TRI_ERR_INVALID_ARG
    assert tri.last_error() != ""


def test_roofline_run_argument_errors():
    L = tri.lib()
    assert L.roofline_run_k(0, 1.0, 0.0, 16, 1024, 4096, 0) == tri.TRI_ERR_INVALID_ARG
    assert L.roofline_run_k((1 << 20) + 1, 1.0, 0.0, 16, 1024, 4096, 0) == tri.TRI_ERR_INVALID_ARG
    assert L.roofline_run(1.0, 16, 0, 4096, 0) == tri.TRI_ERR_INVALID_ARG          # NULL in
    assert L.roofline_run(1.0, 16, 1024 + 4, 4096, 0) == tri.TRI_ERR_ALIGNMENT
    assert L.roofline_run(1.0, 16, 1024, 4096 + 8, 0) == tri.TRI_ERR_ALIGNMENT
    assert L.roofline_run(1.0, 16, 1024, 1024 + 32, 0) == tri.TRI_ERR_INVALID_ARG  # partial overlap
    assert L.roofline_run(1.0, 0, 0, 0, 0) == tri.TRI_OK                            # n == 0: nothing to do


def _gemm_call(fn, m=8, n=64, k=64, x=4096, ldx=None, w=1 << 20, ldw=None, layout=0, y=1 << 22, ldy=None):
    ldx = k if ldx is None else ldx
    ldw = (k if layout == 0 else n) if ldw is None else ldw
    ldy = n if ldy is None else ldy
    return fn(m, n, k, x, ldx, w, ldw, layout, y, ldy, 0)


@pytest.mark.parametrize("name", ["decode_gemv", "prefill_gemm"])
def test_gemm_like_argument_errors(name):
    fn = getattr(tri.lib(), name)
    assert _gemm_call(fn, x=0) == tri.TRI_ERR_INVALID_ARG
    assert _gemm_call(fn, m=0) == tri.TRI_ERR_INVALID_ARG
    assert _gemm_call(fn, n=0) == tri.TRI_ERR_INVALID_ARG
    assert _gemm_call(fn, layout=2) == tri.TRI_ERR_INVALID_ARG
    assert _gemm_call(fn, k=60) == tri.TRI_ERR_UNSUPPORTED_SHAPE
    assert _gemm_call(fn, ldx=56) == tri.TRI_ERR_INVALID_ARG           # ldx < k
    assert _gemm_call(fn, ldw=72 + 4) == tri.TRI_ERR_ALIGNMENT          # ldw % 8 != 0
    assert _gemm_call(fn, x=4096 + 2) == tri.TRI_ERR_ALIGNMENT
    assert _gemm_call(fn, y=4096 + 64) == tri.TRI_ERR_INVALID_ARG       # output inside X
    assert tri.last_error() != ""


def test_decode_gemv_batch_limit():
    fn = tri.lib().decode_gemv
    assert _gemm_call(fn, m=17) == tri.TRI_ERR_INVALID_ARG


def test_trace_argument_errors():
    L = tri.lib()
    assert L.phase_trace_mark(None, 1) == tri.TRI_ERR_INVALID_ARG
    assert L.phase_trace_stop(None, None) == tri.TRI_ERR_INVALID_ARG
    buf = (tri.tri_sample * 4)()
    h = ctypes.c_void_p()
    assert L.phase_trace_start(0, 10, buf, 4, ctypes.byref(h)) == tri.TRI_ERR_INVALID_ARG   # period < 1 ms
    assert L.phase_trace_start(0, 10000, None, 4, ctypes.byref(h)) == tri.TRI_ERR_INVALID_ARG
    assert L.tri_lock_clocks(0, 0, 0) == tri.TRI_ERR_INVALID_ARG
    v = ctypes.c_double()
    assert L.tri_sm_clock_mhz(0, ctypes.byref(v), None) == tri.TRI_ERR_INVALID_ARG


def test_no_gpu_fails_loudly_not_silently():
    """Without a usable sm_100 device a compute call must return an error status (no CPU fallback)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    L = tri.lib()
    st = L.roofline_run(1.0, 16, 1024, 4096, 0)
    assert st in (tri.TRI_ERR_CUDA, tri.TRI_ERR_ARCH)
    st = _gemm_call(L.decode_gemv)
    assert st in (tri.TRI_ERR_CUDA, tri.TRI_ERR_ARCH)


def test_product_does_not_import_oracle():
    """The product path shares nothing with oracle/ (parity rule): no source under the package or
    include/ mentions it."""
    pkg = os.path.join(ROOT, "paper_2606_29629_b200")
    for base, _, files in os.walk(pkg):
        if os.path.basename(base) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(base, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "oracle/" not in text, f


def test_binding_has_every_c_name():
    """The Python binding mirrors the C ABI name for name (argument marshalling only)."""
    assert [n for n in tri.EXPORTS if not hasattr(tri, n)] == []
