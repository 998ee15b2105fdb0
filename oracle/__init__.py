"""ORACLE — test infrastructure, not the product.

Plain, slow CPU definitions (C, gcc) of what the hot path computes, with a ctypes wrapper.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2606_29629_b200 and shares no code with it.

    fma_chain(x, k, a, b)            SURVEY.md §8(c) Oracle A   (oracle/fma_chain.c)
    gemm_rows(a16, w16, rows, ...)   SURVEY.md §8(c) Oracle B   (oracle/gemm_rows.c)
    oracle.dvfs_model                row f3: PAPER.md Eq. 1-6 in plain fp64 Python, Eq. 6 by exhaustive search

Parity pins live in tests/test_oracle_fma.py, tests/test_oracle_gemm.py and tests/test_oracle_dvfs.py; no function here is
"parity unpinned".
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from .build import build as _build

A_DEFAULT = np.float32(0.9990234375)   # 1 - 2^-10 = 0x3F7FC000  (BASELINE.json config 1)
B_DEFAULT = np.float32(0.0009765625)   # 2^-10     = 0x3A800000

W_NK = 0   # physical W[n][k], K contiguous
W_KN = 1   # physical W[k][n], N contiguous

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build())
        L.oracle_fma_chain.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_uint,
                                       ctypes.c_float, ctypes.c_float]
        L.oracle_fma_chain.restype = None
        L.oracle_count_bit_mismatches.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t,
                                                  ctypes.POINTER(ctypes.c_longlong)]
        L.oracle_count_bit_mismatches.restype = ctypes.c_size_t
        L.oracle_f32_to_bf16_rne.argtypes = [ctypes.c_float]
        L.oracle_f32_to_bf16_rne.restype = ctypes.c_uint16
        L.oracle_bf16_to_f32.argtypes = [ctypes.c_uint16]
        L.oracle_bf16_to_f32.restype = ctypes.c_float
        L.oracle_gemm_rows.argtypes = [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_longlong,
                                       ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_int,
                                       ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.oracle_gemm_rows.restype = None
        _lib = L
    return _lib


def num_threads() -> int:
    """Threads the OpenMP loops use (OMP_NUM_THREADS, else the cores this process may run on)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env and env.isdigit() and int(env) > 0:
        return int(env)
    return len(os.sched_getaffinity(0))


def fma_chain(x: np.ndarray, k: int, a=A_DEFAULT, b=B_DEFAULT) -> np.ndarray:
    """out[i] = chain_k(x[i]); fp32 in, fp32 out (new array)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    out = np.empty_like(x)
    lib().oracle_fma_chain(x.ctypes.data, out.ctypes.data, x.size, int(k), float(a), float(b))
    return out


def count_bit_mismatches(x: np.ndarray, y: np.ndarray):
    """(number of differing 32-bit patterns, index of the first one or -1)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    assert x.size == y.size
    first = ctypes.c_longlong(-1)
    bad = lib().oracle_count_bit_mismatches(x.ctypes.data, y.ctypes.data, x.size, ctypes.byref(first))
    return int(bad), int(first.value)


def f32_to_bf16_rne(f: float) -> int:
    return int(lib().oracle_f32_to_bf16_rne(float(f)))


def gemm_rows(a16: np.ndarray, w16: np.ndarray, rows=None, w_layout: int = W_NK):
    """Definition of Y = A·W on the selected rows.

    a16: uint16 [m][k] bf16 bit patterns.  w16: uint16, physical [n][k] (W_NK) or [k][n] (W_KN).
    Returns dict(c64, s64, c32, y16), each [len(rows)][n]."""
    a16 = np.ascontiguousarray(a16, dtype=np.uint16)
    w16 = np.ascontiguousarray(w16, dtype=np.uint16)
    m, k = a16.shape
    if w_layout == W_NK:
        n, kw = w16.shape
    else:
        kw, n = w16.shape
    if kw != k:
        raise ValueError("inner dimensions differ")
    rows = np.arange(m, dtype=np.int32) if rows is None else np.ascontiguousarray(rows, dtype=np.int32)
    if rows.size and (rows.min() < 0 or rows.max() >= m):
        raise ValueError("row index out of range")
    r = rows.size
    c64 = np.empty((r, n), np.float64)
    s64 = np.empty((r, n), np.float64)
    c32 = np.empty((r, n), np.float32)
    y16 = np.empty((r, n), np.uint16)
    lib().oracle_gemm_rows(a16.ctypes.data, k, w16.ctypes.data, w16.shape[1], int(w_layout), n, k,
                           rows.ctypes.data, r, c64.ctypes.data, s64.ctypes.data, c32.ctypes.data,
                           y16.ctypes.data)
    return {"c64": c64, "s64": s64, "c32": c32, "y16": y16}
