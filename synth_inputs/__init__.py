"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side harness.

This module holds NONE of the method's arithmetic (no fma chain, no GEMV/GEMM, no
rounding of results).  It only produces the input arrays BASELINE.json's configs name:

* ``uniform_pm1``      fp32 "uniform in [-1,1] from seed s" (configs 1-2)
* ``normal_bf16``      bf16 "~N(0, std)" arrays (configs 3-4)
* ``stratified_rows``  the "64 seeded sampled rows" of config 4

The generator is counter-based (no state, no dependence on the numpy / torch RNG
version):  ``h = mix64(key(seed, stream) + i)`` where mix64 is the splitmix64 finaliser
(two xor-shift-multiply rounds and a final xor-shift) and
``key(seed, stream) = (seed << 48) + (stream << 40)``, ``i < 2**40``.

These inputs stand in for Qwen2.5-Omni-7B Thinker activations / weights (PAPER.md
lines 52, 90, 202-203); only shapes and value distributions are taken, from
BASELINE.json, since the paper prints no tensor and the model / datasets are absent.
"""
from __future__ import annotations

import numpy as np

_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_CHUNK = 1 << 22


def key(seed: int, stream: int = 0) -> int:
    if not (0 <= seed < (1 << 16) and 0 <= stream < (1 << 8)):
        raise ValueError("seed must be in [0, 2^16), stream in [0, 2^8)")
    return (seed << 48) + (stream << 40)


def mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wraps modulo 2^64)."""
    z = z.astype(np.uint64, copy=True)
    z ^= z >> np.uint64(30)
    z *= _M1
    z ^= z >> np.uint64(27)
    z *= _M2
    z ^= z >> np.uint64(31)
    return z


def _counters(base: int, start: int, count: int) -> np.ndarray:
    return np.arange(start, start + count, dtype=np.uint64) + np.uint64(base)


def uniform_pm1(seed: int, n: int, start: int = 0, stream: int = 0) -> np.ndarray:
    """fp32 values (m - 2^23) * 2^-23, m = top 24 bits of mix64(key + i): the 2^-23 grid
    on [-1, 1 - 2^-23].  Element i depends only on (seed, stream, i)."""
    out = np.empty(n, dtype=np.float32)
    base = key(seed, stream)
    for lo in range(0, n, _CHUNK):
        cnt = min(_CHUNK, n - lo)
        h = mix64(_counters(base, start + lo, cnt))
        m = (h >> np.uint64(40)).astype(np.int64) - (1 << 23)
        out[lo:lo + cnt] = (m.astype(np.float64) * 2.0 ** -23).astype(np.float32)
    return out


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16 bit patterns (uint16).  Input data only; finite values."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    r = (u + np.uint64(0x7FFF) + ((u >> np.uint64(16)) & np.uint64(1))) >> np.uint64(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def normal_f64(seed: int, n: int, start: int = 0, stream: int = 0) -> np.ndarray:
    """Standard normals by Box-Muller in double on two counter-based uniforms per element:
    u1 = (top53(mix64(key+2i)) + 1) * 2^-53 in (0, 1],  u2 = top53(mix64(key+2i+1)) * 2^-53."""
    out = np.empty(n, dtype=np.float64)
    base = key(seed, stream)
    for lo in range(0, n, _CHUNK):
        cnt = min(_CHUNK, n - lo)
        c = _counters(base, 2 * (start + lo), 2 * cnt)
        h = mix64(c) >> np.uint64(11)
        u1 = (h[0::2].astype(np.float64) + 1.0) * 2.0 ** -53
        u2 = h[1::2].astype(np.float64) * 2.0 ** -53
        out[lo:lo + cnt] = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    return out


def normal_bf16(seed: int, shape, std: float = 1.0, stream: int = 0) -> np.ndarray:
    """bf16 bit patterns (uint16) of N(0, std^2): Box-Muller in double -> * std -> fp32 -> bf16 RNE.
    The value at flat index i (row-major over the LOGICAL shape) depends only on (seed, stream, i)."""
    n = int(np.prod(shape))
    z = normal_f64(seed, n, 0, stream) * std
    return f32_to_bf16_bits(z.astype(np.float32)).reshape(shape)


def stratified_rows(seed: int, m: int, count: int = 64) -> np.ndarray:
    """``count`` row indices in [0, m): one per consecutive block of m/count rows, the offset inside
    each block taken from the seeded generator.  Sorted ascending, int32."""
    count = min(count, m)
    edges = (np.arange(count + 1, dtype=np.int64) * m) // count
    h = mix64(_counters(key(seed, 255), 0, count)) >> np.uint64(33)
    width = (edges[1:] - edges[:-1])
    return (edges[:-1] + (h.astype(np.int64) % width)).astype(np.int32)


# ---------------------------------------------------------------------------------------------
# Device-side twins (torch int64 arithmetic; used for the multi-GiB timing buffers so that a
# bench run does not spend its time in numpy).  uniform_pm1_torch is bit-identical to
# uniform_pm1 (pure integer arithmetic; tested).  normal_bf16_torch uses the device's log/cos,
# so it is the same distribution but not bit-pinned: parity inputs always come from the numpy
# functions above.
# ---------------------------------------------------------------------------------------------

def _mix64_torch(z):
    import torch
    def lsr(v, s):
        return (v >> s) & ((1 << (64 - s)) - 1)
    m1 = torch.tensor(0xBF58476D1CE4E5B9 - (1 << 64), dtype=torch.int64, device=z.device)
    m2 = torch.tensor(0x94D049BB133111EB - (1 << 64), dtype=torch.int64, device=z.device)
    z = z ^ lsr(z, 30)
    z = z * m1
    z = z ^ lsr(z, 27)
    z = z * m2
    z = z ^ lsr(z, 31)
    return z


def uniform_pm1_torch(seed: int, n: int, device="cpu", start: int = 0, stream: int = 0, out=None):
    import torch
    if out is None:
        out = torch.empty(n, dtype=torch.float32, device=device)
    base = key(seed, stream)
    if base >= (1 << 63):
        base -= (1 << 64)
    chunk = 1 << 25
    for lo in range(0, n, chunk):
        cnt = min(chunk, n - lo)
        c = torch.arange(start + lo, start + lo + cnt, dtype=torch.int64, device=out.device) + base
        h = _mix64_torch(c)
        m = ((h >> 40) & ((1 << 24) - 1)) - (1 << 23)
        out[lo:lo + cnt] = (m.to(torch.float64) * 2.0 ** -23).to(torch.float32)
    return out


def normal_bf16_torch(seed: int, shape, std: float = 1.0, device="cpu", stream: int = 0):
    import math
    import torch
    n = int(np.prod(shape))
    out = torch.empty(n, dtype=torch.bfloat16, device=device)
    base = key(seed, stream)
    if base >= (1 << 63):
        base -= (1 << 64)
    chunk = 1 << 24
    for lo in range(0, n, chunk):
        cnt = min(chunk, n - lo)
        c = torch.arange(2 * lo, 2 * (lo + cnt), dtype=torch.int64, device=out.device) + base
        h = (_mix64_torch(c) >> 11) & ((1 << 53) - 1)
        u1 = (h[0::2].to(torch.float64) + 1.0) * 2.0 ** -53
        u2 = h[1::2].to(torch.float64) * 2.0 ** -53
        z = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2) * std
        out[lo:lo + cnt] = z.to(torch.float32).to(torch.bfloat16)
    return out.reshape(shape)
