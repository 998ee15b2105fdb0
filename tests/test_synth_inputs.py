"""The seeded input generators (synth_inputs): golden prefixes, grid / range / moments, and the
torch twin used for the multi-GiB timing buffers."""
import os

import numpy as np
import torch

from synth_inputs import (bf16_bits_to_f32, f32_to_bf16_bits, mix64, normal_bf16, normal_bf16_torch,
                          normal_f64, stratified_rows, uniform_pm1, uniform_pm1_torch)

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "synth_inputs_golden.txt")


def _golden():
    out = {}
    for line in open(GOLDEN):
        if line.startswith("#"):
            continue
        *k, = line.split()
        name = " ".join(t for t in k if "=" in t or not all(c in "0123456789ABCDEF" for c in t))
        out[name] = [t for t in k if t not in name.split()]
    return out


def test_mix64_known_vector():
    # splitmix64 with seed 0: first output = mix64(0x9E3779B97F4A7C15) (published test vector)
    assert int(mix64(np.array([0x9E3779B97F4A7C15], np.uint64))[0]) == 0xE220A8397B1DCDAF


def test_golden_prefixes():
    g = _golden()
    for seed in (0, 1):
        got = [f"{x:08X}" for x in uniform_pm1(seed, 8).view(np.uint32)]
        assert got == g[f"uniform_pm1 seed={seed}"]
    got = [f"{x:08X}" for x in uniform_pm1(1, 4, start=(1 << 28) - 4).view(np.uint32)]
    assert got == g["uniform_pm1_tail seed=1"]
    for seed, std, stream in ((2, 1.0, 0), (2, 0.02, 1), (3, 1.0, 0), (3, 0.02, 1)):
        got = [f"{x:04X}" for x in normal_bf16(seed, (8,), std=std, stream=stream)]
        assert got == g[f"normal_bf16 seed={seed} std={std} stream={stream}"]
    assert [str(x) for x in stratified_rows(3, 4096)[:8]] == g["stratified_rows seed=3 m=4096"]


def test_uniform_grid_range_moments_and_offsets():
    x = uniform_pm1(0, 1 << 20)
    assert x.dtype == np.float32 and x.min() >= -1.0 and x.max() <= 1.0 - 2.0 ** -23
    m = x.astype(np.float64) * 2.0 ** 23
    assert (m == np.round(m)).all()
    assert abs(x.mean()) < 3e-3 and abs(x.var() - 1.0 / 3.0) < 3e-3
    # counter-based: any window equals the same window of the whole stream; seeds differ
    assert (uniform_pm1(0, 100, start=5000) == x[5000:5100]).all()
    assert (uniform_pm1(1, 100) != x[:100]).any()


def test_uniform_torch_twin_is_bit_identical():
    for seed, n, start in ((0, 100000, 0), (1, 4097, (1 << 28) - 4097)):
        a = uniform_pm1(seed, n, start=start)
        b = uniform_pm1_torch(seed, n, start=start).numpy()
        assert (a.view(np.uint32) == b.view(np.uint32)).all()


def test_normal_moments_and_bf16():
    z = normal_f64(2, 1 << 20)
    assert abs(z.mean()) < 4e-3 and abs(z.std() - 1.0) < 4e-3 and np.abs(z).max() < 7
    w = bf16_bits_to_f32(normal_bf16(2, (1 << 18,), std=0.02, stream=1)).astype(np.float64)
    assert abs(w.mean()) < 2e-4 and abs(w.std() - 0.02) < 2e-4
    # bf16 round trip of representable values is the identity; RNE on a tie goes to even
    b = normal_bf16(3, (1000,))
    assert (f32_to_bf16_bits(bf16_bits_to_f32(b)) == b).all()
    assert f32_to_bf16_bits(np.array([np.float32(1.00390625)]))[0] == 0x3F80
    assert f32_to_bf16_bits(np.array([np.float32(1.01171875)]))[0] == 0x3F82


def test_normal_torch_twin_same_distribution():
    a = bf16_bits_to_f32(normal_bf16(2, (1 << 16,), std=0.02, stream=1))
    b = normal_bf16_torch(2, (1 << 16,), std=0.02, stream=1).float().numpy()
    # same counters, device libm may differ in the last place before rounding: nearly all equal
    assert (a == b).mean() > 0.999


def test_stratified_rows_cover_every_block():
    r = stratified_rows(3, 4096)
    assert r.size == 64 and (np.diff(r) > 0).all()
    assert (r // 64 == np.arange(64)).all()
    r2 = stratified_rows(3, 10, 64)
    assert (r2 == np.arange(10)).all()
    assert (stratified_rows(4, 4096) != r).any()
