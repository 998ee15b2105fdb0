"""Pins for Oracle B (oracle/gemm_rows.c) — SURVEY.md §8(c) Oracle B; PAPER.md line 90 names the
operators (prefill dense GEMM, decode GEMV); shapes from BASELINE.json configs 3-4."""
from fractions import Fraction

import numpy as np
import pytest
import torch

import oracle
from oracle import W_KN, W_NK
from synth_inputs import bf16_bits_to_f32, f32_to_bf16_bits, normal_bf16
from tests.exact import bits_f32, round_f32_to_bf16_bits


def bf16(x):
    return f32_to_bf16_bits(np.asarray(x, dtype=np.float32))


def test_bf16_rounding_ties_and_edges():
    # RNE fp32 -> bf16 on hand-built patterns: below / at / above the tie,
    # odd and even keepers, carry into the exponent, negative, zero
    for u in (0x3F800000, 0x3F807FFF, 0x3F808000, 0x3F808001, 0x3F818000, 0x3F817FFF, 0x3FFF8000,
              0x3FFFFFFF, 0xBF808000, 0xBF818000, 0x00000000, 0x80000000, 0x7F7F7FFF, 0x00018000):
        f = bits_f32(u)
        assert oracle.f32_to_bf16_rne(f) == round_f32_to_bf16_bits(f), hex(u)
    assert oracle.f32_to_bf16_rne(bits_f32(0x3F808000)) == 0x3F80      # tie -> even (down)
    assert oracle.f32_to_bf16_rne(bits_f32(0x3F818000)) == 0x3F82      # tie -> even (up)


def test_bf16_rounding_matches_torch_conversion():
    # library special case: torch's fp32 -> bfloat16 cast is RNE
    rng = np.random.default_rng(0)
    x = np.concatenate([rng.standard_normal(20000).astype(np.float32) * 3,
                        (rng.integers(0, 1 << 32, 20000, dtype=np.uint64).astype(np.uint32) & 0x7F7FFFFF).view(np.float32)])
    x = x[np.isfinite(x)]
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    got = np.array([oracle.f32_to_bf16_rne(float(v)) for v in x], dtype=np.uint16)
    assert (got == want).all()


@pytest.mark.parametrize("layout", [W_NK, W_KN])
def test_identity_passes_bits_through(layout):
    k = 48
    x = normal_bf16(11, (9, k))
    w = bf16(np.eye(k))
    r = oracle.gemm_rows(x, w, w_layout=layout)
    assert (r["y16"] == x).all()
    assert (r["c64"] == bf16_bits_to_f32(x).astype(np.float64)).all()


@pytest.mark.parametrize("layout", [W_NK, W_KN])
def test_permutation_moves_columns(layout):
    # logical W = P with W[pi(j)][j] = 1  =>  Y[:, j] = X[:, pi(j)]; a transposed operand fails this
    k = 40
    pi = np.random.default_rng(1).permutation(k)
    wl = np.zeros((k, k), np.float32)
    wl[pi, np.arange(k)] = 1.0
    x = normal_bf16(12, (5, k))
    w = bf16(wl.T if layout == W_NK else wl)
    r = oracle.gemm_rows(x, w, w_layout=layout)
    assert (r["y16"] == x[:, pi]).all()
    assert not (r["y16"] == x[:, np.argsort(pi)]).all()


@pytest.mark.parametrize("k", [16, 64, 256, 3584])
def test_ones_give_k_exactly(k):
    x = bf16(np.ones((3, k)))
    w = bf16(np.ones((8, k)))
    r = oracle.gemm_rows(x, w)
    assert (r["c64"] == k).all() and (r["s64"] == k).all() and (r["c32"] == k).all()
    assert (bf16_bits_to_f32(r["y16"]) == k).all()       # k has <= 8 significant bits


def _logical(w16, layout):
    f = bf16_bits_to_f32(w16).astype(np.float64)
    return f.T if layout == W_NK else f


@pytest.mark.parametrize("m,n,k", [(1, 8, 8), (7, 8, 80), (8, 264, 80), (9, 24, 8), (129, 8, 16), (33, 65, 64)])
@pytest.mark.parametrize("layout", [W_NK, W_KN])
def test_against_numpy_float64_matmul(m, n, k, layout):
    # textbook reduction: c64 equals the float64 matmul of the widened inputs to ~1e-13 relative
    x = normal_bf16(20, (m, k))
    w = normal_bf16(21, (n, k) if layout == W_NK else (k, n), std=0.02)
    r = oracle.gemm_rows(x, w, w_layout=layout)
    xf, wf = bf16_bits_to_f32(x).astype(np.float64), _logical(w, layout)
    want = xf @ wf
    s_want = np.abs(xf) @ np.abs(wf)
    assert np.abs(r["c64"] - want).max() <= 1e-13 * s_want.max()
    assert np.abs(r["s64"] - s_want).max() <= 1e-13 * s_want.max()
    # "fp32 from bf16 inputs": sequential fp32 accumulation error <= K 2^-24 sum|ab|
    assert (np.abs(r["c32"].astype(np.float64) - r["c64"]) <= k * 2.0 ** -24 * r["s64"] + 1e-30).all()
    # the definition's own bf16 output meets the north_star tolerance
    y = bf16_bits_to_f32(r["y16"]).astype(np.float64)
    assert (np.abs(y - r["c64"]) <= 2.0 ** -8 * np.abs(r["c64"]) + k * 2.0 ** -24 * r["s64"]).all()


def test_exact_rational_brute_force_tiny():
    x = normal_bf16(30, (3, 8))
    w = normal_bf16(31, (4, 8), std=0.02)
    r = oracle.gemm_rows(x, w)
    xf, wf = bf16_bits_to_f32(x), bf16_bits_to_f32(w)
    for i in range(3):
        for j in range(4):
            exact = sum(Fraction(float(xf[i, kk])) * Fraction(float(wf[j, kk])) for kk in range(8))
            sabs = sum(abs(Fraction(float(xf[i, kk])) * Fraction(float(wf[j, kk]))) for kk in range(8))
            assert abs(Fraction(float(r["c64"][i, j])) - exact) <= Fraction(1, 2 ** 48) * sabs
            assert abs(Fraction(float(r["s64"][i, j])) - sabs) <= Fraction(1, 2 ** 48) * sabs


def test_row_selection_and_layouts_agree():
    m, n, k = 40, 24, 32
    x = normal_bf16(40, (m, k))
    w_kn = normal_bf16(41, (k, n), std=0.02)
    w_nk = np.ascontiguousarray(w_kn.T)
    rows = np.array([3, 0, 39, 17], np.int32)
    full = oracle.gemm_rows(x, w_nk, w_layout=W_NK)
    sel_nk = oracle.gemm_rows(x, w_nk, rows=rows, w_layout=W_NK)
    sel_kn = oracle.gemm_rows(x, w_kn, rows=rows, w_layout=W_KN)
    for key in ("c64", "s64", "c32", "y16"):
        assert (sel_nk[key] == full[key][rows]).all()
        assert (sel_kn[key] == sel_nk[key]).all()
    with pytest.raises(ValueError):
        oracle.gemm_rows(x, w_nk, rows=np.array([m], np.int32))


def test_tolerance_scale_on_configured_distributions():
    # SURVEY §8(c) pin 6: with X~N(0,1), W~N(0,0.02^2), K=3584 the tolerance 1e-3*sum|ab| is ~0.046,
    # bf16 output rounding uses < 0.4 of it, a dropped 64-wide k-block would exceed it
    k, n = 3584, 64
    x = normal_bf16(2, (2, k))
    w = normal_bf16(2, (n, k), std=0.02, stream=1)
    r = oracle.gemm_rows(x, w)
    tol = 1e-3 * r["s64"]
    assert 0.035 < tol.mean() < 0.055
    y = bf16_bits_to_f32(r["y16"]).astype(np.float64)
    assert (np.abs(y - r["c64"]) <= 0.45 * tol).all()
    dropped = oracle.gemm_rows(x[:, 64:], w[:, 64:])["c64"]
    assert (np.abs(dropped - r["c64"]) > tol).mean() > 0.5
