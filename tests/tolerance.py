"""Acceptance bound for the bf16 GEMV / GEMM outputs (test-side only).

BASELINE.json north_star states  |err| <= 1e-3 * sum_k |a_ik * w_kj|  per element, err measured against the
unrounded fp64 product.  That bound is used AS STATED on the configured workloads
(configs 3-4, zero-mean data, K = 3584: sum|ab| ~ 38 x rms(c)).

SURVEY.md §8(c) S9: the stated bound is tighter than the bf16 OUTPUT rounding when there is no cancellation
(half an ulp of bf16 is up to 2^-9 |c| = 1.95e-3 |c|, which exceeds 1e-3 * sum|ab| once |c| > 0.51 sum|ab|);
this happens on the tiny-K ragged-shape cases (K = 8: a single product can dominate).  No kernel that rounds
its output to bf16 can meet it there - the oracle's own bf16 result does not.  For those cases the bound is
widened by exactly the unavoidable part, and only on the elements where it applies (half a bf16 ulp of the exact
value > 1e-3 * sum|ab|): half a bf16 ulp plus the fp32 accumulation bound K * 2^-24 * sum|ab| (any summation order).
Everywhere else the stated bound holds as written, whatever K is.  DESIGN.md lists this reading.
"""
import numpy as np

TOL = 1e-3


def half_ulp_bf16(c64: np.ndarray) -> np.ndarray:
    """Half the bf16 spacing at |c| (8 significant bits: ulp = 2^(floor(log2|c|) - 7))."""
    a = np.maximum(np.abs(c64), 2.0 ** -126)
    return 0.5 * 2.0 ** (np.floor(np.log2(a)) - 7)


def stated_bound(s64: np.ndarray) -> np.ndarray:
    return TOL * s64


def widened_bound(c64: np.ndarray, s64: np.ndarray, k: int) -> np.ndarray:
    """Reading R9 as written: the stated bound everywhere, EXCEPT on the elements where half a bf16 ulp of the exact value
    alone exceeds it (no rounding to bf16 can meet it there); only those get half an ulp plus the fp32 accumulation term.
    A long K (K * 2^-24 > 1e-3 from K = 16778) therefore does not loosen anything by itself."""
    hu = half_ulp_bf16(c64)
    return np.where(hu > TOL * s64, hu * (1.0 + 2.0 ** -6) + k * 2.0 ** -24 * s64, TOL * s64)
