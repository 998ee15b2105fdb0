"""Pins for Oracle A (oracle/fma_chain.c) — SURVEY.md §8(c) Oracle A, BASELINE.json north_star.

None of these re-types the oracle's loop with the same library call: the step is checked against
exact rational arithmetic + one rounding, the chain against its closed form and invariants."""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from synth_inputs import uniform_pm1
from tests.exact import bits_f32, f32_bits, frac_of_f32, fused_step_bits

A = float(oracle.A_DEFAULT)
B = float(oracle.B_DEFAULT)
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def chain_exact_bits(y0: float, k: int, a=A, b=B) -> int:
    y = y0
    for _ in range(k):
        y = bits_f32(fused_step_bits(a, y, b))
    return f32_bits(y)


def test_constants_are_exact():
    assert f32_bits(A) == 0x3F7FC000 and Fraction(A) == 1 - Fraction(1, 1024)
    assert f32_bits(B) == 0x3A800000 and Fraction(B) == Fraction(1, 1024)


def test_fixed_point_for_every_k():
    # b/(1-a) = 1 and fmaf(a, 1, b) = 1 exactly  (SURVEY §8(c) pin 1)
    for k in (0, 1, 2, 3, 4, 16, 64, 1000, 4096):
        out = oracle.fma_chain(np.ones(5, np.float32), k)
        assert (out.view(np.uint32) == 0x3F800000).all()


def test_k0_is_identity():
    x = uniform_pm1(0, 1000)
    assert oracle.count_bit_mismatches(oracle.fma_chain(x, 0), x)[0] == 0


def test_exact_k1_cases():
    # exactly representable results (SURVEY §8(c) pin 5); values follow from a*y+b in rationals
    cases = {-1.0: 0xBF7F8000, 0.0: 0x3A800000, 0.5: 0x3F002000, -0.5: 0xBEFF4000, 0.25: 0x3E806000}
    for y0, bits in cases.items():
        assert Fraction(bits_f32(bits)) == Fraction(A) * Fraction(y0) + Fraction(B)
        got = oracle.fma_chain(np.array([y0], np.float32), 1).view(np.uint32)[0]
        assert got == bits


def test_worked_values_fixture():
    # tests/golden/fma_chain_worked.txt: independent glibc-fmaf values tabulated in SURVEY.md §8(c).6
    rows = [l.split() for l in open(os.path.join(GOLDEN, "fma_chain_worked.txt")) if l.strip() and l[0] != "#"]
    ks = [int(t) for t in rows[0][1:]]
    for r in rows[1:]:
        y0 = float(r[0])
        for k, want in zip(ks, r[1:]):
            got = oracle.fma_chain(np.array([y0], np.float32), k).view(np.uint32)[0]
            assert got == int(want, 16), (y0, k, hex(got), want)
            if k <= 64:   # and the fixture itself agrees with exact arithmetic
                assert chain_exact_bits(y0, k) == int(want, 16)


def test_matches_exact_rational_fused_step_on_random_inputs():
    # a dropped b, a swapped operand, an unfused (two-rounding) step or a wrong k all fail here
    x = uniform_pm1(7, 257)
    for k in (1, 2, 3, 5, 16, 33):
        got = oracle.fma_chain(x, k).view(np.uint32)
        want = np.array([chain_exact_bits(float(v), k) for v in x], dtype=np.uint32)
        assert (got == want).all(), k


def test_fused_differs_from_two_roundings_somewhere():
    # proves the pin above can tell fmaf from (float)(a*y) + b: the two differ on this sample
    x = uniform_pm1(7, 4096)
    fused = oracle.fma_chain(x, 1)
    unfused = (np.float32(A) * x).astype(np.float32) + np.float32(B)
    assert (fused.view(np.uint32) != unfused.astype(np.float32).view(np.uint32)).any()


def test_general_a_b_against_exact():
    x = uniform_pm1(9, 64)
    a, b = 0.75, -0.125
    got = oracle.fma_chain(x, 7, a, b).view(np.uint32)
    want = np.array([chain_exact_bits(float(v), 7, a, b) for v in x], dtype=np.uint32)
    assert (got == want).all()
    # asymmetric in (a, b): swapping them must change the result
    assert (oracle.fma_chain(x, 7, b, a).view(np.uint32) != got).any()


@pytest.mark.parametrize("k", [1, 4, 16, 64, 256, 1024, 4096])
def test_closed_form_within_derived_bound(k):
    # exact-arithmetic y_k = a^k y0 + b (1 - a^k)/(1 - a) = 1 + a^k (y0 - 1); the fp32 chain stays
    # within 2^-25 (1 - a^k)/(1 - a) = 2^-15 (1 - a^k) of it (SURVEY §8(c) pin 2)
    x = uniform_pm1(1, 20000)
    got = oracle.fma_chain(x, k).astype(np.float64)
    ak = float(Fraction(A) ** k)
    want = 1.0 + ak * (x.astype(np.float64) - 1.0)
    bound = 2.0 ** -15 * (1.0 - ak) + 1e-12
    assert np.abs(got - want).max() <= bound
    # and it is a non-trivial statement: the bound is far below the step a chain of k+1 would make
    assert bound < np.abs((1.0 + ak * A * (x.astype(np.float64) - 1.0)) - want).max() or k >= 1024


def test_closed_form_exact_rational_small():
    # rational closed form vs rational recurrence, then oracle within bound of it, for one value
    y0 = Fraction(-3, 8)
    a, b = Fraction(A), Fraction(B)
    y = y0
    for _ in range(50):
        y = a * y + b
    assert y == a ** 50 * y0 + b * (1 - a ** 50) / (1 - a) == 1 + a ** 50 * (y0 - 1)
    got = Fraction(float(oracle.fma_chain(np.array([float(y0)], np.float32), 50)[0]))
    assert abs(got - y) <= Fraction(1, 2 ** 15) * (1 - a ** 50)


def test_composition_bit_for_bit():
    x = uniform_pm1(3, 5000)
    for k1, k2 in ((1, 1), (3, 13), (64, 64), (100, 924)):
        whole = oracle.fma_chain(x, k1 + k2)
        parts = oracle.fma_chain(oracle.fma_chain(x, k1), k2)
        assert oracle.count_bit_mismatches(whole, parts)[0] == 0


def test_monotone_range_no_special_values():
    # y_{s+1} >= y_s, results stay in [-1, 1], never subnormal / zero / NaN (SURVEY §8(c) pin 4)
    x = uniform_pm1(5, 20000)
    prev = x
    for k in (1, 2, 4, 8, 16, 1024):
        cur = oracle.fma_chain(x, k)
        assert (cur >= prev).all() and (cur <= 1.0).all() and (cur >= -1.0).all()
        assert np.isfinite(cur).all()
        assert ((np.abs(cur) >= 2.0 ** -126)).all()
        prev = cur


def test_smallest_first_step_magnitude():
    # the input grid point m = -8200 gives |y1| = 2^-30 exactly (SURVEY §8(c) pin 4)
    y0 = np.array([-8200 * 2.0 ** -23], np.float32)
    assert Fraction(float(oracle.fma_chain(y0, 1)[0])) == Fraction(1, 2 ** 30)


def test_count_bit_mismatches_is_bitwise():
    a = np.array([0.0, 1.0, 2.0], np.float32)
    b = np.array([-0.0, 1.0, 2.5], np.float32)
    assert oracle.count_bit_mismatches(a, b) == (2, 0)      # +0 vs -0 differ in bits
    assert oracle.count_bit_mismatches(a, a) == (0, -1)
