"""Pins of oracle/dvfs_model.py (row f3) against what PAPER.md section III-C and the mathematics fix — not against
itself: hand-worked numbers, closed forms, limits and the paper's qualitative statements about Fig. 3."""
import math

import numpy as np
import pytest

from oracle import dvfs_model as o

ETA, BETA = 0.04, 6.5            # TFLOP/s per MHz, TFLOP/s per (FLOP/B): ridge at ai = eta f / beta


def test_eq1_hand_worked_values():
    # f = 1000 MHz: compute roof 40, ridge at ai = 40 / 6.5.  ai = 2 -> memory bound 13; ai = 10 -> compute bound 40
    assert o.theta(2.0, 1000.0, ETA, BETA) == pytest.approx(13.0, rel=1e-15)
    assert o.theta(10.0, 1000.0, ETA, BETA) == pytest.approx(40.0, rel=1e-15)
    assert o.theta(40.0 / 6.5, 1000.0, ETA, BETA) == pytest.approx(40.0, rel=1e-12)      # the ridge: both branches meet


def test_eq4_saturation_term():
    # omega f^gamma = 0.5 * 1000^0.5 = 15.811...; ai = 50: eta f ai / (ai + 15.81) = 40 * 50 / 65.811 = 30.3899...
    v = o.theta(50.0, 1000.0, ETA, BETA, omega=0.5, gamma=0.5)
    assert v == pytest.approx(40.0 * 50.0 / (50.0 + 0.5 * math.sqrt(1000.0)), rel=1e-15)
    assert v == pytest.approx(30.38988, rel=1e-6)                                          # 2000 / 65.8114
    # "slowly converges to 1 as A.I. increases to infinity, thus reaching the real roofline"
    assert o.theta(1e12, 1000.0, ETA, 1e9, omega=0.5, gamma=0.5) == pytest.approx(40.0, rel=1e-9)
    # omega = 0 reduces Eq. 4 to Eq. 1 exactly
    for ai in (0.25, 3.0, 6.15, 7.0, 1024.0):
        assert o.theta(ai, 1337.0, ETA, BETA, 0.0, 3.0) == o.theta(ai, 1337.0, ETA, BETA)
    # throughput still rises with A.I. in the compute-bound regime and never exceeds either roof
    a = [o.theta(ai, 1000.0, ETA, BETA, 0.5, 0.5) for ai in (20, 40, 80, 160, 320)]
    assert all(x < y for x, y in zip(a, a[1:])) and max(a) < 40.0


def test_eq3_utilisation_peaks_at_the_ridge():
    f = 1500.0
    ridge = ETA * f / BETA
    assert o.phi(ridge, f, ETA, BETA) == pytest.approx(1.0, rel=1e-12)
    assert o.phi(ridge / 4, f, ETA, BETA) == pytest.approx(0.25, rel=1e-12)               # memory bound: beta ai / (eta f)
    assert o.phi(ridge * 4, f, ETA, BETA) == pytest.approx(0.25, rel=1e-12)               # compute bound: eta f / (beta ai)
    xs = np.geomspace(0.1, 1000, 200)
    assert all(0 < o.phi(x, f, ETA, BETA) <= 1 for x in xs)
    # symmetric in log(ai) about the ridge
    assert o.phi(ridge * 3.7, f, ETA, BETA) == pytest.approx(o.phi(ridge / 3.7, f, ETA, BETA), rel=1e-12)


def test_eq2_power_rises_to_the_ridge_then_falls_and_is_capped():
    f, p_idle, p_dyn = 1500.0, 200.0, 600.0
    ridge = ETA * f / BETA
    ais = [ridge / 8, ridge / 2, ridge, ridge * 2, ridge * 8]
    p = [o.power(a, f, p_idle, p_dyn, 1e9, ETA, BETA) for a in ais]
    assert p[0] < p[1] < p[2] > p[3] > p[4]                                               # peak where both are stressed
    assert p[2] == pytest.approx(800.0) and p[0] == pytest.approx(200.0 + 600.0 / 8)
    assert o.power(ridge, f, p_idle, p_dyn, 700.0, ETA, BETA) == 700.0                    # min(., P_TDP)


def test_eq5_duration_weighted_mean():
    assert o.phase_ai([1.0, 3.0], [8.0, 1736.0]) == pytest.approx((8.0 + 3 * 1736.0) / 4)
    assert o.phase_ai([2.0, 2.0, 2.0], [1.0, 2.0, 6.0]) == pytest.approx(3.0)            # equal durations: plain mean
    assert o.phase_ai([5.0], [42.0]) == 42.0
    assert o.phase_ai([0.0, 7.0], [1e9, 3.0]) == 3.0                                      # zero-duration kernels do not count
    assert math.isnan(o.phase_ai([0.0], [1.0]))


def _tables(n=16):
    f = [450.0 + 100.0 * i for i in range(n)]
    p_idle = [60.0 + 0.05 * x for x in f]
    p_dyn = [2e-4 * x * x for x in f]                                                     # ~ f^2: power rises with the clock
    return f, p_idle, p_dyn


def test_eq6_worked_cases():
    f, pi, pd = _tables()
    # memory bound (ai far below every ridge): theta = beta ai at every clock -> the LOWEST clock is feasible and cheapest
    # (Observation 2b: "that same throughput is achievable with the lowest clock")
    assert o.solve_clock(0.25, f, pi, pd, 1e9, ETA, BETA, 0, 0, f[-1], 0.05) == (0, True)
    # compute bound: theta = eta f, need (1 - eps) eta f_max -> lowest clock >= 0.95 * 1950 = 1852.5 -> 1950 only
    assert o.solve_clock(1e4, f, pi, pd, 1e9, ETA, BETA, 0, 0, f[-1], 0.05) == (len(f) - 1, True)
    assert o.solve_clock(1e4, f, pi, pd, 1e9, ETA, BETA, 0, 0, f[-1], 0.11) == (13, True)               # 0.89 * 1950 = 1735.5 -> 1750 = f[13]
    # f_limit below the feasible set: best effort, flagged
    assert o.solve_clock(1e4, f, pi, pd, 1e9, ETA, BETA, 0, 0, 1000.0, 0.05) == (5, False)              # 950 is the highest <= 1000
    # a power cap flattens the top: all capped clocks tie, the HIGHEST of the tying feasible clocks wins
    i, ok = o.solve_clock(1e4, f, pi, pd, 100.0, ETA, BETA, 0, 0, f[-1], 0.5)
    assert ok and i == len(f) - 1


def test_fit_recovers_planted_parameters():
    rng = np.random.default_rng(7)
    eta, beta, omega, gamma = 0.0379, 6.54, 0.02, 0.5        # omega f^gamma ~ 0.85 FLOP/B: the low-A.I. points stay memory bound
    ai = np.array([0.25, 0.5, 1, 2, 64, 128, 256, 512, 1024], float)
    f = rng.uniform(1500, 1965, ai.size)
    th = np.array([o.theta(a, x, eta, beta, omega, gamma) for a, x in zip(ai, f)])
    got = o.fit_theta(ai, f, th, ai_mem=2, ai_cmp=64, gamma=gamma)
    assert got["eta"] == pytest.approx(eta, rel=1e-6) and got["beta"] == pytest.approx(beta, rel=1e-12)
    assert got["omega"] == pytest.approx(omega, rel=1e-5)


def test_fit_power_recovers_a_planted_line():
    """Pin of oracle.fit_power on its own (not against the product): Eq. 2 at one clock is P = P_idle + P_dyn * phi, so
    points planted on that line at the selected clock come back as (P_idle, P_dyn) exactly; points at other clocks and
    points at / above the cap must not enter the fit (above the cap the measured power says nothing about
    P_dyn)."""
    eta, beta = 0.0379, 6.54
    p_idle, p_dyn, cap = 480.0, 770.0, 1000.0
    ai = np.array([0.25, 1, 4, 8, 16, 24, 32, 50, 64, 100, 128, 200, 256, 512, 1024], float)
    f = np.where(ai < 8, 1700.0, 1965.0)                                    # two clock columns; A.I. 8 and 16 at 1965 MHz sit at the cap
    p = np.array([min(p_idle + p_dyn * o.phi(a, x, eta, beta), cap) for a, x in zip(ai, f)])
    got = o.fit_power(ai, f, p, eta, beta, 1965.0, 1.0, cap - 10.0)
    below = int(((f == 1965.0) & (p < cap - 10.0)).sum())
    assert got["n_used"] == below and 2 <= below < int((f == 1965.0).sum())         # the capped points were dropped
    assert got["p_idle_w"] == pytest.approx(p_idle, rel=1e-9) and got["p_dyn_w"] == pytest.approx(p_dyn, rel=1e-9)
    # the other clock column has its own line: a different planted pair is recovered from the same call on that column
    p2 = np.where(f == 1700.0, 300.0 + 500.0 * np.array([o.phi(a, x, eta, beta) for a, x in zip(ai, f)]), p)
    got2 = o.fit_power(ai, f, p2, eta, beta, 1700.0, 1.0, cap)
    assert got2["n_used"] == int((f == 1700.0).sum())
    assert got2["p_idle_w"] == pytest.approx(300.0, rel=1e-9) and got2["p_dyn_w"] == pytest.approx(500.0, rel=1e-9)
    # a dropped intercept or swapped regressors would fail: slope and intercept are distinct and both non-zero
    assert abs(got["p_idle_w"] - got["p_dyn_w"]) > 100.0
    # two points fix the line: hand-worked, phi = 0.5 -> 865 W, phi = 0.25 -> 672.5 W at P_idle 480, P_dyn 770
    a1, a2 = eta * 1965.0 / beta / 0.5, eta * 1965.0 / beta / 0.25          # compute-bound side: phi = eta f / (beta ai)
    g = o.fit_power([a1, a2], [1965.0, 1965.0], [865.0, 672.5], eta, beta, 1965.0, 0.0, cap)
    assert g["p_idle_w"] == pytest.approx(480.0, rel=1e-9) and g["p_dyn_w"] == pytest.approx(770.0, rel=1e-9)


def test_pace_race_hand_worked():
    """P:192.  Levels every 15 MHz from 1005; sustained clocks per A.I. as this repo measured them on B200 (profiles/
    r2b_thermal240.md style): the lowest is 1657 -> the highest level not above it is 1005 + 15 * 43 = 1650.  10 % of a
    2 s prefill = 0.2 s pacing, 1.8 s racing.  And the paper's own figure: if every A.I. sustains >= 1800 and one exactly
    1800, the pace clock is 1800 ("we select a pace frequency of ~1800 MHz")."""
    levels = [1005.0 + 15.0 * i for i in range(65)]                     # 1005 .. 1965
    assert o.pace_race([1965, 1905, 1770, 1657, 1935, 1965], levels, 2.0) == (1650.0, pytest.approx(0.2), pytest.approx(1.8))
    lv = [450.0 + 150.0 * i for i in range(18)]                         # 450 .. 3000, the paper's grid spacing
    assert o.pace_race([2550, 1800, 2100, 1950], lv, 1.0, 0.10)[0] == 1800.0
    assert o.pace_race([2550, 1799, 2100], lv, 1.0)[0] == 1650.0        # just below a level: the next one down
    assert o.pace_race([400.0, 2000.0], lv, 1.0) is None                # nothing is sustainable everywhere
    p, a, b = o.pace_race([1800.0], lv, 0.37, 0.25)
    assert a + b == pytest.approx(0.37) and a == pytest.approx(0.0925)


def test_pace_race_is_the_highest_common_level():
    """Property on random inputs: the pace clock is a level, no sustained clock is below it, and the next level up (if
    any) exceeds at least one sustained clock."""
    rng = np.random.default_rng(7)
    for _ in range(500):
        lv = sorted(set(rng.integers(200, 3000, size=rng.integers(1, 40)).astype(float)))
        sus = list(rng.uniform(150, 3100, size=rng.integers(1, 12)))
        r = o.pace_race(sus, lv, 1.0)
        if r is None:
            assert min(sus) < lv[0]
            continue
        i = lv.index(r[0])
        assert r[0] <= min(sus) and (i == len(lv) - 1 or lv[i + 1] > min(sus))


def test_stall_clocks_are_the_papers():
    assert o.stall_clocks(True) == (210.0, 810.0, False)                # P:132 "210 and 810 MHz ... lowest-level P8"
    assert o.stall_clocks(False) == (0.0, 0.0, True)                    # "we restore auto-boost on exiting it"
    assert o.stall_clocks(True, 345.0, 1593.0) == (345.0, 1593.0, False)
