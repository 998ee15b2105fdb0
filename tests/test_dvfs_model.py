"""Row f3 through the C ABI (host functions, no GPU): tri_model_* / tri_phase_ai / tri_solve_clock / tri_fit_theta against
oracle/dvfs_model.py on seeded random models — the binary search of Eq. 6 against the oracle's exhaustive search."""
import math

import numpy as np
import pytest

import paper_2606_29629_b200 as tri
from oracle import dvfs_model as o


def random_model(rng, n_f=None):
    n_f = n_f or int(rng.integers(1, 40))
    f = np.cumsum(rng.uniform(15.0, 120.0, n_f)) + rng.uniform(200.0, 600.0)
    eta, beta = rng.uniform(0.01, 0.06), rng.uniform(0.5, 8.0)
    omega, gamma = (0.0, 0.0) if rng.random() < 0.3 else (rng.uniform(0.0, 0.05), rng.uniform(0.0, 1.0))
    p_idle = np.sort(rng.uniform(40.0, 150.0, n_f))
    # P_dyn ~ c f^a with a >= 2 keeps P_idle + P_dyn * phi non-decreasing in f on both branches (phi ~ f or 1 / f)
    p_dyn = rng.uniform(1e-5, 4e-4) * f ** rng.uniform(2.0, 3.0)
    p_tdp = rng.choice([1e9, rng.uniform(150.0, 900.0)])
    return dict(eta=eta, beta=beta, omega=omega, gamma=gamma, p_tdp=float(p_tdp), f_mhz=list(f), p_idle_w=list(p_idle), p_dyn_w=list(p_dyn))


def test_model_functions_match_oracle():
    rng = np.random.default_rng(11)
    for _ in range(200):
        kw = random_model(rng)
        m = tri.Model(**kw)
        for ai in np.exp(rng.uniform(math.log(0.1), math.log(4000.0), 8)):
            i = int(rng.integers(0, len(kw["f_mhz"])))
            f = kw["f_mhz"][i]
            assert m.theta(ai, f) == pytest.approx(o.theta(ai, f, kw["eta"], kw["beta"], kw["omega"], kw["gamma"]), rel=1e-13)
            assert m.phi(ai, f) == pytest.approx(o.phi(ai, f, kw["eta"], kw["beta"]), rel=1e-13)
            assert m.power(ai, i) == pytest.approx(o.power(ai, f, kw["p_idle_w"][i], kw["p_dyn_w"][i], kw["p_tdp"], kw["eta"], kw["beta"]), rel=1e-13)
    assert math.isnan(m.theta(-1.0, 1000.0)) and math.isnan(m.power(1.0, 10 ** 6))


def test_phase_ai_matches_oracle_and_config_values():
    rng = np.random.default_rng(12)
    for n in (1, 2, 3, 17, 1000):
        d, a = rng.uniform(0.0, 5.0, n), rng.uniform(0.1, 2000.0, n)
        assert tri.tri_phase_ai(list(d), list(a)) == pytest.approx(o.phase_ai(d, a), rel=1e-12)
    assert math.isnan(tri.tri_phase_ai([0.0, 0.0], [1.0, 2.0]))
    # the three kernels of this library: 2 s of GEMM (A.I. 1736.3) and 2 s of GEMV (7.98) -> 872.1
    assert tri.tri_phase_ai([2.0, 2.0], [1736.275, 7.979]) == pytest.approx(872.127)


def test_solver_binary_search_equals_exhaustive_search():
    rng = np.random.default_rng(13)
    checked = rejected = 0
    for _ in range(3000):
        kw = random_model(rng)
        m = tri.Model(**kw)
        ai = float(np.exp(rng.uniform(math.log(0.1), math.log(4000.0))))
        f_limit = float(rng.choice([kw["f_mhz"][-1], rng.uniform(kw["f_mhz"][0], kw["f_mhz"][-1] + 50.0)]))
        eps = float(rng.choice([0.0, 0.02, 0.05, 0.2, rng.uniform(0.0, 0.9)]))
        try:
            m.validate(ai)                              # once per (model, A.I.): the solver itself does no table scan
        except tri.TriError as e:                       # the library refuses tables on which the binary search is not exact
            assert e.status == tri.TRI_ERR_INVALID_ARG
            f, th = kw["f_mhz"], [o.theta(ai, x, kw["eta"], kw["beta"], kw["omega"], kw["gamma"]) for x in kw["f_mhz"]]
            pw = [o.power(ai, x, kw["p_idle_w"][i], kw["p_dyn_w"][i], kw["p_tdp"], kw["eta"], kw["beta"]) for i, x in enumerate(f)]
            assert any(b < a for a, b in zip(th, th[1:])) or any(b < a for a, b in zip(pw, pw[1:]))
            rejected += 1
            top = max(i for i, x in enumerate(f) if x <= f_limit)
            with pytest.raises(tri.TriError):           # the wrapper validates on first use of an A.I. and refuses too
                m.solve_clock(ai, f_limit, eps)
            idx, _ = m.solve_clock(ai, f_limit, eps, check=False)    # bare C call on unvalidated tables: still a legal index, not necessarily the optimum
            assert 0 <= idx <= top
            continue
        got = m.solve_clock(ai, f_limit, eps)
        want = o.solve_clock(ai, kw["f_mhz"], kw["p_idle_w"], kw["p_dyn_w"], kw["p_tdp"], kw["eta"], kw["beta"], kw["omega"],
                             kw["gamma"], f_limit, eps)
        assert got == want, (kw, ai, f_limit, eps)
        checked += 1
    assert checked > 2000, (checked, rejected)


def test_solver_argument_errors():
    kw = random_model(np.random.default_rng(14), n_f=8)
    m = tri.Model(**kw)
    for bad in [(-1.0, 2000.0, 0.05), (1.0, 2000.0, 1.0), (1.0, 2000.0, -0.1), (1.0, kw["f_mhz"][0] - 1.0, 0.05)]:
        with pytest.raises(tri.TriError):
            m.solve_clock(*bad)
    kw["f_mhz"][3] = kw["f_mhz"][2]                     # not strictly ascending: the validator's business
    with pytest.raises(tri.TriError):
        tri.Model(**kw).validate(1.0)


def test_solver_is_logarithmic_in_the_table_size():
    """"a low-overhead solver ... for every decode period".  tri_solve_clock evaluates the model O(log n_f)
    times and never scans the tables: its time on a 2^20-entry table is within a small factor of a 2^6-entry one, while
    the one-time tri_model_validate grows with n_f."""
    import time

    def model(n):
        f = np.linspace(200.0, 2000.0, n)
        return tri.Model(0.0379, 6.54, 0.02, 0.5, 1e9, list(f), list(60.0 + 0.05 * f), list(2e-4 * f * f))

    def per_call(fn, reps):
        fn()
        t = time.perf_counter()
        for _ in range(reps):
            fn()
        return (time.perf_counter() - t) / reps

    small, big = model(1 << 6), model(1 << 20)
    big.validate(100.0)
    assert small.solve_clock(100.0, 2000.0, 0.05)[1] and big.solve_clock(100.0, 2000.0, 0.05)[1]
    t_small = per_call(lambda: small.solve_clock(100.0, 2000.0, 0.05), 2000)
    t_big = per_call(lambda: big.solve_clock(100.0, 2000.0, 0.05), 2000)
    t_val = per_call(lambda: big.validate(100.0), 3)
    assert t_big < 8 * t_small + 20e-6, (t_small, t_big)          # 20 vs 6 bisection levels plus the ctypes call
    assert t_val > 50 * t_big, (t_val, t_big)                       # the scan is what was moved out of the solver


def test_fit_matches_oracle_on_noisy_sweep():
    rng = np.random.default_rng(15)
    ai = np.array([0.25 * 2 ** i for i in range(13)])
    f = rng.uniform(1550.0, 1965.0, ai.size)
    th = np.array([o.theta(a, x, 0.0379, 6.54, 0.02, 0.5) for a, x in zip(ai, f)]) * rng.uniform(0.97, 1.03, ai.size)
    got = tri.tri_fit_theta(list(ai), list(f), list(th), ai_mem=4.0, ai_cmp=32.0, gamma=0.5)
    want = o.fit_theta(ai, f, th, 4.0, 32.0, 0.5)
    for key in ("eta", "beta", "omega", "gamma"):
        assert got[key] == pytest.approx(want[key], rel=1e-7, abs=1e-12), key
    with pytest.raises(tri.TriError):
        tri.tri_fit_theta([1.0, 2.0], [1000.0, 1000.0], [1.0, 2.0], ai_mem=4.0, ai_cmp=32.0)


def test_power_fit_matches_oracle_and_recovers_planted_line():
    rng = np.random.default_rng(16)
    eta, beta = 0.0379, 6.87
    ai = np.array([0.25, 1, 4, 8, 16, 24, 32, 50, 64, 100, 128, 200, 256, 512, 1024], float)
    f = np.where(ai < 20, rng.uniform(1550.0, 1800.0, ai.size), 1965.0)               # auto-boost: only the compute-bound end at 1965
    p_true = np.array([min(480.0 + 770.0 * o.phi(a, x, eta, beta), 1000.0) for a, x in zip(ai, f)])
    got = tri.tri_fit_power(list(ai), list(f), list(p_true), eta, beta, 1965.0, 1.0, 990.0)
    assert got["n_used"] == int((ai >= 20).sum())
    assert got["p_idle_w"] == pytest.approx(480.0, rel=1e-9) and got["p_dyn_w"] == pytest.approx(770.0, rel=1e-9)
    noisy = p_true * rng.uniform(0.98, 1.02, ai.size)
    got = tri.tri_fit_power(list(ai), list(f), list(noisy), eta, beta, 1965.0, 1.0, 990.0)
    want = o.fit_power(ai, f, noisy, eta, beta, 1965.0, 1.0, 990.0)
    for key in ("p_idle_w", "p_dyn_w", "n_used"):
        assert got[key] == pytest.approx(want[key], rel=1e-8), key
    with pytest.raises(tri.TriError):
        tri.tri_fit_power(list(ai), list(f), list(noisy), eta, beta, 1000.0, 1.0, 990.0)      # no point at that clock


def test_pace_race_equals_the_oracle():
    """P:192 through the C ABI against oracle.pace_race (a scan over the levels; the library bisects) on random level tables and
    sustained clocks, the refusal included; plus the hand-worked B200 case (1657 MHz floor -> 1650 MHz, 0.2 s + 1.8 s)."""
    rng = np.random.default_rng(21)
    refused = 0
    for _ in range(2000):
        lv = sorted(set(rng.integers(200, 3000, size=rng.integers(1, 60)).astype(float)))
        sus = [float(x) for x in rng.uniform(150, 3100, size=rng.integers(1, 12))]
        if rng.random() < 0.3:
            sus[0] = float(rng.choice(lv))                          # a sustained clock exactly on a level
        prefill, frac = float(rng.uniform(0.0, 5.0)), float(rng.choice([0.0, 0.1, 0.25, 1.0]))
        want = o.pace_race(sus, lv, prefill, frac)
        if want is None:
            with pytest.raises(tri.TriError):
                tri.tri_policy_pace_race(sus, lv, prefill, frac)
            refused += 1
            continue
        pace, race = tri.tri_policy_pace_race(sus, lv, prefill, frac)
        assert pace["sm_mhz"] == want[0] and not pace["auto_boost"] and race["auto_boost"] and race["sm_mhz"] == 0.0
        assert pace["duration_s"] == pytest.approx(want[1], abs=1e-12) and race["duration_s"] == pytest.approx(want[2], abs=1e-12)
    assert 20 < refused < 1500
    levels = [1005.0 + 15.0 * i for i in range(65)]
    pace, race = tri.tri_policy_pace_race([1965, 1905, 1770, 1657, 1935, 1965], levels, 2.0)
    assert (pace["sm_mhz"], round(pace["duration_s"], 9), round(race["duration_s"], 9)) == (1650.0, 0.2, 1.8)
    for bad in [([], levels, 1.0, 0.1), ([1800.0], [], 1.0, 0.1), ([1800.0], [900.0, 900.0], 1.0, 0.1), ([1800.0], levels, -1.0, 0.1),
                ([1800.0], levels, 1.0, 1.5), ([float("nan")], levels, 1.0, 0.1)]:
        with pytest.raises(tri.TriError):
            tri.tri_policy_pace_race(*bad)


def test_stall_policy_equals_the_oracle():
    for args in [(True,), (False,), (True, 345.0, 1593.0), (True, 345.0, 0.0)]:
        got = tri.tri_policy_stall(*args)
        sm, mem, boost = o.stall_clocks(args[0], *[a if a > 0 else d for a, d in zip(args[1:], (210.0, 810.0))]) if len(args) > 1 else o.stall_clocks(args[0])
        assert (got["sm_mhz"], got["mem_mhz"], got["auto_boost"], got["duration_s"]) == (sm, mem, boost, 0.0)
    with pytest.raises(tri.TriError):
        tri.tri_policy_stall(True, float("inf"), 0.0)
