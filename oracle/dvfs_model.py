"""ORACLE (test infrastructure) for row f3 — the A.I.-aware frequency selection of PAPER.md section III-C.

Plain fp64 Python, one function per equation, in the paper's notation; the Eq. 6 oracle is BRUTE FORCE over the
clock list (the product uses the paper's binary search).  Imports nothing from paper_2606_29629_b200.

    theta(ai, f, eta, beta, omega, gamma)      Eq. 4; omega = 0 is Eq. 1 (line 142)
    phi(ai, f, eta, beta)                      Eq. 3 (line 154)
    power(ai, f, p_idle, p_dyn, p_tdp, ...)    Eq. 2 (line 148)
    phase_ai(d, ai)                            Eq. 5 (line 173)
    solve_clock(...)                           Eq. 6 (line 182), exhaustive
    fit_theta(...)                             the straight-line fit stated in include/triroof.h, via numpy.polyfit
    pace_race(sustained, f_list, prefill_s, frac)   section III-D (line 192): pace clock, pace seconds, race seconds
    stall_clocks(entering, ...)                     section III-B (lines 130-132): what to lock on sem_wait entry / exit

Pins: tests/test_oracle_dvfs.py (closed forms, limits, the paper's qualitative statements, hand-worked numbers).
"""
from __future__ import annotations

import math

import numpy as np


def theta(ai, f, eta, beta, omega=0.0, gamma=0.0):
    compute = eta * f * (ai / (ai + omega * f ** gamma))
    memory = beta * ai
    return min(compute, memory)


def phi(ai, f, eta, beta):
    return min(eta * f / (beta * ai), beta * ai / (eta * f))


def power(ai, f, p_idle, p_dyn, p_tdp, eta, beta):
    return min(p_idle + p_dyn * phi(ai, f, eta, beta), p_tdp)


def phase_ai(d, ai):
    num = sum(di * ai_i for di, ai_i in zip(d, ai))
    den = sum(d)
    return num / den if den > 0 else math.nan


def solve_clock(ai, f_list, p_idle, p_dyn, p_tdp, eta, beta, omega, gamma, f_limit, eps):
    """Eq. 6 by exhaustive search: (index, feasible).  Least power among the feasible clocks <= f_limit, ties to the
    highest clock; no feasible clock -> the highest clock <= f_limit, feasible False."""
    allowed = [i for i, f in enumerate(f_list) if f <= f_limit]
    need = (1.0 - eps) * theta(ai, f_list[-1], eta, beta, omega, gamma)
    feas = [i for i in allowed if theta(ai, f_list[i], eta, beta, omega, gamma) >= need]
    if not feas:
        return allowed[-1], False
    pw = {i: power(ai, f_list[i], p_idle[i], p_dyn[i], p_tdp, eta, beta) for i in feas}
    pmin = min(pw.values())
    return max(i for i in feas if pw[i] <= pmin), True


def fit_theta(ai, f, th, ai_mem, ai_cmp, gamma):
    ai, f, th = (np.asarray(v, dtype=np.float64) for v in (ai, f, th))
    mem, cmp_ = ai <= ai_mem, ai >= ai_cmp
    beta = float(np.mean(th[mem] / ai[mem]))
    slope, icpt = np.polyfit(f[cmp_] ** gamma / ai[cmp_], f[cmp_] / th[cmp_], 1)
    if slope < 0:
        slope, icpt = 0.0, float(np.mean(f[cmp_] / th[cmp_]))
    return {"eta": 1.0 / icpt, "beta": beta, "omega": slope / icpt, "gamma": gamma}


def fit_power(ai, f, p, eta, beta, f_sel, f_tol, p_cap):
    """Eq. 2 at one clock: numpy.polyfit of p against phi over the points at that clock and below the cap."""
    ai, f, p = (np.asarray(v, dtype=np.float64) for v in (ai, f, p))
    sel = (np.abs(f - f_sel) <= f_tol) & (p < p_cap)
    x = np.array([phi(a, ff, eta, beta) for a, ff in zip(ai[sel], f[sel])])
    slope, icpt = np.polyfit(x, p[sel], 1)
    return {"p_idle_w": float(icpt), "p_dyn_w": float(slope), "n_used": int(sel.sum())}


def pace_race(sustained_mhz, f_list, prefill_s, pace_fraction=0.10):
    """PAPER.md line 192, step by step.  "For the pace frequency, we choose the highest frequency that can run sustainably
    across all A.I.": a clock is sustainable at an A.I. point if it does not exceed the clock that point holds in steady
    state, so among the supported levels f_list the pace clock is the highest one that is <= EVERY entry of sustained_mhz
    (written as that scan, not as a min).  "a pacing duration of 10% of prefill, with 90% racing": pace for
    pace_fraction * prefill_s, then race = auto-boost for the rest.  -> (pace_mhz, pace_s, race_s); None if no level is
    sustainable everywhere."""
    ok = [f for f in f_list if all(f <= s for s in sustained_mhz)]
    if not ok:
        return None
    return max(ok), pace_fraction * prefill_s, prefill_s - pace_fraction * prefill_s


def stall_clocks(entering, idle_sm_mhz=210.0, idle_mem_mhz=810.0):
    """on entering the sem_wait() of a dependency stall lock SM and memory to the clocks of the
    lowest P8 state (210 / 810 MHz in the paper); on leaving it restore auto-boost.  -> (sm_mhz, mem_mhz, auto_boost)."""
    return (idle_sm_mhz, idle_mem_mhz, False) if entering else (0.0, 0.0, True)
