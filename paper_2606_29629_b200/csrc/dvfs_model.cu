// f3. A.I.-aware frequency selection (section III-C; ABI in include/triroof.h): the
// throughput / power models (Eq. 1-4), the phase A.I. (Eq. 5) and the Eq. 6 solver.  Host code: the controller runs
// once per decode period on the CPU next to the NVML calls, there is nothing data-parallel in it.
#include "tri_internal.h"

#include <cmath>

namespace tri {

static bool pos(double v) { return std::isfinite(v) && v > 0.0; }

static double theta(const tri_model *m, double ai, double f)
{
    const double sat = m->omega > 0.0 ? ai / (ai + m->omega * std::pow(f, m->gamma)) : 1.0;
    const double cmp = m->eta * f * sat, mem = m->beta * ai;
    return cmp < mem ? cmp : mem;
}

static double phi(const tri_model *m, double ai, double f)
{
    const double r = m->eta * f / (m->beta * ai);
    return r < 1.0 ? r : 1.0 / r;
}

static double power(const tri_model *m, double ai, int i)
{
    const double p = m->p_idle_w[i] + m->p_dyn_w[i] * phi(m, ai, m->f_mhz[i]);
    return p < m->p_tdp ? p : m->p_tdp;
}

static int check_model(const tri_model *m, bool tables)
{
    if (!m) return fail(TRI_ERR_INVALID_ARG, "model is NULL");
    if (!pos(m->eta) || !pos(m->beta) || !(m->omega >= 0.0) || !std::isfinite(m->omega) || !std::isfinite(m->gamma))
        return fail(TRI_ERR_INVALID_ARG, "eta, beta must be positive, omega >= 0, gamma finite");
    if (!tables) return TRI_OK;
    if (m->n_f < 1 || !m->f_mhz || !m->p_idle_w || !m->p_dyn_w || !pos(m->p_tdp))
        return fail(TRI_ERR_INVALID_ARG, "clock / power tables missing or p_tdp not positive");
    for (int i = 0; i < m->n_f; ++i) {
        if (!pos(m->f_mhz[i]) || !(m->p_idle_w[i] >= 0.0) || !(m->p_dyn_w[i] >= 0.0) || (i && m->f_mhz[i] <= m->f_mhz[i - 1]))
            return fail(TRI_ERR_INVALID_ARG, "clock table must be positive and strictly ascending, powers non-negative");
    }
    return TRI_OK;
}

}  // namespace tri

extern "C" {

double tri_model_theta(const tri_model *m, double ai, double f_mhz)
{
    if (tri::check_model(m, false) != TRI_OK || !tri::pos(ai) || !tri::pos(f_mhz)) return NAN;
    return tri::theta(m, ai, f_mhz);
}

double tri_model_phi(const tri_model *m, double ai, double f_mhz)
{
    if (tri::check_model(m, false) != TRI_OK || !tri::pos(ai) || !tri::pos(f_mhz)) return NAN;
    return tri::phi(m, ai, f_mhz);
}

double tri_model_power(const tri_model *m, double ai, int32_t i)
{
    if (tri::check_model(m, true) != TRI_OK || !tri::pos(ai) || i < 0 || i >= m->n_f) return NAN;
    return tri::power(m, ai, i);
}

double tri_phase_ai(const double *d, const double *ai, size_t n)
{
    if (!d || !ai || n == 0) return NAN;
    double num = 0.0, den = 0.0;
    for (size_t i = 0; i < n; ++i) {
        if (!(d[i] >= 0.0) || !std::isfinite(d[i]) || !std::isfinite(ai[i])) return NAN;
        num += d[i] * ai[i];
        den += d[i];
    }
    return den > 0.0 ? num / den : NAN;
}

int tri_model_validate(const tri_model *m, double ai)
{
    int st = tri::check_model(m, true);
    if (st != TRI_OK) return st;
    if (!tri::pos(ai)) return tri::fail(TRI_ERR_INVALID_ARG, "ai must be positive");
    // the premise of the binary search: throughput and modelled power do not decrease with the clock
    for (int i = 1; i < m->n_f; ++i) {
        if (tri::theta(m, ai, m->f_mhz[i]) < tri::theta(m, ai, m->f_mhz[i - 1]) * (1.0 - 1e-12) ||
            tri::power(m, ai, i) < tri::power(m, ai, i - 1) * (1.0 - 1e-12))
            return tri::fail(TRI_ERR_INVALID_ARG, "model is not monotone in f at A.I. %g (clock %g MHz): binary search does not apply", ai,
                             m->f_mhz[i]);
    }
    return TRI_OK;
}

int tri_solve_clock(const tri_model *m, double ai, double f_limit_mhz, double eps, int32_t *index, int32_t *feasible)
{
    // O(1) checks only: the tables are validated once by tri_model_validate, not per decode period
    int st = tri::check_model(m, false);
    if (st != TRI_OK) return st;
    if (m->n_f < 1 || !m->f_mhz || !m->p_idle_w || !m->p_dyn_w || !tri::pos(m->p_tdp))
        return tri::fail(TRI_ERR_INVALID_ARG, "clock / power tables missing or p_tdp not positive");
    if (!index || !feasible) return tri::fail(TRI_ERR_INVALID_ARG, "index / feasible is NULL");
    if (!tri::pos(ai) || !tri::pos(f_limit_mhz) || !(eps >= 0.0 && eps < 1.0))
        return tri::fail(TRI_ERR_INVALID_ARG, "ai, f_limit must be positive, eps in [0, 1)");
    // hi = the highest supported clock <= f_limit (binary search on the ascending table)
    int lo = 0, hi = m->n_f - 1;
    if (m->f_mhz[0] > f_limit_mhz) return tri::fail(TRI_ERR_INVALID_ARG, "no supported clock <= f_limit = %g MHz", f_limit_mhz);
    while (lo < hi) {
        const int mid = (lo + hi + 1) / 2;
        if (m->f_mhz[mid] <= f_limit_mhz) lo = mid; else hi = mid - 1;
    }
    const int top = lo;
    const double need = (1.0 - eps) * tri::theta(m, ai, m->f_mhz[m->n_f - 1]);
    if (tri::theta(m, ai, m->f_mhz[top]) < need) {           // even the highest allowed clock is too slow
        *index = top;
        *feasible = 0;
        return TRI_OK;
    }
    // lowest feasible clock: theta is non-decreasing in f, so feasibility is a step function of the index
    int a = 0, b = top;
    while (a < b) {
        const int mid = (a + b) / 2;
        if (tri::theta(m, ai, m->f_mhz[mid]) >= need) b = mid; else a = mid + 1;
    }
    // power is non-decreasing in f: the lowest feasible clock has the least power; among the clocks that tie with it
    // (flat stretches, e.g. at the cap) take the highest — again a step function of the index
    const double pmin = tri::power(m, ai, a);
    int c = a, d = top;
    while (c < d) {
        const int mid = (c + d + 1) / 2;
        if (tri::power(m, ai, mid) <= pmin) c = mid; else d = mid - 1;
    }
    *index = c;
    *feasible = 1;
    return TRI_OK;
}

int tri_fit_theta(const double *ai, const double *f_mhz, const double *th, size_t n, double ai_mem, double ai_cmp, double gamma,
                  tri_model *m)
{
    if (!ai || !f_mhz || !th || !m || !std::isfinite(gamma)) return tri::fail(TRI_ERR_INVALID_ARG, "NULL argument or gamma not finite");
    double bsum = 0.0;
    size_t nb = 0, nc = 0;
    double sz = 0.0, sy = 0.0, szz = 0.0, szy = 0.0;
    for (size_t i = 0; i < n; ++i) {
        if (!tri::pos(ai[i]) || !tri::pos(f_mhz[i]) || !tri::pos(th[i])) return tri::fail(TRI_ERR_INVALID_ARG, "point %zu is not positive and finite", i);
        if (ai[i] <= ai_mem) { bsum += th[i] / ai[i]; ++nb; }
        if (ai[i] >= ai_cmp) {
            const double z = std::pow(f_mhz[i], gamma) / ai[i], y = f_mhz[i] / th[i];
            sz += z; sy += y; szz += z * z; szy += z * y; ++nc;
        }
    }
    if (nb < 1 || nc < 2) return tri::fail(TRI_ERR_INVALID_ARG, "need >= 1 memory-bound and >= 2 compute-bound points (have %zu, %zu)", nb, nc);
    const double det = (double)nc * szz - sz * sz;
    if (!(det > 1e-300 * (1.0 + szz * (double)nc))) return tri::fail(TRI_ERR_INVALID_ARG, "compute-bound points share one abscissa: fit is degenerate");
    double slope = ((double)nc * szy - sz * sy) / det, icpt = (sy - slope * sz) / (double)nc;
    if (slope < 0.0) { slope = 0.0; icpt = sy / (double)nc; }          // omega clamped at 0: the line is the mean
    if (!(icpt > 0.0)) return tri::fail(TRI_ERR_INVALID_ARG, "fit is degenerate (1 / eta = %g)", icpt);
    m->eta = 1.0 / icpt;
    m->omega = slope / icpt;
    m->gamma = gamma;
    m->beta = bsum / (double)nb;
    return TRI_OK;
}

int tri_fit_power(const double *ai, const double *f_mhz, const double *p_w, size_t n, const tri_model *m, double f_sel_mhz,
                  double f_tol_mhz, double p_cap_w, double *p_idle_w, double *p_dyn_w, size_t *n_used)
{
    int st = tri::check_model(m, false);
    if (st != TRI_OK) return st;
    if (!ai || !f_mhz || !p_w || !p_idle_w || !p_dyn_w || !tri::pos(f_sel_mhz) || !(f_tol_mhz >= 0.0) || !tri::pos(p_cap_w))
        return tri::fail(TRI_ERR_INVALID_ARG, "NULL argument, or f_sel / p_cap not positive, or f_tol negative");
    size_t k = 0;
    double sx = 0.0, sy = 0.0, sxx = 0.0, sxy = 0.0;
    for (size_t i = 0; i < n; ++i) {
        if (!tri::pos(ai[i]) || !tri::pos(f_mhz[i]) || !std::isfinite(p_w[i])) return tri::fail(TRI_ERR_INVALID_ARG, "point %zu is not finite / positive", i);
        if (std::fabs(f_mhz[i] - f_sel_mhz) > f_tol_mhz || !(p_w[i] < p_cap_w)) continue;
        const double x = tri::phi(m, ai[i], f_mhz[i]);
        sx += x; sy += p_w[i]; sxx += x * x; sxy += x * p_w[i]; ++k;
    }
    if (n_used) *n_used = k;
    const double det = (double)k * sxx - sx * sx;
    if (k < 2 || !(det > 1e-12 * (1.0 + (double)k * sxx))) return tri::fail(TRI_ERR_INVALID_ARG, "%zu usable points: the line is not determined", k);
    *p_dyn_w = ((double)k * sxy - sx * sy) / det;
    *p_idle_w = (sy - *p_dyn_w * sx) / (double)k;
    return TRI_OK;
}

int tri_policy_pace_race(const double *sustained_mhz, size_t n, const double *f_mhz, int32_t n_f, double prefill_s,
                         double pace_fraction, tri_clock_step out[2])
{
    if (!sustained_mhz || !f_mhz || !out || n == 0 || n_f < 1) return tri::fail(TRI_ERR_INVALID_ARG, "NULL argument, n == 0 or n_f < 1");
    if (!(prefill_s >= 0.0) || !std::isfinite(prefill_s) || !(pace_fraction >= 0.0 && pace_fraction <= 1.0))
        return tri::fail(TRI_ERR_INVALID_ARG, "prefill_s must be >= 0 and pace_fraction in [0, 1]");
    // the clock every A.I. point can hold: the lowest of the sustained clocks
    double floor_mhz = INFINITY;
    for (size_t i = 0; i < n; ++i) {
        if (!tri::pos(sustained_mhz[i])) return tri::fail(TRI_ERR_INVALID_ARG, "sustained_mhz[%zu] is not positive and finite", i);
        if (sustained_mhz[i] < floor_mhz) floor_mhz = sustained_mhz[i];
    }
    for (int32_t i = 0; i < n_f; ++i)
        if (!tri::pos(f_mhz[i]) || (i > 0 && !(f_mhz[i] > f_mhz[i - 1])))
            return tri::fail(TRI_ERR_INVALID_ARG, "f_mhz must be positive and strictly ascending (index %d)", (int)i);
    if (f_mhz[0] > floor_mhz)
        return tri::fail(TRI_ERR_INVALID_ARG, "no supported clock is sustainable at every A.I. (lowest level %g MHz > %g MHz)", f_mhz[0], floor_mhz);
    // highest level <= floor_mhz: bisection over the ascending table (f_mhz[lo] <= floor_mhz < f_mhz[hi])
    int32_t lo = 0, hi = n_f;
    while (hi - lo > 1) {
        const int32_t mid = lo + (hi - lo) / 2;
        if (f_mhz[mid] <= floor_mhz) lo = mid;
        else hi = mid;
    }
    const double pace_s = pace_fraction * prefill_s;
    out[0] = tri_clock_step{f_mhz[lo], 0.0, pace_s, 0, 0};
    out[1] = tri_clock_step{0.0, 0.0, prefill_s - pace_s, 1, 0};
    return TRI_OK;
}

int tri_policy_stall(int entering, double idle_sm_mhz, double idle_mem_mhz, tri_clock_step *out)
{
    if (!out) return tri::fail(TRI_ERR_INVALID_ARG, "out is NULL");
    if (!std::isfinite(idle_sm_mhz) || !std::isfinite(idle_mem_mhz)) return tri::fail(TRI_ERR_INVALID_ARG, "idle clocks must be finite");
    if (entering) *out = tri_clock_step{idle_sm_mhz > 0.0 ? idle_sm_mhz : 210.0, idle_mem_mhz > 0.0 ? idle_mem_mhz : 810.0, 0.0, 0, 0};
    else *out = tri_clock_step{0.0, 0.0, 0.0, 1, 0};
    return TRI_OK;
}

}  // extern "C"
