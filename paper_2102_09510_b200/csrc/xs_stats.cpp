// xs_stats.cpp -- a-12: time-to-solution accounting "as the paper defines" (host, tiny).
//
// percentiles TTS_p, P[TTS < TTS_p] = p/100.  L113 Eq.(2): P[TTS > t] =
// exp(-t/tau), tau = mean TTS.  L117/L123: TTS_p = -ln(1 - p/100) tau.  L129-L147: runs with a
// timeout t_max; posterior P(tau | n) = T_tot^n / (n-1)! * exp(-T_tot/tau) / tau^(n+1), i.e.
// an inverse-gamma law of shape n and scale T_tot.  The paper writes T_tot = N_run t_max for
// t_max << tau; here T_tot is the total time actually run, sum_r min(TTS_r, t_max), which
// reduces to the paper's value in that limit and to sum_r TTS_r without a timeout (DESIGN.md
// reading R-ttot).
#include <algorithm>
#include <cmath>
#include <limits>
#include <vector>

#include "xs_internal.h"

namespace {

// Q(n, x) = exp(-x) sum_{k<n} x^k / k!  (upper regularised incomplete gamma, integer shape)
double gamma_q_int(uint32_t n, double x)
{
    if (x <= 0.0) return 1.0;
    const double lx = std::log(x);
    double sum = 0.0;
    for (uint32_t k = 0; k < n; ++k) sum += std::exp(k * lx - x - std::lgamma((double)k + 1.0));
    return std::min(1.0, sum);
}

// x with P[Gamma(n,1) <= x] = q, by bisection.
double gamma_quantile_int(uint32_t n, double q)
{
    double lo = 0.0, hi = (double)n + 12.0 * std::sqrt((double)n) + 60.0;
    for (int it = 0; it < 200; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (1.0 - gamma_q_int(n, mid) < q) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

}  // namespace

extern "C" int xs_tts_stats(const uint32_t* tts, uint32_t n_runs, uint64_t t_max, double* out)
{
    if (!tts || !out || n_runs == 0) return XS_EINVAL;
    const double inf = std::numeric_limits<double>::infinity();
    uint32_t n = 0;
    double t_tot = 0.0;
    std::vector<double> v(n_runs);
    for (uint32_t r = 0; r < n_runs; ++r) {
        const bool solved = tts[r] != XS_NO_HIT && (t_max == 0 || tts[r] <= t_max);
        if (solved) { ++n; t_tot += (double)tts[r]; v[r] = (double)tts[r]; }
        else { t_tot += (double)t_max; v[r] = inf; }
    }
    std::sort(v.begin(), v.end());
    const double tau = n ? t_tot / n : inf;
    out[0] = n;
    out[1] = t_tot;
    out[2] = tau;
    const double ps[3] = {0.50, 0.90, 0.99};
    for (int q = 0; q < 3; ++q) {
        out[3 + q] = n ? -std::log(1.0 - ps[q]) * tau : inf;
        uint32_t rank = (uint32_t)std::ceil(ps[q] * n_runs - 1e-9);   // 1-based order statistic
        rank = std::min(std::max(rank, 1u), n_runs);
        out[6 + q] = v[rank - 1];
    }
    if (n == 0) {
        out[9] = t_tot / std::log(20.0);
        out[10] = inf;
        out[11] = inf;
    } else {
        // tau = T_tot / G, G ~ Gamma(n, 1): the q-quantile of tau is T_tot / (1-q)-quantile of G
        out[9] = t_tot / gamma_quantile_int(n, 1.0 - 0.16);
        out[10] = t_tot / gamma_quantile_int(n, 0.50);
        out[11] = t_tot / gamma_quantile_int(n, 1.0 - 0.84);
    }
    return XS_OK;
}
