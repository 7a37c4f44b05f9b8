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
    // t_max = 0 means "no cap": an unsolved run then has no censoring time to contribute and
    // would silently count as zero cost (tau biased low) -> refuse
    if (t_max == 0)
        for (uint32_t r = 0; r < n_runs; ++r)
            if (tts[r] == XS_NO_HIT) return XS_EINVAL;
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

// ---- cavity free-energy barrier (Eqs. (3)-(4), L171-L208) --------
namespace {

struct CavityPoint { double m, bdf, b; };

// beta (f - f_para) at cavity field h (the saddle-point equations (4) solved for u, b, m given h)
CavityPoint cavity_at(uint32_t K, double beta, double h)
{
    const double th = std::tanh(beta * h);
    const double u = std::atanh(std::tanh(beta) * std::pow(th, (double)K - 1.0)) / beta;
    const double b = h - ((double)K - 1.0) * u;
    const double m = std::tanh(beta * (u + h));
    const double log_zi = std::log(2.0 * std::cosh(beta * (K * u + b))) - K * std::log(2.0 * std::cosh(beta * u));
    const double log_za = std::log(std::cosh(beta)) + std::log1p(std::tanh(beta) * std::pow(th, (double)K));
    const double log_zai = std::log(std::cosh(beta * (u + h))) - std::log(2.0 * std::cosh(beta * u)) -
                           std::log(std::cosh(beta * h));
    const double minus_beta_f = log_zi + log_za - K * log_zai - beta * b * m;
    const double minus_beta_fpara = std::log(2.0 * std::cosh(beta));
    return {m, minus_beta_fpara - minus_beta_f, b};
}

// golden-section search of a maximum (sign = +1) or minimum (sign = -1) of fn on [lo, hi]
template <class F> double golden(F fn, double lo, double hi, double sign)
{
    const double g = 0.5 * (std::sqrt(5.0) - 1.0);
    double a = lo, c = hi, x1 = c - g * (c - a), x2 = a + g * (c - a);
    double f1 = sign * fn(x1), f2 = sign * fn(x2);
    for (int it = 0; it < 200 && c - a > 1e-14; ++it) {
        if (f1 < f2) { a = x1; x1 = x2; f1 = f2; x2 = a + g * (c - a); f2 = sign * fn(x2); }
        else         { c = x2; x2 = x1; f2 = f1; x1 = c - g * (c - a); f1 = sign * fn(x1); }
    }
    return 0.5 * (a + c);
}

}  // namespace

extern "C" int xs_cavity_barrier(uint32_t K, double T, double* out)
{
    if (!out || K < 3 || !(T > 0.0)) return XS_EINVAL;
    const double nan = std::numeric_limits<double>::quiet_NaN();
    for (int i = 0; i < 6; ++i) out[i] = nan;
    // spinodal: smallest beta for which tanh(x) = tanh(beta) tanh((K-1)x)^(K-1) has a solution x > 0
    auto beta_of_x = [&](double x) {
        const double v = std::tanh(x) / std::pow(std::tanh(((double)K - 1.0) * x), (double)K - 1.0);
        return v < 1.0 ? std::atanh(v) : std::numeric_limits<double>::infinity();
    };
    double xb = 0.0, fb = std::numeric_limits<double>::infinity();
    for (int i = 1; i <= 4000; ++i) {                       // coarse scan, then refine
        const double x = 0.0025 * i, f = beta_of_x(x);
        if (f < fb) { fb = f; xb = x; }
    }
    const double xs_ = golden(beta_of_x, std::max(xb - 0.0025, 1e-6), xb + 0.0025, -1.0);
    const double beta_sp = beta_of_x(xs_);
    out[3] = 1.0 / beta_sp;
    const double beta = 1.0 / T;
    if (beta <= beta_sp) return XS_OK;
    // along h: beta Delta f starts at 0 (paramagnet), rises to the barrier (b = 0, unstable),
    // falls to the ferromagnetic state (b = 0, stable) and rises again.
    auto bdf = [&](double h) { return cavity_at(K, beta, h).bdf; };
    const double dh = 1e-3;
    double h_top = 0.0, h_fm = 0.0;
    double prev = 0.0;
    bool rising = true;
    for (int i = 1; i <= 20000; ++i) {
        const double h = dh * i, f = bdf(h);
        if (rising && f < prev) { h_top = h - dh; rising = false; }
        else if (!rising && f > prev) { h_fm = h - dh; break; }
        prev = f;
    }
    if (h_top <= 0.0 || h_fm <= 0.0) return XS_OK;
    const double ht = golden(bdf, std::max(h_top - dh, 1e-9), h_top + dh, +1.0);
    const double hf = golden(bdf, h_fm - dh, h_fm + dh, -1.0);
    const CavityPoint top = cavity_at(K, beta, ht), fm = cavity_at(K, beta, hf);
    out[0] = top.bdf; out[1] = top.m; out[2] = ht;
    out[4] = fm.bdf;  out[5] = fm.m;
    return XS_OK;
}
