// et_gev.cu -- host-side post-processing of the permutation T values:
// "the permutation T distribution can be fitted with a generalised-extreme-value (GEV) function ... The p-value from
// the fitted T distribution can be calculated as the fraction of the integral of the function above the observed T
// value", and its uncertainty "by randomly resampling the fit parameters within their uncertainties, taking into
// account their correlations, and by extracting a p-value for each of these generated T distributions".
// O(nperm) work on <= a few thousand numbers: plain C++ on the host, no kernel.  Not shared with oracle/.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <limits>
#include <vector>

#include "../../include/et.h"

namespace {

// GEV with location mu, scale s > 0, shape xi:  F(x) = exp(-t^(-1/xi)), t = 1 + xi (x - mu) / s > 0;  xi -> 0: Gumbel.
// g(z; xi) = log(t) / xi evaluated smoothly through xi = 0 (= z - xi z^2 / 2 + ...), so that t^(-1/xi) = exp(-g).
inline bool gev_g(double z, double xi, double *g)
{
    const double y = xi * z;
    if (!(y > -1.0)) return false;                     // outside the support
    *g = std::fabs(y) < 1e-5 ? z * (1.0 - y * (0.5 - y / 3.0)) : std::log1p(y) / xi;
    return true;
}

// negative log-likelihood of the sample for theta = (mu, log s, xi); +inf outside the support
double nll(const std::vector<double> &x, const double th[3])
{
    const double mu = th[0], s = std::exp(th[1]), xi = th[2];
    if (!std::isfinite(s) || s <= 0.0) return std::numeric_limits<double>::infinity();
    double acc = 0.0;
    for (double v : x) {
        double g;
        if (!gev_g((v - mu) / s, xi, &g)) return std::numeric_limits<double>::infinity();
        acc += (1.0 + xi) * g + std::exp(-g);          // -log f = log s + (1 + xi) g + e^(-g)
    }
    return acc + (double)x.size() * th[1];
}

// survival function 1 - F(x), accurate in both tails
double gev_sf(double x, double mu, double s, double xi)
{
    double g;
    if (!gev_g((x - mu) / s, xi, &g)) return xi > 0.0 ? 1.0 : 0.0;   // below the lower end point / above the upper one
    return -std::expm1(-std::exp(-g));
}

// Nelder-Mead on three parameters
double nelder_mead(const std::vector<double> &x, double th[3], const double step[3], int max_iter, double tol)
{
    double p[4][3], f[4];
    for (int k = 0; k < 4; ++k) {
        for (int d = 0; d < 3; ++d) p[k][d] = th[d] + (k == d + 1 ? step[d] : 0.0);
        f[k] = nll(x, p[k]);
    }
    for (int it = 0; it < max_iter; ++it) {
        int o[4] = {0, 1, 2, 3};
        std::sort(o, o + 4, [&](int a, int b) { return f[a] < f[b]; });
        const int lo = o[0], hi = o[3], nh = o[2];
        if (std::isfinite(f[hi]) && std::fabs(f[hi] - f[lo]) <= tol * (std::fabs(f[lo]) + 1e-300)) break;
        double c[3] = {0, 0, 0};
        for (int k = 0; k < 4; ++k)
            if (k != hi)
                for (int d = 0; d < 3; ++d) c[d] += p[k][d] / 3.0;
        auto at = [&](double a, double out[3]) {
            for (int d = 0; d < 3; ++d) out[d] = c[d] + a * (p[hi][d] - c[d]);
            return nll(x, out);
        };
        double r[3], e[3];
        const double fr = at(-1.0, r);
        if (fr < f[lo]) {
            const double fe = at(-2.0, e);
            if (fe < fr) { std::copy(e, e + 3, p[hi]); f[hi] = fe; }
            else { std::copy(r, r + 3, p[hi]); f[hi] = fr; }
        } else if (fr < f[nh]) {
            std::copy(r, r + 3, p[hi]); f[hi] = fr;
        } else {
            const double fc = fr < f[hi] ? at(-0.5, e) : at(0.5, e);
            if (fc < std::min(fr, f[hi])) { std::copy(e, e + 3, p[hi]); f[hi] = fc; }
            else
                for (int k = 0; k < 4; ++k)
                    if (k != lo) {
                        for (int d = 0; d < 3; ++d) p[k][d] = p[lo][d] + 0.5 * (p[k][d] - p[lo][d]);
                        f[k] = nll(x, p[k]);
                    }
        }
    }
    int best = 0;
    for (int k = 1; k < 4; ++k)
        if (f[k] < f[best]) best = k;
    std::copy(p[best], p[best] + 3, th);
    return f[best];
}

bool invert3(const double a[9], double inv[9])
{
    const double c00 = a[4] * a[8] - a[5] * a[7], c01 = a[5] * a[6] - a[3] * a[8], c02 = a[3] * a[7] - a[4] * a[6];
    const double det = a[0] * c00 + a[1] * c01 + a[2] * c02;
    if (!(std::fabs(det) > 0.0) || !std::isfinite(det)) return false;
    inv[0] = c00 / det; inv[1] = (a[2] * a[7] - a[1] * a[8]) / det; inv[2] = (a[1] * a[5] - a[2] * a[4]) / det;
    inv[3] = c01 / det; inv[4] = (a[0] * a[8] - a[2] * a[6]) / det; inv[5] = (a[2] * a[3] - a[0] * a[5]) / det;
    inv[6] = c02 / det; inv[7] = (a[1] * a[6] - a[0] * a[7]) / det; inv[8] = (a[0] * a[4] - a[1] * a[3]) / det;
    return true;
}

}  // namespace

extern "C" et_status et_gev_pvalue(const double *T_perm, int64_t nperm, double T_obs, const double *z, int64_t nresample,
                                   et_gev_result *out)
{
    if (!T_perm || !out || nperm < 1 || nresample < 0 || (nresample > 0 && !z) || !std::isfinite(T_obs)) return ET_ERR_INVALID;
    std::vector<double> x;
    x.reserve((size_t)nperm);
    for (int64_t k = 0; k < nperm; ++k)
        if (std::isfinite(T_perm[k])) x.push_back(T_perm[k]);
    const size_t n = x.size();
    if (n < 10) return ET_ERR_DEGENERATE;              // three parameters need a distribution to fit
    double mean = 0.0, var = 0.0;
    for (double v : x) mean += v;
    mean /= (double)n;
    for (double v : x) var += (v - mean) * (v - mean);
    var /= (double)(n - 1);
    if (!(var > 0.0)) return ET_ERR_DEGENERATE;
    // work in standardised units (T is O(1e-7) at large N): y = (x - mean) / sd
    const double sd = std::sqrt(var);
    for (double &v : x) v = (v - mean) / sd;
    // start from the Gumbel moment estimates, polish with restarts of the simplex
    double th[3] = {-0.5772156649015329 * std::sqrt(6.0) / M_PI, std::log(std::sqrt(6.0) / M_PI), 0.0};
    double step[3] = {0.2, 0.2, 0.1};
    double best = std::numeric_limits<double>::infinity();
    bool converged = false;
    for (int round = 0; round < 6; ++round) {
        const double f = nelder_mead(x, th, step, 4000, 1e-14);
        converged = std::isfinite(f) && std::fabs(best - f) <= 1e-10 * (std::fabs(f) + 1.0);
        best = std::min(best, f);
        if (converged && round >= 1) break;
        for (double &s : step) s *= 0.3;
    }
    const double mu_y = th[0], s_y = std::exp(th[1]), xi = th[2];
    // observed information in (mu, s, xi) of the standardised sample by central differences
    auto f3 = [&](double m, double s, double k) {
        const double t[3] = {m, std::log(s), k};
        return nll(x, t);
    };
    const double h[3] = {1e-4 * s_y, 1e-4 * s_y, 1e-4};
    const double q0[3] = {mu_y, s_y, xi};
    double H[9];
    for (int a = 0; a < 3; ++a)
        for (int b = a; b < 3; ++b) {
            double v;
            if (a == b) {
                double p[3] = {q0[0], q0[1], q0[2]}, m[3] = {q0[0], q0[1], q0[2]};
                p[a] += h[a]; m[a] -= h[a];
                v = (f3(p[0], p[1], p[2]) - 2.0 * best + f3(m[0], m[1], m[2])) / (h[a] * h[a]);
            } else {
                double pp[3] = {q0[0], q0[1], q0[2]}, pm[3] = {q0[0], q0[1], q0[2]}, mp[3] = {q0[0], q0[1], q0[2]}, mm[3] = {q0[0], q0[1], q0[2]};
                pp[a] += h[a]; pp[b] += h[b]; pm[a] += h[a]; pm[b] -= h[b]; mp[a] -= h[a]; mp[b] += h[b]; mm[a] -= h[a]; mm[b] -= h[b];
                v = (f3(pp[0], pp[1], pp[2]) - f3(pm[0], pm[1], pm[2]) - f3(mp[0], mp[1], mp[2]) + f3(mm[0], mm[1], mm[2])) / (4.0 * h[a] * h[b]);
            }
            H[a * 3 + b] = H[b * 3 + a] = v;
        }
    double cov_y[9];
    bool cov_ok = invert3(H, cov_y) && cov_y[0] > 0.0 && cov_y[4] > 0.0 && cov_y[8] > 0.0;
    for (int k = 0; k < 9 && cov_ok; ++k) cov_ok = std::isfinite(cov_y[k]);

    et_gev_result r;
    r.mu = mean + sd * mu_y;
    r.sigma = sd * s_y;
    r.xi = xi;
    // back to the units of T: (mu, sigma) scale with sd, xi does not
    const double sc[3] = {sd, sd, 1.0};
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) r.cov[a * 3 + b] = cov_ok ? cov_y[a * 3 + b] * sc[a] * sc[b] : std::numeric_limits<double>::quiet_NaN();
    r.nll = best + (double)n * std::log(sd);
    r.p_value = gev_sf(T_obs, r.mu, r.sigma, r.xi);
    r.n_used = (int64_t)n;
    r.converged = converged && cov_ok ? 1 : 0;
    r.p_lo = r.p_med = r.p_hi = std::numeric_limits<double>::quiet_NaN();
    r.n_resampled = 0;
    if (nresample > 0 && cov_ok) {
        // theta = theta_hat + L z with cov = L L^T (Cholesky), z the caller's standard normal draws [nresample][3]
        double L[9] = {0};
        bool pd = true;
        for (int a = 0; a < 3 && pd; ++a)
            for (int b = 0; b <= a; ++b) {
                double s = r.cov[a * 3 + b];
                for (int k = 0; k < b; ++k) s -= L[a * 3 + k] * L[b * 3 + k];
                if (a == b) { pd = s > 0.0; L[a * 3 + a] = pd ? std::sqrt(s) : 0.0; }
                else L[a * 3 + b] = s / L[b * 3 + b];
            }
        if (pd) {
            std::vector<double> ps;
            ps.reserve((size_t)nresample);
            for (int64_t k = 0; k < nresample; ++k) {
                const double *zz = z + 3 * k;
                const double m = r.mu + L[0] * zz[0];
                const double s = r.sigma + L[3] * zz[0] + L[4] * zz[1];
                const double c = r.xi + L[6] * zz[0] + L[7] * zz[1] + L[8] * zz[2];
                if (s > 0.0 && std::isfinite(m) && std::isfinite(c)) ps.push_back(gev_sf(T_obs, m, s, c));  // sigma <= 0 is no GEV
            }
            if (!ps.empty()) {
                std::sort(ps.begin(), ps.end());
                auto quant = [&](double q) {  // linear interpolation between order statistics
                    const double pos = q * (double)(ps.size() - 1);
                    const size_t i0 = (size_t)pos;
                    const size_t i1 = std::min(i0 + 1, ps.size() - 1);
                    return ps[i0] + (pos - (double)i0) * (ps[i1] - ps[i0]);
                };
                r.p_lo = quant(0.158655253931457);
                r.p_med = quant(0.5);
                r.p_hi = quant(0.841344746068543);
                r.n_resampled = (int64_t)ps.size();
            }
        }
    }
    *out = r;
    return ET_OK;
}
