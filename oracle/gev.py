"""Oracle for the GEV step -- TEST INFRASTRUCTURE ONLY, like the rest of oracle/.

The paper fits the permutation T values with a generalised-extreme-value function, reads the p-value as the integral
of the fitted function above the observed T, and gets its uncertainty by resampling the fitted parameters within their
covariance.  Each step here is a library routine: scipy.stats.genextreme (density and survival function; its shape parameter is c = -xi),
scipy.optimize's Nelder-Mead simplex for the maximum-likelihood fit, a finite-difference Hessian of that log-density, numpy's Cholesky factor and
quantiles.  Shares no code with paper_1612_04705_b200/csrc/et_gev.cu; the normal draws of the resampling are an input
of both sides.
"""
from __future__ import annotations

import numpy as np
from scipy import optimize
from scipy.stats import genextreme


def nll(x, mu: float, sigma: float, xi: float) -> float:
    """Negative log-likelihood of the sample under GEV(mu, sigma, xi), F(x) = exp(-(1 + xi (x - mu)/sigma)^(-1/xi))."""
    if not sigma > 0:
        return float("inf")
    v = -genextreme.logpdf(np.asarray(x, dtype=np.float64), -xi, loc=mu, scale=sigma).sum()
    return float(v) if np.isfinite(v) else float("inf")


def sf(t: float, mu: float, sigma: float, xi: float) -> float:
    """p-value of the fitted function: the fraction of its integral above t."""
    return float(genextreme.sf(t, -xi, loc=mu, scale=sigma))


def fit(x):
    """Maximum-likelihood (mu, sigma, xi) = argmin of `nll`, by scipy's Nelder-Mead simplex with restarts.  The sample is
    standardised first (T is O(1e-7) at large N); several shape starts, the lowest optimum wins.  (scipy's own
    genextreme.fit is not used: from its default start it stops at nll values thousands above the optimum here.)"""
    x = np.asarray(x, dtype=np.float64)
    x = x[np.isfinite(x)]
    m, s = x.mean(), x.std(ddof=1)
    y = (x - m) / s
    f = lambda p: nll(y, p[0], np.exp(p[1]), p[2])
    best = None
    for xi0 in (-0.3, 0.0, 0.3):
        p = np.array([-0.45, np.log(0.78), xi0])      # Gumbel moment estimates of a standardised sample
        step = 0.25
        for _ in range(4):
            simplex = np.vstack([p] + [p + step * np.eye(3)[k] for k in range(3)])
            res = optimize.minimize(f, p, method="Nelder-Mead", options={"initial_simplex": simplex, "xatol": 1e-11, "fatol": 1e-13,
                                                                         "maxiter": 20000, "maxfev": 20000})
            p, step = res.x, step * 0.2
        if np.isfinite(res.fun) and (best is None or res.fun < best[0]):
            best = (res.fun, p)
    assert best is not None
    mu_y, s_y, xi = best[1][0], float(np.exp(best[1][1])), best[1][2]
    return m + s * mu_y, s * s_y, float(xi)


def covariance(x, mu: float, sigma: float, xi: float) -> np.ndarray:
    """Inverse of the observed information in (mu, sigma, xi): central differences of `nll` (relative steps 1e-4)."""
    x = np.asarray(x, dtype=np.float64)
    x = x[np.isfinite(x)]
    p0 = np.array([mu, sigma, xi])
    h = np.array([1e-4 * sigma, 1e-4 * sigma, 1e-4])
    f = lambda p: nll(x, *p)
    H = np.zeros((3, 3))
    f0 = f(p0)
    for a in range(3):
        for b in range(a, 3):
            if a == b:
                e = np.zeros(3); e[a] = h[a]
                H[a, a] = (f(p0 + e) - 2 * f0 + f(p0 - e)) / h[a] ** 2
            else:
                ea = np.zeros(3); ea[a] = h[a]
                eb = np.zeros(3); eb[b] = h[b]
                H[a, b] = H[b, a] = (f(p0 + ea + eb) - f(p0 + ea - eb) - f(p0 - ea + eb) + f(p0 - ea - eb)) / (4 * h[a] * h[b])
    return np.linalg.inv(H)


def resample(t_obs: float, mu: float, sigma: float, xi: float, cov: np.ndarray, z) -> np.ndarray:
    """p-values of the parameter sets theta_hat + L z_k, cov = L L^T; sets with sigma <= 0 dropped."""
    L = np.linalg.cholesky(cov)
    th = np.array([mu, sigma, xi]) + np.asarray(z, dtype=np.float64).reshape(-1, 3) @ L.T
    ok = th[:, 1] > 0
    return np.array([sf(t_obs, *t) for t in th[ok]])
