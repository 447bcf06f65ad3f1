"""GEV step: pins of the oracle (oracle/gev.py, scipy.stats.genextreme) and
parity of the library's host-side et_gev_pvalue with it.  No GPU is needed: the function is host-only."""
import math

import numpy as np
import pytest
from scipy.stats import genextreme

import oracle
from oracle import gev
from paper_1612_04705_b200 import binding, build


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    return binding.lib()


# ------------------------------------------------------------------ pins of the oracle
def test_P15_closed_forms_of_the_gev():
    """F(mu) = exp(-1) for every shape; xi = 0 is the Gumbel law; the support ends at mu - sigma/xi."""
    for xi in (-0.4, -1e-9, 0.0, 0.2, 0.7):
        assert gev.sf(1.5, 1.5, 0.3, xi) == pytest.approx(1 - math.exp(-1), abs=1e-12)
    for zz in (-1.0, 0.3, 4.0, 30.0):
        assert gev.sf(2.0 + 0.5 * zz, 2.0, 0.5, 0.0) == pytest.approx(-math.expm1(-math.exp(-zz)), rel=1e-12)
    assert gev.sf(1.0 + 0.2 / 0.25 + 1e-9, 1.0, 0.2, -0.25) == 0.0       # above the upper end point (xi < 0)
    assert gev.sf(1.0 - 0.2 / 0.25 - 1e-9, 1.0, 0.2, 0.25) == 1.0        # below the lower end point (xi > 0)
    # quantile <-> survival: t^(-1/xi) = -log(1 - p)
    mu, s, xi, p = 3e-7, 1e-7, 0.15, 1e-9
    t = mu + s / xi * ((-math.log1p(-p)) ** (-xi) - 1)
    assert gev.sf(t, mu, s, xi) == pytest.approx(p, rel=1e-6)


def test_P16_fit_recovers_a_known_gev_and_is_stationary():
    rng = np.random.default_rng(3)
    true = (2e-7, 1.1e-7, 0.12)
    x = genextreme.rvs(-true[2], loc=true[0], scale=true[1], size=20000, random_state=rng)
    mu, s, xi = gev.fit(x)
    cov = gev.covariance(x, mu, s, xi)
    err = np.sqrt(np.diag(cov))
    assert abs(mu - true[0]) < 5 * err[0] and abs(s - true[1]) < 5 * err[1] and abs(xi - true[2]) < 5 * err[2]
    assert 0.5 / math.sqrt(20000) < err[2] < 2.0 / math.sqrt(20000)   # the shape error is O(1/sqrt(n))
    f0 = gev.nll(x, mu, s, xi)
    for d in ((1e-3 * s, 0, 0), (0, 1e-3 * s, 0), (0, 0, 1e-3)):
        assert gev.nll(x, mu + d[0], s + d[1], xi + d[2]) >= f0 - 1e-6 and gev.nll(x, mu - d[0], s - d[1], xi - d[2]) >= f0 - 1e-6


# ------------------------------------------------------------------ parity: library vs oracle
@pytest.mark.parametrize("xi_true,n,scale", [(0.1, 1000, 1e-7), (-0.15, 100, 1.0), (0.0, 400, 3e-4)])
def test_gev_pvalue_matches_oracle(xi_true, n, scale):
    rng = np.random.default_rng(int(1000 * abs(xi_true)) + n)
    x = genextreme.rvs(-xi_true, loc=2 * scale, scale=scale, size=n, random_state=rng)
    t_obs = 2 * scale + 7 * scale          # far outside the permutation values, as in the paper's use of the fit
    z = rng.standard_normal((4000, 3))
    got = binding.gev_pvalue(x, t_obs, z)
    mu, s, xi = gev.fit(x)
    assert got.converged and got.n_used == n
    assert got.nll <= gev.nll(x, mu, s, xi) + 1e-7 * n                     # at least as good an optimum as scipy's
    assert got.nll == pytest.approx(gev.nll(x, got.mu, got.sigma, got.xi), abs=1e-8 * n)  # and it is the GEV likelihood
    assert got.mu == pytest.approx(mu, abs=2e-4 * s) and got.sigma == pytest.approx(s, rel=2e-4) and got.xi == pytest.approx(xi, abs=2e-4)
    assert got.p_value == pytest.approx(gev.sf(t_obs, got.mu, got.sigma, got.xi), rel=1e-10, abs=1e-300)
    assert math.log(got.p_value) == pytest.approx(math.log(gev.sf(t_obs, mu, s, xi)), abs=5e-3) if got.p_value > 0 else True
    cov = gev.covariance(x, got.mu, got.sigma, got.xi)
    assert np.allclose(got.cov, cov, rtol=2e-3, atol=1e-6 * np.sqrt(np.outer(np.diag(cov), np.diag(cov))))
    ps = gev.resample(t_obs, got.mu, got.sigma, got.xi, got.cov, z)
    assert got.n_resampled == len(ps)
    lo, med, hi = np.quantile(ps, [0.158655253931457, 0.5, 0.841344746068543])
    assert got.p_lo == pytest.approx(lo, rel=1e-9, abs=1e-300) and got.p_med == pytest.approx(med, rel=1e-9, abs=1e-300)
    assert got.p_hi == pytest.approx(hi, rel=1e-9, abs=1e-300)
    assert got.p_lo <= got.p_med <= got.p_hi


def test_gev_of_a_real_permutation_distribution_agrees_with_counting():
    """T_perm of an oracle permutation test on samples from the same density: the fitted p-value agrees with the
    counted one within its binomial error plus the fit's own band (the paper uses the fit where counting gives 0)."""
    rng = np.random.default_rng(8)
    x, xb = rng.uniform(size=(120, 2)), rng.uniform(size=(140, 2))
    r = oracle.perm_test(x, xb, 0.25, 300, 21)
    g = binding.gev_pvalue(r.T_perm, r.observed.T, rng.standard_normal((2000, 3)))
    assert g.converged
    p = r.count_gt / 300
    assert abs(g.p_value - p) <= 4 * math.sqrt(max(p * (1 - p), 1 / 300) / 300) + (g.p_hi - g.p_lo)
    # an observed T far above every permutation: counting gives 0, the fit a small positive number
    far = r.T_perm.max() + 3 * r.T_perm.std()
    gf = binding.gev_pvalue(r.T_perm, far)
    assert (r.T_perm > far).sum() == 0 and 0 < gf.p_value < 1 / 300 and math.isnan(gf.p_lo)


def test_gev_edge_cases():
    with pytest.raises(binding.EtError) as e:
        binding.gev_pvalue(np.arange(5.0), 1.0)
    assert e.value.status == -4
    with pytest.raises(binding.EtError) as e:
        binding.gev_pvalue(np.ones(50), 1.0)
    assert e.value.status == -4
    with pytest.raises(binding.EtError) as e:
        binding.gev_pvalue(np.arange(50.0), float("nan"))
    assert e.value.status == -1
    x = genextreme.rvs(0.1, size=200, random_state=np.random.default_rng(0))
    a = binding.gev_pvalue(np.concatenate([x, [np.nan, np.inf]]), 3.0)
    b = binding.gev_pvalue(x, 3.0)
    assert a.n_used == 200 and a.p_value == b.p_value and a.mu == b.mu       # non-finite permutation values are skipped
    # affine equivariance: T -> a T + b moves (mu, sigma) and leaves xi and p alone
    c = binding.gev_pvalue(1e-7 * x + 5e-6, 1e-7 * 3.0 + 5e-6)
    assert c.xi == pytest.approx(b.xi, abs=1e-6) and c.p_value == pytest.approx(b.p_value, rel=1e-5)
    assert c.sigma == pytest.approx(1e-7 * b.sigma, rel=1e-5)
