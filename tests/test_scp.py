"""Binned S_CP chi^2 (Eq. 1 at :29): pins of the oracle (oracle/scp.py) against a
hand-evaluated example, scipy's contingency-table chi^2 (alpha = 1), closed forms and invariants; parity of the
library's et_scp with it is in tests/test_gpu_parity.py (-m gpu)."""
import math
import os

import numpy as np
import pytest
from scipy.stats import chi2_contingency, kstest

from oracle import scp as oscp


def _points_in_bins(counts, nb, rng):
    """One point strictly inside bin (a, b) of the nb x nb grid over the unit square per count."""
    pts = []
    for flat, c in enumerate(counts):
        a, b = divmod(flat, nb)
        pts.append((np.array([a, b]) + rng.uniform(0.05, 0.95, size=(c, 2))) / nb)
    return np.vstack(pts)


def _golden(golden_dir):
    vals = {}
    with open(os.path.join(golden_dir, "scp_2x2.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            vals[k] = float(v)
    return vals


def test_S1_hand_evaluated_2x2(golden_dir):
    g = _golden(golden_dir)
    rng = np.random.default_rng(1)
    x = _points_in_bins([6, 2, 3, 1], 2, rng)
    xb = _points_in_bins([2, 2, 1, 1], 2, rng)
    r = oscp.scp(x, xb, [0, 0], [1, 1], [2, 2])
    assert r.Nx.tolist() == [6, 2, 3, 1] and r.Nxbar.tolist() == [2, 2, 1, 1]
    assert r.alpha == g["alpha"] and r.ndf == int(g["ndf"])
    for i in range(4):
        assert r.S[i] == pytest.approx(g[f"S{i}"], rel=1e-15)
    assert r.chi2 == pytest.approx(g["chi2"], rel=1e-15)
    assert r.chi2 == pytest.approx(36 / 35, rel=1e-15)


def test_S2_alpha_one_is_the_contingency_table_chi2():
    """n = nbar: N + alpha^2 Nbar = alpha (N + Nbar), and Eq. 1 summed over the bins is Pearson's homogeneity chi^2 of the
    2 x bins table (scipy.stats.chi2_contingency without Yates' correction), with the same bins - 1 degrees of freedom."""
    rng = np.random.default_rng(2)
    x, xb = rng.uniform(size=(5000, 2)), rng.beta(1.2, 1.0, size=(5000, 2))
    r = oscp.scp(x, xb, [0, 0], [1, 1], [6, 5])
    stat, p, dof, _ = chi2_contingency(np.vstack([r.Nx, r.Nxbar]), correction=False)
    assert r.alpha == 1.0 and r.ndf == dof == 29
    assert r.chi2 == pytest.approx(stat, rel=1e-12)
    assert r.p_value == pytest.approx(p, rel=1e-10)


def test_S3_swap_flips_every_S_and_keeps_chi2():
    rng = np.random.default_rng(3)
    x, xb = rng.uniform(size=(3000, 3)), rng.uniform(size=(4500, 3)) ** 1.1
    a = oscp.scp(x, xb, [0, 0, 0], [1, 1, 1], [4, 3, 2])
    b = oscp.scp(xb, x, [0, 0, 0], [1, 1, 1], [4, 3, 2])
    assert a.alpha == pytest.approx(1 / b.alpha, rel=1e-15)
    np.testing.assert_allclose(a.S, -b.S, rtol=1e-12, atol=0)
    assert a.chi2 == pytest.approx(b.chi2, rel=1e-12)
    # the constraint that ndf = bins - 1 counts (R20)
    assert abs((a.Nx - a.alpha * a.Nxbar).sum()) < 1e-9 * a.n_in_x


def test_S4_p_value_closed_forms():
    """ndf = 2: the chi^2 survival function is exp(-chi^2 / 2); identical samples give chi^2 = 0, p = 1."""
    rng = np.random.default_rng(4)
    x, xb = rng.uniform(size=(900, 1)), rng.uniform(size=(700, 1))
    r = oscp.scp(x, xb, [0], [1], [3])
    assert r.ndf == 2 and r.p_value == pytest.approx(math.exp(-r.chi2 / 2), rel=1e-12)
    same = oscp.scp(x, x, [0], [1], [7])
    assert same.chi2 == 0.0 and same.p_value == 1.0 and same.alpha == 1.0


def test_S5_null_samples_follow_chi2():
    """"In the absence of local CP asymmetries the S_CP^i are distributed according to a Gaussian of unit width and zero
    mean": over 400 null pairs the p-values are uniform and chi^2 / ndf averages 1."""
    rng = np.random.default_rng(5)
    ps, ratio = [], []
    for _ in range(400):
        x, xb = rng.uniform(size=(4000, 2)), rng.uniform(size=(5000, 2))
        r = oscp.scp(x, xb, [0, 0], [1, 1], [5, 4])
        ps.append(r.p_value)
        ratio.append(r.chi2 / r.ndf)
    assert abs(np.mean(ratio) - 1.0) < 4 * math.sqrt(2 / 19 / 400)
    assert kstest(ps, "uniform").pvalue > 1e-3
    # and a local asymmetry is seen
    xb = np.vstack([rng.uniform(size=(4500, 2)), 0.1 * rng.uniform(size=(500, 2))])
    assert oscp.scp(rng.uniform(size=(5000, 2)), xb, [0, 0], [1, 1], [5, 4]).p_value < 1e-6


def test_S6_bin_index_edges_and_histogramdd():
    lo, hi, nb = [0.0, -1.0], [2.0, 1.0], [4, 5]
    pts = np.array([[0.0, -1.0], [2.0, 1.0], [1.999999, 0.999999], [0.5, 0.2], [2.0000001, 0.0], [-1e-12, 0.0], [np.nan, 0.0], [1.0, np.inf]])
    idx = oscp.bin_index(pts, lo, hi, nb)
    assert idx.tolist() == [0, 19, 19, 1 * 5 + 3, -1, -1, -1, -1]
    rng = np.random.default_rng(6)
    x = rng.normal(0.8, 0.9, size=(20000, 2))
    r = oscp.scp(x, x[:10000], lo, hi, nb)
    edges = [np.linspace(lo[k], hi[k], nb[k] + 1) for k in range(2)]
    H, _ = np.histogramdd(x, bins=edges)
    assert (H.reshape(-1).astype(np.int64) == r.Nx).all()
    assert r.n_outside == (20000 - int(H.sum())) + (10000 - int(r.Nxbar.sum()))


def test_S7_empty_bins_are_not_bins():
    """R21: a bin empty in both samples does not enter chi^2 or ndf (the corners of a grid laid over a Dalitz plot)."""
    rng = np.random.default_rng(7)
    x, xb = rng.uniform(0, 0.5, size=(800, 2)), rng.uniform(0, 0.5, size=(900, 2))
    a = oscp.scp(x, xb, [0, 0], [0.5, 0.5], [3, 3])
    b = oscp.scp(x, xb, [0, 0], [1.0, 1.0], [6, 6])  # the same 9 bins plus 27 empty ones
    assert b.bins_used == 9 and b.ndf == a.ndf == 8
    assert b.chi2 == pytest.approx(a.chi2, rel=1e-12)
