"""Parity of et_scp (binned S_CP chi^2, Eq. 1) with oracle/scp.py -- needs a B200 (-m gpu).
Bin contents, in-grid yields, outside counts, ndf: bit-exact (the bin of an event is decided in fp64 by the same
operation order on both sides).  S_CP^i, alpha: the same IEEE operations per bin, compared to 4 ulp.  chi^2: a sum of up
to 2^24 non-negative terms in a different (tree) order, relative 1e-12.  p-value: the library's incomplete-gamma
evaluation against scipy's chi2.sf, relative 1e-9 (absolute 1e-300 in the far tail)."""
import numpy as np
import pytest

from oracle import scp as oscp
from paper_1612_04705_b200 import binding, build
from paper_1612_04705_b200 import datagen as dg

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    build.build()
    c = binding.Context(0)
    yield c
    c.close()


def check(got, exp):
    assert (got.Nx == exp.Nx).all() and (got.Nxbar == exp.Nxbar).all()
    assert (got.n_in_x, got.n_in_xbar, got.n_outside) == (exp.n_in_x, exp.n_in_xbar, exp.n_outside)
    assert (got.ndf, got.bins_used, got.bins_total) == (exp.ndf, exp.bins_used, len(exp.S))
    assert got.alpha == exp.alpha
    np.testing.assert_allclose(got.S, exp.S, rtol=1e-15, atol=0)
    assert got.chi2 == pytest.approx(exp.chi2, rel=1e-12)
    assert got.p_value == pytest.approx(exp.p_value, rel=1e-9, abs=1e-300)


def test_scp_hand_evaluated_2x2(ctx, golden_dir):
    """tests/golden/scp_2x2.txt: chi^2 = 36/35, alpha = 2, ndf = 3."""
    rng = np.random.default_rng(1)
    pts = lambda counts: np.vstack([(np.array(divmod(f, 2)) + rng.uniform(0.05, 0.95, size=(c, 2))) / 2 for f, c in enumerate(counts)])
    r = ctx.scp(pts([6, 2, 3, 1]), pts([2, 2, 1, 1]), [0, 0], [1, 1], [2, 2])
    assert r.Nx.tolist() == [6, 2, 3, 1] and r.Nxbar.tolist() == [2, 2, 1, 1]
    assert r.alpha == 2.0 and r.ndf == 3 and r.chi2 == pytest.approx(36 / 35, rel=1e-15)
    assert r.S == pytest.approx([2 / 14**0.5, -2 / 10**0.5, 1 / 7**0.5, -1 / 5**0.5], rel=1e-15)


@pytest.mark.parametrize("index,nbins", [(0, (6, 5)), (0, (32, 32)), (1, (10, 10)), (1, (100, 100))])
def test_scp_dalitz_configs(ctx, index, nbins):
    """BASELINE configs[0], [1] (Dalitz samples with the injected bump) on grids of O(10) .. O(10^3) .. 10^4 bins
    ("O(10^3) bins", "O(10) to O(10^2)"); the 100 x 100 grid takes the global-atomics histogram."""
    cfg = dg.config(index)
    s = dg.make_sample(cfg)
    lo, hi = [0.9, 0.3], [3.1, 2.0]  # covers the D+ -> K-K+pi+ Dalitz plot; the corners are empty bins (R21)
    got, exp = ctx.scp(s.x, s.xbar, lo, hi, nbins), oscp.scp(s.x, s.xbar, lo, hi, nbins)
    check(got, exp)
    assert got.bins_used < got.bins_total or nbins == (6, 5)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_scp_5d_ragged_with_outside_events_and_edges(ctx, dtype):
    rng = np.random.default_rng(11)
    x = rng.normal(0.5, 0.35, size=(70001, 5)).astype(dtype)
    xb = rng.normal(0.52, 0.35, size=(55555, 5)).astype(dtype)
    x[:5] = [[0, 0, 0, 0, 0], [1, 1, 1, 1, 1], [1, 0, 1, 0, 1], [0.5, 0.5, 0.5, 0.5, 1.0000001], [np.nan, 0.5, 0.5, 0.5, 0.5]]
    xb[0, 2] = np.inf
    got = ctx.scp(x, xb, [0] * 5, [1] * 5, [3, 2, 4, 3, 2])
    exp = oscp.scp(x, xb, [0] * 5, [1] * 5, [3, 2, 4, 3, 2])
    check(got, exp)
    assert got.n_outside > 1000 and got.Nx[0] >= 1 and got.Nx[-1] >= 1


def test_scp_bin_decisions_on_the_edges(ctx):
    """Events placed on (and one ulp around) every bin edge of an awkward grid fall into the oracle's bins."""
    lo, hi, nb = [-0.7], [2.3], [37]
    edges = lo[0] + (hi[0] - lo[0]) * np.arange(38) / 37
    x = np.concatenate([edges, np.nextafter(edges, -np.inf), np.nextafter(edges, np.inf)])[:, None]
    got, exp = ctx.scp(x, x[::2], lo, hi, nb), oscp.scp(x, x[::2], lo, hi, nb)
    check(got, exp)


def test_scp_device_pointers_and_large_grid(ctx):
    import torch

    rng = np.random.default_rng(12)
    x, xb = rng.uniform(size=(200000, 3)), rng.uniform(size=(150000, 3)) ** 1.05
    got = ctx.scp(torch.from_numpy(x).cuda(), torch.from_numpy(xb).cuda(), [0, 0, 0], [1, 1, 1], [64, 64, 32])
    check(got, oscp.scp(x, xb, [0, 0, 0], [1, 1, 1], [64, 64, 32]))
    assert got.bins_total == 131072


def test_scp_null_and_errors(ctx):
    rng = np.random.default_rng(13)
    x = rng.uniform(size=(5000, 2))
    same = ctx.scp(x, x, [0, 0], [1, 1], [4, 4])
    assert same.chi2 == 0.0 and same.p_value == 1.0
    with pytest.raises(binding.EtError) as e:
        ctx.scp(x, x + 5.0, [0, 0], [1, 1], [4, 4])       # xbar entirely outside
    assert e.value.status == -4
    with pytest.raises(binding.EtError) as e:
        ctx.scp(x, x, [0, 0], [1, 1], [1, 1])             # one bin: ndf = 0
    assert e.value.status == -4
    with pytest.raises(binding.EtError) as e:
        ctx.scp(x, x, [0, 1], [1, 1], [4, 4])             # lo == hi
    assert e.value.status == -1
    with pytest.raises(ValueError):
        ctx.scp(x, x, [0, 0], [1, 1], [4096, 4097])       # > 2^24 bins
