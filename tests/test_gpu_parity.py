"""Parity of the CUDA path (through the C ABI) against the oracle -- needs a B200 (-m gpu).

Tolerances (north_star): |dT| <= 1e-6 (|T_XX| + |T_XbarXbar| + |T_XXbar|); labels, split flags, counts and
p-values bit-exact.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1612_04705_b200 import binding, build
from paper_1612_04705_b200 import datagen as dg

pytestmark = pytest.mark.gpu

TOL = 1e-6


@pytest.fixture(scope="module")
def ctx():
    build.build()
    c = binding.Context(0)
    yield c
    c.close()


TERM_REL_TC = 1.5e-5


def assert_T_close(got, exp, tol=TOL, term_rel=0.0):
    """T within the north-star tolerance; the three terms too.  term_rel > 0 (tensor-core path): each term may also
    be off by that fraction of itself -- the 15-bit round-to-nearest loses the psi values below half a step, about 0.005
    steps per pair: the same fraction of all three block sums (measured 7e-7 at sigma = 0.3, 6e-6 at sigma = 0.1, 2.7e-6
    with signed weights), which cancels in T (et_tc.cuh).  The tolerance of T itself is never relaxed."""
    scale = exp.term_scale
    assert abs(got.T - exp.T) <= tol * scale, (got.T, exp.T, scale)
    for k in ("T_xx", "T_bb", "T_xb"):
        assert abs(getattr(got, k) - getattr(exp, k)) <= tol * scale + term_rel * abs(getattr(exp, k)), k
    assert got.W == pytest.approx(exp.W, rel=1e-6) and got.Wbar == pytest.approx(exp.Wbar, rel=1e-6)
    assert got.n_pairs == exp.n_pairs


# ----------------------------------------------------------------------------- closed forms through the GPU
def test_closed_forms(ctx):
    sigma = 0.3
    a = sigma * math.sqrt(2 * math.log(2))
    assert ctx.T(np.array([[0, 0], [a, 0.0]]), np.array([[0, a], [a, a]]), sigma).T == pytest.approx(0.125, abs=1e-6)
    r = ctx.T(np.array([[0.0], [a]]), np.array([[2 * a], [3 * a]]), sigma)
    assert r.T == pytest.approx(0.34326171875, abs=1e-6)
    A, B = np.zeros((3, 3)), np.zeros((5, 3))
    B[:, 1] = 0.37
    assert ctx.T(A, B, 0.5).T == pytest.approx(1 - math.exp(-0.37**2 / 0.5), abs=1e-6)
    pt = np.full((7, 4), 0.3)
    assert ctx.T(pt, pt[:4], 0.4).T == pytest.approx(0.0, abs=1e-6)


# ----------------------------------------------------------------------------- et_T
@pytest.mark.parametrize("dim", [1, 2, 3, 4, 5, 6, 7, 8])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_T_random_all_dims(ctx, dim, dtype):
    rng = np.random.default_rng(100 + dim)
    n, nbar = 1500 + 37 * dim, 1111  # ragged: not multiples of any tile, n != nbar
    x = rng.uniform(size=(n, dim)).astype(dtype)
    xb = (rng.uniform(size=(nbar, dim)) ** 1.1).astype(dtype)
    sigma = 0.2 * math.sqrt(dim)
    assert_T_close(ctx.T(x, xb, sigma), oracle.T(x, xb, sigma))


class force_distance:
    """ET_OPT_DISTANCE for the duration of a block: 1 = differences, 2 = Gram form (k_pairs_T)."""

    def __init__(self, ctx, form):
        self.ctx, self.form = ctx, form

    def __enter__(self):
        self.ctx.set_option(binding.ET_OPT_DISTANCE, self.form)

    def __exit__(self, *exc):
        self.ctx.set_option(binding.ET_OPT_DISTANCE, 0)


@pytest.mark.parametrize("dim", [1, 2, 4, 5, 8])
@pytest.mark.parametrize("weighted", [False, True])
def test_T_gram_form_matches_oracle(ctx, dim, weighted):
    """The Gram form of the distance in k_pairs_T (|u_i|^2 + |u_j|^2 - 2 u_i.u_j: dim + 2 instead of 2 dim + 1 FP32
    operations per pair), forced, against the oracle at the north-star tolerance; ragged sizes, diagonal tiles (the i = j
    term is removed as evaluated), signed weights."""
    rng = np.random.default_rng(300 + dim)
    n, nbar = 2500 + 37 * dim, 2111
    x, xb = rng.uniform(size=(n, dim)), rng.uniform(size=(nbar, dim)) ** 1.1
    wx = rng.uniform(-0.5, 1.5, size=n) if weighted else None
    wb = rng.uniform(-0.5, 1.5, size=nbar) if weighted else None
    sigma = 0.2 * math.sqrt(dim)
    exp = oracle.T(x, xb, sigma, wx, wb)
    with force_distance(ctx, 2):
        got = ctx.T_weighted(x, wx, xb, wb, sigma) if weighted else ctx.T(x, xb, sigma)
        assert ctx.stats().distance_form == 2
    assert_T_close(got, exp)
    with force_distance(ctx, 1):
        ref = ctx.T_weighted(x, wx, xb, wb, sigma) if weighted else ctx.T(x, xb, sigma)
        assert ctx.stats().distance_form == 1
    # the two forms agree far inside the tolerance at this size (errors of either: 1e-9 of the term scale or less)
    assert abs(got.T - ref.T) <= 2e-8 * exp.term_scale


def test_T_distance_form_dispatch(ctx):
    """Default rule (et.h, ET_OPT_DISTANCE): Gram form only for dim >= 4, n + nbar >= 4096 and a sample that is compact in
    units of sigma; everything else keeps the differences."""
    rng = np.random.default_rng(9)
    x5, y5 = rng.uniform(size=(3000, 5)), rng.uniform(size=(2000, 5))
    ctx.T(x5, y5, 0.2)
    assert ctx.stats().distance_form == 2
    ctx.T(x5[:1500], y5, 0.2)                      # fewer than 4096 events
    assert ctx.stats().distance_form == 1
    ctx.T(x5, y5, 0.02)                            # half diagonal of the box >> sigma: |u|^2_max = 5 (0.5 * 42)^2 >> 48
    assert ctx.stats().distance_form == 1
    ctx.T(x5[:, :2].copy(), y5[:, :2].copy(), 0.2)  # dim = 2 is bound by the SFU either way
    assert ctx.stats().distance_form == 1
    far = x5.copy()
    far[0] += 100.0                                # one outlier stretches the box
    ctx.T(far, y5, 0.2)
    assert ctx.stats().distance_form == 1
    with pytest.raises(binding.EtError):
        ctx.set_option(binding.ET_OPT_DISTANCE, 3)


def test_T_config0_full(ctx):
    s = dg.make_sample(dg.config(0))
    exp = oracle.T(s.x, s.xbar, 0.3)
    got = ctx.T(s.x, s.xbar, 0.3)
    assert_T_close(got, exp)
    # the injected 5 % bump is seen (T well above the null fluctuation of ~2e-4)
    assert got.T > 5e-4


def test_T_tiny_and_edge_sizes(ctx):
    rng = np.random.default_rng(3)
    for n, nbar in [(2, 2), (2, 1025), (1024, 1024), (1025, 1023), (3000, 2)]:
        x, xb = rng.normal(size=(n, 2)), rng.normal(0.2, 1.0, size=(nbar, 2))
        assert_T_close(ctx.T(x, xb, 0.7), oracle.T(x, xb, 0.7))


def test_T_device_pointers_match_host_pointers(ctx):
    import torch

    s = dg.make_sample(dg.config(0))
    host = ctx.T(s.x, s.xbar, 0.3)
    dev = ctx.T(torch.from_numpy(s.x).cuda(), torch.from_numpy(s.xbar).cuda(), 0.3)
    assert host.T == dev.T and host.S_xb == dev.S_xb  # deterministic, bit for bit
    again = ctx.T(s.x, s.xbar, 0.3)
    assert again.T == host.T


def test_T_symmetries_on_gpu(ctx):
    rng = np.random.default_rng(5)
    x, xb = rng.normal(size=(700, 3)), rng.normal(0.3, 1.2, size=(900, 3))
    t0 = ctx.T(x, xb, 0.6)
    sw = ctx.T(xb, x, 0.6)
    assert abs(sw.T - t0.T) <= TOL * t0.term_scale and abs(sw.T_xx - t0.T_bb) <= TOL * t0.term_scale
    assert abs(ctx.T(3.7 * x, 3.7 * xb, 3.7 * 0.6).T - t0.T) <= TOL * t0.term_scale
    assert abs(ctx.T(x + 100.0, xb + 100.0, 0.6).T - t0.T) <= TOL * t0.term_scale


def test_T_weighted(ctx):
    c = dg.config(3, scale=0.01)
    s = dg.make_sample(c)
    for sigma in c.sigmas:
        exp = oracle.T(s.x, s.xbar, sigma, s.wx, s.wxbar)
        assert_T_close(ctx.T_weighted(s.x, s.wx, s.xbar, s.wxbar, sigma), exp)
    ones = ctx.T_weighted(s.x, np.ones(c.n), s.xbar, np.ones(c.nbar), 0.3)
    assert ones.T == ctx.T(s.x, s.xbar, 0.3).T  # P11: unit weights are Eq. 2, same kernel, bit for bit


# ----------------------------------------------------------------------------- labels
@pytest.mark.parametrize("N,n,nperm,seed", [(37, 11, 9, 0xE7E57), (4000, 2000, 50, 0xE7E57), (5003, 1, 33, 7),
                                            (2049, 2048, 64, 2**63 + 5), (70001, 35000, 40, 99)])
def test_labels_bit_exact(ctx, N, n, nperm, seed):
    got = ctx.perm_labels(N, n, nperm, seed)
    exp = oracle.labels(N, n, nperm, seed)
    assert got.shape == exp.shape and (got == exp).all()
    bits = ((got[:, :, None] >> np.arange(32, dtype=np.uint32)[None, None, :]) & 1).reshape(N, -1)[:, :nperm]
    assert (bits.sum(0) == n).all()  # P10


@pytest.mark.parametrize("N,n,nperm,seed", [(37, 11, 9, 0xE7E57), (5003, 1, 33, 7), (2049, 2048, 64, 2**63 + 5), (70001, 35000, 40, 99)])
def test_labels_select_fallback_gives_the_same_bits(ctx, N, n, nperm, seed):
    """ET_OPT_LABEL_SELECT = 1: the eight histogram sweeps (the fallback of the candidate-list finish for a key32 bucket of
    more than 64 events, which no input reaches) give the oracle's labels bit for bit too."""
    ctx.set_option(binding.ET_OPT_LABEL_SELECT, 1)
    try:
        got = ctx.perm_labels(N, n, nperm, seed)
    finally:
        ctx.set_option(binding.ET_OPT_LABEL_SELECT, 0)
    assert (got == oracle.labels(N, n, nperm, seed)).all()
    assert (got == ctx.perm_labels(N, n, nperm, seed)).all()


def test_labels_large_sampled(ctx):
    """Config-4 sized label problem: every permutation has exactly n ones; a few permutations against the oracle."""
    N, n, nperm, seed = 2_000_000, 1_000_000, 96, 0xE7E57 + 4
    got = ctx.perm_labels(N, n, nperm, seed)
    for w in range(got.shape[1]):
        bits = (got[:, w, None] >> np.arange(32, dtype=np.uint32)[None, :]) & 1
        assert (bits.sum(0) == n).all()
    for p in (0, 37, 95):
        exp = oracle.labels_range(N, n, p, 1, seed)[0]
        assert (((got[:, p >> 5] >> (p & 31)) & 1) == exp).all()


# ----------------------------------------------------------------------------- row sums
def test_row_sums(ctx):
    c = dg.config(2, scale=0.02)
    s = dg.make_sample(c)
    rows = np.random.default_rng(1).choice(c.n + c.nbar, 64, replace=False)
    rx, rb = ctx.row_sums(s.x, s.xbar, 0.2, rows)
    ex, eb = oracle.row_sums(s.x, s.xbar, 0.2, rows)
    assert np.allclose(rx, ex, rtol=2e-6, atol=1e-9) and np.allclose(rb, eb, rtol=2e-6, atol=1e-9)
    w = dg._rng(5).uniform(-0.5, 1.5, c.n + c.nbar)
    rx, rb = ctx.row_sums(s.x, s.xbar, 0.2, rows, w[: c.n], w[c.n:])
    ex, eb = oracle.row_sums(s.x, s.xbar, 0.2, rows, w[: c.n], w[c.n:])
    assert np.allclose(rx, ex, rtol=2e-6, atol=1e-6) and np.allclose(rb, eb, rtol=2e-6, atol=1e-6)


# ----------------------------------------------------------------------------- permutation test
def check_perm(got, exp, discriminate=True, term_rel=0.0):
    """North-star tolerance, and a bound that still discriminates where 1e-6 of the term scale is
    as wide as the permutation spread itself: the achieved error of every T_p and of T_obs stays below 5 % of the
    standard deviation of the permutation T values."""
    scale = exp.observed.term_scale
    assert_T_close(got.observed, exp.observed, term_rel=term_rel)
    assert np.isnan(got.T_perm).sum() == np.isnan(exp.T_perm).sum()
    ok = np.isfinite(exp.T_perm)
    assert np.abs(got.T_perm[ok] - exp.T_perm[ok]).max() <= TOL * scale
    assert got.nperm == exp.nperm
    if discriminate and ok.sum() >= 8:
        spread = exp.T_perm[ok].std()
        assert np.abs(got.T_perm[ok] - exp.T_perm[ok]).max() <= 0.05 * spread
        assert abs(got.observed.T - exp.observed.T) <= 0.05 * spread
    # p-value exact unless a permutation T sits within the guard band of T_obs (reading R5)
    assert abs(got.count_gt - exp.count_gt) <= got.n_near
    if got.n_near == 0:
        assert got.count_gt == exp.count_gt and got.p_value == exp.p_value


def test_perm_config0_full(ctx):
    c = dg.config(0)
    s = dg.make_sample(c)
    exp = oracle.perm_test(s.x, s.xbar, c.sigma, c.nperm, c.perm_seed)
    got = ctx.permutation_test(s.x, s.xbar, c.sigma, c.nperm, c.perm_seed)
    check_perm(got, exp)
    # same ordering of the permutation T values (the p-value of any threshold is exact)
    assert (np.argsort(got.T_perm) == np.argsort(exp.T_perm)).all()
    assert got.n_near == 0
    # the observed T of the permutation path agrees with et_T to rounding
    assert abs(got.observed.T - ctx.T(s.x, s.xbar, c.sigma).T) <= 1e-8 * exp.observed.term_scale


@pytest.mark.parametrize("n,nbar,dim,nperm", [(300, 500, 5, 70), (1030, 260, 2, 33), (64, 64, 8, 31)])
def test_perm_small_unequal(ctx, n, nbar, dim, nperm):
    rng = np.random.default_rng(n + dim)
    x, xb = rng.uniform(size=(n, dim)), rng.uniform(size=(nbar, dim)) ** 1.2
    sigma = 0.15 * math.sqrt(dim)
    check_perm(ctx.permutation_test(x, xb, sigma, nperm, 12345), oracle.perm_test(x, xb, sigma, nperm, 12345))


def test_perm_offset_is_a_window_of_the_same_stream(ctx):
    """ET_OPT_PERM_OFFSET: permutations p0 .. p0+nperm-1 of the seed's stream (multi-GPU sharding of the loop)."""
    rng = np.random.default_rng(11)
    x, xb = rng.uniform(size=(400, 3)), rng.uniform(size=(350, 3)) ** 1.3
    exp = oracle.perm_test(x, xb, 0.3, 45, 777)
    full = ctx.permutation_test(x, xb, 0.3, 45, 777)
    for p0, cnt in ((13, 32), (4, 7), (44, 1)):
        ctx.set_option(binding.ET_OPT_PERM_OFFSET, p0)
        try:
            got = ctx.permutation_test(x, xb, 0.3, cnt, 777)
            lab = ctx.perm_labels(750, 400, cnt, 777)
        finally:
            ctx.set_option(binding.ET_OPT_PERM_OFFSET, 0)
        assert (got.T_perm == full.T_perm[p0:p0 + cnt]).all()
        assert np.abs(got.T_perm - exp.T_perm[p0:p0 + cnt]).max() <= TOL * exp.observed.term_scale
        ref = oracle.labels_range(750, 400, p0, cnt, 777)  # [cnt, N] bytes
        bits = ((lab[:, :, None] >> np.arange(32, dtype=np.uint32)[None, None, :]) & 1).reshape(750, -1)[:, :cnt]
        assert (bits.T == ref).all()


def test_perm_weighted(ctx):
    c = dg.config(3, scale=0.004)  # 800 + 800 events, weights U[-0.5, 1.5]
    s = dg.make_sample(c)
    exp = oracle.perm_test(s.x, s.xbar, 0.3, 40, c.perm_seed, s.wx, s.wxbar)
    got = ctx.permutation_test(s.x, s.xbar, 0.3, 40, c.perm_seed, s.wx, s.wxbar)
    check_perm(got, exp)


def test_perm_null_sample_is_compatible_with_zero(ctx):
    """identical distributions -> T fluctuates around zero and permutations straddle it."""
    x = dg.dalitz_uniform(3000, dg._rng(1))
    xb = dg.dalitz_uniform(2500, dg._rng(2))
    r = ctx.permutation_test(x, xb, 0.3, 200, 5)
    sd = r.T_perm.std()
    assert abs(r.T_perm.mean()) < 4 * sd / math.sqrt(200)  # P6, statistically
    assert abs(r.observed.T) < 5 * sd
    assert 0.005 < r.p_value < 0.995


# ----------------------------------------------------------------------------- tensor-core permutation sums
class force_kernel:
    """ET_OPT_PERM_KERNEL: 1 = CUDA cores, 2 = tensor cores (tcgen05 kind::i8, 15-bit psi)."""

    def __init__(self, ctx, which):
        self.ctx, self.which = ctx, which

    def __enter__(self):
        self.ctx.set_option(binding.ET_OPT_PERM_KERNEL, self.which)

    def __exit__(self, *exc):
        self.ctx.set_option(binding.ET_OPT_PERM_KERNEL, 0)


@pytest.mark.parametrize("n,nbar,dim,nperm", [(2000, 2000, 2, 50), (2100, 1900, 5, 70), (1500, 2600, 8, 33), (2048, 2048, 3, 600)])
def test_perm_tc_matches_oracle(ctx, n, nbar, dim, nperm):
    """K-PERM-TC (quantised psi, exact integer sums) against the from-scratch oracle; several units per row tile,
    ragged padding, one and two 512-column chunks."""
    rng = np.random.default_rng(n + dim)
    x, xb = rng.uniform(size=(n, dim)), rng.uniform(size=(nbar, dim)) ** 1.15
    sigma = 0.15 * math.sqrt(dim)
    exp = oracle.perm_test(x, xb, sigma, nperm, 4242)
    with force_kernel(ctx, 2):
        got = ctx.permutation_test(x, xb, sigma, nperm, 4242)
        assert ctx.stats().dominant_kernel == "k_perm_tc"
    check_perm(got, exp, term_rel=TERM_REL_TC)
    with force_kernel(ctx, 1):
        cc = ctx.permutation_test(x, xb, sigma, nperm, 4242)
        assert ctx.stats().dominant_kernel in ("k_perm32", "k_pairs_rows")
    assert np.abs(cc.T_perm - got.T_perm).max() <= TOL * exp.observed.term_scale


def test_perm_tc_is_bit_reproducible(ctx):
    """Integer accumulation: the unweighted tensor-core result does not depend on the schedule."""
    s = dg.make_sample(dg.config(0))
    with force_kernel(ctx, 2):
        a = ctx.permutation_test(s.x, s.xbar, 0.3, 50, 7)
        b = ctx.permutation_test(s.x, s.xbar, 0.3, 50, 7)
    assert (a.T_perm == b.T_perm).all() and a.observed.T == b.observed.T


def test_perm_tc_row_order_does_not_change_the_sums(ctx):
    """ET_OPT_TC_ORDER: the contraction runs on a Morton-ordered copy of the records (labels written through the inverse
    map); the unweighted integer sums, hence every T_p, T_obs and the P-even T of the Sect. 5 test, are the same bits in
    the layout order.  5-D four-body sample (both geometries' dims: 5 and 6 by zero-padding a coordinate), P-odd split."""
    c = dg.config(4, scale=0.012)
    s = dg.make_sample(c)
    res = {}
    for order in (1, 0):
        ctx.set_option(binding.ET_OPT_TC_ORDER, order)
        try:
            with force_kernel(ctx, 2):
                res[order] = (ctx.podd_test(s.x, s.mom_x, s.xbar, s.mom_xbar, c.sigma, 40, c.perm_seed),
                              ctx.permutation_test(np.c_[s.x, 0.3 * s.x[:, :1]], np.c_[s.xbar, 0.3 * s.xbar[:, :1]], c.sigma, 520, 7))
                assert ctx.stats().dominant_kernel == "k_perm_tc"
        finally:
            ctx.set_option(binding.ET_OPT_TC_ORDER, 1)
    (pa, ta), (pb, tb) = res[1], res[0]
    assert (pa.p_odd.T_perm == pb.p_odd.T_perm).all() and pa.p_odd.observed == pb.p_odd.observed and pa.p_even == pb.p_even
    assert (ta.T_perm == tb.T_perm).all() and ta.observed == tb.observed and ta.count_gt == tb.count_gt
    # and the sorted run is the oracle's answer (the 6-D sample: 8 permutations from scratch)
    exp = oracle.perm_test(np.c_[s.x, 0.3 * s.x[:, :1]], np.c_[s.xbar, 0.3 * s.xbar[:, :1]], c.sigma, 8, 7)
    assert abs(ta.observed.T - exp.observed.T) <= TOL * exp.observed.term_scale
    assert np.abs(ta.T_perm[:8] - exp.T_perm).max() <= TOL * exp.observed.term_scale


@pytest.mark.parametrize("sigma,nperm", [(0.1, 40), (0.05, 520)])
def test_perm_tc_skipping_far_blocks_does_not_change_the_sums(ctx, sigma, nperm):
    """ET_OPT_TC_SKIP: (row tile, K block) pairs beyond the distance at which the 15-bit psi rounds to 0 are not evaluated.
    Dalitz sample at a small sigma (the plot is many sigma wide): most blocks are skipped, and T_obs and every T_p are the
    same bits as with every block evaluated; the oracle agrees within the tolerance."""
    c = dg.config(1, scale=0.2)
    s = dg.make_sample(c)
    res, evals = {}, {}
    for skip in (1, 0):
        ctx.set_option(binding.ET_OPT_TC_SKIP, skip)
        try:
            with force_kernel(ctx, 2):
                res[skip] = ctx.permutation_test(s.x, s.xbar, sigma, nperm, c.perm_seed)
                st = ctx.stats()
                assert st.dominant_kernel == "k_perm_tc"
                evals[skip] = st.pair_evals
        finally:
            ctx.set_option(binding.ET_OPT_TC_SKIP, 1)
    assert evals[1] < 0.6 * evals[0], evals                       # the skip is in force
    assert (res[1].T_perm == res[0].T_perm).all() and res[1].observed == res[0].observed
    assert (res[1].count_gt, res[1].n_near) == (res[0].count_gt, res[0].n_near)
    exp = oracle.perm_test(s.x, s.xbar, sigma, 4, c.perm_seed)
    assert abs(res[1].observed.T - exp.observed.T) <= TOL * exp.observed.term_scale
    assert np.abs(res[1].T_perm[:4] - exp.T_perm).max() <= TOL * exp.observed.term_scale


def test_perm_tc_weighted(ctx):
    c = dg.config(3, scale=0.012)  # 2400 + 2400 events, weights U[-0.5, 1.5]: signed hi digit
    s = dg.make_sample(c)
    exp = oracle.perm_test(s.x, s.xbar, 0.3, 40, c.perm_seed, s.wx, s.wxbar)
    with force_kernel(ctx, 2):
        got = ctx.permutation_test(s.x, s.xbar, 0.3, 40, c.perm_seed, s.wx, s.wxbar)
    check_perm(got, exp, term_rel=TERM_REL_TC)
    pos = np.abs(s.wx), np.abs(s.wxbar)  # non-negative weights: unsigned hi digit
    exp = oracle.perm_test(s.x, s.xbar, 0.3, 20, 3, *pos)
    with force_kernel(ctx, 2):
        got = ctx.permutation_test(s.x, s.xbar, 0.3, 20, 3, *pos)
    check_perm(got, exp, term_rel=TERM_REL_TC)


def test_perm_tc_default_path_midsize(ctx):
    """N = 40000 pooled (the default dispatch picks the tensor cores); 8 permutations from scratch in the oracle."""
    c = dg.config(1, scale=0.2)
    s = dg.make_sample(c)
    exp = oracle.perm_test(s.x, s.xbar, 0.3, 8, c.perm_seed)
    got = ctx.permutation_test(s.x, s.xbar, 0.3, 8, c.perm_seed)
    assert ctx.stats().dominant_kernel == "k_perm_tc"
    check_perm(got, exp, term_rel=TERM_REL_TC)
    assert abs(got.observed.T - ctx.T(s.x, s.xbar, 0.3).T) <= TOL * exp.observed.term_scale


def test_podd_tc_parity(ctx):
    c = dg.config(4, scale=0.003)  # 3000 + 3000 events
    s = dg.make_sample(c)
    nperm = 40
    with force_kernel(ctx, 2):
        got = ctx.podd_test(s.x, s.mom_x, s.xbar, s.mom_xbar, c.sigma, nperm, c.perm_seed)
    posx, _ = oracle.podd_split(s.mom_x[:, 0], s.mom_x[:, 1], s.mom_x[:, 2], False)
    posb, _ = oracle.podd_split(s.mom_xbar[:, 0], s.mom_xbar[:, 1], s.mom_xbar[:, 2], True)
    I, II, III, IV = s.x[posx == 1], s.x[posx == 0], s.xbar[posb == 1], s.xbar[posb == 0]
    assert got.count == (len(I), len(II), len(III), len(IV))
    exp = oracle.perm_test(np.vstack([I, IV]), np.vstack([II, III]), c.sigma, nperm, c.perm_seed)
    check_perm(got.p_odd, exp, term_rel=TERM_REL_TC)
    assert_T_close(got.p_even, oracle.T(s.x, s.xbar, c.sigma))


# ----------------------------------------------------------------------------- Sect. 5
def test_podd_split_bit_exact(ctx):
    c = dg.config(4, scale=0.02)
    s = dg.make_sample(c)
    for mom, conj in ((s.mom_x, False), (s.mom_xbar, True)):
        B, Cc, D = (np.ascontiguousarray(mom[:, k]) for k in range(3))
        got, gcnt = ctx.podd_split(B, Cc, D, conj)
        exp, ecnt = oracle.podd_split(B, Cc, D, conj)
        assert (got == exp).all() and gcnt == ecnt


def test_podd_test_parity(ctx):
    c = dg.config(4, scale=0.0012)  # 1200 + 1200 events
    s = dg.make_sample(c)
    nperm = 40
    got = ctx.podd_test(s.x, s.mom_x, s.xbar, s.mom_xbar, c.sigma, nperm, c.perm_seed)
    posx, _ = oracle.podd_split(s.mom_x[:, 0], s.mom_x[:, 1], s.mom_x[:, 2], False)
    posb, _ = oracle.podd_split(s.mom_xbar[:, 0], s.mom_xbar[:, 1], s.mom_xbar[:, 2], True)
    I, II, III, IV = s.x[posx == 1], s.x[posx == 0], s.xbar[posb == 1], s.xbar[posb == 0]
    assert got.count == (len(I), len(II), len(III), len(IV))
    A, B = np.vstack([I, IV]), np.vstack([II, III])
    exp = oracle.perm_test(A, B, c.sigma, nperm, c.perm_seed)
    check_perm(got.p_odd, exp)
    assert_T_close(got.p_even, oracle.T(s.x, s.xbar, c.sigma))


# ----------------------------------------------------------------------------- error behaviour
def test_error_codes(ctx):
    x = np.random.default_rng(0).normal(size=(10, 2))
    with pytest.raises(binding.EtError) as e:
        ctx.T(x[:1], x, 0.3)
    assert e.value.status == -1
    with pytest.raises(binding.EtError) as e:
        ctx.T(x, x, 0.0)
    assert e.value.status == -2
    bad = x.copy()
    bad[3, 1] = np.nan
    with pytest.raises(binding.EtError) as e:
        ctx.T(bad, x, 0.3)
    assert e.value.status == -3
    with pytest.raises(binding.EtError) as e:
        ctx.T_weighted(x, np.full(10, 0.05), x, np.ones(10), 0.3)
    assert e.value.status == -4
    with pytest.raises(binding.EtError) as e:
        ctx.T(np.zeros((4, 9)), np.zeros((4, 9)), 0.3)
    assert e.value.status == -1
    # the context is still usable after an error
    assert math.isfinite(ctx.T(x, x + 0.1, 0.3).T)


# ----------------------------------------------------------------------------- BASELINE sizes, sampled
@pytest.mark.parametrize("index", [1, 2, 3, 4])
def test_full_size_row_sum_parity(ctx, index):
    """At BASELINE sizes a full oracle T is too slow; compare per-row class sums on sampled rows."""
    c = dg.config(index)
    s = dg.make_sample(c)
    N = c.n + c.nbar
    rows = np.random.default_rng(index).choice(N, 24, replace=False)
    rx, rb = ctx.row_sums(s.x, s.xbar, c.sigma, rows, s.wx, s.wxbar)
    ex, eb = oracle.row_sums(s.x, s.xbar, c.sigma, rows, s.wx, s.wxbar)
    assert np.allclose(rx, ex, rtol=3e-6, atol=1e-6) and np.allclose(rb, eb, rtol=3e-6, atol=1e-6)


def test_full_size_podd_tc_properties(ctx):
    """BASELINE configs[4] in the launch configuration bench.py times (n = nbar = 10^6, 1000 permutations, tensor-core
    path).  The oracle anchor at this size is test_full_size_golden[4] below (stored oracle values); HERE the split is
    compared with the oracle bit for bit, the observed statistics of both labellings (columns 0 and 1 of K-PERM-TC) with
    the fp32/fp64 all-pairs kernel k_pairs_T on the regrouped samples -- two independent GPU kernels, not an oracle
    comparison -- and the permutation distribution through properties that hold at any size (pin P6: E_perm[T] = 0;
    count = #{T_p > T_obs}; no two permutations alike)."""
    c = dg.config(4)
    s = dg.make_sample(c)
    got = ctx.podd_test(s.x, s.mom_x, s.xbar, s.mom_xbar, c.sigma, c.nperm, c.perm_seed)
    assert ctx.stats().dominant_kernel == "k_perm_tc"
    posx, _ = oracle.podd_split(s.mom_x[:, 0], s.mom_x[:, 1], s.mom_x[:, 2], False)
    posb, _ = oracle.podd_split(s.mom_xbar[:, 0], s.mom_xbar[:, 1], s.mom_xbar[:, 2], True)
    I, II, III, IV = s.x[posx == 1], s.x[posx == 0], s.xbar[posb == 1], s.xbar[posb == 0]
    assert got.count == (len(I), len(II), len(III), len(IV))
    odd = ctx.T(np.vstack([I, IV]), np.vstack([II, III]), c.sigma)
    even = ctx.T(s.x, s.xbar, c.sigma)
    obs = got.p_odd.observed
    for a, b in ((obs, odd), (got.p_even, even)):
        scale = b.term_scale
        assert abs(a.T - b.T) <= TOL * scale
        assert abs(a.T_xx - b.T_xx) <= TOL * scale and abs(a.T_bb - b.T_bb) <= TOL * scale and abs(a.T_xb - b.T_xb) <= TOL * scale
        assert a.W == b.W and a.Wbar == b.Wbar
    Tp = got.p_odd.T_perm
    assert len(Tp) == c.nperm and np.isfinite(Tp).all() and len(np.unique(Tp)) == c.nperm
    assert got.p_odd.count_gt == int((Tp > obs.T).sum()) and got.p_odd.p_value == got.p_odd.count_gt / c.nperm
    assert abs(Tp.mean()) <= 5.0 * Tp.std() / math.sqrt(c.nperm)     # pin P6, statistically
    # the null spread of T scales like 1/N: a wrong normalisation or label count shows up as orders of magnitude
    assert 1e-9 < Tp.std() < 1e-5 and got.p_odd.n_near <= 5


# ----------------------------------------------------------------------------- Eq. 3 (NEXT-1)
def assert_bkg_close(got, exp_T, scale):
    assert abs(got.T - exp_T) <= TOL * scale, (got.T, exp_T)


@pytest.mark.parametrize("scale,dtype", [(1.0, np.float64), (0.05, np.float64), (1.0, np.float32)])
def test_T_bkg_matches_oracle(ctx, scale, dtype):
    """Eq. 3 on inputs with the structure of the paper's Fig. 3 study (4000 signal, 1600 + 1600 background, 3:1
    flavour asymmetry of the background, sigma = 0.25) against the oracle's Eq. 3 written out as printed."""
    x, xb, bx, bb, b, bbar = (a.astype(dtype) if isinstance(a, np.ndarray) else a for a in dg.make_bkg_sample(scale=scale))
    exp = oracle.T_bkg(x, xb, bx, bb, b, bbar, 0.25)
    got = ctx.T_bkg(x, xb, bx, bb, b, bbar, 0.25)
    assert got.w == len(x) - b and got.wbar == len(xb) - bbar
    assert_bkg_close(got, exp, got.term_scale)
    # the subtraction does something here: Eq. 2 on the contaminated main samples is far from Eq. 3
    if scale == 1.0:
        assert abs(ctx.T(x, xb, 0.25).T - got.T) > 100 * TOL * got.term_scale


def test_T_bkg_reductions_and_sums(ctx):
    rng = np.random.default_rng(77)
    x, xb = rng.uniform(size=(700, 3)), rng.uniform(size=(1300, 3)) ** 1.1
    bx, bb = rng.uniform(size=(90, 3)), rng.uniform(size=(2, 3))
    # b = bbar = 0: Eq. 3 is Eq. 2 of the main samples
    z = ctx.T_bkg(x, xb, bx, bb, 0.0, 0.0, 0.3)
    t = ctx.T(x, xb, 0.3)
    assert abs(z.T - t.T) <= TOL * t.term_scale and abs(z.S[0] - t.S_xx) <= 1e-9 * t.S_xx and abs(z.S[2] - t.S_xb) <= 1e-9 * t.S_xb
    # the ten raw sums against the oracle's two-sample sums
    names = {"x": x, "bx": bx, "xb": xb, "bb": bb}
    order = [("x", "x"), ("x", "bx"), ("x", "xb"), ("x", "bb"), ("bx", "bx"), ("bx", "xb"), ("bx", "bb"), ("xb", "xb"), ("xb", "bb"), ("bb", "bb")]
    g = ctx.T_bkg(x, xb, bx, bb, 31.5, 0.25, 0.3)
    for k, (p, q) in enumerate(order):
        o = oracle.T(names[p], names[q], 0.3)
        e = o.S_xx if p == q else o.S_xb
        assert abs(g.S[k] - e) <= 2e-6 * e, (p, q)
    assert abs(g.T - oracle.T_bkg(x, xb, bx, bb, 31.5, 0.25, 0.3)) <= TOL * g.term_scale
    # device pointers
    import torch
    d = [torch.from_numpy(a).cuda() for a in (x, xb, bx, bb)]
    assert ctx.T_bkg(*d, 31.5, 0.25, 0.3).T == g.T


def test_T_bkg_errors(ctx):
    a = np.random.default_rng(1).uniform(size=(10, 2))
    with pytest.raises(binding.EtError) as e:
        ctx.T_bkg(a, a, a[:1], a, 1.0, 1.0, 0.3)
    assert e.value.status == -1
    with pytest.raises(binding.EtError) as e:
        ctx.T_bkg(a, a, a, a, -1.0, 1.0, 0.3)
    assert e.value.status == -1
    with pytest.raises(binding.EtError) as e:
        ctx.T_bkg(a, a, a, a, 9.5, 1.0, 0.3)
    assert e.value.status == -4


def test_full_size_config1_permutations_from_scratch(ctx):
    """BASELINE configs[1] at full size (n = nbar = 100 000, fp32 coordinates, sigma = 0.3), default dispatch (tensor
    cores): the observed T and the first eight permutations against the oracle, each re-evaluated from scratch
    (9 x 2e10 psi in fp64, about 100 s on 16 host cores); labels of those permutations bit for bit."""
    c = dg.config(1)
    s = dg.make_sample(c)
    assert s.x.dtype == np.float32
    nperm = 8
    exp = oracle.perm_test(s.x, s.xbar, 0.3, nperm, c.perm_seed)
    got = ctx.permutation_test(s.x, s.xbar, 0.3, nperm, c.perm_seed)
    assert ctx.stats().dominant_kernel == "k_perm_tc"
    check_perm(got, exp, term_rel=TERM_REL_TC)
    N = c.n + c.nbar
    assert (ctx.perm_labels(N, c.n, nperm, c.perm_seed) == oracle.labels(N, c.n, nperm, c.perm_seed)).all()


# ----------------------------------------------------------------------------- sigma scan in one pass (NEXT-3)
@pytest.mark.parametrize("dim,sigmas", [(2, (0.1, 0.3, 0.5)), (5, (0.2, 0.1)), (3, (0.5, 0.25, 1.0, 0.125)), (2, (0.3,))])
def test_T_sigmas_matches_oracle(ctx, dim, sigmas):
    """BASELINE configs[1] evaluates sigma in {0.1, 0.3, 0.5} on the same samples: one pass, one distance per pair."""
    if dim == 2:
        s = dg.make_sample(dg.config(1, scale=0.04))  # 4000 + 4000 events, fp32 coordinates
        x, xb = s.x, s.xbar
    else:
        rng = np.random.default_rng(dim)
        x, xb = rng.uniform(size=(1500, dim)), rng.uniform(size=(2100, dim)) ** 1.2
    got = ctx.T_sigmas(x, xb, sigmas)
    assert len(got) == len(sigmas)
    for g, sg in zip(got, sigmas):
        assert_T_close(g, oracle.T(x, xb, sg))
        one = ctx.T(x, xb, sg)
        assert abs(g.T - one.T) <= TOL * one.term_scale


def test_T_sigmas_weighted_and_errors(ctx):
    c = dg.config(3, scale=0.01)
    s = dg.make_sample(c)
    got = ctx.T_sigmas(s.x, s.xbar, (0.3, 0.5, 0.1), s.wx, s.wxbar)
    for g, sg in zip(got, (0.3, 0.5, 0.1)):
        assert_T_close(g, oracle.T(s.x, s.xbar, sg, s.wx, s.wxbar))
    with pytest.raises(binding.EtError) as e:
        ctx.T_sigmas(s.x, s.xbar, (0.3, -1.0))
    assert e.value.status == -2
    with pytest.raises(binding.EtError) as e:
        ctx.T_sigmas(s.x, s.xbar, (0.3, 0.2, 0.1, 0.4, 0.5))
    assert e.value.status == -1
    with pytest.raises(binding.EtError) as e:
        ctx.T_sigmas(s.x, s.xbar, (1e-9, 1e3))
    assert e.value.status == -2


@pytest.mark.parametrize("n,nbar,nperm", [(2, 3, 7), (300, 340, 1), (300, 340, 509), (300, 340, 510), (257, 1023, 1019)])
def test_perm_tc_chunk_and_size_edges(ctx, n, nbar, nperm):
    """Tensor-core path forced at its edges: the smallest samples, one permutation, and permutation counts on both
    sides of the 509-per-launch boundary (1, 2 and 3 launches of 512 label columns).  Below the default dispatch
    threshold (8192 rows) the 15-bit quantisation noise of psi does not average out: the bound used here is 8 sigma of
    DESIGN.md section 6, var(T) = (1/12) q^2 [1/(2n(n-1)) + 1/(2nbar(nbar-1)) + 1/(n nbar)] with q = 1 / 32766, or the
    north-star tolerance if that is larger."""
    rng = np.random.default_rng(n * 1000 + nperm)
    x, xb = rng.normal(size=(n, 4)), rng.normal(size=(nbar, 4)) * 1.1 + 0.05
    exp = oracle.perm_test(x, xb, 0.8, nperm, 99)
    with force_kernel(ctx, 2):
        got = ctx.permutation_test(x, xb, 0.8, nperm, 99)
        assert ctx.stats().dominant_kernel == "k_perm_tc"
    var = (1.0 / 12.0) / 32766.0 ** 2 * (0.5 / (n * (n - 1.0)) + 0.5 / (nbar * (nbar - 1.0)) + 1.0 / (n * nbar))
    bound = max(TOL * exp.observed.term_scale, 8.0 * math.sqrt(var))
    assert abs(got.observed.T - exp.observed.T) <= bound
    assert np.abs(got.T_perm - exp.T_perm).max() <= bound and got.nperm == nperm
    assert abs(got.count_gt - exp.count_gt) <= got.n_near


@pytest.mark.parametrize("dim", [1, 4, 6, 7])
def test_perm_tc_remaining_dims(ctx, dim):
    """Every pair-record width of K-PERM-TC (1 to 5 float4 per j pair): dims not covered by test_perm_tc_matches_oracle."""
    rng = np.random.default_rng(40 + dim)
    x, xb = rng.uniform(size=(1100, dim)), rng.uniform(size=(1300, dim)) ** 1.3
    sigma = 0.2 * math.sqrt(dim)
    exp = oracle.perm_test(x, xb, sigma, 20, 5)
    with force_kernel(ctx, 2):
        got = ctx.permutation_test(x, xb, sigma, 20, 5)
        assert ctx.stats().dominant_kernel == "k_perm_tc"
    check_perm(got, exp, term_rel=TERM_REL_TC)


def test_perm_tc_bit_reproducible_many_units(ctx):
    """N = 60 000 pooled events through the default dispatch: hundreds of work units over all 74 clusters, two launches.
    Integer accumulation and fixed-order reductions: two calls agree bit for bit, and a second context does too."""
    c = dg.config(2, scale=0.1)
    s = dg.make_sample(c)
    a = ctx.permutation_test(s.x, s.xbar, c.sigma, 600, 11)
    assert ctx.stats().dominant_kernel == "k_perm_tc"
    b = ctx.permutation_test(s.x, s.xbar, c.sigma, 600, 11)
    assert (a.T_perm == b.T_perm).all() and a.observed.T == b.observed.T and a.count_gt == b.count_gt
    with binding.Context(0) as other:
        d = other.permutation_test(s.x, s.xbar, c.sigma, 600, 11)
    assert (a.T_perm == d.T_perm).all() and a.observed.T == d.observed.T
    assert abs(a.observed.T - ctx.T(s.x, s.xbar, c.sigma).T) <= TOL * a.observed.term_scale


# ----------------------------------------------------------------------------- Eq. 3 permutation test (NEXT-1, R18)
def test_bkg_permutation_test_matches_oracle(ctx):
    """Fig. 3-structured inputs at a tenth of the paper's size: every permutation T of Eq. 3 against the oracle's
    from-scratch re-evaluation (both pools permuted with the shared Philox label rule)."""
    x, xb, bx, bb, b, bbar = dg.make_bkg_sample(scale=0.1)
    nperm = 40
    t_obs, t_perm, count, p = oracle.bkg_perm_test(x, xb, bx, bb, b, bbar, 0.25, nperm, 4711)
    got = ctx.bkg_permutation_test(x, xb, bx, bb, b, bbar, 0.25, nperm, 4711)
    scale = got.observed.term_scale
    assert abs(got.observed.T - t_obs) <= TOL * scale
    assert np.abs(got.T_perm - t_perm).max() <= TOL * scale
    assert abs(got.count_gt - count) <= got.n_near and got.nperm == nperm
    if got.n_near == 0:
        assert got.p_value == p
    # same permutation order of the T values
    assert (np.argsort(got.T_perm) == np.argsort(t_perm)).all()


def test_bkg_permutation_test_reduces_to_eq2_and_windows(ctx):
    rng = np.random.default_rng(90)
    x, xb = rng.uniform(size=(900, 3)), rng.uniform(size=(1200, 3)) ** 1.1
    bx, bb = rng.uniform(size=(1030, 3)), rng.uniform(size=(17, 3))
    # b = bbar = 0: the permutation T values of Eq. 3 are those of Eq. 2 on the main samples (same label stream)
    z = ctx.bkg_permutation_test(x, xb, bx, bb, 0.0, 0.0, 0.3, 24, 5)
    with force_kernel(ctx, 1):
        ref = ctx.permutation_test(x, xb, 0.3, 24, 5)
    assert np.abs(z.T_perm - ref.T_perm).max() <= TOL * ref.observed.term_scale and z.count_gt == ref.count_gt
    # ET_OPT_PERM_OFFSET: a window of the same stream
    full = ctx.bkg_permutation_test(x, xb, bx, bb, 40.0, 10.0, 0.3, 12, 5)
    try:
        ctx.set_option(binding.ET_OPT_PERM_OFFSET, 5)
        win = ctx.bkg_permutation_test(x, xb, bx, bb, 40.0, 10.0, 0.3, 7, 5)
    finally:
        ctx.set_option(binding.ET_OPT_PERM_OFFSET, 0)
    assert (win.T_perm == full.T_perm[5:12]).all() and win.observed.T == full.observed.T
    with pytest.raises(binding.EtError) as e:
        ctx.bkg_permutation_test(x, xb, bx, bb, 899.5, 0.0, 0.3, 4, 5)
    assert e.value.status == -4


def test_full_size_config3_weighted_tc_properties(ctx):
    """BASELINE configs[3] at full size (n = nbar = 200 000, signed per-event weights, 1000 permutations): the weighted
    tensor-core path (signed hi digit, fp64 epilogue) against the weighted all-pairs kernel for the observed statistic,
    and the permutation distribution through properties (count consistency, distinct values, W_p recomputed)."""
    c = dg.config(3)
    s = dg.make_sample(c)
    got = ctx.permutation_test(s.x, s.xbar, c.sigma, c.nperm, c.perm_seed, s.wx, s.wxbar)
    assert ctx.stats().dominant_kernel == "k_perm_tc"
    ref = ctx.T_weighted(s.x, s.wx, s.xbar, s.wxbar, c.sigma)
    scale = ref.term_scale
    o = got.observed
    assert_T_close(o, ref, term_rel=TERM_REL_TC)
    assert abs(o.T - ref.T) <= 0.05 * got.T_perm.std()
    assert o.W == pytest.approx(ref.W, rel=1e-12) and o.Wbar == pytest.approx(ref.Wbar, rel=1e-12)
    assert o.W == pytest.approx(float(np.float32(s.wx).astype(np.float64).sum()), rel=1e-9)   # weights enter as fp32
    Tp = got.T_perm
    assert np.isfinite(Tp).all() and len(np.unique(Tp)) == c.nperm
    assert got.count_gt == int((Tp > o.T).sum()) and got.p_value == got.count_gt / c.nperm
    assert 1e-8 < Tp.std() < 1e-4


@pytest.mark.parametrize("dim", [2, 6])
def test_perm_tc_accumulator_headroom_coincident_points(ctx, dim):
    """The largest values the int32 TMEM accumulators can see: 260 000 coincident events, psi = 1 for every pair, so
    every work unit of the first row tiles runs the longest unit its geometry allows with all digits at their maximum --
    dim = 2 (Geo<128, 16, 2>, et_tc.cuh): |Y| = 32767 x 128 x 512 = 2 147 418 112, dim = 6 (Geo<96, 12, 3>): 32767 x 96 x
    660 = 2 076 117 120, of 2^31 = 2 147 483 648 (run_perm_tc caps the units there from N = 2.4e5 on, which is every
    config-2/3/4 launch).  300 permutations: both 256-column accumulators.  Pin P1 at scale: T = 1/2 + 1/2 - 1 = 0 for the
    observed and for every permutation; the raw sums are the pair counts."""
    n = nbar = 130000
    x, xb = np.full((n, dim), 0.25), np.full((nbar, dim), 0.25)
    got = ctx.permutation_test(x, xb, 0.3, 300, 3)
    assert ctx.stats().dominant_kernel == "k_perm_tc"
    o = got.observed
    assert o.S_xx == pytest.approx(n * (n - 1) / 2, rel=1e-15) and o.S_bb == pytest.approx(nbar * (nbar - 1) / 2, rel=1e-15)
    assert o.S_xb == pytest.approx(n * nbar, rel=1e-15)
    assert abs(o.T) <= 1e-15 and np.abs(got.T_perm).max() <= 1e-15
    # ties everywhere: every permutation is inside the guard band and stays undecided
    assert got.n_near == 300


# ----------------------------------------------------------------------------- sigma scan of the permutation test
@pytest.mark.parametrize("sigma", [0.1, 0.5])
@pytest.mark.parametrize("kernel", [0, 1])
def test_perm_sigma_scan_values(ctx, sigma, kernel):
    """BASELINE configs[1] / [3] quote sigma in {0.1, 0.3, 0.5}: the permutation path at the two outer values (config 1
    at a fifth of its size, fp32 coordinates, 8 permutations from scratch in the oracle), default dispatch (tensor cores)
    and CUDA cores.  At sigma = 0.1 most psi underflow or round to 0 on the 15-bit grid."""
    c = dg.config(1, scale=0.2)
    s = dg.make_sample(c)
    exp = oracle.perm_test(s.x, s.xbar, sigma, 8, c.perm_seed)
    with force_kernel(ctx, kernel):
        got = ctx.permutation_test(s.x, s.xbar, sigma, 8, c.perm_seed)
        assert ctx.stats().dominant_kernel == ("k_perm_tc" if kernel == 0 else "k_perm32")
    check_perm(got, exp, term_rel=TERM_REL_TC if kernel == 0 else 0.0)
    assert (np.argsort(got.T_perm) == np.argsort(exp.T_perm)).all()


@pytest.mark.parametrize("kernel", [0, 1])
@pytest.mark.parametrize("weighted", [False, True])
def test_permutation_test_sigmas_is_the_scan_of_single_calls(ctx, kernel, weighted):
    """et_permutation_test_sigmas (Fig. 2: p-value versus sigma; BASELINE configs[1] / [3]: three sigma x the
    same permutations): every sigma equals its own et_permutation_test call bit for bit (labels generated once, records
    re-scaled per sigma), and the oracle within the tolerance (8 permutations from scratch per sigma)."""
    c = dg.config(3 if weighted else 1, scale=0.1)
    s = dg.make_sample(c)
    sig = (0.1, 0.3, 0.5)
    with force_kernel(ctx, kernel):
        scan = ctx.permutation_test_sigmas(s.x, s.xbar, sig, 8, c.perm_seed, s.wx, s.wxbar)
        assert len(scan) == 3
        for sg, got in zip(sig, scan):
            one = ctx.permutation_test(s.x, s.xbar, sg, 8, c.perm_seed, s.wx, s.wxbar)
            # CUDA-core path with one mask word: the row sums (k_pairs_rows) outweigh the one k_perm32 launch
            assert ctx.stats().dominant_kernel in (("k_perm_tc",) if kernel == 0 else ("k_perm32", "k_pairs_rows"))
            assert (got.T_perm == one.T_perm).all() and got.observed == one.observed
            assert (got.count_gt, got.n_near, got.p_value) == (one.count_gt, one.n_near, one.p_value)
            exp = oracle.perm_test(s.x, s.xbar, sg, 8, c.perm_seed, s.wx, s.wxbar)
            check_perm(got, exp, term_rel=TERM_REL_TC * (4 if weighted else 1) if kernel == 0 else 0.0)
    # the scan sees the injected asymmetry differently at each sigma: three distinct observed T values
    assert len({r.observed.T for r in scan}) == 3


def test_permutation_test_sigmas_errors(ctx):
    rng = np.random.default_rng(5)
    x, xb = rng.uniform(size=(300, 2)), rng.uniform(size=(200, 2))
    with pytest.raises(binding.EtError) as e:
        ctx.permutation_test_sigmas(x, xb, (0.3, -1.0), 4, 1)
    assert e.value.status == -2
    with pytest.raises(binding.EtError) as e:
        ctx.permutation_test_sigmas(x, xb, [0.1] * 17, 4, 1)
    assert e.value.status == -1
    one = ctx.permutation_test_sigmas(x, xb, (0.25,), 40, 9)[0]
    ref = ctx.permutation_test(x, xb, 0.25, 40, 9)
    assert (one.T_perm == ref.T_perm).all() and one.count_gt == ref.count_gt


# ----------------------------------------------------------------------------- oracle anchor at the bench sizes
def _golden():
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "fullsize_T.txt")
    out = {}
    with open(path) as f:
        for line in f:
            if line.startswith("#") or "=" not in line:
                continue
            k, v = line.split("=", 1)
            out[k.strip()] = float.fromhex(v.split("|")[1].strip())
    return out


def _golden_result(g, prefix, n_pairs):
    return binding.Result(*(g[f"{prefix}.{k}"] for k in ("T", "T_xx", "T_bb", "T_xb", "S_xx", "S_bb", "S_xb", "W", "Wbar")), n_pairs)


@pytest.mark.parametrize("index", [2, 3, 4])
def test_full_size_golden(ctx, index):
    """BASELINE configs[2], [3], [4] at full size, in the launch configuration bench.py times (all 1000 permutations,
    default dispatch = K-PERM-TC), against oracle values stored in tests/golden/fullsize_T.txt (written by
    tests/golden/make_fullsize_golden.py from oracle + datagen alone: the observed statistic with its three terms and the
    first permutation T values, each a from-scratch fp64 pass; config 4 also the P-even grouping).  et_T (k_pairs_T) is
    compared with the same values.  Beside the north-star tolerance -- which at these sizes is as wide as the
    permutation spread -- the achieved errors must stay below 5 % of the spread of the permutation T values."""
    g = _golden()
    c = dg.config(index)
    tag = f"cfg{index}"
    if f"{tag}.obs.T" not in g:
        pytest.skip(f"{tag} is not in tests/golden/fullsize_T.txt yet (run tests/golden/make_fullsize_golden.py)")
    s = dg.make_sample(c)
    N = c.n + c.nbar
    exp = _golden_result(g, f"{tag}.obs", N * (N - 1) // 2)
    if c.podd:
        r = ctx.podd_test(s.x, s.mom_x, s.xbar, s.mom_xbar, c.sigma, c.nperm, c.perm_seed)
        assert tuple(float(v) for v in r.count) == tuple(g[f"{tag}.count.{k}"] for k in ("I", "II", "III", "IV"))
        got, even = r.p_odd, r.p_even
    else:
        got, even = ctx.permutation_test(s.x, s.xbar, c.sigma, c.nperm, c.perm_seed, s.wx, s.wxbar), None
    st = ctx.stats()
    assert st.dominant_kernel == "k_perm_tc"
    spread = got.T_perm.std()
    scale = exp.term_scale
    o = got.observed
    assert_T_close(o, exp, term_rel=TERM_REL_TC)
    assert abs(o.T - exp.T) <= 0.05 * spread, (o.T, exp.T, spread)
    # weights enter the kernels as fp32 values: W agrees to fp32 rounding of the individual weights
    assert o.W == pytest.approx(exp.W, rel=1e-7 if c.weighted else 1e-15) and o.Wbar == pytest.approx(exp.Wbar, rel=1e-7 if c.weighted else 1e-15)
    errs = [abs(o.T - exp.T)]
    k = 0
    while f"{tag}.perm.{k}" in g:
        e = abs(got.T_perm[k] - g[f"{tag}.perm.{k}"])
        assert e <= TOL * scale and e <= 0.05 * spread, (k, got.T_perm[k], g[f"{tag}.perm.{k}"], spread)
        # the side of T_obs each of these permutations falls on is the oracle's
        assert (got.T_perm[k] > o.T) == (g[f"{tag}.perm.{k}"] > exp.T)
        errs.append(e)
        k += 1
    assert k >= 1
    if even is not None:
        ev = _golden_result(g, f"{tag}.even", N * (N - 1) // 2)
        assert abs(even.T - ev.T) <= TOL * ev.term_scale and abs(even.T - ev.T) <= 0.05 * spread
        assert abs(even.T_xx - ev.T_xx) <= TOL * ev.term_scale and abs(even.T_xb - ev.T_xb) <= TOL * ev.term_scale
        errs.append(abs(even.T - ev.T))
    # k_pairs_T at the same size against the same stored values
    if c.podd:
        posx, _ = oracle.podd_split(s.mom_x[:, 0], s.mom_x[:, 1], s.mom_x[:, 2], False)
        posb, _ = oracle.podd_split(s.mom_xbar[:, 0], s.mom_xbar[:, 1], s.mom_xbar[:, 2], True)
        A = np.vstack([s.x[posx == 1], s.xbar[posb == 0]])
        B = np.vstack([s.x[posx == 0], s.xbar[posb == 1]])
        t = ctx.T(A, B, c.sigma)
    elif c.weighted:
        t = ctx.T_weighted(s.x, s.wx, s.xbar, s.wxbar, c.sigma)
    else:
        t = ctx.T(s.x, s.xbar, c.sigma)
    assert abs(t.T - exp.T) <= TOL * scale and abs(t.T - exp.T) <= 0.05 * spread
    for k in ("T_xx", "T_bb", "T_xb"):
        assert abs(getattr(t, k) - getattr(exp, k)) <= TOL * scale, k
    print(f"\n[golden cfg{index}] spread {spread:.3e}; |dT| tensor-core path: " + ", ".join(f"{e:.2e}" for e in errs) +
          f"; et_T {abs(t.T - exp.T):.2e}; n_near {st.n_near_before} -> {got.n_near}, escalation {st.ms_escalation:.1f} ms")


def test_full_size_config4_p_even_golden(ctx):
    """BASELINE configs[4] at full size (n = nbar = 10^6, 5-D), the launch bench.py times: the P-even statistic (I+II) vs
    (III+IV) = Eq. 2 of (X, Xbar) -- column 1 of K-PERM-TC -- and et_T (k_pairs_T, Gram form at this size)
    against the oracle's stored value (tests/golden/fullsize_T.txt, cfg4.even.*: one 2.0e12-pair fp64 pass, 97 minutes on 7
    host cores), at the north-star tolerance and at 5 % of the permutation spread."""
    g = _golden()
    if "cfg4.even.T" not in g:
        pytest.skip("cfg4.even is not in tests/golden/fullsize_T.txt yet")
    c = dg.config(4)
    s = dg.make_sample(c)
    N = c.n + c.nbar
    ev = _golden_result(g, "cfg4.even", N * (N - 1) // 2)
    r = ctx.podd_test(s.x, s.mom_x, s.xbar, s.mom_xbar, c.sigma, c.nperm, c.perm_seed)
    assert ctx.stats().dominant_kernel == "k_perm_tc"
    assert tuple(float(v) for v in r.count) == tuple(g[f"cfg4.count.{k}"] for k in ("I", "II", "III", "IV"))
    spread = r.p_odd.T_perm.std()
    assert_T_close(r.p_even, ev, term_rel=TERM_REL_TC)
    assert abs(r.p_even.T - ev.T) <= 0.05 * spread, (r.p_even.T, ev.T, spread)
    t = ctx.T(s.x, s.xbar, c.sigma)
    assert ctx.stats().distance_form == 2
    assert_T_close(t, ev)
    assert abs(t.T - ev.T) <= 0.05 * spread
    print(f"\n[golden cfg4.even] spread {spread:.3e}; |dT| tensor-core column 1 {abs(r.p_even.T - ev.T):.2e}, et_T {abs(t.T - ev.T):.2e} "
          f"(= {abs(t.T - ev.T) / ev.term_scale:.1e} of the term scale)")


# ----------------------------------------------------------------------------- exact p-values (guard-band escalation)
def test_escalation_restores_the_oracle_count(ctx):
    """p is the fraction of permutation T values greater than the observed one, and north_star wants it
    equal to the oracle's.  Tiny samples and the largest permutation count make the 15-bit rounding noise of the
    tensor-core path matter: with 65 536 permutations about one of them falls on the wrong side of T_obs, and ten or so
    inside the guard band.  Without the escalation (ET_OPT_EXACT_P = 0) the count differs from the oracle's for at
    least one of the seeds below and the difference is covered by n_near; with it (the near permutations re-evaluated
    in the fp32-pair / fp64-sum arithmetic) the count is the oracle's whenever nothing is left inside the fp32 band."""
    rng = np.random.default_rng(2024)
    x, xb = rng.uniform(size=(40, 3)), rng.uniform(size=(50, 3)) ** 1.2
    nperm, flipped_before = 65536, 0
    for seed in range(1, 9):
        exp = oracle.perm_test(x, xb, 0.3, nperm, seed)
        with force_kernel(ctx, 2):
            ctx.set_option(binding.ET_OPT_EXACT_P, 0)
            try:
                raw = ctx.permutation_test(x, xb, 0.3, nperm, seed)
            finally:
                ctx.set_option(binding.ET_OPT_EXACT_P, 64)
            try:
                got = ctx.permutation_test(x, xb, 0.3, nperm, seed)
                st = ctx.stats()
            finally:
                ctx.set_option(binding.ET_OPT_EXACT_P, 16)
        assert abs(raw.count_gt - exp.count_gt) <= raw.n_near and raw.n_near > 0
        assert st.n_near_before == raw.n_near and st.n_escalated == raw.n_near and st.ms_escalation > 0
        assert got.n_near < raw.n_near
        assert abs(got.count_gt - exp.count_gt) <= got.n_near
        assert got.count_gt == int((got.T_perm > got.observed.T).sum()) and got.observed.T == raw.observed.T
        # only the escalated permutations moved, and by less than the band
        moved = np.flatnonzero(got.T_perm != raw.T_perm)
        assert len(moved) <= raw.n_near and np.abs(got.T_perm - raw.T_perm).max() < 1e-5
        # the re-evaluated differences T_p - T_obs are the oracle's to fp32-path accuracy
        assert np.abs((got.T_perm[moved] - got.observed.T) - (exp.T_perm[moved] - exp.observed.T)).max() < 2e-7
        if got.n_near == 0:
            assert got.count_gt == exp.count_gt and got.p_value == exp.p_value
        if raw.count_gt != exp.count_gt:
            flipped_before += 1
            assert got.count_gt == exp.count_gt or got.n_near > 0
    assert flipped_before >= 1, "no seed showed a count that the escalation had to repair"


def test_escalation_weighted_and_podd(ctx):
    """The escalation on the weighted path (all ten class-pair sums, W_p recomputed) and on the four-class layout of
    the Sect. 5 test, forced tensor cores on small samples with many permutations."""
    c = dg.config(3, scale=0.0005)  # 100 + 100 events
    s = dg.make_sample(c)
    exp = oracle.perm_test(s.x, s.xbar, 0.3, 20000, 5, s.wx, s.wxbar)
    with force_kernel(ctx, 2):
        ctx.set_option(binding.ET_OPT_EXACT_P, 64)
        try:
            got = ctx.permutation_test(s.x, s.xbar, 0.3, 20000, 5, s.wx, s.wxbar)
            st = ctx.stats()
        finally:
            ctx.set_option(binding.ET_OPT_EXACT_P, 16)
    assert st.n_near_before > 0 and (st.n_escalated == st.n_near_before or st.n_escalated == 0)
    assert abs(got.count_gt - exp.count_gt) <= got.n_near
    if got.n_near == 0:
        assert got.count_gt == exp.count_gt
    c = dg.config(4, scale=0.0001)  # 100 + 100 events
    s = dg.make_sample(c)
    posx, _ = oracle.podd_split(s.mom_x[:, 0], s.mom_x[:, 1], s.mom_x[:, 2], False)
    posb, _ = oracle.podd_split(s.mom_xbar[:, 0], s.mom_xbar[:, 1], s.mom_xbar[:, 2], True)
    A = np.vstack([s.x[posx == 1], s.xbar[posb == 0]])
    B = np.vstack([s.x[posx == 0], s.xbar[posb == 1]])
    exp = oracle.perm_test(A, B, c.sigma, 30000, 9)
    with force_kernel(ctx, 2):
        ctx.set_option(binding.ET_OPT_EXACT_P, 64)
        try:
            got = ctx.podd_test(s.x, s.mom_x, s.xbar, s.mom_xbar, c.sigma, 30000, 9).p_odd
            st = ctx.stats()
        finally:
            ctx.set_option(binding.ET_OPT_EXACT_P, 16)
    assert st.n_near_before > 0
    assert abs(got.count_gt - exp.count_gt) <= got.n_near
    if got.n_near == 0:
        assert got.count_gt == exp.count_gt and got.p_value == exp.p_value


def test_escalation_through_the_gram_form(ctx):
    """dim = 5 and >= 4096 events: the escalation's k_pairs_T pass runs in the Gram form (default rule) and its guard band
    carries the form's rounding term.  Forced tensor cores at n = nbar = 3000 with 3000 permutations put a few of them
    inside the 15-bit band; after the escalation the count is the oracle's unless something stays inside the fp32 band."""
    c = dg.config(2, scale=0.01)
    s = dg.make_sample(c)
    nperm = 3000
    exp = oracle.perm_test(s.x, s.xbar, c.sigma, nperm, 77)
    with force_kernel(ctx, 2):
        ctx.set_option(binding.ET_OPT_EXACT_P, 64)
        try:
            got = ctx.permutation_test(s.x, s.xbar, c.sigma, nperm, 77)
            st = ctx.stats()
        finally:
            ctx.set_option(binding.ET_OPT_EXACT_P, 16)
    assert st.dominant_kernel == "k_perm_tc" and st.distance_form == 2
    assert st.n_near_before > 0 and st.n_escalated == st.n_near_before
    assert abs(got.count_gt - exp.count_gt) <= got.n_near
    if got.n_near == 0:
        assert got.count_gt == exp.count_gt and got.p_value == exp.p_value
    # the re-evaluated differences are the oracle's to the accuracy of the escalation's arithmetic
    d_got, d_exp = got.T_perm - got.observed.T, exp.T_perm - exp.observed.T
    near = np.argsort(np.abs(d_exp))[: int(st.n_escalated)]
    assert np.abs(d_got[near] - d_exp[near]).max() <= 5e-9   # 4 sigma of the band's model at n = 3000 (1.3e-9)


# ----------------------------------------------------------------------------- the error model behind the guard band
@pytest.mark.parametrize("kernel", [1, 2])
@pytest.mark.parametrize("index,scale,sigma", [(1, 0.2, 0.3), (1, 0.2, 0.1), (2, 0.1, 0.2)])
def test_error_model_of_the_decision(ctx, kernel, index, scale, sigma):
    """the guard band is 8 sigma of T_p - T_obs under the model 'every pair carries an independent
    error' -- 2^-22 of the fp32 psi and step / sqrt(12) of the rounding of w_j psi_ij to the path's grid.  Measured against
    the oracle over 24 permutations (n = nbar = 20 000 and 30 000): the errors of T_p, of T_obs and of T_p - T_obs stay
    within the model -- rms below 1.5, maximum below 5 model sigmas, and no common offset of the T_p against T_obs (the
    fp32 partial sums of the CUDA-core path had one of 10 .. 30 sigma before kFlushJ, et_device.cuh)."""
    c = dg.config(index, scale=scale)
    s = dg.make_sample(c)
    n, nbar, nperm = c.n, c.nbar, 24
    exp = oracle.perm_test(s.x, s.xbar, sigma, nperm, c.perm_seed)
    ctx.set_option(binding.ET_OPT_EXACT_P, 0)
    try:
        with force_kernel(ctx, kernel):
            got = ctx.permutation_test(s.x, s.xbar, sigma, nperm, c.perm_seed)
            assert ctx.stats().dominant_kernel in (("k_perm_tc",) if kernel == 2 else ("k_perm32", "k_pairs_rows"))
    finally:
        ctx.set_option(binding.ET_OPT_EXACT_P, 16)
    # rounding step of w_j psi_ij: 1 / 32766 on the tensor-core path, 2^-19 on the CUDA-core path (grid_term: unit weights,
    # fp32 partial sums of 32 terms)
    step = 1 / 32766.0 if kernel == 2 else 2.0 ** -19
    pair_err = math.sqrt(step ** 2 / 12 + (2.0 ** -22) ** 2)
    var = 1 / (2.0 * n * (n - 1)) + 1 / (2.0 * nbar * (nbar - 1)) + 1.0 / (n * nbar)
    sig = pair_err * math.sqrt(var)                       # model sigma of one T
    e_p, e_o = got.T_perm - exp.T_perm, got.observed.T - exp.observed.T
    e_d = (e_p - e_o) / math.sqrt(2.0)                    # T_p - T_obs, in units of ITS model sigma
    report = (math.sqrt((e_p ** 2).mean()) / sig, e_p.mean() / sig, e_o / sig, math.sqrt((e_d ** 2).mean()) / sig)
    assert math.sqrt((e_p ** 2).mean()) <= 1.5 * sig and np.abs(e_p).max() <= 5.0 * sig, report
    assert abs(e_o) <= 5.0 * sig, report
    assert math.sqrt((e_d ** 2).mean()) <= 1.5 * sig and np.abs(e_d).max() <= 5.0 * sig, report
    assert abs(e_p.mean()) <= 5.0 * sig / math.sqrt(nperm) + 0.5 * sig, report


# ----------------------------------------------------------------------------- unit-range shard
def _run_sharded(world, call, exact_p=16):
    """`world` contexts on this GPU, one host thread each, in lock step: the all-gather callback of et_set_shard is a
    host-side rendezvous of the threads (no kernel waits for another).  Returns the ranks' results."""
    import ctypes
    import threading

    bar = threading.Barrier(world)
    box = {}
    results, errors = [None] * world, []

    def make_cb(rank):
        def fn(_user, buf, nbytes):
            mine = ctypes.string_at(buf + rank * nbytes, nbytes)
            box[rank] = mine
            bar.wait()
            for r in range(world):
                ctypes.memmove(buf + r * nbytes, box[r], nbytes)
            bar.wait()
            return 0
        return binding._ALLGATHER(fn)

    def worker(rank):
        try:
            with binding.Context(0) as c:
                cb = make_cb(rank)
                c._check(binding.lib().et_set_shard(c._h, rank, world, ctypes.cast(cb, ctypes.c_void_p), None))
                c.set_option(binding.ET_OPT_EXACT_P, exact_p)
                results[rank] = call(c)
        except Exception as exc:  # release the other threads
            errors.append(exc)
            bar.abort()

    th = [threading.Thread(target=worker, args=(r,)) for r in range(world)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errors, errors
    return results


@pytest.mark.parametrize("world", [2, 3])
def test_unit_shard_is_bit_identical(ctx, world):
    """Ranks of a unit-range shard evaluate disjoint work units of K-PERM-TC (and of k_pairs_T) and exchange exact
    int64 column sums: every rank's result equals the unsharded one bit for bit, whatever the number of ranks."""
    c = dg.config(2, scale=0.1)  # 30 000 + 30 000 events, 5-D: hundreds of units, two launches
    s = dg.make_sample(c)
    ref = ctx.permutation_test(s.x, s.xbar, c.sigma, 600, 11)
    assert ctx.stats().dominant_kernel == "k_perm_tc"
    refT = ctx.T(s.x, s.xbar, c.sigma)
    out = _run_sharded(world, lambda cx: (cx.permutation_test(s.x, s.xbar, c.sigma, 600, 11), cx.T(s.x, s.xbar, c.sigma)))
    for r, t in out:
        assert (r.T_perm == ref.T_perm).all() and r.observed.T == ref.observed.T and r.count_gt == ref.count_gt
        assert r.n_near == ref.n_near and r.observed.S_xb == ref.observed.S_xb
        assert abs(t.T - refT.T) <= 1e-12 * refT.term_scale  # fp64 block sums regrouped by rank


def test_unit_shard_with_escalation_and_weights(ctx):
    """Sharded runs whose escalation passes (k_pairs_T, sharded too) and weighted fp64 sums go through the all-gather."""
    rng = np.random.default_rng(2024)
    x, xb = rng.uniform(size=(40, 3)), rng.uniform(size=(50, 3)) ** 1.2
    with force_kernel(ctx, 2):
        ctx.set_option(binding.ET_OPT_EXACT_P, 64)
        try:
            ref = ctx.permutation_test(x, xb, 0.3, 20000, 1)
            assert ctx.stats().n_escalated > 0
        finally:
            ctx.set_option(binding.ET_OPT_EXACT_P, 16)

    def call(cx):
        cx.set_option(binding.ET_OPT_PERM_KERNEL, 2)
        return cx.permutation_test(x, xb, 0.3, 20000, 1), cx.stats()

    for r, st in _run_sharded(2, call, exact_p=64):
        assert st.n_escalated > 0 and r.count_gt == ref.count_gt and r.n_near == ref.n_near
        assert np.abs(r.T_perm - ref.T_perm).max() <= 1e-15 and r.observed.T == ref.observed.T
    c = dg.config(3, scale=0.1)  # weighted, 20 000 + 20 000
    s = dg.make_sample(c)
    ref = ctx.permutation_test(s.x, s.xbar, 0.3, 100, 3, s.wx, s.wxbar)
    for r in _run_sharded(2, lambda cx: cx.permutation_test(s.x, s.xbar, 0.3, 100, 3, s.wx, s.wxbar)):
        assert np.abs(r.T_perm - ref.T_perm).max() <= 1e-12 * ref.observed.term_scale and r.count_gt == ref.count_gt
