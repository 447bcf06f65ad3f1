"""Pins for the oracle (oracle/et_oracle.c) -- CPU only.

Each test checks the oracle against something other than itself: a value that
follows from the paper's equations by hand (tests/golden/closed_forms.txt), an
invariant of Eq. 2, a textbook/library routine (scipy cdist, cuRAND's host
Philox, numpy sort), brute force on tiny inputs.  Pin numbers P1..P14 are those
of SURVEY.md 8(c) / DESIGN.md.
"""
import ctypes
import itertools
import math
import os

import numpy as np
import pytest
from scipy.spatial.distance import cdist
from scipy.special import erf

import oracle

A_OF = lambda sigma: sigma * math.sqrt(2.0 * math.log(2.0))  # psi(k a) = 2^(-k^2)


def lib_T(x, xbar, sigma, wx=None, wxbar=None):
    """Eq. 2 through a library distance routine (scipy cdist) -- independent of the oracle's loops."""
    x, xbar = np.atleast_2d(np.asarray(x, float)), np.atleast_2d(np.asarray(xbar, float))
    wx = np.ones(len(x)) if wx is None else np.asarray(wx, float)
    wb = np.ones(len(xbar)) if wxbar is None else np.asarray(wxbar, float)
    k = lambda a, b: np.exp(-cdist(a, b, "sqeuclidean") / (2 * sigma**2))
    Kxx, Kbb, Kxb = k(x, x), k(xbar, xbar), k(x, xbar)
    sxx = (np.triu(Kxx, 1) * np.outer(wx, wx)).sum()
    sbb = (np.triu(Kbb, 1) * np.outer(wb, wb)).sum()
    sxb = (Kxb * np.outer(wx, wb)).sum()
    W, Wb = wx.sum(), wb.sum()
    return sxx / (W * (W - 1)) + sbb / (Wb * (Wb - 1)) - sxb / (W * Wb)


def read_golden(golden_dir, name):
    rows = []
    with open(os.path.join(golden_dir, name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append(line.split())
    return rows


# ------------------------------------------------------------------ P1..P4
def test_P1_psi_zero_and_symmetry():
    rng = np.random.default_rng(1)
    a, b = rng.normal(size=5), rng.normal(size=5)
    assert oracle.psi(a, a, 0.3) == 1.0
    assert oracle.psi(a, b, 0.3) == oracle.psi(b, a, 0.3)
    d2 = ((a - b) ** 2).sum()
    assert oracle.psi(a, b, 0.7) == pytest.approx(math.exp(-d2 / (2 * 0.49)), rel=1e-15)


@pytest.mark.parametrize("n,nbar", [(2, 2), (3, 7), (10, 4)])
def test_P1_coincident_points_give_zero(n, nbar):
    # all psi = 1: T = n(n-1)/2/(n(n-1)) + 1/2 - 1 = 0   (reading R1: within terms are half-means)
    pt = np.array([[0.3, -1.2, 2.0]])
    r = oracle.T(np.repeat(pt, n, 0), np.repeat(pt, nbar, 0), 0.4)
    assert r.T == pytest.approx(0.0, abs=1e-15)
    assert r.T_xx == pytest.approx(0.5) and r.T_bb == pytest.approx(0.5) and r.T_xb == pytest.approx(1.0)
    assert r.n_pairs == n * (n - 1) // 2 + nbar * (nbar - 1) // 2 + n * nbar


def test_P2_P3_closed_forms(golden_dir):
    gold = {r[0]: float(r[1]) for r in read_golden(golden_dir, "closed_forms.txt")}
    for sigma in (0.3, 1.7):
        a = A_OF(sigma)
        r = oracle.T([[0, 0], [a, 0]], [[0, a], [a, a]], sigma)
        assert r.T == pytest.approx(gold["P2_square_2plus2"], abs=1e-15)
        # collinear, embedded in D = 1, 2 and 5 by zero padding
        for dim in (1, 2, 5):
            pad = lambda v: [[t] + [0.0] * (dim - 1) for t in v]
            r = oracle.T(pad([0, a]), pad([2 * a, 3 * a]), sigma)
            assert r.T == pytest.approx(gold["P3_collinear_2plus2"], abs=1e-15)


@pytest.mark.parametrize("n,nbar,d", [(3, 5, 0.37), (6, 2, 1.1), (4, 4, 50.0)])
def test_P4_two_clusters(n, nbar, d):
    sigma = 0.5
    A, B = np.zeros((n, 3)), np.zeros((nbar, 3))
    B[:, 1] = d
    r = oracle.T(A, B, sigma)
    assert r.T == pytest.approx(1.0 - math.exp(-d * d / (2 * sigma**2)), abs=1e-14)


# ------------------------------------------------------------------ P5 symmetries
def test_P5_symmetries_and_limits():
    rng = np.random.default_rng(5)
    x, xb = rng.normal(size=(23, 3)), rng.normal(0.3, 1.2, size=(31, 3))
    s = 0.6
    t0 = oracle.T(x, xb, s)
    assert oracle.T(xb, x, s).T == pytest.approx(t0.T, abs=1e-15)  # swap
    assert oracle.T(xb, x, s).T_xx == pytest.approx(t0.T_bb, abs=1e-15)
    assert oracle.T(x + 7.5, xb + 7.5, s).T == pytest.approx(t0.T, abs=1e-13)  # translation
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    assert oracle.T(x @ q, xb @ q, s).T == pytest.approx(t0.T, abs=1e-14)  # rotation
    assert oracle.T(x[::-1], xb[rng.permutation(31)], s).T == pytest.approx(t0.T, abs=1e-15)  # reordering
    assert oracle.T(3.7 * x, 3.7 * xb, 3.7 * s).T == pytest.approx(t0.T, abs=1e-14)  # scale
    assert abs(oracle.T(x, xb, 1e6).T) < 1e-9  # sigma -> inf: all psi -> 1
    assert oracle.T(x, xb, 1e-6).T == 0.0  # sigma -> 0: all psi -> 0 (distinct points)


def test_library_routine_agrees():
    # special case that reduces to a library routine: squared-distance matrix via scipy
    rng = np.random.default_rng(11)
    for dim in (1, 2, 5, 8):
        x, xb = rng.uniform(size=(40, dim)), rng.uniform(size=(57, dim))
        assert oracle.T(x, xb, 0.25).T == pytest.approx(lib_T(x, xb, 0.25), abs=1e-14)
        wx, wb = rng.uniform(-0.5, 1.5, 40), rng.uniform(-0.5, 1.5, 57)
        assert oracle.T(x, xb, 0.25, wx, wb).T == pytest.approx(lib_T(x, xb, 0.25, wx, wb), abs=1e-13)


def test_term_signs_and_factors():
    # a dropped 1/2, a wrong sign of the cross term or a transposed normalisation fails here
    x = np.array([[0.0], [1.0], [2.0]])
    xb = np.array([[0.5], [4.0]])
    s = 1.0
    e = lambda d: math.exp(-d * d / 2)
    sxx = e(1) + e(2) + e(1)
    sbb = e(3.5)
    sxb = e(0.5) + e(4) + e(0.5) + e(3) + e(1.5) + e(2)
    r = oracle.T(x, xb, s)
    assert r.S_xx == pytest.approx(sxx) and r.S_bb == pytest.approx(sbb) and r.S_xb == pytest.approx(sxb)
    assert r.T == pytest.approx(sxx / 6 + sbb / 2 - sxb / 6, abs=1e-15)


# ------------------------------------------------------------------ P6 exhaustive mean
@pytest.mark.parametrize("N,n", [(8, 3), (7, 2)])
def test_P6_exhaustive_permutation_mean_is_zero(N, n):
    rng = np.random.default_rng(6)
    z = rng.normal(size=(N, 2))
    tot, cnt = 0.0, 0
    for sel in itertools.combinations(range(N), n):
        m = np.zeros(N, bool)
        m[list(sel)] = True
        tot += oracle.T(z[m], z[~m], 0.8).T
        cnt += 1
    assert cnt == math.comb(N, n)
    assert abs(tot / cnt) < 1e-15


# ------------------------------------------------------------------ P9 Philox
def test_P9_philox_known_answers(golden_dir):
    for row in read_golden(golden_dir, "philox4x32_10_kat.txt"):
        v = [int(t, 16) for t in row]
        out = oracle.philox4x32_10(v[0:4], v[4:6])
        assert [int(t) for t in out] == v[6:10]


def test_P9_philox_matches_curand_host_generator():
    """cuRAND's host Philox4_32_10 generator, an independent library implementation: with seed s its k-th
    block of four outputs is philox(ctr = (k >> 16, 0, k & 0xffff, 0), key = (s_lo, s_hi)) -- cuRAND walks 65536
    subsequences (counter word 2) before advancing the offset (counter word 0); mapping found by search."""
    try:
        cr = ctypes.CDLL("libcurand.so.10")
    except OSError:
        try:
            cr = ctypes.CDLL("/usr/local/cuda/lib64/libcurand.so.10")
        except OSError:
            pytest.skip("libcurand not available")
    gen = ctypes.c_void_p()
    CURAND_RNG_PSEUDO_PHILOX4_32_10 = 161
    if cr.curandCreateGeneratorHost(ctypes.byref(gen), CURAND_RNG_PSEUDO_PHILOX4_32_10) != 0:
        pytest.skip("cuRAND host generator unavailable")
    nblk = 65536 + 3
    for seed in (0, 0xE7E57, 0x1234_5678_9ABC_DEF0):
        assert cr.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
        assert cr.curandSetGeneratorOffset(gen, ctypes.c_ulonglong(0)) == 0
        buf = (ctypes.c_uint32 * (4 * nblk))()
        assert cr.curandGenerate(gen, buf, ctypes.c_size_t(4 * nblk)) == 0
        got = np.frombuffer(buf, dtype=np.uint32).reshape(nblk, 4)
        for k in list(range(16)) + [4097, 65535, 65536, 65537, 65538]:
            exp = oracle.philox4x32_10([k >> 16, 0, k & 0xFFFF, 0], [seed & 0xFFFFFFFF, seed >> 32])
            assert (got[k] == exp).all(), (seed, k)
    cr.curandDestroyGenerator(gen)


def py_philox(ctr, key):
    """Independent restatement of the round function (Salmon et al.), for the label pins below."""
    c, k = [int(v) for v in ctr], [int(v) for v in key]
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return c


def test_py_philox_restatement_hits_known_answers(golden_dir):
    for row in read_golden(golden_dir, "philox4x32_10_kat.txt"):
        v = [int(t, 16) for t in row]
        assert py_philox(v[0:4], v[4:6]) == v[6:10]


# ------------------------------------------------------------------ P10 labels
@pytest.mark.parametrize("N,n,nperm,seed", [(37, 11, 9, 0xE7E57), (64, 32, 33, 5), (10, 0, 3, 1), (10, 10, 3, 1)])
def test_P10_labels_rule_and_counts(N, n, nperm, seed):
    a = oracle.labels_range(N, n, 0, nperm, seed)
    assert a.shape == (nperm, N)
    assert (a.sum(1) == n).all()
    # reading R4 re-derived with numpy sort and the python Philox restatement
    for p in range(nperm):
        K = [(py_philox([i, 0, p >> 2, 0], [seed & 0xFFFFFFFF, seed >> 32])[p & 3] << 32) | i for i in range(N)]
        order = np.argsort(np.array(K, dtype=np.uint64), kind="stable")
        exp = np.zeros(N, np.uint8)
        exp[order[:n]] = 1
        assert (a[p] == exp).all()
    # packed form, and a sub-range equals the same permutations of the full range
    mask = oracle.labels(N, n, nperm, seed)
    for p in range(nperm):
        assert (((mask[:, p >> 5] >> (p & 31)) & 1) == a[p]).all()
    assert (oracle.labels_range(N, n, 2, 1, seed)[0] == a[2]).all()


def test_P8_label_histogram_uniform_over_splits():
    # 2+2 problem: the C(4,2) = 6 splits must be equally likely (chi^2, 5 dof; 20.5 is p = 0.001)
    nperm = 6000
    a = oracle.labels_range(4, 2, 0, nperm, 0xE7E57)
    codes = (a * np.array([1, 2, 4, 8])).sum(1)
    vals, counts = np.unique(codes, return_counts=True)
    assert len(vals) == 6
    chi2 = ((counts - nperm / 6) ** 2 / (nperm / 6)).sum()
    assert chi2 < 20.5
    # each event is in X half of the time, pairs 1/6 of the time
    assert abs(a.mean() - 0.5) < 1e-12
    # successive permutations are not copies of each other
    assert (a[1:] != a[:-1]).any(1).mean() > 0.7


# ------------------------------------------------------------------ P8 brute-force p-value, P7 identity
@pytest.mark.parametrize("weighted", [False, True])
def test_P8_permutation_test_brute_force(weighted):
    rng = np.random.default_rng(8)
    n, nbar, nperm, seed, sigma = 3, 4, 40, 77, 0.9
    x, xb = rng.normal(size=(n, 2)), rng.normal(0.8, 1.0, size=(nbar, 2))
    wx = rng.uniform(0.6, 1.5, n) if weighted else None  # sums stay > 1 for every split of 3+4
    wb = rng.uniform(0.6, 1.5, nbar) if weighted else None
    res = oracle.perm_test(x, xb, sigma, nperm, seed, wx, wb)
    z = np.vstack([x, xb])
    w = None if not weighted else np.concatenate([wx, wb])
    a = oracle.labels_range(n + nbar, n, 0, nperm, seed).astype(bool)
    t_obs = lib_T(x, xb, sigma, wx, wb)
    assert res.observed.T == pytest.approx(t_obs, abs=1e-14)
    tp = np.array([lib_T(z[m], z[~m], sigma, None if w is None else w[m], None if w is None else w[~m]) for m in a])
    assert np.allclose(res.T_perm, tp, atol=1e-14, rtol=0)
    assert res.count_gt == int((tp > t_obs).sum())  # strict >, reading R3
    assert res.p_value == res.count_gt / nperm and res.nperm == nperm


def test_P7_QRS_identity_against_from_scratch():
    """S_XX = Q, S_bb = S - R + Q, S_xb = R - 2Q with Q = sum_{i<j} a_i a_j Psi'_ij, R = sum_i a_i r_i."""
    rng = np.random.default_rng(7)
    N, n, sigma = 16, 7, 0.7
    z = rng.normal(size=(N, 3))
    w = rng.uniform(-0.5, 1.5, N)  # signed weights
    done = 0
    psi = np.exp(-cdist(z, z, "sqeuclidean") / (2 * sigma**2)) * np.outer(w, w)
    np.fill_diagonal(psi, 0.0)
    S, r = psi.sum() / 2, psi.sum(1)
    for p in range(8):
        a = oracle.labels_range(N, n, p, 1, 3)[0].astype(float)
        Q, R = a @ psi @ a / 2, a @ r
        m = a.astype(bool)
        if w[m].sum() <= 1 or w[~m].sum() <= 1:
            continue
        done += 1
        res = oracle.T(z[m], z[~m], sigma, w[m], w[~m])
        assert res.S_xx == pytest.approx(Q, abs=1e-12)
        assert res.S_bb == pytest.approx(S - R + Q, abs=1e-12)
        assert res.S_xb == pytest.approx(R - 2 * Q, abs=1e-12)
        assert res.W == pytest.approx(a @ w)
    assert done >= 5


def test_degenerate_weighted_split_is_nan_not_counted():
    # weights chosen so that some splits have W_p <= 1 (reading R10)
    x, xb = np.array([[0.0], [1.0]]), np.array([[2.0], [3.0], [4.0]])
    wx, wb = np.array([1.2, 1.1]), np.array([0.1, 0.1, 2.0])
    res = oracle.perm_test(x, xb, 1.0, 60, 9, wx, wb)
    assert np.isnan(res.T_perm).any() and np.isfinite(res.T_perm).any()
    finite = res.T_perm[np.isfinite(res.T_perm)]
    assert res.count_gt == int((finite > res.observed.T).sum())


# ------------------------------------------------------------------ P11, P12 weights
def test_P11_unit_weights_and_duplicated_events():
    rng = np.random.default_rng(12)
    x, xb = rng.normal(size=(9, 2)), rng.normal(0.4, 1.0, size=(7, 2))
    s = 0.8
    plain = oracle.T(x, xb, s)
    ones = oracle.T(x, xb, s, np.ones(9), np.ones(7))
    assert ones.T == plain.T and ones.S_xx == plain.S_xx
    # integer weights k_i == each event repeated k_i times, minus the coincident (psi = 1) pairs
    kx, kb = rng.integers(1, 4, 9), rng.integers(1, 4, 7)
    wres = oracle.T(x, xb, s, kx.astype(float), kb.astype(float))
    dup = oracle.T(np.repeat(x, kx, 0), np.repeat(xb, kb, 0), s)
    assert dup.S_xx == pytest.approx(wres.S_xx + (kx * (kx - 1) // 2).sum(), abs=1e-12)
    assert dup.S_bb == pytest.approx(wres.S_bb + (kb * (kb - 1) // 2).sum(), abs=1e-12)
    assert dup.S_xb == pytest.approx(wres.S_xb, abs=1e-12)
    assert dup.W == wres.W and dup.Wbar == wres.Wbar


def test_P12_eq3_is_weighted_form_up_to_self_term():
    """Reading R7: weights {+1 main, -b/b_s background sample} reproduce Eq. 3 except the bkg-bkg self term,
    where Eq. 3 has b(b+1)/(b_s(b_s-1)) and the weighted form (b/b_s)^2 (per sum over i != j)."""
    rng = np.random.default_rng(13)
    s = 0.25
    x, xb = rng.uniform(size=(30, 2)), rng.uniform(size=(26, 2))
    bx, bb = rng.uniform(size=(12, 2)), rng.uniform(size=(9, 2))
    b, bbar = 5.0, 4.0
    t3 = oracle.T_bkg(x, xb, bx, bb, b, bbar, s)
    wx = np.concatenate([np.ones(30), np.full(12, -b / 12)])
    wb = np.concatenate([np.ones(26), np.full(9, -bbar / 9)])
    tw = oracle.T(np.vstack([x, bx]), np.vstack([xb, bb]), s, wx, wb)
    assert tw.W == pytest.approx(30 - b) and tw.Wbar == pytest.approx(26 - bbar)
    k = lambda a: np.exp(-cdist(a, a, "sqeuclidean") / (2 * s * s)).sum() - len(a)  # sum over i != j
    w, wbar = 30 - b, 26 - bbar
    corr = (b * (b + 1) / (12 * 11) - (b / 12) ** 2) * k(bx) / (2 * w * (w - 1)) + (
        bbar * (bbar + 1) / (9 * 8) - (bbar / 9) ** 2
    ) * k(bb) / (2 * wbar * (wbar - 1))
    assert t3 == pytest.approx(tw.T + corr, abs=1e-14)


def test_eq3_without_background_is_eq2():
    rng = np.random.default_rng(14)
    x, xb = rng.uniform(size=(15, 2)), rng.uniform(size=(11, 2))
    bx, bb = rng.uniform(size=(4, 2)), rng.uniform(size=(5, 2))
    assert oracle.T_bkg(x, xb, bx, bb, 0.0, 0.0, 0.3) == pytest.approx(oracle.T(x, xb, 0.3).T, abs=1e-15)


def test_eq3_direct_restatement():
    """Eq. 3 typed again with library distance matrices (readings R8, R9, R16)."""
    rng = np.random.default_rng(15)
    s = 0.4
    x, xb = rng.uniform(size=(14, 3)), rng.uniform(size=(10, 3))
    bx, bb = rng.uniform(size=(6, 3)), rng.uniform(size=(7, 3))
    b, bbar = 3.0, 2.5
    K = lambda a, c: np.exp(-cdist(a, c, "sqeuclidean") / (2 * s * s)).sum()
    ne = lambda a: K(a, a) - len(a)
    w, wbar, bs, bsb = 14 - b, 10 - bbar, 6, 7
    t = (ne(x) - 2 * b / bs * K(x, bx) + b * (b + 1) / (bs * (bs - 1)) * ne(bx)) / (2 * w * (w - 1))
    t += (ne(xb) - 2 * bbar / bsb * K(xb, bb) + bbar * (bbar + 1) / (bsb * (bsb - 1)) * ne(bb)) / (2 * wbar * (wbar - 1))
    t -= (K(x, xb) - bbar / bsb * K(x, bb) - b / bs * K(xb, bx) + b * bbar / (bs * bsb) * K(bx, bb)) / (w * wbar)
    assert oracle.T_bkg(x, xb, bx, bb, b, bbar, s) == pytest.approx(t, abs=1e-14)


# ------------------------------------------------------------------ P13 statistical pin
def test_P13_unit_cube_expectation():
    # E[psi] for two independent uniform points in the unit D-cube: g(sigma)^D
    D, sigma, n = 5, 0.2, 3000
    g = sigma * math.sqrt(2 * math.pi) * erf(1 / (sigma * math.sqrt(2))) - 2 * sigma**2 * (1 - math.exp(-1 / (2 * sigma**2)))
    rng = np.random.default_rng(130)
    x, xb = rng.uniform(size=(n, D)), rng.uniform(size=(n, D))
    r = oracle.T(x, xb, sigma)
    tol = 6.0 / math.sqrt(n)
    assert r.T_xb == pytest.approx(g**D, rel=tol)  # full mean
    assert r.T_xx == pytest.approx(0.5 * g**D, rel=tol)  # half-mean (reading R1)
    assert r.T_bb == pytest.approx(0.5 * g**D, rel=tol)


# ------------------------------------------------------------------ row sums
def test_row_sums_compose_to_block_sums():
    rng = np.random.default_rng(21)
    x, xb = rng.normal(size=(13, 2)), rng.normal(size=(17, 2))
    wx, wb = rng.uniform(0.2, 1.5, 13), rng.uniform(0.2, 1.5, 17)
    for W in ((None, None), (wx, wb)):
        res = oracle.T(x, xb, 0.7, *W)
        rx, rb = oracle.row_sums(x, xb, 0.7, np.arange(30), *W)
        ux = np.ones(13) if W[0] is None else wx
        ub = np.ones(17) if W[1] is None else wb
        assert 0.5 * (ux * rx[:13]).sum() == pytest.approx(res.S_xx, abs=1e-12)
        assert 0.5 * (ub * rb[13:]).sum() == pytest.approx(res.S_bb, abs=1e-12)
        assert (ux * rb[:13]).sum() == pytest.approx(res.S_xb, abs=1e-12)
        assert (ub * rx[13:]).sum() == pytest.approx(res.S_xb, abs=1e-12)


# ------------------------------------------------------------------ P14 triple product
def test_P14_triple_product_split():
    rng = np.random.default_rng(14)
    n = 500
    B, Cc, D = rng.normal(size=(n, 3)), rng.normal(size=(n, 3)), rng.normal(size=(n, 3))
    pos, cnt = oracle.podd_split(B, Cc, D, False)
    det = np.linalg.det(np.stack([B, Cc, D], axis=1))  # library determinant = B . (C x D)
    assert (pos == (det > 0)).all() and cnt == int((det > 0).sum())
    assert (oracle.podd_split(Cc, B, D, False)[0] == 1 - pos).all()  # odd under a swap
    assert (oracle.podd_split(-B, -Cc, -D, False)[0] == 1 - pos).all()  # odd under parity
    assert (oracle.podd_split(Cc, D, B, False)[0] == pos).all()  # cyclic
    assert (oracle.podd_split(B, Cc, D, True)[0] == 1 - pos).all()  # -Cbar_T > 0
    # C_T == 0 exactly goes to the negative class for both flavours (reading R11)
    z = np.zeros((1, 3))
    assert oracle.podd_split(z, z, z, False)[0][0] == 0 and oracle.podd_split(z, z, z, True)[0][0] == 0


def test_P14_peven_from_four_classes_is_default_test():
    """(I+II) vs (III+IV) is the default X vs Xbar comparison."""
    rng = np.random.default_rng(140)
    x, xb = rng.uniform(size=(40, 5)), rng.uniform(size=(35, 5))
    px, pb = rng.normal(size=(40, 3, 3)), rng.normal(size=(35, 3, 3))
    posx, _ = oracle.podd_split(px[:, 0], px[:, 1], px[:, 2], False)
    posb, _ = oracle.podd_split(pb[:, 0], pb[:, 1], pb[:, 2], True)
    I, II, III, IV = x[posx == 1], x[posx == 0], xb[posb == 1], xb[posb == 0]
    assert len(I) + len(II) == 40 and len(III) + len(IV) == 35
    even = oracle.T(np.vstack([I, II]), np.vstack([III, IV]), 0.2)
    assert even.T == pytest.approx(oracle.T(x, xb, 0.2).T, abs=1e-15)


# ------------------------------------------------------------------ argument checking
def test_oracle_rejects_bad_arguments():
    x = np.zeros((3, 2))
    with pytest.raises(ValueError):
        oracle.T(x[:1], x, 0.3)
    with pytest.raises(ValueError):
        oracle.T(x, x, 0.0)
    with pytest.raises(ValueError):
        oracle.T(x, x, float("nan"))
    with pytest.raises(ValueError):
        oracle.T(x, x, 0.3, np.array([0.2, 0.2, 0.2]), np.ones(3))  # W <= 1


def test_eq3_permutations_without_background_are_eq2_permutations():
    """Reading R18 pinned to the Eq. 2 permutation oracle: with b = bbar = 0 the background samples drop out of Eq. 3
    and every permutation T equals the one of `perm_test` on the main samples (same label stream, same order)."""
    rng = np.random.default_rng(31)
    x, xb = rng.uniform(size=(14, 2)), rng.uniform(size=(11, 2))
    bx, bb = rng.uniform(size=(5, 2)), rng.uniform(size=(4, 2))
    t_obs, t_perm, count, p = oracle.bkg_perm_test(x, xb, bx, bb, 0.0, 0.0, 0.3, 12, 77)
    ref = oracle.perm_test(x, xb, 0.3, 12, 77)
    assert t_obs == pytest.approx(ref.observed.T, abs=1e-15)
    assert np.allclose(t_perm, ref.T_perm, rtol=0, atol=1e-15) and count == ref.count_gt


def test_eq3_permutations_keep_sizes_and_equalise_the_purity():
    """Flat signal and flat background with a 3:1 flavour asymmetry of the background only: Eq. 2 on the main samples
    is blind to it (same density), and under permutation the expected background counts are proportional to the
    sample sizes: the mean of the permutation T of Eq. 3 is compatible with zero."""
    rng = np.random.default_rng(32)
    sig, bkg, side = rng.uniform(size=(60, 2)), rng.uniform(size=(40, 2)), rng.uniform(size=(40, 2))
    fl, flb, fls = rng.random(60) < 0.5, rng.random(40) < 0.75, rng.random(40) < 0.75
    x, xb = np.vstack([sig[fl], bkg[flb]]), np.vstack([sig[~fl], bkg[~flb]])
    t_obs, t_perm, count, p = oracle.bkg_perm_test(x, xb, side[fls], side[~fls], float(flb.sum()), float((~flb).sum()), 0.25, 60, 5)
    assert np.isfinite(t_perm).all() and len(np.unique(t_perm)) == 60
    assert abs(t_perm.mean()) < 4 * t_perm.std() / np.sqrt(60)
    assert 0 <= p <= 1 and count == int((t_perm > t_obs).sum())


def test_R18_purity_of_permuted_samples_by_enumeration():
    """Pin of reading R18's b': tag b + bbar of the n + nbar pooled main events as background,
    enumerate ALL C(n + nbar, n) reassignments to samples of sizes (n, nbar) and average the number of tagged events
    that land in X' and in Xbar'.  n != nbar, so that b' = b, swapped sizes or a plain half all fail."""
    import itertools

    n, nbar, b, bbar = 5, 3, 2, 1
    N = n + nbar
    tagged = np.zeros(N, dtype=bool)
    tagged[[0, 3, 6]] = True  # b + bbar = 3 background events somewhere in the pool
    in_x = []
    for sel in itertools.combinations(range(N), n):
        in_x.append(tagged[list(sel)].sum())
    mean_x = float(np.mean(in_x))
    bp, bbp = oracle.bkg_perm_purity(b, bbar, n, nbar)
    assert bp == pytest.approx(mean_x, abs=1e-14) and bbp == pytest.approx((b + bbar) - mean_x, abs=1e-14)
    assert bp == pytest.approx(15 / 8) and bbp == pytest.approx(9 / 8)
    # the plausible mistakes are different numbers here
    for wrong in ((b, bbar), (bbp, bp), ((b + bbar) / 2, (b + bbar) / 2)):
        assert abs(wrong[0] - mean_x) > 0.1


def _eq3_perm_mean(x, xb, bx, bb, b, bbar, sigma, nperm, seed, purity):
    """Mean and standard error of the Eq. 3 permutation T values with the permuted samples' background counts given
    by `purity(b, bbar, n, nbar)`; the reassignment is R18's (labels_range from `seed` and `seed ^ BKG_SEED_XOR`)."""
    n, nbar, bs, bsb = len(x), len(xb), len(bx), len(bb)
    main, side = np.vstack([x, xb]), np.vstack([bx, bb])
    am = oracle.labels_range(n + nbar, n, 0, nperm, seed)
    ab = oracle.labels_range(bs + bsb, bs, 0, nperm, seed ^ oracle.BKG_SEED_XOR)
    bp, bbp = purity(b, bbar, n, nbar)
    t = np.array([oracle.T_bkg(main[am[p] == 1], main[am[p] == 0], side[ab[p] == 1], side[ab[p] == 0], bp, bbp, sigma)
                  for p in range(nperm)])
    return t, t.mean(), t.std(ddof=1) / np.sqrt(nperm)


def test_R18_wrong_purity_biases_the_permutation_T():
    """Second pin of R18's b': background whose density differs from the signal's (a cluster on a flat signal), unequal
    sample sizes (305 : 135) and a background that sits mostly in the smaller sample (5 : 35).  Eq. 3 removes the
    background on average only when the permuted samples are evaluated with the background counts they have on average,
    (b + bbar) n / (n + nbar) and (b + bbar) nbar / (n + nbar): then the permutation T values scatter around zero, and
    `bkg_perm_test` reproduces them.  With b' = b, bbar' = bbar (the observed counts) or with the sizes swapped the mean
    permutation T is tens of standard errors away from zero.  (R18 uses the EXPECTED counts; the hypergeometric
    fluctuation of the actual counts around them leaves a second-order term ~ var / w^2 in the mean, which this setup
    -- a broad cluster, 9 % background -- keeps below the permutation spread: measured +1.5 standard errors.)"""
    rng = np.random.default_rng(1805)
    nsig_x, nsig_b, b, bbar, bs, bsb = 300, 100, 5, 35, 60, 60
    sig = rng.uniform(size=(nsig_x + nsig_b, 2))
    cl = lambda m: 0.5 + 0.15 * rng.normal(size=(m, 2))  # the background: a cluster
    x = np.vstack([sig[:nsig_x], cl(b)])
    xb = np.vstack([sig[nsig_x:], cl(bbar)])
    bx, bb = cl(bs), cl(bsb)
    nperm, seed, sigma = 300, 99, 0.2
    t, m, se = _eq3_perm_mean(x, xb, bx, bb, b, bbar, sigma, nperm, seed, oracle.bkg_perm_purity)
    assert abs(m) < 4 * se, (m, se)
    _, m_obs, se_obs = _eq3_perm_mean(x, xb, bx, bb, b, bbar, sigma, nperm, seed, lambda b, bbar, n, nbar: (b, bbar))
    assert abs(m_obs) > 8 * se_obs, (m_obs, se_obs)
    _, m_sw, se_sw = _eq3_perm_mean(x, xb, bx, bb, b, bbar, sigma, nperm, seed,
                                    lambda b, bbar, n, nbar: ((b + bbar) * nbar / (n + nbar), (b + bbar) * n / (n + nbar)))
    assert abs(m_sw) > 8 * se_sw, (m_sw, se_sw)
    # bkg_perm_test is this loop with R18's purity
    t_obs, t_perm, count, p = oracle.bkg_perm_test(x, xb, bx, bb, b, bbar, sigma, 40, seed)
    assert np.allclose(t_perm, t[:40], rtol=0, atol=1e-13) and count == int((t_perm > t_obs).sum())  # OpenMP sum order
