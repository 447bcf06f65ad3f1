"""Seeded input generators: determinism, kinematics, the shapes BASELINE.json names."""
import numpy as np

from paper_1612_04705_b200 import datagen as dg


def test_configs_match_baseline_sizes():
    sizes = [(2000, 2, 50), (100_000, 2, 1000), (300_000, 5, 1000), (200_000, 2, 1000), (1_000_000, 5, 1000)]
    for i, (n, dim, nperm) in enumerate(sizes):
        c = dg.config(i)
        assert (c.n, c.nbar, c.dim, c.nperm) == (n, n, dim, nperm)
    assert dg.config(1).sigmas == (0.1, 0.3, 0.5) and dg.config(1).coord_dtype == "f32"
    assert dg.config(3).weighted and dg.config(4).podd and dg.config(0).sigma == 0.3


def test_dalitz_deterministic_and_inside():
    s1, s2 = dg.make_sample(dg.config(0)), dg.make_sample(dg.config(0))
    assert (s1.x == s2.x).all() and (s1.xbar == s2.xbar).all()
    assert s1.x.shape == (2000, 2) and s1.x.dtype == np.float64
    assert dg.dalitz_inside(s1.x[:, 0], s1.x[:, 1]).all() and dg.dalitz_inside(s1.xbar[:, 0], s1.xbar[:, 1]).all()
    # bounding box of SURVEY 8(d) and the bump centre inside the boundary (reading R14)
    (a, b), (c, d) = dg.dalitz_box()
    assert np.allclose([a, b, c, d], [0.974868, 2.993211, 0.401002, 1.893329], atol=2e-6)
    assert dg.dalitz_inside(1.04, 1.5)
    # the 5 % bump is visible near (1.04, 1.5) in Xbar only
    near = lambda z: (np.hypot(z[:, 0] - 1.04, z[:, 1] - 1.5) < 0.1).sum()
    assert near(s1.xbar) > near(s1.x) + 40


def test_fourbody_kinematics():
    coords, P, E = dg.fourbody_phase_space(20000, dg._rng(7))
    assert np.abs(P.sum(1)).max() < 1e-12 and np.abs(E.sum(1) - dg.M_D0).max() < 1e-12
    m = np.sqrt(E**2 - (P**2).sum(2))
    assert np.allclose(m, np.array(dg.FOURBODY_MASSES)[None, :], atol=1e-9)
    assert coords.min() > 0 and coords.max() < 1  # unit range by kinematic limits (reading R15)
    assert np.allclose(coords.mean(0), [0.28, 0.26, 0.62, 0.63, 0.28], atol=0.01)


def test_fourbody_weight_bound():
    r = dg._rng(2)
    tk = dg.M_D0 - sum(dg.FOURBODY_MASSES)
    rr = np.sort(r.uniform(0, 1, (500000, 2)), axis=1)
    m12 = 2 * dg.M_K + rr[:, 0] * tk
    m123 = 2 * dg.M_K + dg.M_PI + rr[:, 1] * tk
    wt = dg._q(dg.M_D0, m123, dg.M_PI) * dg._q(m123, m12, dg.M_PI) * dg._q(m12, dg.M_K, dg.M_K)
    assert wt.max() < dg.FOURBODY_WMAX


def test_small_scaled_configs():
    c = dg.config(3, scale=0.01)
    s = dg.make_sample(c)
    assert s.x.dtype == np.float32 and s.wx.shape == (2000,) and s.wx.min() >= -0.5 and s.wx.max() <= 1.5
    c = dg.config(4, scale=0.002)
    s = dg.make_sample(c)
    assert s.mom_x.shape == (2000, 3, 3) and s.mom_xbar.shape == (2000, 3, 3)
    ct = np.einsum("ij,ij->i", s.mom_x[:, 0], np.cross(s.mom_x[:, 1], s.mom_x[:, 2]))
    assert 0.4 < (ct > 0).mean() < 0.6


def test_bkg_sample_structure():
    x, xb, bx, bb, b, bbar = dg.make_bkg_sample()
    assert b + bbar == 1600 and len(bx) + len(bb) == 1600 and len(x) + len(xb) == 5600
    assert 0.70 < b / 1600 < 0.80 and 0.70 < len(bx) / 1600 < 0.80  # 3:1 flavour asymmetry of the background
    assert dg.dalitz_inside(x[:, 0], x[:, 1]).all() and dg.dalitz_inside(bb[:, 0], bb[:, 1]).all()
    again = dg.make_bkg_sample()
    assert (again[0] == x).all() and again[4] == b
