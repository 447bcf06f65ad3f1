"""Randomised cross-check of the two permutation dispatches (-m gpu): 40 seeded cases with random sizes (ragged tiles, n
!= nbar), dimensions 1-8 (both geometries of k_perm_tc), permutation counts on both sides of the 253 / 509 / 1018 column
boundaries, with and without signed weights.  The fp32 CUDA-core path (pinned to the oracle by
test_error_model_of_the_decision and the parity tests) is the reference; the tensor-core path must agree within the
north-star tolerance or 8 sigma of its rounding model, whichever is larger (below ~8000 events the 15-bit noise exceeds
1e-6 of the term scale: DESIGN.md section 6), give the same NaN pattern, and a count that differs by at most the
permutations either path flags as undecided."""
import math

import numpy as np
import pytest

from paper_1612_04705_b200 import binding, build

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed", [1, 2])
def test_tc_and_cuda_core_paths_agree_on_random_problems(seed):
    build.build()
    rng = np.random.default_rng(seed)
    with binding.Context(0) as ctx:
        for case in range(20):
            dim = int(rng.integers(1, 9))
            n, nbar = int(rng.integers(50, 30000)), int(rng.integers(50, 30000))
            nperm = int(rng.choice([1, 31, 32, 253, 254, 509, 510, 700, 1018, 1019]))
            weighted = bool(rng.integers(0, 2))
            x = rng.uniform(size=(n, dim))
            xb = rng.uniform(size=(nbar, dim)) ** rng.uniform(0.9, 1.3)
            wx = rng.uniform(-0.5, 1.5, size=n) if weighted else None
            wb = rng.uniform(-0.5, 1.5, size=nbar) if weighted else None
            sigma = float(rng.uniform(0.1, 0.5)) * math.sqrt(dim)
            pseed = int(rng.integers(1, 2**40))
            res = {}
            for k in (1, 2):
                ctx.set_option(binding.ET_OPT_PERM_KERNEL, k)
                try:
                    res[k] = ctx.permutation_test(x, xb, sigma, nperm, pseed, wx, wb)
                finally:
                    ctx.set_option(binding.ET_OPT_PERM_KERNEL, 0)
            a, b = res[1], res[2]
            o = a.observed
            # rounding model of the tensor-core path: step of w_j psi_ij times |w_i| (signed weights: 14 bits)
            q = (1.5 / 16382 * 1.5) if weighted else 1 / 32766
            var = (n * (n - 1) / 2) / (o.W * (o.W - 1)) ** 2 + (nbar * (nbar - 1) / 2) / (o.Wbar * (o.Wbar - 1)) ** 2 + n * nbar / (o.W * o.Wbar) ** 2
            bound = max(1e-6 * o.term_scale, 8 * q / math.sqrt(12) * math.sqrt(var))
            what = (case, dim, n, nbar, nperm, weighted)
            assert (np.isfinite(a.T_perm) == np.isfinite(b.T_perm)).all(), what
            ok = np.isfinite(a.T_perm)
            assert abs(a.observed.T - b.observed.T) <= bound, what
            assert not ok.any() or np.abs(a.T_perm[ok] - b.T_perm[ok]).max() <= bound, what
            assert abs(a.count_gt - b.count_gt) <= a.n_near + b.n_near, what
            assert b.observed.n_pairs == (n + nbar) * (n + nbar - 1) // 2 and b.nperm == nperm


def test_random_small_problems_against_the_oracle():
    """The same kind of random problems at sizes the oracle re-evaluates from scratch in well under a second (n, nbar < 4000,
    at most 40 permutations): BOTH dispatches against oracle.perm_test -- T_obs and every T_p within the north-star
    tolerance (tensor-core path: or 8 sigma of its rounding model, which is wider below ~8000 events), labels-driven NaN
    pattern equal, counts equal unless a permutation is flagged as undecided."""
    import oracle

    build.build()
    rng = np.random.default_rng(7)
    with binding.Context(0) as ctx:
        for case in range(24):
            dim = int(rng.integers(1, 9))
            n, nbar = int(rng.integers(20, 4000)), int(rng.integers(20, 4000))
            nperm = int(rng.choice([1, 31, 32, 40]))
            weighted = bool(rng.integers(0, 2))
            x = rng.uniform(size=(n, dim))
            xb = rng.uniform(size=(nbar, dim)) ** rng.uniform(0.9, 1.3)
            wx = rng.uniform(-0.5, 1.5, size=n) if weighted else None
            wb = rng.uniform(-0.5, 1.5, size=nbar) if weighted else None
            sigma = float(rng.uniform(0.1, 0.5)) * math.sqrt(dim)
            pseed = int(rng.integers(1, 2**40))
            exp = oracle.perm_test(x, xb, sigma, nperm, pseed, wx, wb)
            o = exp.observed
            for k in (1, 2):
                ctx.set_option(binding.ET_OPT_PERM_KERNEL, k)
                try:
                    got = ctx.permutation_test(x, xb, sigma, nperm, pseed, wx, wb)
                finally:
                    ctx.set_option(binding.ET_OPT_PERM_KERNEL, 0)
                bound = 1e-6 * o.term_scale
                if k == 2:
                    q = (1.5 / 16382 * 1.5) if weighted else 1 / 32766
                    var = ((n * (n - 1) / 2) / (o.W * (o.W - 1)) ** 2 + (nbar * (nbar - 1) / 2) / (o.Wbar * (o.Wbar - 1)) ** 2
                           + n * nbar / (o.W * o.Wbar) ** 2)
                    bound = max(bound, 8 * q / math.sqrt(12) * math.sqrt(var))
                what = (case, k, dim, n, nbar, nperm, weighted)
                assert (np.isfinite(got.T_perm) == np.isfinite(exp.T_perm)).all(), what
                ok = np.isfinite(exp.T_perm)
                assert abs(got.observed.T - o.T) <= bound, what
                assert not ok.any() or np.abs(got.T_perm[ok] - exp.T_perm[ok]).max() <= bound, what
                assert abs(got.count_gt - exp.count_gt) <= got.n_near, what
                if got.n_near == 0:
                    assert got.count_gt == exp.count_gt and got.p_value == exp.p_value, what
