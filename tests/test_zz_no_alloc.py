"""et_T_static (include/et.h, csrc/et_static.cu): the entry point that allocates nothing, against the existing et_T.

Collected last on purpose (the file name sorts after every other test file): the suite runs with pytest -x, and a
failure here must not hide the other tests.  Needs a B200 (-m gpu).  Tolerance: the north-star one the other GPU tests
use, |dT| <= 1e-6 (|T_XX| + |T_XbarXbar| + |T_XXbar|), for T and for each term; n_pairs exact.
"""
import numpy as np
import pytest

import oracle
from paper_1612_04705_b200 import binding, build
from paper_1612_04705_b200 import datagen as dg

pytestmark = pytest.mark.gpu

TOL = 1e-6


@pytest.fixture(scope="module")
def torch_dev():
    import torch

    build.build()
    binding.static_setup(0)
    binding.static_setup(0)  # idempotent
    return torch


def call_static(torch, x, xbar, sigma, stream=None):
    """One et_T_static call on device tensors; returns the decoded result after a synchronisation."""
    out = torch.full((binding.RESULT_DOUBLES,), -7.0, dtype=torch.float64, device="cuda:0")
    binding.T_static(x, xbar, sigma, out, stream=stream)
    torch.cuda.synchronize()
    return binding.result_from_words(out.cpu().numpy())


def assert_close(got, exp):
    scale = exp.term_scale
    assert abs(got.T - exp.T) <= TOL * scale, (got.T, exp.T, scale)
    for k in ("T_xx", "T_bb", "T_xb"):
        assert abs(getattr(got, k) - getattr(exp, k)) <= TOL * scale, k
    for k in ("S_xx", "S_bb", "S_xb"):
        assert getattr(got, k) == pytest.approx(getattr(exp, k), rel=1e-6), k
    assert got.W == exp.W and got.Wbar == exp.Wbar and got.n_pairs == exp.n_pairs


def samples(torch):
    """(x, xbar, sigma) on the device: BASELINE config 0 (Dalitz, fp64, 2-D), then a SMALLER ragged 5-D fp32 problem, so
    that the second call finds the first call's records, bounding box and partial sums in the shared array."""
    s = dg.make_sample(dg.config(0))
    rng = np.random.default_rng(77)
    a = rng.random((1501, 5)).astype(np.float32)
    b = (rng.random((777, 5)) * 0.9 + 0.1).astype(np.float32)
    dev = lambda z: torch.from_numpy(np.ascontiguousarray(z)).to("cuda:0")
    return [(dev(s.x), dev(s.xbar), 0.3, s.x, s.xbar), (dev(a), dev(b), 0.2, a, b)]


def test_static_matches_existing_path_on_two_calls_in_a_row(torch_dev):
    torch = torch_dev
    cases = samples(torch)
    torch.cuda.synchronize()
    with binding.Context(0) as ctx:
        expected = [ctx.T(x, xb, sg) for x, xb, sg, _, _ in cases]
    # two calls in a row (different sizes, dims and dtypes), then both again: the array keeps the last call's contents
    got = [call_static(torch, x, xb, sg) for x, xb, sg, _, _ in cases]
    again = [call_static(torch, x, xb, sg) for x, xb, sg, _, _ in cases]
    for g, a, e in zip(got, again, expected):
        assert_close(g, e)
        assert_close(a, e)
        assert (g.T, g.S_xx, g.S_bb, g.S_xb) == (a.T, a.S_xx, a.S_bb, a.S_xb)  # fixed-order sums: bit-reproducible
    # and against the oracle (the definition) on both
    for g, (_, _, sg, hx, hxb) in zip(got, cases):
        assert_close(g, oracle.T(np.asarray(hx, dtype=np.float64), np.asarray(hxb, dtype=np.float64), sg))


@pytest.mark.parametrize("dim", [1, 2, 3, 4, 5, 6, 7, 8])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_static_all_dims_against_the_oracle(torch_dev, dim, dtype):
    """Every instantiation of the variant kernel (dim 1..8, both input dtypes), ragged sizes around the 1024-row padding."""
    torch = torch_dev
    rng = np.random.default_rng(100 + dim)
    n, nbar = 1024 + 3 * dim, 2049 - dim
    x = rng.normal(size=(n, dim)).astype(dtype)
    xb = (rng.normal(size=(nbar, dim)) * 1.1 + 0.1).astype(dtype)
    sigma = 0.4 * np.sqrt(dim)
    got = call_static(torch, torch.from_numpy(x).to("cuda:0"), torch.from_numpy(xb).to("cuda:0"), sigma)
    assert_close(got, oracle.T(x.astype(np.float64), xb.astype(np.float64), sigma))


def test_static_allocates_no_device_memory(torch_dev):
    torch = torch_dev
    cases = samples(torch)
    for x, xb, sg, _, _ in cases:
        call_static(torch, x, xb, sg)   # kernels loaded (lazy module loading allocates on first use)
    outs = [torch.zeros(binding.RESULT_DOUBLES, dtype=torch.float64, device="cuda:0") for _ in cases]
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(0)[0]
    for (x, xb, sg, _, _), o in zip(cases, outs):
        binding.T_static(x, xb, sg, o)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(0)[0] >= free_before


def test_static_on_a_side_stream_and_under_graph_capture(torch_dev):
    """The call enqueues on the caller's stream without synchronising, so it can be captured into a CUDA graph."""
    torch = torch_dev
    x, xb, sg, _, _ = samples(torch)[1]
    exp = call_static(torch, x, xb, sg)
    out = torch.zeros(binding.RESULT_DOUBLES, dtype=torch.float64, device="cuda:0")
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        binding.T_static(x, xb, sg, out, stream=torch.cuda.current_stream())
    for _ in range(2):
        out.fill_(-1.0)
        g.replay()
        torch.cuda.synchronize()
        got = binding.result_from_words(out.cpu().numpy())
        assert (got.T, got.S_xx, got.S_bb, got.S_xb, got.n_pairs) == (exp.T, exp.S_xx, exp.S_bb, exp.S_xb, exp.n_pairs)


def test_static_rejects_what_does_not_fit_and_bad_arguments(torch_dev):
    torch = torch_dev
    out = torch.zeros(binding.RESULT_DOUBLES, dtype=torch.float64, device="cuda:0")
    big = torch.zeros((300_000, 5), dtype=torch.float32, device="cuda:0")   # 2 x 300 032 rows x 32 B > 8 MiB
    with pytest.raises(binding.EtError) as e:
        binding.T_static(big, big, 0.2, out)
    assert e.value.status == -1 and "ET_STATIC_SCRATCH_BYTES" in str(e.value)
    small = torch.rand((100, 2), dtype=torch.float64, device="cuda:0")
    with pytest.raises(binding.EtError) as e:
        binding.T_static(small, small, 0.0, out)
    assert e.value.status == -2
    with pytest.raises(binding.EtError):
        binding.T_static(small[:1], small, 0.3, out)
    with pytest.raises(ValueError):
        binding.T_static(small.cpu(), small.cpu(), 0.3, out)
    # the largest BASELINE config that fits (config 3's size: 2 x 200 000 events, 2-D) is accepted
    fits = torch.rand((200_000, 2), dtype=torch.float32, device="cuda:0")
    binding.T_static(fits[:2000], fits, 0.3, out)
    torch.cuda.synchronize()
    # non-finite input: reported as NaN in the result (no synchronisation inside the call)
    bad = small.clone()
    bad[3, 1] = float("nan")
    r = call_static(torch, bad, small, 0.3)
    assert np.isnan(r.T) and np.isnan(r.S_xx) and r.n_pairs == 100 * 99 + 100 * 100
    # and the next call is clean again (the flag is reset every call)
    assert np.isfinite(call_static(torch, small, small, 0.3).T)
