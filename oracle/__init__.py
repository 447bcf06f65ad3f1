"""TEST INFRASTRUCTURE ONLY -- ctypes front of ``oracle/et_oracle.c``.

The oracle is the plain double-precision CPU statement of the energy-test hot
path (see the header of ``et_oracle.c``).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It imports nothing from
``paper_1612_04705_b200`` and shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "et_oracle.c")
_LIB = os.path.join(_HERE, "libet_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
        )
    return _LIB


class _Result(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("T", "T_xx", "T_bb", "T_xb", "S_xx", "S_bb", "S_xb", "W", "Wbar")] + [
        ("n_pairs", C.c_int64)
    ]


class _PermResult(C.Structure):
    _fields_ = [("observed", _Result), ("p_value", C.c_double), ("count_gt", C.c_int64), ("nperm", C.c_int64)]


@dataclass
class Result:
    T: float
    T_xx: float
    T_bb: float
    T_xb: float
    S_xx: float
    S_bb: float
    S_xb: float
    W: float
    Wbar: float
    n_pairs: int

    @property
    def term_scale(self) -> float:
        """|T_XX| + |T_XbarXbar| + |T_XXbar|, the scale of the north-star tolerance."""
        return abs(self.T_xx) + abs(self.T_bb) + abs(self.T_xb)


@dataclass
class PermResult:
    observed: Result
    p_value: float
    count_gt: int
    nperm: int
    T_perm: np.ndarray


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.oracle_psi.restype = C.c_double
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def _res(r: _Result) -> Result:
    return Result(*(getattr(r, k) for k, _ in _Result._fields_))


def _f64(a, dim=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if dim is not None:
        a = a.reshape(-1, dim)
    return a


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"{what} failed with oracle status {rc}")


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def psi(a, b, sigma: float) -> float:
    a, b = _f64(a).ravel(), _f64(b).ravel()
    return float(lib().oracle_psi(_p(a), _p(b), C.c_int(a.size), C.c_double(sigma)))


def T(x, xbar, sigma: float, wx=None, wxbar=None) -> Result:
    """Eq. 2; with weights, its per-event-weighted form (reading R7)."""
    x, xbar = np.atleast_2d(_f64(x)), np.atleast_2d(_f64(xbar))
    dim = x.shape[1]
    assert xbar.shape[1] == dim
    wx = None if wx is None else _f64(wx).ravel()
    wxbar = None if wxbar is None else _f64(wxbar).ravel()
    out = _Result()
    rc = lib().oracle_T_weighted(_p(x), _p(wx), C.c_int64(len(x)), _p(xbar), _p(wxbar), C.c_int64(len(xbar)),
                                 C.c_int(dim), C.c_double(sigma), C.byref(out))
    _check(rc, "oracle_T_weighted")
    return _res(out)


def row_sums(x, xbar, sigma: float, rows, wx=None, wxbar=None):
    """Per-row class sums of psi (weighted by w_j) for the listed pooled rows."""
    x, xbar = np.atleast_2d(_f64(x)), np.atleast_2d(_f64(xbar))
    dim = x.shape[1]
    wx = None if wx is None else _f64(wx).ravel()
    wxbar = None if wxbar is None else _f64(wxbar).ravel()
    rows = np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
    rx, rb = np.zeros(len(rows)), np.zeros(len(rows))
    rc = lib().oracle_row_sums(_p(x), _p(wx), C.c_int64(len(x)), _p(xbar), _p(wxbar), C.c_int64(len(xbar)),
                               C.c_int(dim), C.c_double(sigma), _p(rows), C.c_int64(len(rows)), _p(rx), _p(rb))
    _check(rc, "oracle_row_sums")
    return rx, rb


def philox4x32_10(ctr, key) -> np.ndarray:
    ctr = np.ascontiguousarray(np.asarray(ctr, dtype=np.uint32))
    key = np.ascontiguousarray(np.asarray(key, dtype=np.uint32))
    assert ctr.size == 4 and key.size == 2
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(ctr), _p(key), _p(out))
    return out


def labels_range(N: int, n: int, p_begin: int, p_count: int, seed: int) -> np.ndarray:
    """Byte labels a[q, i] (1 = sample X) of permutations p_begin .. p_begin+p_count-1."""
    a = np.zeros((p_count, N), dtype=np.uint8)
    rc = lib().oracle_labels_range(C.c_int64(N), C.c_int64(n), C.c_int64(p_begin), C.c_int64(p_count),
                                   C.c_uint64(seed), _p(a))
    _check(rc, "oracle_labels_range")
    return a


def labels(N: int, n: int, nperm: int, seed: int) -> np.ndarray:
    """Bit-packed labels mask[i, p >> 5] bit (p & 31)."""
    mask = np.zeros((N, (nperm + 31) // 32), dtype=np.uint32)
    rc = lib().oracle_labels(C.c_int64(N), C.c_int64(n), C.c_int64(nperm), C.c_uint64(seed), _p(mask))
    _check(rc, "oracle_labels")
    return mask


def perm_test(x, xbar, sigma: float, nperm: int, seed: int, wx=None, wxbar=None) -> PermResult:
    """Permutation test of PAPER.md:67, every permutation re-evaluated from scratch."""
    x, xbar = np.atleast_2d(_f64(x)), np.atleast_2d(_f64(xbar))
    dim = x.shape[1]
    wx = None if wx is None else _f64(wx).ravel()
    wxbar = None if wxbar is None else _f64(wxbar).ravel()
    Tp = np.zeros(nperm)
    out = _PermResult()
    rc = lib().oracle_perm_test(_p(x), _p(wx), C.c_int64(len(x)), _p(xbar), _p(wxbar), C.c_int64(len(xbar)),
                                C.c_int(dim), C.c_double(sigma), C.c_int64(nperm), C.c_uint64(seed), _p(Tp),
                                C.byref(out))
    _check(rc, "oracle_perm_test")
    return PermResult(_res(out.observed), out.p_value, out.count_gt, out.nperm, Tp)


def podd_split(pB, pC, pD, is_conjugate: bool):
    """Sect. 5 / Eq. 4 sign split; returns (positive[n] uint8, n_positive)."""
    pB, pC, pD = _f64(pB, 3), _f64(pC, 3), _f64(pD, 3)
    pos = np.zeros(len(pB), dtype=np.uint8)
    cnt = C.c_int64(0)
    rc = lib().oracle_podd_split(_p(pB), _p(pC), _p(pD), C.c_int64(len(pB)), C.c_int(int(is_conjugate)), _p(pos),
                                 C.byref(cnt))
    _check(rc, "oracle_podd_split")
    return pos, int(cnt.value)


def T_bkg(x, xbar, bx, bxbar, b: float, bbar: float, sigma: float) -> float:
    """Eq. 3, background-sample-subtracted T."""
    x, xbar, bx, bxbar = (np.atleast_2d(_f64(a)) for a in (x, xbar, bx, bxbar))
    dim = x.shape[1]
    out = C.c_double(0.0)
    rc = lib().oracle_T_bkg(_p(x), C.c_int64(len(x)), _p(xbar), C.c_int64(len(xbar)), _p(bx), C.c_int64(len(bx)),
                            _p(bxbar), C.c_int64(len(bxbar)), C.c_double(b), C.c_double(bbar), C.c_int(dim),
                            C.c_double(sigma), C.byref(out))
    _check(rc, "oracle_T_bkg")
    return float(out.value)


BKG_SEED_XOR = 0x9E3779B97F4A7C15  # reading R18: the background pool draws from the stream of seed ^ this constant


def bkg_perm_purity(b: float, bbar: float, n: int, nbar: int):
    """Reading R18: the numbers of background events (b', bbar') that Eq. 3 subtracts from the PERMUTED main samples.
    A random reassignment of the n + nbar pooled main events, b + bbar of which are background, to samples of sizes n
    and nbar puts (b + bbar) n / (n + nbar) background events into X' and (b + bbar) nbar / (n + nbar) into Xbar' on
    average (the purities are consistent for the permuted samples).  Pinned in tests/test_oracle_pins.py by
    enumerating every split of a tagged pool (n != nbar, so that a swapped formula fails)."""
    tot = b + bbar
    return tot * n / (n + nbar), tot * nbar / (n + nbar)


def bkg_perm_test(x, xbar, bx, bxbar, b: float, bbar: float, sigma: float, nperm: int, seed: int):
    """Permutation test with Eq. 3 as the statistic ("using the same method to remove background from the
    randomly permuted samples"; reading R18).  Permutation p reassigns the pooled main events to main samples of sizes
    (n, nbar) with the labels of reading R4 from `seed`, and the pooled background-sample events to samples of sizes
    (bs, bsbar) with the labels from `seed ^ BKG_SEED_XOR`; a random flavour gives both main samples the same purity, so
    the permuted samples are evaluated with b' = (b + bbar) n / (n + nbar), bbar' = (b + bbar) nbar / (n + nbar).
    Every T_p is Eq. 3 from scratch (`T_bkg`).  Returns (T_obs, T_perm, count_gt, p_value)."""
    x, xbar, bx, bxbar = (np.atleast_2d(_f64(a)) for a in (x, xbar, bx, bxbar))
    n, nbar, bs, bsbar = len(x), len(xbar), len(bx), len(bxbar)
    t_obs = T_bkg(x, xbar, bx, bxbar, b, bbar, sigma)
    main, side = np.vstack([x, xbar]), np.vstack([bx, bxbar])
    am = labels_range(n + nbar, n, 0, nperm, seed)
    ab = labels_range(bs + bsbar, bs, 0, nperm, seed ^ BKG_SEED_XOR)
    bp, bbp = bkg_perm_purity(b, bbar, n, nbar)
    t_perm = np.empty(nperm)
    for p in range(nperm):
        t_perm[p] = T_bkg(main[am[p] == 1], main[am[p] == 0], side[ab[p] == 1], side[ab[p] == 0], bp, bbp, sigma)
    count = int((t_perm > t_obs).sum())
    return t_obs, t_perm, count, count / nperm
