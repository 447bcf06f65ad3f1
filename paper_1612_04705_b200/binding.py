"""Thin ctypes front of libet.so (include/et.h): argument marshalling only.

Every step of the path runs inside the CUDA library; this module turns numpy
arrays (host memory) or torch CUDA tensors (device memory) into the plain
pointers and sizes of the C ABI and copies the result structs into dataclasses.
There is no CPU fallback: if libet.so is missing, cannot be loaded, or no CUDA
device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libet.so")

ET_OK = 0
ET_F32, ET_F64 = 0, 1
ET_HOST, ET_DEVICE = 0, 1
ET_OPT_PERM_KERNEL = 0
ET_OPT_PERM_OFFSET = 1
ET_OPT_EXACT_P = 2
ET_OPT_DISTANCE = 3
ET_OPT_LABEL_SELECT = 4
ET_OPT_TC_ORDER = 5
ET_OPT_TC_SKIP = 6
STATUS_NAMES = {0: "ET_OK", -1: "ET_ERR_INVALID", -2: "ET_ERR_SIGMA", -3: "ET_ERR_NONFINITE", -4: "ET_ERR_DEGENERATE",
                -5: "ET_ERR_NOMEM", -6: "ET_ERR_CUDA"}

# every symbol include/et.h declares (tests/test_abi.py checks the library exports them all)
SYMBOLS = ["et_create", "et_destroy", "et_last_error", "et_set_option", "et_set_shard", "et_get_stats", "et_version", "et_T",
           "et_T_weighted", "et_T_sigmas", "et_T_bkg", "et_bkg_permutation_test", "et_gev_pvalue", "et_permutation_test", "et_permutation_test_sigmas", "et_podd_split", "et_podd_test", "et_perm_labels", "et_row_sums", "et_scp",
           "et_static_setup", "et_T_static", "et_static_last_error"]


class EtError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


class _Result(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("T", "T_xx", "T_bb", "T_xb", "S_xx", "S_bb", "S_xb", "W", "Wbar")] + [
        ("n_pairs", C.c_int64)]


class _PermResult(C.Structure):
    _fields_ = [("observed", _Result), ("p_value", C.c_double), ("count_gt", C.c_int64), ("n_near", C.c_int64),
                ("nperm", C.c_int64)]


class _PoddResult(C.Structure):
    _fields_ = [("count", C.c_int64 * 4), ("p_even", _Result), ("p_odd", _PermResult)]


class _BkgResult(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("T", "T_xx", "T_bb", "T_xb")] + [("S", C.c_double * 10), ("w", C.c_double),
                                                                        ("wbar", C.c_double), ("n_pairs", C.c_int64)]


class _BkgPermResult(C.Structure):
    _fields_ = [("observed", _BkgResult), ("p_value", C.c_double), ("count_gt", C.c_int64), ("n_near", C.c_int64),
                ("nperm", C.c_int64)]


class _GevResult(C.Structure):
    _fields_ = ([(k, C.c_double) for k in ("mu", "sigma", "xi")] + [("cov", C.c_double * 9)] +
                [(k, C.c_double) for k in ("nll", "p_value", "p_lo", "p_med", "p_hi")] +
                [(k, C.c_int64) for k in ("n_used", "converged", "n_resampled")])


class _ScpResult(C.Structure):
    _fields_ = [("chi2", C.c_double), ("ndf", C.c_int64), ("p_value", C.c_double), ("alpha", C.c_double),
                ("n_in_x", C.c_int64), ("n_in_xbar", C.c_int64), ("n_outside", C.c_int64), ("bins_used", C.c_int64),
                ("bins_total", C.c_int64)]


class _Stats(C.Structure):
    _fields_ = [("ms_total", C.c_double), ("ms_pairs", C.c_double), ("ms_labels", C.c_double), ("launches", C.c_int64),
                ("pair_evals", C.c_int64), ("ms_dominant", C.c_double), ("dominant_launches", C.c_int64),
                ("dominant_ops", C.c_int64), ("dominant_kernel", C.c_char * 32), ("dominant_ops_executed", C.c_int64),
                ("ms_escalation", C.c_double), ("n_near_before", C.c_int64), ("n_escalated", C.c_int64),
                ("distance_form", C.c_int64)]


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
        return abs(self.T_xx) + abs(self.T_bb) + abs(self.T_xb)


@dataclass
class PermResult:
    observed: Result
    p_value: float
    count_gt: int
    n_near: int
    nperm: int
    T_perm: np.ndarray


@dataclass
class PoddResult:
    count: tuple
    p_even: Result
    p_odd: PermResult


@dataclass
class BkgResult:
    T: float
    T_xx: float
    T_bb: float
    T_xb: float
    S: tuple  # XX, XBx, XXbar, XBxbar, BxBx, BxXbar, BxBxbar, XbarXbar, XbarBxbar, BxbarBxbar
    w: float
    wbar: float
    n_pairs: int

    @property
    def term_scale(self) -> float:
        return abs(self.T_xx) + abs(self.T_bb) + abs(self.T_xb)


@dataclass
class BkgPermResult:
    observed: BkgResult
    p_value: float
    count_gt: int
    n_near: int
    nperm: int
    T_perm: np.ndarray


@dataclass
class GevResult:
    mu: float
    sigma: float
    xi: float
    cov: np.ndarray
    nll: float
    p_value: float
    p_lo: float
    p_med: float
    p_hi: float
    n_used: int
    converged: bool
    n_resampled: int


def gev_pvalue(T_perm, T_obs: float, z=None) -> GevResult:
    """GEV fit of the permutation T values and the fitted p-value of T_obs (host-only; z: [nresample, 3] standard
    normal draws for the parameter resampling, or None)."""
    tp = np.ascontiguousarray(np.asarray(T_perm, dtype=np.float64))
    zz = None if z is None else np.ascontiguousarray(np.asarray(z, dtype=np.float64).reshape(-1, 3))
    out = _GevResult()
    L = lib()
    st = L.et_gev_pvalue(tp.ctypes.data_as(C.c_void_p), len(tp), float(T_obs), None if zz is None else zz.ctypes.data_as(C.c_void_p),
                         0 if zz is None else len(zz), C.byref(out))
    if st != ET_OK:
        raise EtError(st, "et_gev_pvalue: needs >= 10 finite permutation T values with non-zero spread and a finite T_obs")
    return GevResult(out.mu, out.sigma, out.xi, np.array(out.cov).reshape(3, 3), out.nll, out.p_value, out.p_lo, out.p_med,
                     out.p_hi, out.n_used, bool(out.converged), out.n_resampled)


@dataclass
class ScpResult:
    chi2: float
    ndf: int
    p_value: float
    alpha: float
    n_in_x: int
    n_in_xbar: int
    n_outside: int
    bins_used: int
    bins_total: int
    S: np.ndarray
    Nx: np.ndarray
    Nxbar: np.ndarray


@dataclass
class Stats:
    ms_total: float
    ms_pairs: float
    ms_labels: float
    launches: int
    pair_evals: int
    ms_dominant: float = 0.0
    dominant_launches: int = 0
    dominant_ops: int = 0
    dominant_kernel: str = ""
    dominant_ops_executed: int = 0
    ms_escalation: float = 0.0
    n_near_before: int = 0
    n_escalated: int = 0
    distance_form: int = 0


_lib = None


def lib():
    """Loads libet.so; raises if the CUDA extension has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1612_04705_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i64, u64, dbl, ci = C.c_void_p, C.c_int64, C.c_uint64, C.c_double, C.c_int
        L.et_last_error.restype = C.c_char_p
        L.et_version.restype = C.c_char_p
        L.et_static_last_error.restype = C.c_char_p
        L.et_destroy.restype = None
        # the argument types of EVERY entry point of include/et.h, in its order (a missing one would let ctypes pass a
        # Python int as a 32-bit C int and truncate an int64 silently)
        sample = [vp, i64, vp, i64]                       # x, n, xbar, nbar
        wsample = [vp, vp, i64, vp, vp, i64]              # x, wx, n, xbar, wxbar, nbar
        tail = [ci, ci, ci, dbl]                          # dim, dtype, mem, sigma
        bkg = [vp] + sample + [vp, i64, vp, i64, dbl, dbl] + tail
        for name, args in {
            "et_create": [C.POINTER(vp), ci, vp], "et_destroy": [vp], "et_last_error": [vp], "et_version": [],
            "et_set_option": [vp, ci, i64], "et_set_shard": [vp, ci, ci, vp, vp], "et_get_stats": [vp, vp],
            "et_T": [vp] + sample + tail + [vp],
            "et_T_weighted": [vp] + wsample + tail + [vp],
            "et_T_sigmas": [vp] + wsample + [ci, ci, ci, vp, ci, vp],
            "et_T_bkg": bkg + [vp],
            "et_bkg_permutation_test": bkg + [i64, u64, vp, vp],
            "et_gev_pvalue": [vp, i64, dbl, vp, i64, vp],
            "et_permutation_test": [vp] + wsample + tail + [i64, u64, vp, vp],
            "et_permutation_test_sigmas": [vp] + wsample + [ci, ci, ci, vp, ci, i64, u64, vp, vp],
            "et_podd_split": [vp, vp, vp, vp, i64, ci, ci, vp, vp],
            "et_podd_test": [vp] + wsample + tail + [i64, u64, vp, vp],
            "et_perm_labels": [vp, i64, i64, i64, u64, ci, vp],
            "et_row_sums": [vp] + wsample + tail + [vp, i64, vp, vp],
            "et_scp": [vp] + sample + [ci, ci, ci, vp, vp, vp, vp, vp, vp, vp],
            "et_static_setup": [ci], "et_T_static": [ci, vp] + sample + [ci, ci, dbl, vp], "et_static_last_error": [],
        }.items():
            getattr(L, name).argtypes = args
        assert all(getattr(L, n).argtypes is not None for n in SYMBOLS)
        _lib = L
    return _lib


def _res(r: _Result) -> Result:
    return Result(*(getattr(r, k) for k, _ in _Result._fields_))


class _Arr:
    """A pointer plus what the ABI needs to know about it."""

    def __init__(self, ptr, dtype, mem, shape, keep):
        self.ptr, self.dtype, self.mem, self.shape, self.keep = ptr, dtype, mem, shape, keep


def _is_torch(a) -> bool:
    return type(a).__module__.startswith("torch")


def _marshal(a, want=None) -> _Arr:
    """numpy array -> host pointer; torch CUDA tensor -> device pointer.  `want` forces a dtype ("f64")."""
    if a is None:
        return _Arr(None, None, None, None, None)
    if _is_torch(a):
        import torch

        if want == "f64" and a.dtype != torch.float64:
            a = a.double()
        if a.dtype not in (torch.float32, torch.float64, torch.uint8, torch.int32, torch.uint32):
            a = a.double()
        a = a.contiguous()
        mem = ET_DEVICE if a.is_cuda else ET_HOST
        dt = ET_F32 if a.dtype == torch.float32 else ET_F64
        return _Arr(C.c_void_p(a.data_ptr()), dt, mem, tuple(a.shape), a)
    a = np.asarray(a)
    if want == "f64" or a.dtype not in (np.float32, np.float64):
        a = a.astype(np.float64, copy=False)   # no copy when it already is float64: a pinned buffer stays the caller's pinned buffer
    a = np.ascontiguousarray(a)
    dt = ET_F32 if a.dtype == np.float32 else ET_F64
    return _Arr(C.c_void_p(a.ctypes.data), dt, ET_HOST, a.shape, a)


def _aux(a, shape, mem, what, device=None) -> _Arr:
    """A double-precision companion array (weights, momenta): must have exactly `shape` and live where the coordinates
    live, or the library would read past its end."""
    r = _marshal(a, "f64")
    if r.ptr is None:
        return r
    if tuple(r.shape) != tuple(shape):
        raise ValueError(f"{what} must have shape {tuple(shape)}, got {tuple(r.shape)}")
    if r.mem != mem:
        raise ValueError(f"{what} must live where the coordinates live")
    if device is not None and r.mem == ET_DEVICE and r.keep.device.index != device:
        raise ValueError(f"{what} is on cuda:{r.keep.device.index}, the coordinates on cuda:{device}")
    return r


def _coords(x, xbar):
    ax, ab = _marshal(x), _marshal(xbar)
    if ax.mem != ab.mem or ax.dtype != ab.dtype:
        raise ValueError("x and xbar must share memory space and dtype")
    if len(ax.shape) == 1:
        ax.shape, ab.shape = (ax.shape[0], 1), (ab.shape[0], 1)
    if len(ax.shape) != 2 or len(ab.shape) != 2 or ax.shape[1] != ab.shape[1]:
        raise ValueError("x and xbar must be [n, dim] and [nbar, dim]")
    if ax.mem == ET_DEVICE and ax.keep.device != ab.keep.device:
        raise ValueError("x and xbar must be on the same CUDA device")
    return ax, ab


def _weights(ax, ab, wx, wxbar):
    if (wx is None) != (wxbar is None):
        raise ValueError("give both weight arrays or neither")
    dev = ax.keep.device.index if ax.mem == ET_DEVICE else None
    return _aux(wx, (ax.shape[0],), ax.mem, "wx", dev), _aux(wxbar, (ab.shape[0],), ax.mem, "wxbar", dev)


_ALLGATHER = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_int64)


def make_allgather(rank: int, world: int, group=None):
    """The et_allgather_fn of include/et.h on torch.distributed: buf is host memory [world][nbytes] with slice `rank`
    filled in; on return every slice holds that rank's bytes.  Pure data movement (no arithmetic): the library sums the
    slices on the device.  NCCL moves device tensors, so there the slices travel through a small CUDA staging tensor."""
    def fn(_user, buf, nbytes):
        try:
            import torch
            import torch.distributed as dist

            raw = (C.c_uint8 * (world * nbytes)).from_address(buf)
            host = torch.frombuffer(raw, dtype=torch.uint8).view(world, nbytes)
            if dist.get_backend(group) == "nccl":
                mine = host[rank].cuda()
                parts = torch.empty(world, nbytes, dtype=torch.uint8, device=mine.device)
                dist.all_gather_into_tensor(parts, mine, group=group)
                host.copy_(parts.cpu())
            else:
                parts = [torch.empty(nbytes, dtype=torch.uint8) for _ in range(world)]
                dist.all_gather(parts, host[rank].clone(), group=group)
                for r in range(world):
                    host[r].copy_(parts[r])
            return 0
        except Exception:  # an exception must not unwind through the C caller
            import traceback

            traceback.print_exc()
            return 1
    return fn


# ---- the entry point that allocates nothing (include/et.h, csrc/et_static.cu) -------------------------------------
STATIC_SCRATCH_BYTES = 8 << 20
RESULT_DOUBLES = C.sizeof(_Result) // 8   # a device et_result is this many 8-byte words (the last one an int64)


def static_setup(device: int = 0) -> None:
    """Once per device, outside any graph capture: resolves the device address of the library's static scratch."""
    st = lib().et_static_setup(C.c_int(device))
    if st != ET_OK:
        raise EtError(st, lib().et_static_last_error().decode())


def T_static(x, xbar, sigma: float, out, stream=None) -> None:
    """et_T_static: x, xbar are CUDA tensors [n, dim] (float32 or float64, same device), `out` a CUDA float64 tensor of
    RESULT_DOUBLES elements on that device (the device et_result).  Enqueues on `stream` (None: the legacy default
    stream) and returns without synchronising; decode a host copy of `out` with result_from_words."""
    ax, ab = _coords(x, xbar)
    if ax.mem != ET_DEVICE:
        raise ValueError("T_static takes device tensors (there is no staging: the call allocates nothing)")
    import torch

    if not (_is_torch(out) and out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= RESULT_DOUBLES
            and out.device.index == ax.keep.device.index):
        raise ValueError(f"out must be a contiguous CUDA float64 tensor of >= {RESULT_DOUBLES} elements on the inputs' device")
    sp = None if stream is None else C.c_void_p(int(getattr(stream, "cuda_stream", stream)))
    st = lib().et_T_static(C.c_int(ax.keep.device.index), sp, ax.ptr, C.c_int64(ax.shape[0]), ab.ptr, C.c_int64(ab.shape[0]),
                           C.c_int(ax.shape[1]), C.c_int(ax.dtype), C.c_double(sigma), C.c_void_p(out.data_ptr()))
    if st != ET_OK:
        raise EtError(st, lib().et_static_last_error().decode())


def result_from_words(words) -> Result:
    """A host copy (numpy float64[RESULT_DOUBLES]) of a device et_result -> Result."""
    w = np.ascontiguousarray(np.asarray(words, dtype=np.float64)[:RESULT_DOUBLES])
    return _res(_Result.from_buffer_copy(w.tobytes()))


class Context:
    """One et_ctx: a device, a stream and the scratch of the library.  Not thread-safe."""

    def __init__(self, device: int = 0, stream=None):
        self._h = C.c_void_p()
        L = lib()
        sp = None
        if stream is not None:
            sp = C.c_void_p(int(getattr(stream, "cuda_stream", stream)))
        st = L.et_create(C.byref(self._h), device, sp)
        if st != ET_OK:
            self._h = C.c_void_p()
            raise EtError(st, "et_create failed (no CUDA device? there is no CPU fallback)")

    def close(self):
        if self._h:
            lib().et_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check(self, st):
        if st != ET_OK:
            raise EtError(st, lib().et_last_error(self._h).decode())

    def set_option(self, opt: int, value: int):
        self._check(lib().et_set_option(self._h, C.c_int(opt), C.c_int64(value)))

    def set_shard(self, rank: int, world: int, group=None):
        """Unit-range shard over the ranks of a torch.distributed process group (et_set_shard): this context evaluates
        every world-th work unit of the O(N^2) kernels, and the library's partial sums are completed by an all-gather on
        `group` (NCCL or gloo).  world = 1 switches the shard off."""
        if world <= 1:
            self._shard_cb = None
            self._check(lib().et_set_shard(self._h, 0, 1, None, None))
            return
        self._shard_cb = _ALLGATHER(make_allgather(rank, world, group))
        self._check(lib().et_set_shard(self._h, rank, world, C.cast(self._shard_cb, C.c_void_p), None))

    def stats(self) -> Stats:
        s = _Stats()
        self._check(lib().et_get_stats(self._h, C.byref(s)))
        return Stats(s.ms_total, s.ms_pairs, s.ms_labels, s.launches, s.pair_evals, s.ms_dominant, s.dominant_launches,
                     s.dominant_ops, s.dominant_kernel.decode(), s.dominant_ops_executed, s.ms_escalation, s.n_near_before,
                     s.n_escalated, s.distance_form)

    # ---------------------------------------------------------------- Eq. 2
    def T(self, x, xbar, sigma: float) -> Result:
        ax, ab = _coords(x, xbar)
        out = _Result()
        self._check(lib().et_T(self._h, ax.ptr, C.c_int64(ax.shape[0]), ab.ptr, C.c_int64(ab.shape[0]), C.c_int(ax.shape[1]),
                               C.c_int(ax.dtype), C.c_int(ax.mem), C.c_double(sigma), C.byref(out)))
        return _res(out)

    def T_weighted(self, x, wx, xbar, wxbar, sigma: float) -> Result:
        ax, ab = _coords(x, xbar)
        if wx is None or wxbar is None:
            raise ValueError("T_weighted needs both weight arrays")
        awx, awb = _weights(ax, ab, wx, wxbar)
        out = _Result()
        self._check(lib().et_T_weighted(self._h, ax.ptr, awx.ptr, C.c_int64(ax.shape[0]), ab.ptr, awb.ptr, C.c_int64(ab.shape[0]),
                                        C.c_int(ax.shape[1]), C.c_int(ax.dtype), C.c_int(ax.mem), C.c_double(sigma), C.byref(out)))
        return _res(out)

    def T_sigmas(self, x, xbar, sigmas, wx=None, wxbar=None) -> list:
        """Eq. 2 (weighted if wx, wxbar are given) for up to four sigma values from one pass over the pairs."""
        ax, ab = _coords(x, xbar)
        awx, awb = _weights(ax, ab, wx, wxbar)
        sg = np.ascontiguousarray(np.asarray(sigmas, dtype=np.float64))
        out = (_Result * max(len(sg), 1))()
        self._check(lib().et_T_sigmas(self._h, ax.ptr, awx.ptr, C.c_int64(ax.shape[0]), ab.ptr, awb.ptr, C.c_int64(ab.shape[0]),
                                      C.c_int(ax.shape[1]), C.c_int(ax.dtype), C.c_int(ax.mem), sg.ctypes.data_as(C.c_void_p),
                                      C.c_int(len(sg)), out))
        return [_res(out[k]) for k in range(len(sg))]

    def T_bkg(self, x, xbar, bx, bxbar, b: float, bbar: float, sigma: float) -> BkgResult:
        """Eq. 3: background-sample-subtracted T (main samples x, xbar; background samples bx, bxbar)."""
        ax, ab = _coords(x, xbar)
        abx, abb = _coords(bx, bxbar)
        if (abx.mem, abx.dtype, abx.shape[1]) != (ax.mem, ax.dtype, ax.shape[1]):
            raise ValueError("background samples must share memory space, dtype and dim with the main samples")
        out = _BkgResult()
        self._check(lib().et_T_bkg(self._h, ax.ptr, C.c_int64(ax.shape[0]), ab.ptr, C.c_int64(ab.shape[0]), abx.ptr,
                                   C.c_int64(abx.shape[0]), abb.ptr, C.c_int64(abb.shape[0]), C.c_double(b), C.c_double(bbar),
                                   C.c_int(ax.shape[1]), C.c_int(ax.dtype), C.c_int(ax.mem), C.c_double(sigma), C.byref(out)))
        return BkgResult(out.T, out.T_xx, out.T_bb, out.T_xb, tuple(out.S), out.w, out.wbar, out.n_pairs)

    def bkg_permutation_test(self, x, xbar, bx, bxbar, b: float, bbar: float, sigma: float, nperm: int, seed: int) -> BkgPermResult:
        """Permutation test with Eq. 3 as the statistic (main and background pools permuted independently)."""
        ax, ab = _coords(x, xbar)
        abx, abb = _coords(bx, bxbar)
        if (abx.mem, abx.dtype, abx.shape[1]) != (ax.mem, ax.dtype, ax.shape[1]):
            raise ValueError("background samples must share memory space, dtype and dim with the main samples")
        Tp = np.zeros(max(int(nperm), 1), dtype=np.float64)
        out = _BkgPermResult()
        self._check(lib().et_bkg_permutation_test(
            self._h, ax.ptr, C.c_int64(ax.shape[0]), ab.ptr, C.c_int64(ab.shape[0]), abx.ptr, C.c_int64(abx.shape[0]), abb.ptr,
            C.c_int64(abb.shape[0]), C.c_double(b), C.c_double(bbar), C.c_int(ax.shape[1]), C.c_int(ax.dtype), C.c_int(ax.mem),
            C.c_double(sigma), C.c_int64(nperm), C.c_uint64(seed), Tp.ctypes.data_as(C.c_void_p), C.byref(out)))
        o = out.observed
        return BkgPermResult(BkgResult(o.T, o.T_xx, o.T_bb, o.T_xb, tuple(o.S), o.w, o.wbar, o.n_pairs), out.p_value,
                             out.count_gt, out.n_near, out.nperm, Tp)

    # ---------------------------------------------------------------- permutation test
    def permutation_test(self, x, xbar, sigma: float, nperm: int, seed: int, wx=None, wxbar=None) -> PermResult:
        ax, ab = _coords(x, xbar)
        awx, awb = _weights(ax, ab, wx, wxbar)
        Tp = np.zeros(max(int(nperm), 1), dtype=np.float64)
        out = _PermResult()
        self._check(lib().et_permutation_test(self._h, ax.ptr, awx.ptr, C.c_int64(ax.shape[0]), ab.ptr, awb.ptr,
                                              C.c_int64(ab.shape[0]), C.c_int(ax.shape[1]), C.c_int(ax.dtype), C.c_int(ax.mem),
                                              C.c_double(sigma), C.c_int64(nperm), C.c_uint64(seed),
                                              Tp.ctypes.data_as(C.c_void_p), C.byref(out)))
        return PermResult(_res(out.observed), out.p_value, out.count_gt, out.n_near, out.nperm, Tp)

    def permutation_test_sigmas(self, x, xbar, sigmas, nperm: int, seed: int, wx=None, wxbar=None) -> list:
        """The permutation test at several sigma (the scan of Fig. 2): one PermResult per sigma, labels generated once."""
        ax, ab = _coords(x, xbar)
        awx, awb = _weights(ax, ab, wx, wxbar)
        sg = np.ascontiguousarray(np.asarray(sigmas, dtype=np.float64).reshape(-1))
        Tp = np.zeros((max(len(sg), 1), max(int(nperm), 1)), dtype=np.float64)
        out = (_PermResult * max(len(sg), 1))()
        self._check(lib().et_permutation_test_sigmas(
            self._h, ax.ptr, awx.ptr, C.c_int64(ax.shape[0]), ab.ptr, awb.ptr, C.c_int64(ab.shape[0]), C.c_int(ax.shape[1]),
            C.c_int(ax.dtype), C.c_int(ax.mem), sg.ctypes.data_as(C.c_void_p), C.c_int(len(sg)), C.c_int64(nperm), C.c_uint64(seed),
            Tp.ctypes.data_as(C.c_void_p), out))
        return [PermResult(_res(out[k].observed), out[k].p_value, out[k].count_gt, out[k].n_near, out[k].nperm, Tp[k].copy())
                for k in range(len(sg))]

    # ---------------------------------------------------------------- Sect. 5
    def podd_split(self, pB, pC, pD, is_conjugate: bool):
        aB, aC, aD = _marshal(pB, "f64"), _marshal(pC, "f64"), _marshal(pD, "f64")
        n = aB.shape[0]
        if not (tuple(aB.shape) == tuple(aC.shape) == tuple(aD.shape) == (n, 3)) or not (aB.mem == aC.mem == aD.mem):
            raise ValueError("pB, pC, pD must be [n, 3] arrays in the same memory space")
        cnt = C.c_int64(0)
        if aB.mem == ET_DEVICE:
            import torch

            pos = torch.empty(n, dtype=torch.uint8, device=aB.keep.device)
            pp = C.c_void_p(pos.data_ptr())
        else:
            pos = np.zeros(n, dtype=np.uint8)
            pp = pos.ctypes.data_as(C.c_void_p)
        self._check(lib().et_podd_split(self._h, aB.ptr, aC.ptr, aD.ptr, C.c_int64(n), C.c_int(int(is_conjugate)),
                                        C.c_int(aB.mem), pp, C.byref(cnt)))
        return pos, int(cnt.value)

    def podd_test(self, x, mom_x, xbar, mom_xbar, sigma: float, nperm: int, seed: int) -> PoddResult:
        ax, ab = _coords(x, xbar)
        dev = ax.keep.device.index if ax.mem == ET_DEVICE else None
        amx = _aux(mom_x, (ax.shape[0], 3, 3), ax.mem, "mom_x", dev)
        amb = _aux(mom_xbar, (ab.shape[0], 3, 3), ax.mem, "mom_xbar", dev)
        if amx.ptr is None or amb.ptr is None:
            raise ValueError("podd_test needs the momenta of both samples")
        Tp = np.zeros(max(int(nperm), 1), dtype=np.float64)
        out = _PoddResult()
        self._check(lib().et_podd_test(self._h, ax.ptr, amx.ptr, C.c_int64(ax.shape[0]), ab.ptr, amb.ptr, C.c_int64(ab.shape[0]),
                                       C.c_int(ax.shape[1]), C.c_int(ax.dtype), C.c_int(ax.mem), C.c_double(sigma),
                                       C.c_int64(nperm), C.c_uint64(seed), Tp.ctypes.data_as(C.c_void_p), C.byref(out)))
        po = out.p_odd
        return PoddResult(tuple(out.count), _res(out.p_even),
                          PermResult(_res(po.observed), po.p_value, po.count_gt, po.n_near, po.nperm, Tp))

    # ---------------------------------------------------------------- test hooks
    def perm_labels(self, N: int, n: int, nperm: int, seed: int) -> np.ndarray:
        mask = np.zeros((N, (nperm + 31) // 32), dtype=np.uint32)
        self._check(lib().et_perm_labels(self._h, C.c_int64(N), C.c_int64(n), C.c_int64(nperm), C.c_uint64(seed),
                                         C.c_int(ET_HOST), mask.ctypes.data_as(C.c_void_p)))
        return mask

    def row_sums(self, x, xbar, sigma: float, rows, wx=None, wxbar=None):
        ax, ab = _coords(x, xbar)
        awx, awb = _weights(ax, ab, wx, wxbar)
        rows = np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
        rx, rb = np.zeros(len(rows)), np.zeros(len(rows))
        self._check(lib().et_row_sums(self._h, ax.ptr, awx.ptr, C.c_int64(ax.shape[0]), ab.ptr, awb.ptr, C.c_int64(ab.shape[0]),
                                      C.c_int(ax.shape[1]), C.c_int(ax.dtype), C.c_int(ax.mem), C.c_double(sigma),
                                      rows.ctypes.data_as(C.c_void_p), C.c_int64(len(rows)),
                                      rx.ctypes.data_as(C.c_void_p), rb.ctypes.data_as(C.c_void_p)))
        return rx, rb

    # ---------------------------------------------------------------- Sect. 2.1
    def scp(self, x, xbar, lo, hi, nbins) -> ScpResult:
        """Binned S_CP chi^2 (Eq. 1) on a uniform grid: axis k has nbins[k] equal bins over [lo[k], hi[k]]."""
        ax, ab = _coords(x, xbar)
        dim = ax.shape[1]
        alo = np.ascontiguousarray(np.asarray(lo, dtype=np.float64).reshape(-1))
        ahi = np.ascontiguousarray(np.asarray(hi, dtype=np.float64).reshape(-1))
        anb = np.ascontiguousarray(np.asarray(nbins, dtype=np.int32).reshape(-1))
        if not (len(alo) == len(ahi) == len(anb) == dim):
            raise ValueError(f"lo, hi, nbins must have one entry per axis ({dim})")
        if (anb < 1).any() or int(np.prod(anb.astype(np.int64))) > 1 << 24:
            raise ValueError("nbins must be >= 1 per axis and at most 2^24 bins in total")
        total = int(np.prod(anb.astype(np.int64)))
        S, Nx, Nb = np.zeros(total), np.zeros(total, dtype=np.int64), np.zeros(total, dtype=np.int64)
        out = _ScpResult()
        self._check(lib().et_scp(self._h, ax.ptr, C.c_int64(ax.shape[0]), ab.ptr, C.c_int64(ab.shape[0]), C.c_int(dim),
                                 C.c_int(ax.dtype), C.c_int(ax.mem), alo.ctypes.data_as(C.c_void_p), ahi.ctypes.data_as(C.c_void_p),
                                 anb.ctypes.data_as(C.c_void_p), S.ctypes.data_as(C.c_void_p), Nx.ctypes.data_as(C.c_void_p),
                                 Nb.ctypes.data_as(C.c_void_p), C.byref(out)))
        return ScpResult(out.chi2, out.ndf, out.p_value, out.alpha, out.n_in_x, out.n_in_xbar, out.n_outside, out.bins_used,
                         out.bins_total, S, Nx, Nb)
