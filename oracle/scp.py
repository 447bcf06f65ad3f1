"""Oracle for the binned S_CP chi^2 (Sect. 2.1, Eq. 1 at :29) -- TEST INFRASTRUCTURE ONLY, like the
rest of oracle/.

Eq. 1:  S_CP^i = (N^i(X) - alpha N^i(Xbar)) / sqrt(N^i(X) + alpha^2 N^i(Xbar)),  alpha = N_tot(X) / N_tot(Xbar),
chi^2 = sum_i (S_CP^i)^2, "number of degrees of freedom; here equal to number of bins-1", the p-value
"computed directly from the observed chi^2 value and the number of degrees of freedom".

The paper leaves the binning to the analyst; readings R19-R21 fix what it does not say:
  R19  bins are a uniform rectangular grid: axis k has nbins[k] equal bins over [lo[k], hi[k]], bin index
       floor(((x - lo) / (hi - lo)) * nbins) evaluated in fp64 in exactly this order, x == hi falls into the last bin,
       an event outside the box on any axis (or not finite) is left out and counted in `n_outside`;
  R20  N_tot are the yields INSIDE the grid (the sums of the bin contents), so that sum_i (N^i(X) - alpha N^i(Xbar)) = 0,
       the one linear constraint that "bins - 1" counts;
  R21  a bin that is empty in both samples (outside the kinematic boundary on a rectangular grid) has 0/0 in Eq. 1: it
       is not a bin -- S = 0, not counted in ndf.
Steps: the bin index of every event by the formula of R19 (numpy fp64 elementwise arithmetic), numpy.bincount as the
counting primitive, Eq. 1 bin by bin, scipy.stats.chi2.sf for the p-value.  Shares no code with
paper_1612_04705_b200/csrc.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
from scipy.stats import chi2 as _chi2


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
    S: np.ndarray        # [prod(nbins)] S_CP^i, 0 in empty bins
    Nx: np.ndarray       # [prod(nbins)] int64
    Nxbar: np.ndarray    # [prod(nbins)] int64


def bin_index(x, lo, hi, nbins):
    """Flat bin index of every event (axis 0 slowest ... last axis fastest), -1 outside the grid (R19)."""
    x = np.asarray(x, dtype=np.float64)
    lo = np.asarray(lo, dtype=np.float64)
    hi = np.asarray(hi, dtype=np.float64)
    nbins = np.asarray(nbins, dtype=np.int64)
    n, dim = x.shape
    flat = np.zeros(n, dtype=np.int64)
    inside = np.ones(n, dtype=bool)
    for k in range(dim):
        with np.errstate(invalid="ignore"):
            t = (x[:, k] - lo[k]) / (hi[k] - lo[k])
            b = np.floor(t * float(nbins[k]))
        ok = np.isfinite(x[:, k]) & (x[:, k] >= lo[k]) & (x[:, k] <= hi[k])
        b = np.where(ok, b, 0.0).astype(np.int64)
        b = np.minimum(b, nbins[k] - 1)  # x == hi, or the product rounding up to nbins
        inside &= ok
        flat = flat * nbins[k] + b
    return np.where(inside, flat, -1)


def scp(x, xbar, lo, hi, nbins) -> ScpResult:
    """Eq. 1 on a uniform grid."""
    nb = int(np.prod(np.asarray(nbins, dtype=np.int64)))
    ix, ib = bin_index(x, lo, hi, nbins), bin_index(xbar, lo, hi, nbins)
    Nx = np.bincount(ix[ix >= 0], minlength=nb).astype(np.int64)
    Nb = np.bincount(ib[ib >= 0], minlength=nb).astype(np.int64)
    ntx, ntb = int(Nx.sum()), int(Nb.sum())
    alpha = ntx / ntb if ntb > 0 else float("nan")
    S = np.zeros(nb, dtype=np.float64)
    chi2 = 0.0
    used = 0
    for i in range(nb):
        if Nx[i] == 0 and Nb[i] == 0:
            continue
        used += 1
        S[i] = (Nx[i] - alpha * Nb[i]) / np.sqrt(Nx[i] + alpha * alpha * Nb[i])
        chi2 += S[i] * S[i]
    ndf = used - 1
    p = float(_chi2.sf(chi2, ndf)) if ndf > 0 and np.isfinite(chi2) else float("nan")
    return ScpResult(chi2, ndf, p, alpha, ntx, ntb, int((ix < 0).sum() + (ib < 0).sum()), used, S, Nx, Nb)
