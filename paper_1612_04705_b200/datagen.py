"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module serves BOTH the oracle and the CUDA path (tests, bench, smoke) and
therefore holds none of the method's arithmetic: no psi, no T, no labels.  It
only makes event samples with the shapes, sizes and value distributions of the
paper's workloads (PAPER.md:39, 105, 203 give sizes and decay channels; the
Laura++ / MINT samples themselves are not available, so uniform phase space
plus a localised bump stands in for them -- DESIGN.md "Input recipe").

Everything is drawn from ``numpy.random.Generator(numpy.random.Philox(seed))``
in a fixed batch schedule, so a (config, seed) pair always yields the same bytes.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# PDG-style masses in GeV, as fixed by BASELINE.json configs[0] and configs[2].
M_DPLUS = 1.86966
M_D0 = 1.86484
M_K = 0.493677
M_PI = 0.13957


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(seed))


# --------------------------------------------------------------------------- #
# 3-body Dalitz plot: D+ -> K-(1) K+(2) pi+(3), coordinates (m^2_12, m^2_23)
# --------------------------------------------------------------------------- #
def dalitz_box(M=M_DPLUS, m1=M_K, m2=M_K, m3=M_PI):
    """Bounding box of the Dalitz region in (s12, s23)."""
    return ((m1 + m2) ** 2, (M - m3) ** 2), ((m2 + m3) ** 2, (M - m1) ** 2)


def dalitz_inside(s12, s23, M=M_DPLUS, m1=M_K, m2=M_K, m3=M_PI):
    """Kinematic boundary of a three-body decay (two-body-subsystem form)."""
    s12 = np.asarray(s12, dtype=np.float64)
    s23 = np.asarray(s23, dtype=np.float64)
    (lo12, hi12), _ = dalitz_box(M, m1, m2, m3)
    ok = (s12 > lo12) & (s12 < hi12)
    s = np.where(ok, s12, 0.5 * (lo12 + hi12))
    rt = np.sqrt(s)
    e2 = (s - m1 * m1 + m2 * m2) / (2.0 * rt)
    e3 = (M * M - s - m3 * m3) / (2.0 * rt)
    p2 = np.sqrt(np.maximum(e2 * e2 - m2 * m2, 0.0))
    p3 = np.sqrt(np.maximum(e3 * e3 - m3 * m3, 0.0))
    lo = (e2 + e3) ** 2 - (p2 + p3) ** 2
    hi = (e2 + e3) ** 2 - (p2 - p3) ** 2
    return ok & (s23 > lo) & (s23 < hi)


def dalitz_uniform(n: int, rng: np.random.Generator) -> np.ndarray:
    """n points uniform inside the D+ -> K-K+pi+ Dalitz boundary (accept-reject)."""
    (lo12, hi12), (lo23, hi23) = dalitz_box()
    out = np.empty((n, 2), dtype=np.float64)
    have = 0
    while have < n:
        m = max(1024, int((n - have) * 2.0))
        a = rng.uniform(lo12, hi12, m)
        b = rng.uniform(lo23, hi23, m)
        keep = dalitz_inside(a, b)
        a, b = a[keep], b[keep]
        k = min(n - have, a.size)
        out[have:have + k, 0] = a[:k]
        out[have:have + k, 1] = b[:k]
        have += k
    return out


def dalitz_with_bump(n: int, rng: np.random.Generator, frac: float, centre=(1.04, 1.5), width=0.05) -> np.ndarray:
    """Reading R14: each event is, with probability ``frac``, drawn from an isotropic
    normal (std ``width`` GeV^2 per axis) at ``centre``, redrawn until inside the
    boundary; otherwise from the uniform generator."""
    out = dalitz_uniform(n, rng)
    is_bump = rng.uniform(0.0, 1.0, n) < frac
    idx = np.flatnonzero(is_bump)
    todo = idx
    while todo.size:
        a = rng.normal(centre[0], width, todo.size)
        b = rng.normal(centre[1], width, todo.size)
        keep = dalitz_inside(a, b)
        out[todo[keep], 0] = a[keep]
        out[todo[keep], 1] = b[keep]
        todo = todo[~keep]
    return out


# --------------------------------------------------------------------------- #
# 4-body flat phase space: D0 -> K-(1) K+(2) pi+(3) pi-(4)
# --------------------------------------------------------------------------- #
def _q(M, m1, m2):
    """Two-body break-up momentum."""
    t = (M * M - (m1 + m2) ** 2) * (M * M - (m1 - m2) ** 2)
    return np.sqrt(np.maximum(t, 0.0)) / (2.0 * M)


def _iso(n, rng):
    c = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2.0 * np.pi, n)
    s = np.sqrt(1.0 - c * c)
    return np.stack([s * np.cos(ph), s * np.sin(ph), c], axis=1)


def _boost(p, e, beta_vec, gamma):
    """Boost (p, e) by velocity beta_vec (each row)."""
    b2 = np.sum(beta_vec * beta_vec, axis=1)
    bp = np.sum(beta_vec * p, axis=1)
    g2 = np.where(b2 > 0, (gamma - 1.0) / np.where(b2 > 0, b2, 1.0), 0.0)
    p_new = p + (g2 * bp + gamma * e)[:, None] * beta_vec
    e_new = gamma * (e + bp)
    return p_new, e_new


FOURBODY_MASSES = (M_K, M_K, M_PI, M_PI)
FOURBODY_WMAX = 0.0270  # >= max of q(M;m123,m4) q(m123;m12,m3) q(m12;m1,m2) over the allowed masses (checked in tests)


def fourbody_limits(M=M_D0, masses=FOURBODY_MASSES):
    """Kinematic limits of (m^2_12, m^2_34, m^2_123, m^2_234, m^2_14), reading R15."""
    m1, m2, m3, m4 = masses
    return np.array(
        [
            [(m1 + m2) ** 2, (M - m3 - m4) ** 2],
            [(m3 + m4) ** 2, (M - m1 - m2) ** 2],
            [(m1 + m2 + m3) ** 2, (M - m4) ** 2],
            [(m2 + m3 + m4) ** 2, (M - m1) ** 2],
            [(m1 + m4) ** 2, (M - m2 - m3) ** 2],
        ]
    )


def fourbody_phase_space(n: int, rng: np.random.Generator, M=M_D0, masses=FOURBODY_MASSES):
    """n flat-phase-space events by sequential two-body decays
    M -> R123 + 4, R123 -> R12 + 3, R12 -> 1 + 2, isotropic in each rest frame,
    accept-reject on the product of break-up momenta.

    Returns (coords[n,5] mapped to the unit range, p[n,4,3] momenta and e[n,4]
    energies of particles 1..4 in the mother rest frame)."""
    m1, m2, m3, m4 = masses
    tkin = M - (m1 + m2 + m3 + m4)
    P = np.empty((n, 4, 3))
    E = np.empty((n, 4))
    have = 0
    while have < n:
        m = max(1024, int((n - have) * 1.8))
        r = np.sort(rng.uniform(0.0, 1.0, (m, 2)), axis=1)
        m12 = m1 + m2 + r[:, 0] * tkin
        m123 = m1 + m2 + m3 + r[:, 1] * tkin
        q4 = _q(M, m123, m4)
        q3 = _q(m123, m12, m3)
        q2 = _q(m12, m1, m2)
        wt = q4 * q3 * q2
        u = rng.uniform(0.0, FOURBODY_WMAX, m)
        d4, d3, d2 = _iso(m, rng), _iso(m, rng), _iso(m, rng)
        keep = u < wt
        m12, m123, q4, q3, q2 = m12[keep], m123[keep], q4[keep], q3[keep], q2[keep]
        d4, d3, d2 = d4[keep], d3[keep], d2[keep]
        k = min(n - have, m12.size)
        m12, m123, q4, q3, q2, d4, d3, d2 = (a[:k] for a in (m12, m123, q4, q3, q2, d4, d3, d2))
        # mother frame: particle 4 and R123 back to back
        p4 = q4[:, None] * d4
        e4 = np.sqrt(q4 * q4 + m4 * m4)
        pR3 = -p4
        eR3 = np.sqrt(q4 * q4 + m123 * m123)
        # R123 frame: particle 3 and R12
        p3 = q3[:, None] * d3
        e3 = np.sqrt(q3 * q3 + m3 * m3)
        pR2 = -p3
        eR2 = np.sqrt(q3 * q3 + m12 * m12)
        # R12 frame: particles 1, 2
        p1 = q2[:, None] * d2
        e1 = np.sqrt(q2 * q2 + m1 * m1)
        p2 = -p1
        e2 = np.sqrt(q2 * q2 + m2 * m2)
        # boost 1, 2 from the R12 frame to the R123 frame
        b2 = pR2 / eR2[:, None]
        g2 = eR2 / m12
        p1, e1 = _boost(p1, e1, b2, g2)
        p2, e2 = _boost(p2, e2, b2, g2)
        # boost 1, 2, 3 from the R123 frame to the mother frame
        b3 = pR3 / eR3[:, None]
        g3 = eR3 / m123
        p1, e1 = _boost(p1, e1, b3, g3)
        p2, e2 = _boost(p2, e2, b3, g3)
        p3, e3 = _boost(p3, e3, b3, g3)
        sl = slice(have, have + k)
        P[sl, 0], P[sl, 1], P[sl, 2], P[sl, 3] = p1, p2, p3, p4
        E[sl, 0], E[sl, 1], E[sl, 2], E[sl, 3] = e1, e2, e3, e4
        have += k

    def m2_of(idx):
        e = sum(E[:, i] for i in idx)
        p = sum(P[:, i] for i in idx)
        return e * e - np.sum(p * p, axis=1)

    raw = np.stack([m2_of((0, 1)), m2_of((2, 3)), m2_of((0, 1, 2)), m2_of((1, 2, 3)), m2_of((0, 3))], axis=1)
    lim = fourbody_limits(M, masses)
    coords = (raw - lim[:, 0]) / (lim[:, 1] - lim[:, 0])
    return coords, P, E


# --------------------------------------------------------------------------- #
# The five configurations
# --------------------------------------------------------------------------- #
@dataclass
class Config:
    index: int
    name: str
    n: int
    nbar: int
    dim: int
    sigmas: tuple
    nperm: int
    coord_dtype: str  # "f64" or "f32": the dtype the coordinates are supplied in
    weighted: bool = False
    podd: bool = False
    bump_frac: float = 0.0
    perm_seed: int = field(default=0)

    @property
    def sigma(self) -> float:
        """Headline sigma of the configuration."""
        return self.sigmas[len(self.sigmas) // 2] if len(self.sigmas) > 1 else self.sigmas[0]


def config(index: int, scale: float = 1.0) -> Config:
    """BASELINE.json configs[index]; ``scale`` shrinks n and nbar (tests only)."""
    base = {
        0: Config(0, "dalitz3_2k", 2000, 2000, 2, (0.3,), 50, "f64", bump_frac=0.05),
        1: Config(1, "dalitz3_100k_f32", 100_000, 100_000, 2, (0.1, 0.3, 0.5), 1000, "f32", bump_frac=0.01),
        2: Config(2, "kkpipi_300k_5d", 300_000, 300_000, 5, (0.2,), 1000, "f64"),
        3: Config(3, "dalitz3_200k_weighted", 200_000, 200_000, 2, (0.1, 0.3, 0.5), 1000, "f32", weighted=True,
                  bump_frac=0.01),
        4: Config(4, "kkpipi_1m_podd", 1_000_000, 1_000_000, 5, (0.2,), 1000, "f64", podd=True),
    }[index]
    base.perm_seed = 0xE7E57 + index
    if scale != 1.0:
        base.n = max(2, int(round(base.n * scale)))
        base.nbar = max(2, int(round(base.nbar * scale)))
    return base


@dataclass
class Sample:
    cfg: Config
    x: np.ndarray  # [n, dim]     sample X  (particle)
    xbar: np.ndarray  # [nbar, dim]  sample Xbar (anti-particle)
    wx: np.ndarray | None = None  # per-event weights (config 3)
    wxbar: np.ndarray | None = None
    mom_x: np.ndarray | None = None  # [n, 3, 3] momenta (B, C, D) for the triple product (config 4)
    mom_xbar: np.ndarray | None = None


def make_sample(cfg: Config) -> Sample:
    """Seeds: 1000+config for X, 2000+config for Xbar, 3000/4000+config for weights."""
    rx, rb = _rng(1000 + cfg.index), _rng(2000 + cfg.index)
    if cfg.dim == 2:
        x = dalitz_uniform(cfg.n, rx)
        xbar = dalitz_with_bump(cfg.nbar, rb, cfg.bump_frac)
        s = Sample(cfg, x, xbar)
    elif cfg.dim == 5:
        x, Px, _ = fourbody_phase_space(cfg.n, rx)
        xbar, Pb, _ = fourbody_phase_space(cfg.nbar, rb)
        s = Sample(cfg, x, xbar)
        if cfg.podd:
            # (B, C, D) = particles (2, 3, 4): (K+, pi+, pi-) for D0 and, with the
            # C-conjugate particle numbering of the Dbar0 sample, (K-, pi-, pi+).
            s.mom_x = np.ascontiguousarray(Px[:, 1:4, :])
            s.mom_xbar = np.ascontiguousarray(Pb[:, 1:4, :])
    else:
        raise ValueError("unsupported dim")
    if cfg.coord_dtype == "f32":
        s.x = s.x.astype(np.float32)
        s.xbar = s.xbar.astype(np.float32)
    if cfg.weighted:
        s.wx = _rng(3000 + cfg.index).uniform(-0.5, 1.5, cfg.n)
        s.wxbar = _rng(4000 + cfg.index).uniform(-0.5, 1.5, cfg.nbar)
    return s


def make_bkg_sample(seed: int = 5000, n_sig: int = 4000, n_bkg: int = 1600, asym: float = 0.75, scale: float = 1.0):
    """Inputs with the structure of the paper's Fig. 3 study for Eq. 3: `n_sig` signal events with a
    random 50 % flavour, `n_bkg` background events flat over the Dalitz plot contaminating the main samples with a
    3:1 flavour asymmetry, and `n_bkg` more with the same asymmetry as the background samples.  The paper's signal model
    (its Ref. [13]) is not available: the stand-in signal is the bumped Dalitz density of the other configs (no CP
    violation: both flavours are drawn from it).  Returns (x, xbar, bx, bxbar, b, bbar) with b, bbar the numbers of
    background events that went into the main samples."""
    rng = _rng(seed)
    n_sig, n_bkg = max(8, int(n_sig * scale)), max(8, int(n_bkg * scale))
    sig = dalitz_with_bump(n_sig, rng, 0.3)
    fl = rng.random(n_sig) < 0.5
    bkg = dalitz_uniform(n_bkg, rng)
    flb = rng.random(n_bkg) < asym
    side = dalitz_uniform(n_bkg, rng)
    fls = rng.random(n_bkg) < asym
    x = np.ascontiguousarray(np.vstack([sig[fl], bkg[flb]]))
    xbar = np.ascontiguousarray(np.vstack([sig[~fl], bkg[~flb]]))
    return x, xbar, np.ascontiguousarray(side[fls]), np.ascontiguousarray(side[~fls]), float(flb.sum()), float((~flb).sum())
