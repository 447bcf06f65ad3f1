#!/usr/bin/env python
"""Writes tests/golden/fullsize_T.txt: oracle values at the sizes bench.py times (BASELINE configs[2], [3], [4]).

    python tests/golden/make_fullsize_golden.py [--configs 3,2,4] [--out tests/golden/fullsize_T.txt]

Imports ONLY `oracle` (the plain fp64 CPU statement of Eq. 2 and of the permutation test) and
`paper_1612_04705_b200.datagen` (seeded inputs, none of the method's arithmetic).  Nothing here touches the CUDA path:
the stored numbers are what tests/test_gpu_parity.py compares `et_permutation_test` / `et_podd_test` / `et_T` with at
full size, where an in-test oracle run is too slow (config 4: 2.0e12 psi evaluations per T).

Entries (one per line, `key = decimal | hex-float`; a key that is already in the file is not recomputed, so the script
can be interrupted and restarted):
  cfgC.obs.{T,T_xx,T_bb,T_xb,S_xx,S_bb,S_xb,W,Wbar}   observed statistic of the step bench.py times
                                                       (config 4: the P-odd grouping (I+IV) vs (II+III))
  cfgC.perm.K                                          T of permutation K (from scratch, labels of reading R4, the
                                                       config's permutation seed), K < 2 (config 4: K = 0)
  cfgC.perm.K (K >= the count above, --extra-perm)     the same quantity for one more permutation, evaluated as
                                                       oracle.T on the split that oracle.labels gives (one pass instead
                                                       of re-running the whole block)
  cfg4.even.{...}                                      P-even grouping (I+II) vs (III+IV) = Eq. 2 of (X, Xbar)
  cfg4.count.{I,II,III,IV}                             class sizes of the Sect. 5 split
Each block is preceded by a comment line with the host cores used and the wall time.
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1612_04705_b200 import datagen as dg  # noqa: E402

FIELDS = ("T", "T_xx", "T_bb", "T_xb", "S_xx", "S_bb", "S_xb", "W", "Wbar")


def read_existing(path):
    have = {}
    if os.path.exists(path):
        with open(path) as f:
            for line in f:
                if line.startswith("#") or "=" not in line:
                    continue
                k, v = line.split("=", 1)
                have[k.strip()] = float.fromhex(v.split("|")[1].strip())
    return have


class Out:
    def __init__(self, path):
        self.path, self.have = path, read_existing(path)

    def comment(self, text):
        with open(self.path, "a") as f:
            f.write(f"# {text}\n")

    def put(self, key, value):
        value = float(value)
        with open(self.path, "a") as f:
            f.write(f"{key} = {value!r} | {value.hex()}\n")
        self.have[key] = value

    def put_result(self, prefix, r):
        for k in FIELDS:
            self.put(f"{prefix}.{k}", getattr(r, k))


def run_two_sample(out: Out, tag: str, a, b, sigma, wa, wb, nperm, seed):
    """Observed T and the first `nperm` permutation T values, every one a from-scratch pass (oracle.perm_test)."""
    keys = [f"{tag}.obs.{k}" for k in FIELDS] + [f"{tag}.perm.{k}" for k in range(nperm)]
    if all(k in out.have for k in keys):
        return
    t0 = time.time()
    r = oracle.perm_test(a, b, sigma, nperm, seed, wa, wb)
    dt = time.time() - t0
    N = len(a) + len(b)
    out.comment(f"{tag}: oracle.perm_test n={len(a)} nbar={len(b)} dim={a.shape[1]} sigma={sigma} nperm={nperm} seed={seed:#x}; "
                f"{(nperm + 1) * N * (N - 1) // 2:.3e} psi evaluations, {oracle.num_threads()} host cores, {dt:.0f} s wall")
    out.put_result(f"{tag}.obs", r.observed)
    for k in range(nperm):
        out.put(f"{tag}.perm.{k}", r.T_perm[k])


def run_extra_perm(out: Out, tag: str, a, b, sigma, wa, wb, k, seed):
    """T of permutation k alone: the pooled events split by oracle.labels (reading R4), Eq. 2 by oracle.T."""
    key = f"{tag}.perm.{k}"
    if key in out.have:
        return
    pooled = np.vstack([a, b])
    w = None if wa is None else np.concatenate([wa, wb])
    N, n = len(pooled), len(a)
    lab = (oracle.labels(N, n, k + 1, seed)[:, k >> 5] >> (k & 31)) & 1
    t0 = time.time()
    r = oracle.T(pooled[lab == 1], pooled[lab == 0], sigma, None if w is None else w[lab == 1], None if w is None else w[lab == 0])
    out.comment(f"{key}: oracle.labels + oracle.T on the permuted split ({int(lab.sum())} + {N - int(lab.sum())} events), "
                f"{oracle.num_threads()} host cores, {time.time() - t0:.0f} s wall")
    out.put(key, r.T)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="3,2,4")
    ap.add_argument("--out", default=os.path.join(ROOT, "tests", "golden", "fullsize_T.txt"))
    ap.add_argument("--scale", type=float, default=1.0, help="shrink n, nbar (dry runs only; the committed file is scale 1)")
    ap.add_argument("--extra-perm", type=int, default=-1, help="also store T of this permutation index (one oracle.T pass)")
    args = ap.parse_args()
    out = Out(args.out)
    if not out.have:
        out.comment("written by tests/golden/make_fullsize_golden.py (oracle + datagen only); see its docstring for the keys")
    for index in (int(c) for c in args.configs.split(",")):
        cfg = dg.config(index, scale=args.scale)
        tag = f"cfg{index}" if args.scale == 1.0 else f"cfg{index}@{args.scale}"
        s = dg.make_sample(cfg)
        if not cfg.podd:
            run_two_sample(out, tag, s.x, s.xbar, cfg.sigma, s.wx, s.wxbar, 2, cfg.perm_seed)
            if args.extra_perm >= 0:
                run_extra_perm(out, tag, s.x, s.xbar, cfg.sigma, s.wx, s.wxbar, args.extra_perm, cfg.perm_seed)
            continue
        posx, _ = oracle.podd_split(s.mom_x[:, 0], s.mom_x[:, 1], s.mom_x[:, 2], False)
        posb, _ = oracle.podd_split(s.mom_xbar[:, 0], s.mom_xbar[:, 1], s.mom_xbar[:, 2], True)
        I, II, III, IV = s.x[posx == 1], s.x[posx == 0], s.xbar[posb == 1], s.xbar[posb == 0]
        for name, part in (("I", I), ("II", II), ("III", III), ("IV", IV)):
            if f"{tag}.count.{name}" not in out.have:
                out.put(f"{tag}.count.{name}", len(part))
        if not all(f"{tag}.even.{k}" in out.have for k in FIELDS):
            t0 = time.time()
            r = oracle.T(s.x, s.xbar, cfg.sigma)
            out.comment(f"{tag}.even: oracle.T n={cfg.n} nbar={cfg.nbar}; {oracle.num_threads()} host cores, {time.time() - t0:.0f} s wall")
            out.put_result(f"{tag}.even", r)
        run_two_sample(out, tag, np.vstack([I, IV]), np.vstack([II, III]), cfg.sigma, None, None, 1, cfg.perm_seed)
        if args.extra_perm >= 0:
            run_extra_perm(out, tag, np.vstack([I, IV]), np.vstack([II, III]), cfg.sigma, None, None, args.extra_perm, cfg.perm_seed)


if __name__ == "__main__":
    main()
