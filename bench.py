#!/usr/bin/env python
"""bench.py -- throughput of the energy-test hot path (arXiv:1612.04705) on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A step is one pass of the WHOLE hot path of SURVEY.md 8(a) over one synthetic sample: H0 split (config 4), H1 prep,
H4 labels, H2/H3 all-pairs psi + block sums, H5 permutation sums for all `nperm` permutations, H6 statistic and
p-value -- i.e. one `et_permutation_test` (configs 0-3) or one `et_podd_test` (config 4) through the C ABI.
The default workload is BASELINE.json configs[4], the one the north-star target is quoted on (n = nbar = 10^6, 5-D,
1000 permutations); it fits one GPU.

metric = pair-evaluations/s = unordered event pairs that enter T, N(N-1)/2, divided by the step time (every pair is
counted once however often a kernel touches it).  `value` is timed with the inputs resident in HBM (CUDA events on
the library's stream); `e2e` is the same call with pinned HOST buffers, the host->device staging inside the timed
region.  N > 1 (under torchrun, or `--gpus N` alone, which re-launches itself through torch.distributed.run): the
UNIT RANGE of the O(N^2) kernels is sharded (et_set_shard: rank r evaluates every N-th work unit for all label columns
and the ranks exchange exact int64 column sums through one small all-gather per launch), the same test on N GPUs --
strong scaling; value = pairs / max-over-ranks time.

`--impl reference` times the oracle (oracle/, plain fp64 CPU loops) on the host cores on a bounded row subset of the
same workload; it is the only place besides `cpu_baseline` where this file executes anything under oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

NUM_SMS = 148
SM_MAX_MHZ_FALLBACK = 1965.0


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    # fallback stated in /opt/skills/guides/B200_PROFILING.md
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": SM_MAX_MHZ_FALLBACK,
            "_source": "fallback"}


def alu_roofline_pairs_per_s(dim: int, sm_mhz: float) -> float:
    """FP32/SFU pipe roofline of the psi evaluation: per pair 2D+1 FP32-pipe instructions and
    one MUFU.EX2; 128 FP32 lanes and 16 SFU lanes per SM per clock, 148 SMs."""
    return min(128.0 / (2 * dim + 1), 16.0) * NUM_SMS * sm_mhz * 1e6


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md, the clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device: int):
        self.device, self.rows, self.proc = device, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.device), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self, peaks):
        sm, reasons, mx, pw = [], set(), peaks.get("sm_max_mhz", SM_MAX_MHZ_FALLBACK), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                pw.append(float(r[2]))
                for k, nm in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        reasons.add(nm)
            except (ValueError, IndexError):
                continue
        busy = [v for v, p in zip(sm, pw) if p > 0.5 * max(pw)] if pw else sm
        return {"sm_mhz": float(np.median(busy)) if busy else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(pw) if pw else None}


TRAFFIC_CSV = "r02_traffic_k_perm_tc_cfg4.csv"


def ncu_traffic(kernel: str, cfg_index: int, default_nperm: bool):
    """DRAM bytes per launch (read + write) of `kernel` from the COMMITTED ncu capture of this workload (a static figure,
    not measured in this run), or None.  Only the default configs[4] workload has one (profiles/r02_README.md names the
    command)."""
    path = os.path.join(ROOT, "profiles", TRAFFIC_CSV)
    if kernel != "k_perm_tc" or cfg_index != 4 or not default_nperm or not os.path.exists(path):
        return None, None
    import csv

    per_launch = {}
    with open(path) as f:
        lines = [ln for ln in f if not ln.startswith("==")]   # ncu's own log lines precede the CSV header
        for r in csv.DictReader(lines):
            if r.get("Metric Name") in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                per_launch[r["ID"]] = per_launch.get(r["ID"], 0.0) + float(r["Metric Value"].replace(",", ""))
    if not per_launch:
        return None, None
    return sum(per_launch.values()) / len(per_launch), f"profiles/{TRAFFIC_CSV} (ncu, bytes per launch)"


def pinned(a: np.ndarray):
    """Copy of `a` in page-locked host memory (torch owns it); returns (numpy view, keep-alive)."""
    import torch

    t = torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    return t.numpy(), t


def n_pairs(n, nbar):
    N = n + nbar
    return N * (N - 1) // 2


# ---------------------------------------------------------------------------------------------------------- ours
def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_1612_04705_b200 import binding, build, datagen as dg

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")          # the communicator line (nranks) stays in the log
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    if rank == 0:
        build.build()      # one rank (re)builds libet.so if it is stale; the others wait
    if world > 1:
        dist.barrier()
    peaks = load_peaks()

    cfg = dg.config(args.config)
    if args.nperm:
        cfg.nperm = args.nperm
    s = dg.make_sample(cfg)
    sigma = cfg.sigma
    # BASELINE configs[1] / [3] are a sigma scan (three sigma x the same 1000 permutations): the step is the whole scan,
    # one et_permutation_test_sigmas call, and every (pair, sigma) counts as a pair evaluation
    scan = list(getattr(cfg, "sigmas", ()) or ()) if not args.one_sigma else []
    scan = scan if len(scan) > 1 else []
    pairs1 = n_pairs(cfg.n, cfg.nbar)
    pairs = pairs1 * max(len(scan), 1)
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream(dev)
    ctx = binding.Context(local, stream=stream)
    if world > 1:
        ctx.set_shard(rank, world)

    def to_dev(a):
        return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev)

    d = {k: to_dev(getattr(s, k)) for k in ("x", "xbar", "wx", "wxbar", "mom_x", "mom_xbar")}
    h_keep = []
    h = {}
    for k in ("x", "xbar", "wx", "wxbar", "mom_x", "mom_xbar"):
        v = getattr(s, k)
        if v is None:
            h[k] = None
        else:
            h[k], keep = pinned(v)
            h_keep.append(keep)

    def step(src):
        if cfg.podd:
            r = ctx.podd_test(src["x"], src["mom_x"], src["xbar"], src["mom_xbar"], sigma, cfg.nperm, cfg.perm_seed)
            return r.p_odd
        if scan:
            rs = ctx.permutation_test_sigmas(src["x"], src["xbar"], scan, cfg.nperm, cfg.perm_seed, src["wx"], src["wxbar"])
            return rs[scan.index(sigma)] if sigma in scan else rs[0]
        return ctx.permutation_test(src["x"], src["xbar"], sigma, cfg.nperm, cfg.perm_seed, src["wx"], src["wxbar"])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def timed(src, steps):
        """CUDA events on the library's stream around exactly `steps` calls; ms of the slowest rank."""
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        agg = {"ms_pairs": 0.0, "ms_labels": 0.0, "ms_dom": 0.0, "launches": 0, "pair_evals": 0, "ms_esc": 0.0}
        barrier()
        e0.record(stream)
        for _ in range(steps):
            res = step(src)
            st = ctx.stats()
            agg["ms_pairs"] += st.ms_pairs
            agg["ms_labels"] += st.ms_labels
            agg["ms_dom"] += st.ms_dominant
            agg["launches"] += st.launches
            agg["pair_evals"] += st.pair_evals
            agg["dom_launches"] = st.dominant_launches
            agg["dom_kernel"] = st.dominant_kernel
            agg["dom_ops"] = st.dominant_ops
            agg["dom_ops_exec"] = st.dominant_ops_executed
            agg["ms_esc"] += st.ms_escalation
            agg["n_near_before"] = st.n_near_before
            agg["n_escalated"] = st.n_escalated
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms, agg, res

    # L2 flush between timed steps is unnecessary here: every step re-stages and re-prepares its records and the
    # O(N^2) kernels stream label/row data far larger than L2 at the bench sizes; stated in config.
    for _ in range(args.warmup):
        step(d)
    with ClockSampler(local) as cs:
        ms, agg, res = timed(d, args.steps)
    clocks = cs.summary(peaks)
    for _ in range(1):
        step(h)
    ms_e2e, _, res_h = timed(h, args.steps)
    ms_step = ms / args.steps
    value = pairs / (ms_step * 1e-3)   # one test on `world` GPUs (unit-range shard): strong scaling
    e2e_value = pairs / (ms_e2e / args.steps * 1e-3)
    h2d = sum(v.nbytes for v in h.values() if v is not None)
    d2h = (cfg.nperm * 8 + 256) * max(len(scan), 1)

    # et_T alone (H1-H3, H6): the psi kernel against the FP32/SFU roofline
    def T_only():
        if cfg.weighted:
            return ctx.T_weighted(d["x"], d["wx"], d["xbar"], d["wxbar"], sigma)
        return ctx.T(d["x"], d["xbar"], sigma)

    for _ in range(2):
        T_only()
    msT, msT_k, nT = 0.0, 0.0, 3
    for _ in range(nT):
        T_only()
        st = ctx.stats()
        msT += st.ms_total
        msT_k += st.ms_pairs
        formT = st.distance_form
    sm_mhz_max = peaks.get("sm_max_mhz", SM_MAX_MHZ_FALLBACK)
    roofT = alu_roofline_pairs_per_s(cfg.dim, sm_mhz_max)
    et_T = {"pairs_per_s": pairs1 / (msT / nT * 1e-3), "kernel_pairs_per_s": pairs1 / (msT_k / nT * 1e-3),
            "ms": msT / nT, "roofline_pairs_per_s": roofT, "frac": pairs1 / (msT_k / nT * 1e-3) / roofT,
            "frac_at_sampled_clock": (pairs1 / (msT_k / nT * 1e-3) / alu_roofline_pairs_per_s(cfg.dim, clocks["sm_mhz"])
                                      if clocks.get("sm_mhz") else None),
            "peak_model": "min(128/(2D+1),16) pairs/clk/SM x 148 SMs x sm_max_mhz (FP32/SFU pipes): the difference form of "
                          "the distance, 2D+1 FP32 lane-ops and one MUFU.EX2 per pair (SURVEY 8(d))",
            # the Gram form (ET_OPT_DISTANCE, default for D >= 4) needs D+2 lane-ops per pair: its own bound is
            # min(128/(D+2),16), the SFU's 16 pairs/clk/SM for every D <= 6
            "distance_form": {1: "differences", 2: "gram"}.get(formT, "?"),
            "pairs_per_clk_per_sm": pairs1 / (msT_k / nT * 1e-3) / (NUM_SMS * sm_mhz_max * 1e6),
            "frac_of_form_roofline": pairs1 / (msT_k / nT * 1e-3) / (min(128.0 / ((cfg.dim + 2) if formT == 2 else (2 * cfg.dim + 1)), 16.0)
                                                                     * NUM_SMS * sm_mhz_max * 1e6)}

    # sigma scan (configs with several sigma values, BASELINE configs[1] / [3]): one fused pass against separate et_T calls
    sigma_scan = None
    if len(getattr(cfg, "sigmas", ()) or ()) > 1:
        sg = list(cfg.sigmas)

        def ms_of(fn, reps=3):
            fn()
            t = 0.0
            for _ in range(reps):
                fn()
                t += ctx.stats().ms_total
            return t / reps

        fused = ms_of(lambda: ctx.T_sigmas(d["x"], d["xbar"], sg, d["wx"], d["wxbar"]))
        if cfg.weighted:
            sep = sum(ms_of(lambda v=v: ctx.T_weighted(d["x"], d["wx"], d["xbar"], d["wxbar"], v)) for v in sg)
        else:
            sep = sum(ms_of(lambda v=v: ctx.T(d["x"], d["xbar"], v)) for v in sg)
        sigma_scan = {"sigmas": sg, "ms_fused": fused, "ms_separate": sep, "pair_sigma_evals_per_s": len(sg) * pairs1 / (fused * 1e-3)}

    # binned S_CP chi^2 of the same samples (Eq. 1; NEXT-4): the paper's O(N) comparison method on a uniform
    # grid over the bounding box, about 10 bins per axis in 2-D ("O(10) to O(10^2)" bins), 3 per axis in 5-D
    try:
        nb = [10] * cfg.dim if cfg.dim <= 2 else [3] * cfg.dim
        lo = np.minimum(s.x.min(axis=0), s.xbar.min(axis=0)).astype(np.float64)
        hi = np.maximum(s.x.max(axis=0), s.xbar.max(axis=0)).astype(np.float64)
        ctx.scp(d["x"], d["xbar"], lo, hi, nb)
        sc_ = ctx.scp(d["x"], d["xbar"], lo, hi, nb)
        scp = {"chi2": sc_.chi2, "ndf": sc_.ndf, "p_value": sc_.p_value, "bins": sc_.bins_total, "ms": ctx.stats().ms_total}
    except (binding.EtError, ValueError) as exc:
        scp = {"error": str(exc)}

    # GEV fit of this step's permutation T values: the p-value where counting gives 0 (host-only, ~ms)
    try:
        g = binding.gev_pvalue(res.T_perm, res.observed.T, np.random.default_rng(12345).standard_normal((2000, 3)))
        gev = {"p_value": g.p_value, "p_lo": g.p_lo, "p_hi": g.p_hi, "mu": g.mu, "sigma": g.sigma, "xi": g.xi, "converged": g.converged}
    except binding.EtError as exc:
        gev = {"error": str(exc)}

    # roofline of the dominant kernel of the step (the one with the largest share of ms_pairs)
    dom_ms = agg["ms_dom"] / (args.steps * max(agg["dom_launches"], 1))
    if agg["dom_kernel"].startswith("k_perm_tc"):
        # int8 tensor-core contraction: ops = 2 * MACs; peak = measured bf16 peak x nominal int8:bf16 ratio (2)
        # algorithmic ops: 2 digits x 2 x unordered pairs x the label columns the test needs (nperm
        # permutations + observed + second labelling + ones), summed over the launches of one step, per launch
        nl = max(agg["dom_launches"], 1)
        ops = agg["dom_ops"] / nl
        ach = ops / (dom_ms * 1e-3) / 1e12
        ach_padded = agg["dom_ops_exec"] / nl / (dom_ms * 1e-3) / 1e12
        peak = 2.0 * peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"])
        traffic, traffic_src = ncu_traffic(agg["dom_kernel"], cfg.index, not args.nperm and world == 1)
        # distinct operand bytes of one launch: its 512-column label chunk (64 B per padded row), the records and the
        # pair records
        npad = cfg.n + cfg.nbar + 4096
        fl = 4 * ((cfg.dim + 1 + 3) // 4)
        algo_bytes = npad * (64 + 4 * fl + 8 * ((cfg.dim + 2) // 2))
        roofline = {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TOP/s (int8)", "frac": ach / peak,
                    "ops": ops, "launch_ms": dom_ms, "launches_per_step": nl, "frac_padded": ach_padded / peak,
                    "traffic": traffic, "traffic_static": True, "traffic_source": traffic_src,
                    "traffic_ratio": (traffic / algo_bytes if traffic else None), "algorithmic_bytes": algo_bytes,
                    "kernel": agg["dom_kernel"],
                    # context: the measured bf16 peak is a power-throttled cuBLAS GEMM (1.34 GHz), this kernel runs its int8
                    # MMAs at ~1.9 GHz, so frac can pass 1; against the burst figure and the nominal dense int8 (4.5 POP/s):
                    "frac_of_burst": ach / (2.0 * peaks["bf16_tflops"]),
                    "frac_of_nominal_int8": ach / 4500.0,
                    "peak_source": f"{peaks['_source']} bf16 sustained x 2 (nominal int8:bf16)"}
    else:
        # CUDA-core kernels: FP32-pipe thread-instructions per second
        ach = agg["dom_ops"] / max(agg["dom_launches"], 1) / (dom_ms * 1e-3) / 1e12
        peak = 128.0 * NUM_SMS * sm_mhz_max * 1e6 / 1e12
        roofline = {"bound": "alu", "achieved": ach, "peak": peak, "unit": "Tinst/s (FP32 pipe)", "frac": ach / peak,
                    "traffic": None, "kernel": agg["dom_kernel"],
                    "peak_source": "128 FP32 lanes x 148 SMs x sm_max_mhz (DESIGN.md)"}

    out = {
        "metric": "energy_test_pair_evaluations_per_s", "value": value, "unit": "pairs/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "strong", "vs_baseline": None, "dtype": "f32 psi / f64 or exact-int sums", "data": "synthetic",
        "config": {"workload": f"BASELINE configs[{cfg.index}] {cfg.name}: n={cfg.n} nbar={cfg.nbar} dim={cfg.dim} "
                               f"sigma={scan if scan else sigma} nperm={cfg.nperm}", "n": cfg.n, "nbar": cfg.nbar, "dim": cfg.dim,
                   "nperm": cfg.nperm, "sigma": scan if scan else sigma, "l2": "inputs and label matrix larger than L2; records re-prepared every step",
                   "parallelism": f"work units of the O(N^2) kernels sharded over {world} GPU(s), one all-gather of 2 x 512 "
                                  f"int64 column sums per launch"},
        "permutations_per_s": cfg.nperm * max(len(scan), 1) / (ms_step * 1e-3),
        "pair_perm_updates_per_s": cfg.nperm * pairs / (ms_step * 1e-3),
        "effective_pairs_per_s": (cfg.nperm + 1) * pairs / (ms_step * 1e-3),  # what one pass per permutation would need
        "p_value": res.p_value, "count_gt": res.count_gt, "T_obs": res.observed.T, "n_near": res.n_near,
        # exact p-value: permutations inside the guard band of the tensor-core pass, re-evaluated in the
        # fp32-pair / fp64-sum arithmetic inside the timed step
        "escalation": {"n_near_before": agg.get("n_near_before", 0), "n_escalated": agg.get("n_escalated", 0),
                       "n_near_after": res.n_near, "escalation_ms": agg["ms_esc"] / args.steps},
        "gev": gev,
        "scp": scp,
        "et_T": et_T,
        "sigma_scan": sigma_scan,
        "share_pairs_kernels": agg["ms_pairs"] / ms, "share_labels": agg["ms_labels"] / ms,
        "e2e": {"value": e2e_value, "unit": "pairs/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": ms_e2e / args.steps},
        "gpu_launches": agg["launches"],
        "clocks": clocks,
        "roofline": roofline,
    }
    if world > 1:
        # every rank holds the complete result; they must agree bit for bit (integer column sums, fixed-order reductions)
        sig = torch.tensor([float(res.observed.T), float(res.count_gt), float(np.asarray(res.T_perm).sum())], device=dev, dtype=torch.float64)
        lo, hi = sig.clone(), sig.clone()
        dist.all_reduce(lo, op=dist.ReduceOp.MIN)
        dist.all_reduce(hi, op=dist.ReduceOp.MAX)
        out["ranks_agree"] = bool((lo == hi).all().item())
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(s, cfg, sigma, args.cpu_rows)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    if rank == 0:
        sys.stdout.flush()
        print(json.dumps(out), flush=True)


# ---------------------------------------------------------------------------------------------------------- oracle
def cpu_baseline(s, cfg, sigma, nrows):
    """The oracle as it stands on the host cores, on a bounded sample: `nrows` random pooled rows against all N
    columns (oracle.row_sums), i.e. nrows * N psi evaluations in fp64 with libm exp."""
    import oracle

    N = cfg.n + cfg.nbar
    if nrows <= 0:
        nrows = int(max(16, min(N, 6e9 // N)))
    rows = np.random.default_rng(7).choice(N, min(nrows, N), replace=False)
    oracle.row_sums(s.x[:64], s.xbar[:64], sigma, np.arange(8))  # load + first touch
    t0 = time.perf_counter()
    oracle.row_sums(s.x, s.xbar, sigma, rows, s.wx, s.wxbar)
    dt = time.perf_counter() - t0
    rate = len(rows) * (N - 1) / dt  # psi evaluations per second
    # The metric is unordered pairs / time of the WHOLE step (the permutation test).  The oracle re-evaluates every
    # permutation from scratch (oracle O4), so its step is nperm + 1 passes over the pairs: exact N^2 scaling.
    step_s = n_pairs(cfg.n, cfg.nbar) * (cfg.nperm + 1) / rate
    return {"value": rate / (cfg.nperm + 1), "unit": "pairs/s", "cores": oracle.num_threads(), "kind": "oracle",
            "psi_evaluations_per_s": rate,
            "sample": f"{len(rows)} random pooled rows x all {N} columns ({len(rows) * (N - 1):.3g} psi evaluations in "
                      f"{dt:.1f} s = {rate:.3g}/s); the step (T_obs + {cfg.nperm} permutations, each from scratch) "
                      f"extrapolated = pairs*(nperm+1)/rate = {step_s / 3600:.1f} h, value = pairs / that"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1612_04705_b200 import datagen as dg  # seeded inputs only (holds none of the method's arithmetic)

    cfg = dg.config(args.config)
    s = dg.make_sample(cfg)
    N = cfg.n + cfg.nbar
    nrows = args.cpu_rows if args.cpu_rows > 0 else int(max(16, min(N, 2e9 // N)))
    for _ in range(args.warmup):
        cpu_baseline(s, cfg, cfg.sigma, max(8, nrows // 8))
    vals, t0 = [], time.perf_counter()
    for _ in range(args.steps):
        b = cpu_baseline(s, cfg, cfg.sigma, nrows)
        vals.append(b["value"])
    dt = time.perf_counter() - t0
    v = float(np.mean(vals))
    b["value"] = v
    print(json.dumps({
        "impl": "reference", "metric": "energy_test_pair_evaluations_per_s", "value": v, "unit": "pairs/s",
        "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / args.steps * 1e3,  # wall time of one bounded sample, NOT of a whole step:
        "ms_per_step_extrapolated": n_pairs(cfg.n, cfg.nbar) / v * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE configs[{cfg.index}] {cfg.name}: n={cfg.n} nbar={cfg.nbar} dim={cfg.dim} "
                               f"sigma={cfg.sigma} nperm={cfg.nperm} (oracle timed on a row subset, the step of "
                               f"nperm + 1 from-scratch passes extrapolated)", "n": cfg.n, "nbar": cfg.nbar,
                   "dim": cfg.dim, "nperm": cfg.nperm, "sigma": cfg.sigma},
        "cpu_baseline": b,
        "e2e": {"value": v, "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--nperm", type=int, default=0, help="override the configuration's permutation count (experiments)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-rows", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--one-sigma", action="store_true", help="configs 1 / 3: time the middle sigma alone instead of the scan")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "RANK" not in os.environ:
        # started as plain `python bench.py --gpus N`: one rank per GPU through torch.distributed.run (the launch the
        # driver uses itself); fail loudly instead of running one rank and printing n_gpus = 1
        import socket

        import torch

        have = torch.cuda.device_count()
        if have < args.gpus:
            sys.exit(f"bench.py --gpus {args.gpus}: only {have} CUDA device(s) visible")
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if args.gpus > 1 and int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        sys.exit(f"bench.py --gpus {args.gpus} under a launcher with WORLD_SIZE={os.environ.get('WORLD_SIZE')}")
    run_ours(args)


if __name__ == "__main__":
    main()
