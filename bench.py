#!/usr/bin/env python
"""bench.py -- site-updates/s of the fused spin-2 QLGA step on B200 (one lattice per GPU).

    python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path
    python bench.py --impl reference --steps K --warmup W     # the CPU oracle on a bounded sample

One bench "step" = one pass of the whole hot path over the lattice: `--inner` time
steps of eq. (112)/(108) (fused y pass + x pass kernels), one observables reduction
and one lattice-vorticity evaluation (2D).  Metric: lattice-site updates per second
(GSUP/s), one site-update = one full time step of one site, all five fields.
Default workload: BASELINE.json configs[4] (2D 8192x8192, fp64, interleaved), the
largest single-GPU configuration and the one the north-star target is stated on.
Prints ONE JSON line on rank 0.  See DESIGN.md "Measurement".
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

from paper_1907_12834_b200 import inputs  # noqa: E402  (generators only: no method arithmetic)

METRIC = "site-updates/sec (GSUP/s) on 1 B200 and % of HBM roofline (fp64/fp32)"
UNIT = "GSUP/s"

WORKLOADS = {
    "cfg1": dict(ndim=1, gen=lambda L: inputs.config1(L=L or 1024), L=1024),
    "cfg2": dict(ndim=1, gen=lambda L: inputs.config2(L=L or 65536), L=65536),
    "cfg3": dict(ndim=1, gen=lambda L: inputs.config3(L=L or (1 << 22)), L=1 << 22),
    "cfg4": dict(ndim=2, gen=lambda L: inputs.config4(L=L or 2048), L=2048),
    "cfg5": dict(ndim=2, gen=lambda L: inputs.config5(L=L or 8192), L=8192),
    "cfg3d": dict(ndim=3, gen=lambda L: inputs.config3d(L=L or 256), L=256),   # SURVEY 8(f) row 3, not a BASELINE config
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", choices=sorted(WORKLOADS))
    ap.add_argument("--precision", default="f64", choices=["f64", "f32", "f32x"])
    ap.add_argument("--order", default="interleaved", choices=["interleaved", "plain"])
    ap.add_argument("--inner", type=int, default=0, help="time steps per bench step (0 = auto)")
    ap.add_argument("--lattice", type=int, default=0, help="override the lattice edge (testing)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    ap.add_argument("--tile-y", type=int, default=0)
    ap.add_argument("--threads-x", type=int, default=0)
    ap.add_argument("--threads-y", type=int, default=0)
    ap.add_argument("--steps-per-launch", type=int, default=0, help="QLGA_OPT_STEPS_PER_LAUNCH (1D)")
    ap.add_argument("--tol-log2", type=int, default=0, help="QLGA_OPT_EXP_TOL_LOG2 override (experiments only)")
    ap.add_argument("--no-variants", action="store_true",
                    help="skip the `variants` record (the other precisions / orderings / config 3, a few bench steps each)")
    ap.add_argument("--variant-steps", type=int, default=2)
    ap.add_argument("--mod-shift", type=int, default=-1, help="QLGA_OPT_EXP_MOD_SHIFT override (experiments only)")
    ap.add_argument("--band", type=int, default=-1, choices=[-1, 0, 1, 2],
                    help="QLGA_OPT_BAND (plain ordering, 2D): -1 = the library's default (band pipelining through L2 where it "
                         "pays), 0 = two launches per step, 1 = bands on the library's streams, 2 = replayed as a CUDA graph")
    ap.add_argument("--band-rows", type=int, default=0, help="QLGA_OPT_BAND_ROWS (0 = auto)")
    ap.add_argument("--band-slots", type=int, default=0, help="QLGA_OPT_BAND_SLOTS (0 = auto)")
    ap.add_argument("--band-trace", action="store_true",
                    help="band mode, library built with QLGA_NVCC_EXTRA=-DQLGA_TRACE: add the timeline of one band step "
                         "(first CTA start / last CTA end of every y and x kernel, %%globaltimer) to the JSON line")
    ap.add_argument("--profiler-range", action="store_true",
                    help="bracket the timed region with cudaProfilerStart / Stop (for `ncu --replay-mode app-range`, "
                         "which measures the DRAM traffic of the whole region with its kernels running side by side)")
    ap.add_argument("--slab", action="store_true",
                    help="one lattice cut into slabs along its slowest axis, one slab per GPU, 4-layer halo exchange "
                         "per step (paper_1907_12834_b200/slab.py); weak scaling: every rank owns the workload's lattice "
                         "of a lattice N times as long.  Default is independent replicas (DESIGN.md section 11)")
    return ap.parse_args()


def load_traffic(workload, precision, order):
    """{kernel: (dram bytes per launch, FP instr per site per launch)} from the committed ncu
    capture (profiles/r2_traffic.csv), or {} when this workload was not captured."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    out = {}
    if os.path.exists(path):
        import csv
        with open(path) as f:
            for row in csv.DictReader(f):
                if (row["workload"], row["precision"], row["order"]) == (workload, precision, order):
                    fpi = row["fp_thread_instr_per_site_per_launch"]
                    out[row["kernel"]] = (float(row["dram_bytes_per_launch"]), float(fpi) if fpi else None)
    return out


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured", float(p.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback", 1965.0


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx = gpu_index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200",
                 "-i", str(self.idx)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "power_w_max": float(max(pw)) if pw else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------
# models: algorithmic bytes and FP instructions per site-update
# ---------------------------------------------------------------------------
def bytes_per_site_update(precision):
    """One read + one write of the 20 reals of a site: SURVEY.md section 8(d)."""
    return 320.0 if precision == "f64" else 160.0          # f32 and f32x store fp32


def fp_instr_per_site_update(ndim, order, degree, precision="f64"):
    """FP instructions (FMA/ADD/MUL, one per lane) per site-update of the fused step,
    counted from qlga_math.cuh: one U of polynomial degree p costs
    180 + 156 p in fp64 (densities and spin 52, spin gauge 59, scalar phase 29, output 40; per
    Horner stage and spinor vector 68 + 10) and 120 + 196 p in fp32 (no gauge: 88 + 10 per stage),
    one kinetic factor 40, the final scaling 20 per pass.  ncu at config 5 (fp64): 7860 per
    site-update without the halo recompute; this model gives 7800 at the mean degree 4.85."""
    n_fac = 4 * ndim
    n_u = n_fac if order == "interleaved" else 1
    per_u = (180.0 + 156.0 * degree) if precision == "f64" else (120.0 + 196.0 * degree)
    return n_u * per_u + n_fac * 40.0 + 20.0 * ndim


def mean_degree(sim):
    """Mean per-site polynomial degree of U on the CURRENT (evolved) state, from the library's own degree
    lookup (qlga_angle_stats): the degree the ALU model charges."""
    st = sim.angle_stats()
    hist = st["degree_hist"]
    n = sum(hist)
    # sites beyond the split angle ([0]) take the general path: charge them the top degree
    return (sum(p * c for p, c in enumerate(hist) if p > 0) + 12 * hist[0]) / max(n, 1), st


_ALU_PEAKS = {}


def alu_peak(qlga, precision):
    """Measured issue rate of the binding FP pipe (qlga_issue_peak, live in this run): thread-instructions per
    second and per SM cycle.  fp64 arithmetic: DFMA.  fp32: the larger of the FFMA and packed FFMA2 lane rates."""
    kinds = ("dfma",) if precision in ("f64", "f32x") else ("ffma", "ffma2")
    best = None
    for k in kinds:
        if k not in _ALU_PEAKS:
            _ALU_PEAKS[k] = qlga.issue_peak(k)
        if best is None or _ALU_PEAKS[k]["instr_per_s"] > best[1]["instr_per_s"]:
            best = (k, _ALU_PEAKS[k])
    return best


# ---------------------------------------------------------------------------
# the oracle arm: cpu_baseline (inside the normal run) and --impl reference
# ---------------------------------------------------------------------------
def oracle_sample(w, ndim, order, target_seconds):
    """A periodic crop of the workload's lattice sized for ~target_seconds of oracle time."""
    nx, ny = w.dims[0], w.dims[1]
    if ndim == 3:
        edge = min(nx, 40)
        o = nx // 2 - edge // 2
        psi = w.psi[:, o:o + edge, o:o + edge, o:o + edge]
    elif ndim == 2:
        edge = min(nx, 256)
        y0, x0 = ny // 2 - edge // 2, nx // 2 - edge // 2
        psi = w.psi[:, y0:y0 + edge, x0:x0 + edge]
    else:
        edge = min(nx, 1 << 16)
        x0 = nx // 4 - edge // 2 if nx > edge else 0
        psi = w.psi[:, :, x0:x0 + edge]
    q = np.ascontiguousarray(np.repeat(psi[:, None] / 2, 2, axis=1))
    return q, edge


def time_oracle(w, ndim, order, target_seconds):
    from oracle.qlga_oracle import Oracle     # test infrastructure: allowed here (cpu_baseline / reference arm)
    orc = Oracle("double")
    q, edge = oracle_sample(w, ndim, order, target_seconds)
    sites = int(np.prod(q.shape[2:]))
    o = 1 if order == "interleaved" else 0
    t0 = time.perf_counter()
    q = orc.step(q, ndim, w.couplings, o, 1)
    t1 = time.perf_counter() - t0
    nsteps = max(1, int(target_seconds / max(t1, 1e-6)) - 1)
    t0 = time.perf_counter()
    orc.step(q, ndim, w.couplings, o, nsteps)
    dt = time.perf_counter() - t0
    rate = sites * nsteps / dt
    sample = (f"periodic {'x'.join([str(edge)] * ndim)} crop" if ndim >= 2 else f"periodic {edge}-site crop") + \
             f" of the workload's input, {nsteps} time steps, {dt:.1f} s"
    return rate, sample, sites, nsteps


def run_reference(args, w, ndim, config):
    """--impl reference: the oracle as it stands on the host cores, same metric/config."""
    from oracle.qlga_oracle import Oracle
    orc = Oracle("double")
    q, edge = oracle_sample(w, ndim, args.order, 0)
    sites = int(np.prod(q.shape[2:]))
    o = 1 if args.order == "interleaved" else 0
    t0 = time.perf_counter()
    q = orc.step(q, ndim, w.couplings, o, 1)
    t1 = time.perf_counter() - t0
    budget = 120.0 / max(1, args.steps + args.warmup)              # whole run within a few minutes
    inner = max(1, int(budget / max(t1, 1e-6)))
    for _ in range(args.warmup):
        q = orc.step(q, ndim, w.couplings, o, inner)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        q = orc.step(q, ndim, w.couplings, o, inner)
    dt = time.perf_counter() - t0
    val = sites * inner * args.steps / dt / 1e9
    sample = (f"periodic {'x'.join([str(edge)] * ndim)} crop" if ndim >= 2 else f"periodic {edge}-site crop") + \
             f" of the workload's input, {inner} time steps per bench step"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---------------------------------------------------------------------------
# multi-GPU plumbing: replicas only -- one lattice per rank, no
# data-path collective; torch.distributed serves the barrier and the max over ranks
# ---------------------------------------------------------------------------
def max_over_ranks(ms, world, device=None):
    """Largest per-rank duration (the job is as slow as its slowest replica)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_gsups(sites_per_rank, time_steps, world, ms):
    """Whole-job site-updates per second (GSUP/s): every rank advances its own lattice."""
    return sites_per_rank * time_steps * world / (ms * 1e-3) / 1e9


def build_roofline(qlga, prof, ndim, sites, time_steps, precision, order, deg_info, clocks, captured):
    """Both rooflines of the dominant pass kernel; the binding one (larger fraction) on top.
    HBM: algorithmic bytes per launch / launch time against the measured copy bandwidth.  ALU: FP instructions
    per launch (model of fp_instr_per_site_update at the mean per-site degree of the evolved state) / launch time
    against the issue rate measured live by qlga_issue_peak."""
    hbm_peak, peak_kind, sm_max = load_peaks()
    bps = bytes_per_site_update(precision)
    kinds = {k: v for k, v in prof.items() if v[1] > 0}
    if not kinds:
        return None
    dom = max(kinds, key=lambda k: kinds[k][0])
    dms, dn = kinds[dom]
    per_launch_ms = dms / dn
    # a pass launch advances every site by 1/ndim of a time step (times the fused steps in 1D)
    per_step = 1 if dom == "x_pass" else max(1, ndim - 1)    # the y_pass timer covers the y and z passes
    units = sites * time_steps * per_step / (ndim * dn)       # site-updates per launch
    if dom == "band_step":                                    # band mode: one graph replay = one whole time step
        units = float(sites)
    deg, stats = deg_info
    arith = "f64" if precision in ("f64", "f32x") else "f32"
    fpi = fp_instr_per_site_update(ndim, order, deg, arith)
    kind, pk = alu_peak(qlga, precision)
    alu_peak_t = pk["instr_per_s"] / 1e12
    alu_ach = units * fpi / (per_launch_ms * 1e-3) / 1e12
    hbm_ach = units * bps / (per_launch_ms * 1e-3) / 1e9
    traffic = captured.get(dom, (None, None))[0]
    roof_hbm = {"bound": "hbm", "achieved": hbm_ach, "peak": hbm_peak, "unit": "GB/s",
                "frac": hbm_ach / hbm_peak, "traffic": traffic, "peak_kind": peak_kind,
                "kernel": dom, "ms_per_launch": per_launch_ms,
                "model": f"{bps:.0f} B per site-update x {units:.3g} site-updates per launch"}
    roof_alu = {"bound": "alu", "achieved": alu_ach, "peak": alu_peak_t, "unit": "Tinstr/s",
                "frac": alu_ach / alu_peak_t, "traffic": traffic, "kernel": dom, "peak_kind": "measured",
                "ms_per_launch": per_launch_ms,
                "model": f"{fpi:.0f} FP instr per site-update (mean degree {deg:.2f} on the evolved state, "
                         f"theta_max {stats['theta_max']:.3g}) x {units:.3g} site-updates per launch; peak = {kind.upper()} issue "
                         f"microbenchmark in this run: {pk['instr_per_clk_per_sm']:.1f} instr/clk/SM, {alu_peak_t:.2f} Tinstr/s "
                         f"(spec: 148 SMs x {64 if arith == 'f64' else 128} lanes x clock)"}
    roof = roof_alu if roof_alu["frac"] > roof_hbm["frac"] else roof_hbm
    if roof is roof_alu:
        roof["hbm_model"] = roof_hbm
    else:
        roof["alu_model"] = roof_alu
    return roof


def default_inner(sites, order, ndim):
    """Time steps per bench step: about 0.5 s of GPU work for the interleaved ordering; four times as many steps for the
    plain ordering in 2D / 3D, whose steps are four times cheaper (and whose first step of every qlga_step call cannot
    take the band pipeline: its U has not been applied by a previous step)."""
    inner = max(1, min(1000, int(6.0e8 / sites)))
    return min(1000, 4 * inner) if (order == "plain" and ndim >= 2) else inner


def band_timeline(qlga, sim, torch):
    """Timeline of one band step with the trailing U (QLGA_OPT_BAND; debug build of the library with -DQLGA_TRACE):
    per band the first CTA start and last CTA end of its y kernel and its x kernel, microseconds from the first."""
    import ctypes
    lib = qlga._lib
    if not hasattr(lib, "qlga_debug_trace"):
        return {"error": "libqlga.so was not built with -DQLGA_TRACE"}
    buf = (ctypes.c_ulonglong * (2 * 8192))()
    torch.cuda.synchronize()
    lib.qlga_debug_trace(buf, 1)
    sim.step(3)                     # two-launch step, band step with the trailing U (graph 0), last band step
    torch.cuda.synchronize()
    lib.qlga_debug_trace(buf, 0)
    full = np.array(buf, dtype=np.uint64).reshape(-1, 2).astype(np.int64)
    # graph n of the context traces into ids [2048 n, 2048 n + 2 bands): take the first region that was written
    # (the band step with the trailing U is the first of the three steps)
    a = None
    for base in range(0, 8192, 2048):
        reg = full[base:base + 2048]
        if (reg[:, 1] > 0).sum() >= 16:
            if a is None or reg[reg[:, 1] > 0, 0].min() < a[a[:, 1] > 0, 0].min():
                a = reg
    if a is None:
        return {"error": "no band step traced"}
    nb = int((a[:, 1] > 0).sum()) // 2
    t0 = a[:2 * nb, 0].min()
    y0, y1, x0, x1 = ((a[0:2 * nb:2, 0] - t0) / 1e3, (a[0:2 * nb:2, 1] - t0) / 1e3,
                      (a[1:2 * nb:2, 0] - t0) / 1e3, (a[1:2 * nb:2, 1] - t0) / 1e3)
    mid = slice(nb // 4, 3 * nb // 4)
    return {"bands": nb, "step_us": float(x1.max()), "period_us": float(np.diff(x0[mid]).mean()),
            "y_kernel_us": float((y1 - y0)[mid].mean()), "x_kernel_us": float((x1 - x0)[mid].mean()),
            "x_overlap_with_next_x_us": float((x1[mid][:-1] - x0[mid][1:]).mean()),
            "sample": [[round(float(v), 1) for v in (y0[k], y1[k], x0[k], x1[k])] for k in range(nb // 2, nb // 2 + 6)],
            "columns": "y_start, y_end, x_start, x_end (us) of six consecutive bands"}


# the other precisions / orderings of the headline workload and config 3 (the large 1D lattice), a few bench
# steps each, so that they are measured by whoever runs bench.py and not only quoted in DESIGN.md
VARIANTS = (("cfg5", "f32", "interleaved"), ("cfg5", "f32x", "interleaved"), ("cfg5", "f64", "plain"),
            ("cfg5", "f32", "plain"), ("cfg5", "f32x", "plain"), ("cfg5", "f64", "plain+two-launch"), ("cfg5", "f32", "plain+two-launch"),
            ("cfg3", "f64", "interleaved"), ("cfg3", "f32", "interleaved"),
            ("cfg3", "f64", "plain"), ("cfg3", "f32", "plain"),
            ("cfg4", "f64", "interleaved"), ("cfg2", "f64", "interleaved"), ("cfg1", "f64", "interleaved"),
            ("cfg3d", "f64", "interleaved"))


def run_variant(qlga, torch, dev, local_rank, workload, precision, order, psi_dev, w, steps, lattice):
    """One variant: `steps` bench steps (same definition of a step as the headline) after 3 warm-up steps,
    CUDA events on the library's stream, clocks sampled during the timed region, both rooflines."""
    ndim = WORKLOADS[workload]["ndim"]
    sites = int(np.prod(w.dims))
    inner = default_inner(sites, order.split("+")[0], ndim)
    two_launch = order.endswith("+two-launch")     # plain ordering with band mode off (QLGA_OPT_BAND = 0): the comparison
    tag, order = order, order.split("+")[0]
    sim = qlga.Qlga(ndim, w.dims, w.couplings, order=order, precision=precision, device=dev)
    if two_launch:
        sim.set_option(qlga.OPT_BAND, 0)
    cdt = torch.complex128 if precision == "f64" else torch.complex64
    sim.set_state_psi(psi_dev.to(cdt))
    omega = (torch.empty((5, sim.ny, sim.nx), dtype=sim.rdtype, device=dev) if ndim == 2 else None)

    def step():
        sim.step(inner)
        ob = sim.observables()
        if omega is not None:
            sim.vorticity(omega)
        return ob

    ob0 = sim.observables()
    for _ in range(3):
        step()
    sim.profile_enable(True)
    sampler = ClockSampler(local_rank)
    torch.cuda.synchronize()
    sampler.start()
    n0 = sim.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        ob = step()
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    prof = sim.profile_read()
    deg_info = mean_degree(sim)
    launches = sim.launch_count() - n0
    roof = build_roofline(qlga, prof, ndim, sites, inner * steps, precision, order, deg_info, clocks,
                          load_traffic(workload, precision, order) if not lattice else {})
    value = sites * inner * steps / (ms * 1e-3) / 1e9
    out = {"workload": workload, "lattice": list(w.dims), "precision": precision, "order": tag, "value": value, "unit": UNIT,
           "steps": steps, "time_steps_per_bench_step": inner, "ms_per_step": ms / steps, "clocks": clocks,
           "gpu_launches": launches, "roofline": roof,
           "hbm_model_frac": value * 1e9 * bytes_per_site_update(precision) / (load_peaks()[0] * 1e9),
           "kernel_ms": {k: {"ms_total": v[0], "launches": v[1]} for k, v in prof.items() if v[1]},
           "norm_q_drift": ob["norm_q"] / ob0["norm_q"] - 1.0}
    sim.close()
    del sim, omega
    torch.cuda.empty_cache()
    return out


# ---------------------------------------------------------------------------
# this repo's arm
# ---------------------------------------------------------------------------
def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    wl = WORKLOADS[args.workload]
    ndim = wl["ndim"]

    if args.impl == "reference" and rank != 0:
        return                                              # rank 0 alone runs the oracle arm
    w = wl["gen"](args.lattice)
    nx, ny = w.dims[0], w.dims[1]
    sites = int(np.prod(w.dims))
    lat = tuple(reversed(w.dims)) if ndim == 3 else (ny, nx)        # array shape of one plane
    cfg_tag = (f"BASELINE.json configs[{int(args.workload[3]) - 1}]" if args.workload[3:].isdigit()
               else "SURVEY.md 8(f) row 3, not a BASELINE.json config")
    inner = args.inner or default_inner(sites, args.order, ndim)
    config = {"workload": f"{w.name} ({cfg_tag}): "
                          f"{ndim}D periodic {'x'.join(str(v) for v in w.dims[:max(2, ndim)])}, {args.precision}, "
                          f"{args.order} ordering (eq. {'112' if args.order == 'interleaved' else '108'})",
              "lattice": list(w.dims), "precision": args.precision, "order": args.order,
              "couplings": list(w.couplings), "time_steps_per_bench_step": inner,
              "per_bench_step": f"{inner} time steps + 1 observables reduction" + (" + 1 vorticity map" if ndim == 2 else ""),
              "l2_policy": "state (%.1f GB per buffer) larger than the 126 MB L2" % (sites * 160 / 1e9 * (1 if args.precision == 'f64' else 0.5))
                           if sites * 80 > 126e6 else "state fits in L2 (latency-bound workload; no HBM claim)",
              "parallelism": (f"slabs x{args.gpus} of one lattice {args.gpus} times as long along its slowest axis, "
                              "ring exchange of 4 ghost layers per side per time step (NCCL P2P; device copy at N=1)"
                              if args.slab else
                              f"replicas x{args.gpus} (one lattice per GPU, no data-path collective)")}
    if args.impl == "reference":
        run_reference(args, w, ndim, config)
        return

    import torch
    from paper_1907_12834_b200 import qlga                  # fails loudly without libqlga.so
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device; there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cdt = torch.complex128 if args.precision == "f64" else torch.complex64
    # host input in pinned memory: q1 = q2 = psi/2 (reading R6)
    q_host = torch.empty((5, 2) + lat, dtype=cdt, pin_memory=True)
    half = torch.from_numpy(w.psi / 2).to(cdt)
    q_host[:, 0] = half
    q_host[:, 1] = half
    del half
    out_host = torch.empty_like(q_host, pin_memory=True) if not args.no_e2e else None

    ss = None
    if args.slab:
        # every rank owns the workload's lattice; the global lattice is that tile repeated along the slab
        # axis (continuous: the tile is periodic), so the extended slab is the tile plus its own wrap
        from paper_1907_12834_b200 import slab
        args.no_e2e = True
        gdims = tuple(w.dims[:ndim - 1]) + (w.dims[ndim - 1] * world,)
        ss = slab.SlabQlga(ndim, gdims, w.couplings, order=args.order, precision=args.precision,
                           rank=rank, world=world, device=dev)
        sim = ss.sim
        n_own = w.dims[ndim - 1]
        ext = (np.arange(-slab.GHOST, n_own + slab.GHOST)) % n_own
        q_ext = np.ascontiguousarray(np.take(q_host.numpy(), ext, axis=-ndim))
    else:
        sim = qlga.Qlga(ndim, w.dims, w.couplings, order=args.order, precision=args.precision, device=dev)
    if args.tile_y:
        sim.set_option(qlga.OPT_TILE_Y, args.tile_y)
    if args.threads_x:
        sim.set_option(qlga.OPT_THREADS_X, args.threads_x)
    if args.threads_y:
        sim.set_option(qlga.OPT_THREADS_Y, args.threads_y)
    if args.steps_per_launch:
        sim.set_option(qlga.OPT_STEPS_PER_LAUNCH, args.steps_per_launch)
    if args.tol_log2:
        sim.set_option(qlga.OPT_EXP_TOL_LOG2, args.tol_log2)
    if args.mod_shift >= 0:
        sim.set_option(qlga.OPT_EXP_MOD_SHIFT, args.mod_shift)
    if args.band >= 0 or args.band_rows or args.band_slots:
        sim.set_option(qlga.OPT_BAND, args.band)
        sim.set_option(qlga.OPT_BAND_ROWS, args.band_rows)
        sim.set_option(qlga.OPT_BAND_SLOTS, args.band_slots)
        config["band"] = {"mode": args.band, "rows": args.band_rows, "slots": args.band_slots}
    omega_dev = (torch.empty((5, sim.ny, nx), dtype=torch.float64 if args.precision == "f64" else torch.float32,
                             device=dev) if ndim == 2 else None)
    state_bytes = q_host.numel() * q_host.element_size()

    def hot_path_step():
        if ss is not None:
            ss.step(inner)                   # inner x (library step on the extended slab + halo exchange)
            obs = ss.observables()           # owned-layer sums, all-reduced over the slabs
        else:
            sim.step(inner)
            obs = sim.observables()
        if omega_dev is not None:
            sim.vorticity(omega_dev)
        return obs

    # ---- device-resident measurement -------------------------------------------------
    sim.set_state_q(q_ext if ss is not None else q_host.numpy())
    obs0 = ss.observables() if ss is not None else sim.observables()
    for _ in range(max(3, args.warmup)):
        hot_path_step()
    sim.profile_enable(True)
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    launches0 = sim.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if args.profiler_range:
        torch.cuda.profiler.start()
    ev0.record()
    for _ in range(args.steps):
        obs = hot_path_step()
    ev1.record()
    barrier()
    if args.profiler_range:
        torch.cuda.profiler.stop()
    clocks = sampler.stop()
    launches = sim.launch_count() - launches0
    ms = ev0.elapsed_time(ev1)
    prof = sim.profile_read()
    sim.profile_enable(False)
    deg_info = mean_degree(sim)
    ms = max_over_ranks(ms, world, dev)
    value = aggregate_gsups(sites, inner * args.steps, world, ms)
    band_trace = band_timeline(qlga, sim, torch) if args.band_trace else None

    # ---- end to end through the C ABI with host buffers ---------------------------------
    # The user-facing call: upload the five wavefunctions psi_m (the paper's initial condition, split as
    # q1 = q2 = psi/2 on the device, reading R6), step, reduce the observables, download psi_m.  A second
    # record moves the full two-spinor state q (what a checkpoint / restart of the run needs) both ways.
    e2e = None
    e2e_q = None
    if not args.no_e2e:
        # the psi buffers alias the first half of the pinned q buffers (the full-state record runs first)
        psi_host = q_host.view(-1)[:5 * sites].view((5,) + lat)
        psi_out = out_host.view(-1)[:5 * sites].view((5,) + lat)
        psi_bytes = psi_host.numel() * psi_host.element_size()

        def e2e_psi():
            sim.set_state_psi(psi_host.numpy())             # H2D from pinned host memory + split on the device
            sim.step(inner)
            o = sim.observables()
            sim.get_state_psi(psi_out.numpy())              # sum on the device + D2H of the step's result
            return o

        def e2e_full():
            sim.set_state_q(q_host.numpy())
            sim.step(inner)
            o = sim.observables()
            sim.get_state_q(out_host.numpy())
            return o

        def timed(fn, h2d, d2h, call):
            fn()
            barrier()
            t0 = time.perf_counter()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(args.e2e_steps):
                fn()
            e1.record()
            barrier()
            wall = time.perf_counter() - t0
            ems = max_over_ranks(max(e0.elapsed_time(e1), 0.0), world, dev)
            return {"value": aggregate_gsups(sites, inner * args.e2e_steps, world, ems), "unit": UNIT,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h + 168,
                    "steps": args.e2e_steps, "ms_per_step": ems / args.e2e_steps,
                    "wall_ms_per_step": wall * 1e3 / args.e2e_steps, "call": call}

        e2e_q = timed(e2e_full, state_bytes, state_bytes,
                      "qlga_set_state_q(host) + qlga_step(n) + qlga_observables + qlga_get_state_q(host)")
        psi_host.copy_(torch.from_numpy(w.psi).to(cdt))
        e2e = timed(e2e_psi, psi_bytes, psi_bytes,
                    "qlga_set_state_psi(host) + qlga_step(n) + qlga_observables + qlga_get_state_psi(host)")

    if rank != 0:
        return

    # ---- roofline of the dominant kernel (the pass kernels) -----------------------------
    hbm_peak = load_peaks()[0]
    bps = bytes_per_site_update(args.precision)
    roof = build_roofline(qlga, prof, ndim, sites, inner * args.steps, args.precision, args.order, deg_info, clocks,
                          load_traffic(args.workload, args.precision, args.order) if not args.lattice else {})

    # ---- variants (rank 0, one GPU): free the headline's buffers first ------------------------------
    variants = None
    if world == 1 and not args.no_variants and not args.slab:
        sim.close()
        del sim, omega_dev, q_host, out_host
        torch.cuda.empty_cache()
        variants = []
        psi_cache = {}
        for vw, vp, vo in VARIANTS:
            if (vw, vp, vo) == (args.workload, args.precision, args.order):
                continue
            if vw not in psi_cache:
                psi_cache.clear()
                torch.cuda.empty_cache()
                ww = w if vw == args.workload else WORKLOADS[vw]["gen"](args.lattice if vw == args.workload else 0)
                psi_cache[vw] = (ww, torch.from_numpy(ww.psi).to(dev))
            ww, psi_dev = psi_cache[vw]
            try:
                variants.append(run_variant(qlga, torch, dev, local_rank, vw, vp, vo, psi_dev, ww, args.variant_steps,
                                            args.lattice if vw == args.workload else 0))
            except Exception as exc:                       # a failed variant must not lose the headline line
                variants.append({"workload": vw, "precision": vp, "order": vo, "error": repr(exc)})
        psi_cache.clear()

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        rate, sample, _, _ = time_oracle(w, ndim, args.order, args.cpu_seconds)
        cpu = {"value": rate / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
            "config": config, "clocks": clocks, "e2e": e2e, "e2e_full_state": e2e_q, "gpu_launches": launches,
            "roofline": roof, "cpu_baseline": cpu, "variants": variants,
            "hbm_model_frac": value / world * 1e9 * bps / (hbm_peak * 1e9),
            "kernel_ms": {k: {"ms_total": v[0], "launches": v[1]} for k, v in prof.items()},
            "pass_kernel_share_of_step": sum(v[0] for v in prof.values()) / ms if ms > 0 else None,
            "norm_q_drift": obs["norm_q"] / obs0["norm_q"] - 1.0,
            "sim_step": obs["step"]}
    if band_trace is not None:
        line["band_trace"] = band_trace
    line["issue_peaks"] = {k: {"instr_per_clk_per_sm": v["instr_per_clk_per_sm"], "tinstr_per_s": v["instr_per_s"] / 1e12}
                           for k, v in _ALU_PEAKS.items()}          # qlga_issue_peak, measured in this run
    if ss is not None:
        halo = 2 * ss.edge_lo.numel() * ss.edge_lo.element_size()
        line["slab"] = {"ghost_layers": 4, "owned_layers": int(w.dims[ndim - 1]),
                        "halo_bytes_sent_per_rank_per_time_step": halo,
                        "transport": "torch.distributed P2P (NCCL)" if world > 1 else "device copy (one slab, its own wrap)"}
    print(json.dumps(line))


if __name__ == "__main__":
    main()
