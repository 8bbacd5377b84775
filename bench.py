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
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", choices=sorted(WORKLOADS))
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--order", default="interleaved", choices=["interleaved", "plain"])
    ap.add_argument("--inner", type=int, default=0, help="time steps per bench step (0 = auto)")
    ap.add_argument("--lattice", type=int, default=0, help="override the lattice edge (testing)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    ap.add_argument("--tile-y", type=int, default=0)
    ap.add_argument("--threads-x", type=int, default=0)
    return ap.parse_args()


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
    return 320.0 if precision == "f64" else 160.0


def fp_instr_per_site_update(ndim, order, degree):
    """FP instructions (FMA/ADD/MUL, one per lane) per site-update of the fused step,
    counted from qlga_math.cuh: one U of polynomial degree p
    costs about 140 + 200 p, one kinetic factor 40, the final scaling 20 per pass."""
    n_fac = 4 * ndim
    n_u = n_fac if order == "interleaved" else 1
    return n_u * (140.0 + 200.0 * degree) + n_fac * 40.0 + 20.0 * ndim


def expected_degree(w, ndim, order, precision):
    """Degree the kernel's order selection picks on the workload's background state
    (same rule as build_exp_table / interaction(): theta = s (2|c1||F| + |c2| rho / 5))."""
    psi = w.psi.reshape(5, -1)
    idx = np.linspace(0, psi.shape[1] - 1, 4096).astype(np.int64)
    p5 = psi[:, idx]
    n = np.abs(p5) ** 2
    rho = n.sum(0)
    fz = 2 * (n[0] - n[4]) + n[1] - n[3]
    fp = (2 * (np.conj(p5[0]) * p5[1] + np.conj(p5[3]) * p5[4])
          + np.sqrt(6.0) * (np.conj(p5[1]) * p5[2] + np.conj(p5[2]) * p5[3]))
    fabs = np.sqrt(fz ** 2 + np.abs(fp) ** 2)
    s = 1.0 / (4 * ndim) if order == "interleaved" else 1.0
    c0, c1, c2 = w.couplings
    theta = s * (2 * abs(c1) * fabs + abs(c2) / 5 * rho)
    tol = 2.0 ** (-56 if precision == "f64" else -27)
    deg = np.ones_like(theta)
    fact = 2.0
    for p in range(1, 18):
        fact_p = float(np.prod(np.arange(1, p + 2)))
        thr = (tol * fact_p) ** (1.0 / (p + 1)) * 0.999
        deg += theta > thr
    return float(np.percentile(deg, 90))


# ---------------------------------------------------------------------------
# the oracle arm: cpu_baseline (inside the normal run) and --impl reference
# ---------------------------------------------------------------------------
def oracle_sample(w, ndim, order, target_seconds):
    """A periodic crop of the workload's lattice sized for ~target_seconds of oracle time."""
    nx, ny = w.dims
    if ndim == 2:
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
    sites = q.shape[2] * q.shape[3]
    o = 1 if order == "interleaved" else 0
    t0 = time.perf_counter()
    q = orc.step(q, ndim, w.couplings, o, 1)
    t1 = time.perf_counter() - t0
    nsteps = max(1, int(target_seconds / max(t1, 1e-6)) - 1)
    t0 = time.perf_counter()
    orc.step(q, ndim, w.couplings, o, nsteps)
    dt = time.perf_counter() - t0
    rate = sites * nsteps / dt
    sample = (f"periodic {edge}x{edge} crop" if ndim == 2 else f"periodic {edge}-site crop") + \
             f" of the workload's input, {nsteps} time steps, {dt:.1f} s"
    return rate, sample, sites, nsteps


def run_reference(args, w, ndim, config):
    """--impl reference: the oracle as it stands on the host cores, same metric/config."""
    from oracle.qlga_oracle import Oracle
    orc = Oracle("double")
    q, edge = oracle_sample(w, ndim, args.order, 0)
    sites = q.shape[2] * q.shape[3]
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
    sample = (f"periodic {edge}x{edge} crop" if ndim == 2 else f"periodic {edge}-site crop") + \
             f" of the workload's input, {inner} time steps per bench step"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
