#!/usr/bin/env python
"""bench.py — grid-point RK4 updates/s of libadsc on B200, with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl reference]

One bench "step" = `--rk4-per-step` (default 100) classical RK4 steps of the whole ensemble
through ONE adsc_step call: every row of SURVEY.md 8(a) (a1-a6) runs 4x per RK4 step.
The N=1 workload is BASELINE.json configs[1] (1024 members, N=4097).  Prints ONE JSON line.
See DESIGN.md "Measurement" for the definitions used here.
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
sys.path.insert(0, ROOT)

METRIC = "grid-point RK4 updates/s (fp64, batched)"
UNIT = "updates/s"

# Algorithmic cost per grid point per RK4 step:
#   resident regime: FP64-pipe instruction slots (FMA/ADD/MUL = 1 slot); reported as
#   TFLOP/s with 2 flop per slot so that it is commensurate with the DFMA peak.
SLOTS_PER_POINT_STEP = 250.0
#   streaming regime: bytes of HBM traffic with classical RK4 and one fused pass per stage.
BYTES_PER_POINT_STEP = 384.0
# FP64 ALU peak: 148 SMs x 64 DFMA lanes/clk x sm_max_mhz (derived in DESIGN.md; the
# measured DFMA issue rate on this pool is recorded there too).
FP64_LANES_PER_SM = 64
N_SMS = 148


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="adsc", choices=["adsc", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--rk4-per-step", type=int, default=0, help="RK4 steps per bench step (0 = workload default)")
    ap.add_argument("--batch", type=int, default=0, help="override the ensemble size (0 = workload default)")
    ap.add_argument("--path", type=int, default=0, help="0 auto, 1 streaming, 2 resident")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


RK4_PER_STEP = {"cfg1": 2000, "cfg2": 100, "cfg3": 50, "cfg4": 20, "cfg5": 100}
WORKLOAD_DESC = {
    "cfg1": "configs[0]: 1 member, N=1025, Gaussian Pi sigma=1/16 eps=1",
    "cfg2": "configs[1]: amplitude ensemble, 1024 members, N=4097, Gaussian Pi sigma=1/16 eps~U[0.5,5]",
    "cfg3": "configs[2]: two-mode ensemble, 4096 members, N=8193",
    "cfg4": "configs[3]: single large grid, 1 member, N=2^20+1",
    "cfg5": "configs[4]: wide-pulse ensemble, 16384 members, N=2049",
}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), src="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, src="fallback")


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.2] or [r for (_, r) in self.rows]
        for r in rows:
            c = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_rate(name, N, seconds, rk4_cap=None):
    """Time the oracle as it stands on the host cores on a bounded sample of the workload:
    2 x cores members (or the whole batch if smaller), enough RK4 steps for ~`seconds`."""
    import oracle
    from paper_1706_07413_b200 import inputs
    cores = os.cpu_count() or 1
    thr = min(cores, oracle.max_threads())
    Bfull = inputs.CONFIGS[name]["B"]
    B = min(Bfull, 2 * thr)
    thr = min(thr, B)
    Phi, Pi, _ = inputs.make(name, B=B)
    ev = oracle.Evolution(Phi, Pi, nthreads=thr)
    t = time.perf_counter(); ev.step(2); cal = (time.perf_counter() - t) / 2
    n = max(2, int(seconds / max(cal, 1e-9)))
    if rk4_cap:
        n = min(n, rk4_cap)
    t = time.perf_counter(); ev.step(n); el = time.perf_counter() - t
    rate = B * N * n / el
    return dict(value=rate, unit=UNIT, cores=thr, kind="oracle",
                sample=f"{B} members of {name} (N={N}) x {n} RK4 steps, {el:.1f} s, oracle/adsc_oracle.c "
                       f"gcc -O2 -ffp-contract=off, OpenMP over members"), el, n, B
