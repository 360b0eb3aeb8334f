#!/usr/bin/env python
"""bench.py — grid-point RK4 updates/s of libadsc on B200, with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl reference]

One bench "step" = `--rk4-per-step` (default: RK4_PER_STEP below, 1200 for cfg2) classical RK4 steps of the whole
ensemble through ONE adsc_step call: every row of SURVEY.md 8(a) (a1-a6) runs 4x per RK4 step.  The defaults
give >= 2 s of timed GPU work with --steps 20 (SURVEY.md 8(d) protocol).
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
#   fixed background: no f, scan, exp, A update: per stage fluxes 3 + D4 H 4 +
#   cot^2 D4 F 5 + 2 x KO 14 + RK combine of Phi, Pi 4 = 30, x 4 stages.
SLOTS_PER_POINT_STEP_FIXED = 120.0
#   streaming regime: bytes of HBM traffic with classical RK4 and one fused pass per stage.
BYTES_PER_POINT_STEP = 384.0
# FP64 ALU peak: 148 SMs x 64 DFMA lanes/clk x sm_max_mhz (derived in DESIGN.md; the
# measured DFMA issue rate on this pool is recorded there too).
FP64_LANES_PER_SM = 64
N_SMS = 148
# Global-memory bytes per point per RK stage the persistent streaming kernel provably moves (u^n and accumulator
# in the permuted arrays; the stage state never leaves shared memory): classical RK4 = 24 (stage 1: accumulator
# written) + 72 + 72 (u^n read, accumulator read and written) + 48 (accumulator read, u^n written) = 216 B per
# point per step, plus 3 coefficient tables x 8 B per stage staged by bulk copies.
STREAM_BYTES_STAGE_FIRST, STREAM_BYTES_STAGE_MID, STREAM_BYTES_STAGE_LAST, STREAM_BYTES_TABLES = 24.0, 72.0, 48.0, 24.0
L2_BYTES = 126e6


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="adsc", choices=["adsc", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "paper32k"])
    ap.add_argument("--rk4-per-step", type=int, default=0, help="RK4 steps per bench step (0 = workload default)")
    ap.add_argument("--batch", type=int, default=0, help="override the ensemble size (0 = workload default)")
    ap.add_argument("--grid-points", type=int, default=0, metavar="N",
                    help="override the grid size N of the workload's data family (diagnosis only: the line then no "
                         "longer describes a BASELINE.json config; config.N says what ran)")
    ap.add_argument("--path", type=int, default=0, help="0 auto, 1 persistent streaming, 2 resident, 3 generic streaming")
    ap.add_argument("--fixed-background", action="store_true",
                    help="time the fixed-background variant (A = 1, delta = 0 held fixed; PAPER.md:177 Table II)")
    ap.add_argument("--rk-order", type=int, default=0, choices=[0, 2, 3, 4],
                    help="Runge-Kutta order (PAPER.md:57; 3 and 2 run on the streaming paths); the metric then counts "
                         "grid-point steps of that rule and the algorithmic cost scales with the stage count "
                         "(0 = workload default: 4, except paper32k: 3)")
    ap.add_argument("--masked-fraction", type=float, default=0.0,
                    help="force this fraction of the members to collapse during warm-up (Pi x 1000): shows that masked "
                         "members cost nothing; the metric then counts the members still active (SURVEY.md 8(d))")
    ap.add_argument("--e2e-parts", type=int, default=8, help="sub-batches (handles, streams) of the e2e leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle sample")
    ap.add_argument("--spread", action="store_true",
                    help="ADSC_OPT_SPREAD: latency mode for ensembles that do not fill the device (more, shorter CTAs per member)")
    ap.add_argument("--mode-energies", type=int, default=0, metavar="J",
                    help="also time adsc_mode_energies(J) (SURVEY.md 8(f) f3) on the evolved ensemble and add a "
                         "`mode_energies` object with its own roofline to the line")
    ap.add_argument("--extra-workloads", default="cfg3,cfg5,cfg4,paper32k:1", metavar="LIST",
                    help="comma list of name[:path] also timed at N=1 (device-resident, own roofline) and reported in "
                         "`workloads`: the other configs the 60 %% target is stated on, cfg4, and the paper's "
                         "production shape forced onto the streaming kernel (the one workload that leaves L2); '' = none")
    ap.add_argument("--extra-seconds", type=float, default=1.0, help="timed window of each extra workload")
    ap.add_argument("--probe-ms", type=float, default=50.0, help="duration of each roofline-denominator probe (0 = skip)")
    a = ap.parse_args()
    if a.rk_order == 0:
        a.rk_order = 3 if a.workload == "paper32k" else 4
    return a


# RK steps per bench step: >= 100 ms per adsc_step call, so that --steps 20 times >= 2 s of GPU work
RK4_PER_STEP = {"cfg1": 25000, "cfg2": 1200, "cfg3": 150, "cfg4": 1500, "cfg5": 200, "paper32k": 2000}
WORKLOAD_DESC = {
    "cfg1": "configs[0]: 1 member, N=1025, Gaussian Pi sigma=1/16 eps=1",
    "cfg2": "configs[1]: amplitude ensemble, 1024 members, N=4097, Gaussian Pi sigma=1/16 eps~U[0.5,5]",
    "cfg3": "configs[2]: two-mode ensemble, 4096 members, N=8193",
    "cfg4": "configs[3]: single large grid, 1 member, N=2^20+1",
    "cfg5": "configs[4]: wide-pulse ensemble, 16384 members, N=2049",
    "paper32k": "the paper's production shape (PAPER.md:57, 115, 123): 64 amplitudes of the k_d=3, mu=1 family of "
                "eq (13), N=2^15+1, RK3",
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


def oracle_rate(name, N, seconds, rk4_cap=None, fixed=False, rk_order=4, threads=None):
    """Time the oracle as it stands on the host cores on a bounded sample of the workload:
    2 x cores members (or the whole batch if smaller), enough RK4 steps for ~`seconds`.
    threads=1: the one-core, one-member leg of SURVEY.md 8(d)(i)."""
    import oracle
    from paper_1706_07413_b200 import inputs
    cores = os.cpu_count() or 1
    thr = min(cores, oracle.max_threads()) if threads is None else threads
    Bfull = inputs.CONFIGS[name]["B"]
    B = min(Bfull, 2 * thr) if threads is None else threads
    thr = min(thr, B)
    Phi, Pi, _ = inputs.make(name, B=B, N=N)
    ev = oracle.Evolution(Phi, Pi, nthreads=thr, fixed_background=fixed, rk_order=rk_order)
    t = time.perf_counter(); ev.step(2); cal = (time.perf_counter() - t) / 2
    n = max(2, int(seconds / max(cal, 1e-9)))
    if rk4_cap:
        n = min(n, rk4_cap)
    t = time.perf_counter(); ev.step(n); el = time.perf_counter() - t
    rate = B * N * n / el
    return dict(value=rate, unit=UNIT, cores=thr, kind="oracle",
                sample=f"{B} members of {name} (N={N}) x {n} RK4 steps, {el:.1f} s, oracle/adsc_oracle.c "
                       f"gcc -O2 -ffp-contract=off, OpenMP over members"), el, n, B


def fast_build_rate(name, N, seconds, fixed, rk_order):
    """The oracle's source compiled for throughput (gcc -O3 -march=native -ffp-contract=fast; oracle.build_fast) on the
    same sample and cores, checked against the oracle over 20 steps first.  Reported beside the oracle's rate: the
    oracle is the unoptimised checker, this is the same program as a compiler makes it fast."""
    import oracle
    from paper_1706_07413_b200 import inputs
    try:
        thr = min(os.cpu_count() or 1, oracle.max_threads())
        B = min(inputs.CONFIGS[name]["B"], thr)
        thr = min(thr, B)
        Phi, Pi, _ = inputs.make(name, B=B, N=N)
        ref = oracle.Evolution(Phi, Pi, nthreads=thr, fixed_background=fixed, rk_order=rk_order).step(20)
        oracle.use_build("fast")
        ev = oracle.Evolution(Phi, Pi, nthreads=thr, fixed_background=fixed, rk_order=rk_order).step(20)
        diff = float(max(np.max(np.abs(ev.Phi - ref.Phi)), np.max(np.abs(ev.Pi - ref.Pi)), np.max(np.abs(ev.A - ref.A))))
        t = time.perf_counter(); ev.step(2); cal = (time.perf_counter() - t) / 2
        n = max(2, int(seconds / max(cal, 1e-9)))
        t = time.perf_counter(); ev.step(n); el = time.perf_counter() - t
        return {"value": B * N * n / el, "unit": UNIT, "cores": thr, "flags": " ".join(oracle.FAST_FLAGS),
                "max_abs_diff_vs_oracle_20_steps": diff,
                "sample": f"{B} members of {name} (N={N}) x {n} steps, {el:.1f} s"}
    except Exception as e:                                  # (a missing -march=native target etc.: no fast figure)
        return {"value": None, "error": str(e)[:200]}
    finally:
        oracle.use_build("oracle")


def make_roofline(path, B, N, NS, fixed, per_gpu_rate, rk4, launches_per_step, probe, peaks, probe_ms):
    """The `roofline` object of one workload on one GPU: resident path = FP64 ALU bound,
    streaming paths = the [NS] HBM line with the ALU fraction beside it."""
    peak_tf = N_SMS * FP64_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6 * 2 / 1e12
    slots = (SLOTS_PER_POINT_STEP_FIXED if fixed else SLOTS_PER_POINT_STEP) * NS / 4.0
    ach_tf = per_gpu_rate * slots * 2 / 1e12
    peak_src = (f"derived: {N_SMS} SMs x {FP64_LANES_PER_SM} DFMA lanes x {peaks['sm_max_mhz']:.0f} MHz x 2 flop "
                f"(DESIGN.md Roofline); peak_measured: adsc_probe(FP64_FMA) run for {probe_ms:.0f} ms before "
                f"the timed region")
    fp64_meas = probe["fp64_fma_tflops"] if probe else None
    if path == 2:
        return {"bound": "alu", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": ach_tf / peak_tf,
                "peak_measured": fp64_meas, "frac_of_measured": (ach_tf / fp64_meas) if fp64_meas else None,
                "shared_load_tbs_measured": probe["shared_load_tbs"] if probe else None,
                "traffic": 6.0 * B * N * 8,
                "traffic_unit": "global-memory bytes per launch: the three fields are loaded once and stored once, whatever "
                                "the number of steps in the launch (the ncu dram figures are in profiles/)",
                "kernel": f"k_resident3 (whole RK steps on chip; {launches_per_step} launch per adsc_step)",
                "peak_src": peak_src,
                "algorithmic": f"{slots:.0f} FP64-pipe instr per point per step"}
    # [NS]/SURVEY.md 8(d) streaming roofline: bytes per point per step with one fused pass per stage:
    # first and last stage 72 B, every middle stage 120 B
    bytes_step = 72.0 * 2 + 120.0 * (NS - 2)
    if fixed:
        bytes_step *= 2.0 / 3.0                       # two evolved fields instead of three
    ach = per_gpu_rate * bytes_step / 1e9
    kern_bytes = (STREAM_BYTES_STAGE_FIRST + STREAM_BYTES_STAGE_LAST + STREAM_BYTES_STAGE_MID * (NS - 2)
                  + STREAM_BYTES_TABLES * NS)
    wset = 9.0 * B * N * 8 + 3.0 * N * 8
    return {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
            "frac": ach / peaks["hbm_gbs"],
            "traffic": (kern_bytes * rk4 + 48.0) * B * N if path == 1 else None,
            "traffic_unit": "global-memory bytes per launch the kernel provably requests (u^n, accumulator, tables; "
                            "load + store of the fields once); see l2_resident",
            "kernel_bytes_per_point_step": kern_bytes if path == 1 else None,
            "working_set_bytes": wset, "l2_resident": bool(wset < L2_BYTES),
            "alu": {"achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach_tf / peak_tf,
                    "peak_measured": fp64_meas, "frac_of_measured": (ach_tf / fp64_meas) if fp64_meas else None},
            "note": ("the [NS] streaming roofline (algorithmic bytes over the HBM copy peak); when l2_resident is true "
                     "the working set never leaves the 126 MB L2, HBM is not the binding resource and the `alu` "
                     "fraction is the one that measures the kernel"),
            "kernel": ("k_stream_async (stage state in shared memory, tables staged by cp.async.bulk rings, "
                       "u^n/accumulator through L2; 1 cooperative launch per adsc_step)" if path == 1 else
                       "k_stream_rhs (+ k_stream_I, k_stream_carry: 3 launches per RK stage)"),
            "peak_src": f"{peaks['src']} copy bandwidth (MEASURED_PEAKS.json); alu: " + peak_src,
            "algorithmic": f"{bytes_step:.0f} B per point per step"}


def time_extra_workload(torch, binding, inputs, dev, index, flush, name, path_opt, seconds, probe, peaks, probe_ms):
    """One more BASELINE.json config (or the paper's production shape) at full size on this GPU, by the protocol of the
    headline: 3 warm-up adsc_step calls, then enough calls for >= `seconds` of device time, L2 flushed before each,
    CUDA events on the stream the kernels run on, clocks sampled during the window.  Device-resident only (no e2e,
    no CPU leg: those belong to the headline workload)."""
    cfg = inputs.CONFIGS[name]
    N, B = cfg["N"], cfg["B"]
    order = 3 if name == "paper32k" else 4
    rk4 = RK4_PER_STEP[name]
    Phi, Pi, _ = inputs.make(name, B=B, N=N)
    ens = binding.Ensemble(N, B, device=dev, path=path_opt, rk_order=(order if order != 4 else None))
    path, cluster = ens.path
    ens.set_initial(torch.from_numpy(np.ascontiguousarray(Phi)).to(dev), torch.from_numpy(np.ascontiguousarray(Pi)).to(dev))
    del Phi, Pi
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ms1 = 0.0
    for _ in range(3):                                           # warm-up (the last one also sizes the window)
        a.record(); ens.step(rk4); b.record(); torch.cuda.synchronize(dev)
        ms1 = a.elapsed_time(b)
    K = max(3, min(40, int(np.ceil(seconds * 1e3 / max(ms1, 1e-3)))))
    l0 = ens.launch_count
    sampler = ClockSampler(index)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    t0 = time.time()
    for a, b in evs:
        flush.fill_(1)
        a.record(); ens.step(rk4); b.record()
    torch.cuda.synchronize(dev)
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    launches = ens.launch_count - l0
    ms = sum(a.elapsed_time(b) for a, b in evs)
    d = ens.diagnostics()
    value = float(B) * N * rk4 * K / (ms * 1e-3)
    out = {"workload": WORKLOAD_DESC[name], "name": name, "N": N, "batch": B, "rk_order": order, "rk_steps_per_step": rk4,
           "path": {1: "streaming-persistent", 2: "resident", 3: "streaming-generic"}[path], "ctas_per_member": cluster,
           "value": value, "unit": UNIT, "steps": K, "warmup": 3, "ms_per_step": ms / K, "timed_region_s": ms * 1e-3,
           "active_fraction": float((d["collapsed"] == 0).mean()), "gpu_launches": int(launches),
           "roofline": make_roofline(path, B, N, order, False, value, rk4, launches // K, probe, peaks, probe_ms),
           "clocks": clocks}
    ens.close()
    del ens
    torch.cuda.empty_cache()
    return out


# ----------------------------------------------------------------------------- reference arm
def run_reference(args):
    """`--impl reference`: the oracle as it stands on the host cores, same config/metric/unit.
    Each bench step is a bounded sample: min(B, 2 x cores) members x n RK4 steps (n sized from a
    calibration so that warmup+steps stay within ~cpu-seconds each ... a few minutes in total)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from paper_1706_07413_b200 import inputs
    name = args.workload
    N = inputs.CONFIGS[name]["N"]
    cores = os.cpu_count() or 1
    thr = min(cores, oracle.max_threads())
    B = min(inputs.CONFIGS[name]["B"], 2 * thr)
    thr = min(thr, B)
    Phi, Pi, _ = inputs.make(name, B=B)
    ev = oracle.Evolution(Phi, Pi, nthreads=thr, fixed_background=args.fixed_background, rk_order=args.rk_order)
    t = time.perf_counter(); ev.step(2); cal = (time.perf_counter() - t) / 2
    budget = max(1.0, min(args.cpu_seconds, 150.0 / max(1, args.steps + args.warmup)))
    n = max(1, int(budget / max(cal, 1e-9)))
    for _ in range(args.warmup):
        ev.step(n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ev.step(n)
    el = time.perf_counter() - t0
    rate = B * N * n * args.steps / el
    sample = (f"{B} members of {name} (N={N}) x {n} RK4 steps per bench step, oracle/adsc_oracle.c "
              f"gcc -O2 -ffp-contract=off, OpenMP over members")
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic (seeded, paper_1706_07413_b200/inputs.py)",
        "config": {"workload": WORKLOAD_DESC[name], "N": N, "batch_sampled": B, "rk4_per_step": n,
                   "courant": 0.25, "ko_eps": 0.1, "fixed_background": bool(args.fixed_background)},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- product arm
def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_1706_07413_b200 import binding, inputs, shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libadsc has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    name = args.workload
    cfg = inputs.CONFIGS[name]
    N = args.grid_points or cfg["N"]
    B = args.batch or cfg["B"]              # members PER GPU (weak scaling: members are independent)
    rk4 = args.rk4_per_step or RK4_PER_STEP[name]
    K, W = args.steps, max(args.warmup, 0)

    # Rank r evolves members [r*B, (r+1)*B) of the (tiled) seeded ensemble: no exchange step.
    lo, hi = shard.member_range(rank, world, B * world)
    Phi_all, Pi_all, _ = inputs.make(name, B=hi, lo=lo, N=N)  # this rank's members only
    if args.masked_fraction > 0.0:
        bidx = np.arange(lo, hi)
        forced = np.floor((bidx + 1) * args.masked_fraction) > np.floor(bidx * args.masked_fraction)
        Pi_all[forced] *= 1.0e3                   # collapses within the first warm-up steps
    Phi_h = torch.from_numpy(np.ascontiguousarray(Phi_all)).pin_memory()
    Pi_h = torch.from_numpy(np.ascontiguousarray(Pi_all)).pin_memory()
    del Phi_all, Pi_all

    ens = binding.Ensemble(N, B, device=dev, path=args.path, spread=args.spread,
                           fixed_background=args.fixed_background, rk_order=(args.rk_order if args.rk_order != 4 else None))
    path, cluster = ens.path
    Phi_d, Pi_d = Phi_h.to(dev), Pi_h.to(dev)
    ens.set_initial(Phi_d, Pi_d)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- roofline denominators measured on this device, before the timed region (adsc_probe)
    probe = None
    if args.probe_ms > 0.0 and rank == 0:
        probe = {"fp64_fma_tflops": binding.adsc_probe(binding.ADSC_PROBE_FP64_FMA, args.probe_ms) / 1e12,
                 "shared_load_tbs": binding.adsc_probe(binding.ADSC_PROBE_SHARED_LOAD, args.probe_ms) / 1e12}

    # ---- device-resident timing: K bench steps, each one adsc_step(rk4) call
    for _ in range(W):
        ens.step(rk4)
    barrier()
    l0 = ens.launch_count
    sampler = ClockSampler(local_rank) if rank == 0 else None
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    t0 = time.time()
    for a, b in evs:
        flush.fill_(1)                      # L2 flush between timed iterations (outside the events)
        a.record()
        ens.step(rk4)
        b.record()
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if sampler else None
    launches = ens.launch_count - l0
    ms = sum(a.elapsed_time(b) for a, b in evs)
    d = ens.diagnostics()
    active_frac = float((d["collapsed"] == 0).mean())
    if dist is not None:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    n_active = float((d["collapsed"] == 0).sum())
    if dist is not None:
        t = torch.tensor([n_active], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        n_active = float(t.item())
    # members still active x N x RK4 steps; without forced collapses every member is active
    updates = (n_active if args.masked_fraction > 0.0 else float(B) * world) * N * rk4 * K
    value = updates / (ms * 1e-3)

    # ---- f3: normal-mode projection of the evolved ensemble (off the per-step path; its own roofline)
    modes = None
    if args.mode_energies > 0:
        J = args.mode_energies
        ens.mode_energies(J)                               # warm-up
        torch.cuda.synchronize(dev)
        tm0 = time.perf_counter()
        reps = 5
        for _ in range(reps):
            ens.mode_energies(J)                           # two kernels + D2H of [B][J]; synchronises
        tm = (time.perf_counter() - tm0) / reps
        # per point: sincospi and the j-independent weights (~45 FP64-pipe instr), per point and mode: two Jacobi
        # recurrences (6) + two projections (4)
        m_slots = 45.0 + 10.0 * J
        modes = {"J": J, "ms_per_call": tm * 1e3, "points_per_s": B * N / tm, "algorithmic": f"{m_slots:.0f} FP64-pipe instr per point",
                 "achieved_tflops": B * N / tm * m_slots * 2 / 1e12}

    # ---- end to end through the C ABI with HOST buffers: H2D of Phi, Pi + step + D2H of the fields
    Phi_o = torch.empty_like(Phi_h).pin_memory(); Pi_o = torch.empty_like(Phi_h).pin_memory()
    A_o = torch.empty_like(Phi_h).pin_memory()
    Ke = max(1, min(K, 5))
    out = {"Phi": Phi_o, "Pi": Pi_o, "A": A_o}
    # The user-facing way to run a batch from host memory: sub-batches on their own handles and streams, so that one
    # sub-batch's transfers overlap the other's kernels (binding.PipelinedEnsemble; members are independent).
    parts = max(1, min(args.e2e_parts, B // 32))
    pe = binding.PipelinedEnsemble(N, B, parts=parts, device=dev, path=args.path, spread=args.spread,
                                   fixed_background=args.fixed_background,
                                   rk_order=(args.rk_order if args.rk_order != 4 else None))
    for _ in range(1):
        pe.set_initial(Phi_h, Pi_h); pe.step(rk4); pe.get_fields_host(out); pe.synchronize()
    barrier()
    te0 = time.perf_counter()
    for _ in range(Ke):
        pe.set_initial(Phi_h, Pi_h)
        pe.step(rk4)
        pe.get_fields_host(out)              # enqueued; diagnostics() synchronises every stream
        dd = pe.diagnostics()
    barrier()
    e2e_s = time.perf_counter() - te0
    if dist is not None:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e_value = (updates / K) * Ke / e2e_s
    h2d = 2 * B * N * 8
    d2h = 3 * B * N * 8 + B * binding.DIAG_DTYPE.itemsize

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    peaks = load_peaks()
    roof = make_roofline(path, B, N, args.rk_order, args.fixed_background, value / world, rk4, launches // max(K, 1),
                         probe, peaks, args.probe_ms)

    # ---- the other configs the north_star target is stated on, by the same protocol, each with its own roofline
    extra = None
    if args.extra_workloads and world == 1:
        del ens, pe, Phi_d, Pi_d, Phi_h, Pi_h, Phi_o, Pi_o, A_o, out
        torch.cuda.empty_cache()
        extra = []
        for spec in args.extra_workloads.split(","):
            wname, _, wpath = spec.partition(":")
            if wname == name and int(wpath or 0) == args.path:
                continue
            extra.append(time_extra_workload(torch, binding, inputs, dev, local_rank, flush, wname, int(wpath or 0),
                                             args.extra_seconds, probe, peaks, args.probe_ms))

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        cpu, _, _, _ = oracle_rate(name, N, args.cpu_seconds, fixed=args.fixed_background, rk_order=args.rk_order)
        one, _, _, _ = oracle_rate(name, N, min(5.0, args.cpu_seconds), fixed=args.fixed_background,
                                   rk_order=args.rk_order, threads=1)
        cpu["one_core"] = {"value": one["value"], "unit": UNIT, "cores": 1, "sample": one["sample"]}
        cpu["fast_build"] = fast_build_rate(name, N, min(5.0, args.cpu_seconds), args.fixed_background, args.rk_order)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "timed_region_s": ms * 1e-3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic (seeded, paper_1706_07413_b200/inputs.py)",
        "config": {"workload": WORKLOAD_DESC[name], "N": N, "batch_per_gpu": B, "global_batch": B * world,
                   "rk4_per_step": rk4, "courant": 0.25, "ko_eps": 0.1, "fixed_background": bool(args.fixed_background), "rk_order": args.rk_order,
                   "path": {1: "streaming-persistent", 2: "resident", 3: "streaming-generic"}[path],
                   "ctas_per_member": cluster, "spread": bool(args.spread),
                   "parallelism": f"members sharded over {world} GPU(s), no collective",
                   "l2": "flushed between timed iterations (256 MiB fill)",
                   "active_fraction": active_frac, "masked_fraction_forced": args.masked_fraction},
        "roofline": roof,
        "cpu_baseline": cpu,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": Ke, "what": "adsc_set_initial_host + adsc_step + adsc_get_fields_host_async(Phi,Pi,A) + adsc_diagnostics, "
                        f"{parts} sub-batch(es) on separate streams (binding.PipelinedEnsemble)"},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    if extra is not None:
        line["workloads"] = extra
    if modes is not None:
        peak_tf = N_SMS * FP64_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6 * 2 / 1e12
        modes["roofline"] = {"bound": "alu", "achieved": modes.pop("achieved_tflops"), "peak": peak_tf, "unit": "TFLOP/s"}
        modes["roofline"]["frac"] = modes["roofline"]["achieved"] / peak_tf
        line["mode_energies"] = modes
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
