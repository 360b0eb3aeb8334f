"""Run a BASELINE.json configuration IN FULL on the GPU ("full run for CFG 1, 3, 4; ... unless actually run").

    python -m paper_1706_07413_b200.run_config cfg2 [--chunk-steps 50000] [--steps N]

Evolves the whole seeded ensemble of the configuration (inputs.make) for its full number of steps with per-member
collapse detection, looking at the diagnostics every `--chunk-steps` steps, and prints one JSON line: wall-clock and
device time, grid-point updates/s over the members still active, collapse count, mass drift and constraint residual.
All stepping and all reductions run in libadsc; this file only drives it.
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np


def run(name: str, steps: int | None = None, chunk_steps: int = 50000, device: str = "cuda:0"):
    import torch
    from . import binding, inputs
    cfg = inputs.CONFIGS[name]
    N, B = cfg["N"], cfg["B"]
    nsteps = int(steps if steps else cfg["steps"])
    rk = 3 if name == "paper32k" else None
    Phi, Pi, _ = inputs.make(name)
    ens = binding.Ensemble(N, B, device=device, rk_order=rk)
    ens.set_initial(torch.from_numpy(Phi).to(device), torch.from_numpy(Pi).to(device))
    d0 = ens.diagnostics()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    gpu_ms, done, updates = 0.0, 0, 0.0
    d = d0
    while done < nsteps:
        n = min(chunk_steps, nsteps - done)
        active = float((d["collapsed"] == 0).sum())
        ev0.record(); ens.step(n); ev1.record()
        d = ens.diagnostics()                      # synchronises
        gpu_ms += ev0.elapsed_time(ev1)
        updates += active * N * n                  # (upper bound: members that collapse inside the chunk stop early)
        done += n
        if d["collapsed"].all():
            break
    wall = time.perf_counter() - t0
    alive = d["collapsed"] == 0
    out = {
        "config": name, "N": N, "members": B, "steps": done, "t_end": float(done * ens.dt), "path": list(ens.path),
        "wall_s": wall, "gpu_s": gpu_ms * 1e-3, "updates_per_s": updates / (gpu_ms * 1e-3),
        "collapsed": int(d["collapsed"].sum()),
        "max_rel_mass_drift": float(np.max(np.abs(d["mass"][alive] - d0["mass"][alive]) / np.abs(d0["mass"][alive]))) if alive.any() else None,
        "max_constraint_residual": float(np.max(d["constraint_residual"][alive])) if alive.any() else None,
        "min_A": float(np.min(d["min_A"])),
    }
    ens.close()
    return out


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("config", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "paper32k"])
    ap.add_argument("--steps", type=int, default=0, help="0 = the configuration's own number of steps")
    ap.add_argument("--chunk-steps", type=int, default=50000)
    a = ap.parse_args(argv)
    print(json.dumps(run(a.config, a.steps or None, a.chunk_steps)))
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
