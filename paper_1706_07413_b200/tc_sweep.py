"""t_c(eps) driver for the paper's data families (eq (13), Fig. 3).

One ensemble member per amplitude eps of a family A_k = eps exp(-mu |k - k_d|) (Phi(x,0) = 0); the
ensemble is evolved on the GPU until t_max or until every member has collapsed (min A < threshold,
PAPER.md:85: the paper records t_c at 0.01), and the collapse time and the mass loss |M(t)-M(0)|/M(0)
 are tabulated.  All stepping and all diagnostics run in libadsc; this file only builds
the initial data and prints the table.

    python -m paper_1706_07413_b200.tc_sweep --kd 3 --mu 1.0 --eps 0.3,0.4,0.5 --N 4097 --tmax 50
"""
from __future__ import annotations

import argparse

import numpy as np


def sweep(eps, mu: float, kd: int, N: int = 4097, tmax: float = 500.0, threshold: float = 0.01,
          courant: float = 0.25, ko_eps: float = 0.1, chunk_steps: int = 2000, device: str = "cuda:0",
          rk_order: int = 4):
    """Returns a dict of arrays over the amplitudes: eps, t_collapse (NaN if none by t_max), collapsed,
    t (time reached), mass0, mass, mass_loss, min_A."""
    import torch
    from . import binding, inputs
    eps = np.atleast_1d(np.asarray(eps, dtype=np.float64))
    Phi, Pi, _ = inputs.qp_family(N, eps, mu, kd)
    ens = binding.Ensemble(N, len(eps), courant=courant, ko_eps=ko_eps, device=device, threshold=threshold,
                           rk_order=(rk_order if rk_order != 4 else None))
    ens.set_initial(torch.from_numpy(Phi).to(device), torch.from_numpy(Pi).to(device))
    d0 = ens.diagnostics()
    nsteps = int(np.ceil(tmax / ens.dt))            # reading R18
    done = 0
    d = d0
    while done < nsteps:
        n = min(chunk_steps, nsteps - done)
        ens.step(n)
        done += n
        d = ens.diagnostics()
        if d["collapsed"].all():
            break
    out = dict(eps=eps, t_collapse=d["t_collapse"].copy(), collapsed=d["collapsed"].copy(), t=d["t"].copy(),
               mass0=d0["mass"].copy(), mass=d["mass"].copy(), min_A=d["min_A"].copy())
    out["path"] = ens.path
    out["mass_loss"] = np.abs(out["mass"] - out["mass0"]) / np.abs(out["mass0"])
    ens.close()
    return out


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--kd", type=int, default=3)
    ap.add_argument("--mu", type=float, default=1.0)
    ap.add_argument("--eps", default="0.3,0.4,0.5,0.6", help="comma-separated amplitudes")
    ap.add_argument("--N", type=int, default=4097)
    ap.add_argument("--tmax", type=float, default=50.0)
    ap.add_argument("--threshold", type=float, default=0.01, help="collapse when min A < this (PAPER.md:85)")
    ap.add_argument("--rk-order", type=int, default=4, choices=[2, 3, 4], help="the paper's production runs used 3 (PAPER.md:57)")
    ap.add_argument("--chunk-steps", type=int, default=2000, help="RK steps between two looks at the collapse flags")
    a = ap.parse_args(argv)
    eps = [float(v) for v in a.eps.split(",")]
    r = sweep(eps, a.mu, a.kd, N=a.N, tmax=a.tmax, threshold=a.threshold, rk_order=a.rk_order, chunk_steps=a.chunk_steps)
    print(f"# family k_d={a.kd} mu={a.mu} N={a.N} t_max={a.tmax} threshold={a.threshold} rk_order={a.rk_order} "
          f"path={r['path'][0]} ctas_per_member={r['path'][1]}")
    print("# eps        1/eps^2      t_collapse   t_reached    mass_loss    min_A")
    for i in range(len(eps)):
        print(f"{r['eps'][i]:10.4e} {1.0 / r['eps'][i] ** 2:12.4e} {r['t_collapse'][i]:12.5f} {r['t'][i]:12.5f} "
              f"{r['mass_loss'][i]:12.3e} {r['min_A'][i]:10.3e}")
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
