"""Parity table of BASELINE.md / profiles/: max |Delta| GPU vs oracle per config shape, on the GPU box.

    python tests/parity_report.py            # prints a markdown table (needs a B200 and the built library)

Not a pytest module: the assertions live in tests/test_gpu_parity.py; this script only reports the numbers.  It runs the
full grid size of every BASELINE.json config with a reduced batch (the oracle finishes each in seconds to a minute).
"""
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

CASES = [  # name, B, steps, rk_order
    ("cfg1", 1, 1000, 4), ("cfg2", 8, 1000, 4), ("cfg3", 8, 1000, 4), ("cfg4", 1, 20, 4), ("cfg5", 8, 1000, 4),
    ("paper32k", 2, 200, 3),
    # the configs' own run lengths (BASELINE.json: cfg1 to t = 10, cfg3 20000 steps, cfg4 1000 steps): information only,
    # the [NS] tolerance is stated for 1000 steps
    ("cfg1", 1, 26076, 4), ("cfg3", 4, 20000, 4), ("cfg4", 1, 1000, 4),
]


def main():
    import torch
    import oracle
    from paper_1706_07413_b200 import binding, inputs
    print("| workload | N | members | steps | path (CTAs/member) | max abs diff Phi | Pi | A | delta | oracle s |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for name, B, steps, order in CASES:
        Phi, Pi, _ = inputs.make(name, B=B)
        N = Phi.shape[1]
        ens = binding.Ensemble(N, B, rk_order=(order if order != 4 else None))
        ens.set_initial(torch.from_numpy(Phi).cuda(), torch.from_numpy(Pi).cuda())
        ens.step(steps)
        f = {k: v.cpu().numpy() for k, v in ens.get_fields().items()}
        t = time.time()
        ev = oracle.Evolution(Phi, Pi, nthreads=min(B, 8), rk_order=order).step(steps)
        el = time.time() - t
        err = [float(np.max(np.abs(f[k] - r))) for k, r in (("Phi", ev.Phi), ("Pi", ev.Pi), ("A", ev.A), ("delta", ev.delta))]
        p, cl = ens.path
        print(f"| {name} | {N} | {B} | {steps} (RK{order}) | {p} ({cl}) | " + " | ".join(f"{e:.1e}" for e in err) + f" | {el:.1f} |")


if __name__ == "__main__":
    main()
