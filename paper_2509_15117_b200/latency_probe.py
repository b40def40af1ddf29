"""Latency of one RK step against the number of warps that share an SM sub-partition, for both lane layouts.

    python -m paper_2509_15117_b200.latency_probe [t_max_rf]

One long-lived initial condition (a complex still bound at t_max, found by running a 128 x 128 map of config 1 once)
is replicated N times, so that every trajectory of a launch takes exactly the same steps; N is chosen to give 1/4 ...
4 warps per sub-partition in the cooperative layout (ten trajectories per warp, IA_PATH_COOP_ONLY) and 1/4 ... 3 in
the bulk layout (32 per warp, IA_PATH_BULK_ONLY).  Prints the launch time, the time per step of a trajectory and the
aggregate step rate.  This is the measurement behind the straggler chain's stages.
Marshalling and timing only: every step runs in the library's kernels.
"""
from __future__ import annotations

import os
import sys
from dataclasses import replace

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402


def main():
    import torch

    import ia_inputs as I
    import paper_2509_15117_b200 as P

    t_max = float(sys.argv[1]) if len(sys.argv) > 1 else 60.0
    cell = I.config1(128)
    cell = replace(cell, params=replace(cell.params, t_max_rf=t_max))
    with P.Context(cell.params) as ctx:
        n_sm = ctx.kernel_info["bulk"]["n_sm"]
        rec, _, ic = ctx.run_sync(replace(cell.launch, path=P.IA_PATH_BULK_ONLY), want_ic=True)
        bound = np.nonzero(rec["status"] == 1)[0]
        steps_all = rec["steps_acc"].astype(np.int64) + rec["steps_rej"]
        j = bound[np.argmax(steps_all[bound])]
        steps = int(steps_all[j])
        print(f"{len(bound)} trajectories of the 128 x 128 map still bound at {t_max:g} T_rf; replicating number {j}: "
              f"{steps} attempted steps, {rec['n_coll'][j]} bounces")
        lat = P.ia_fp64_latency(0)
        print(f"dependent DFMA: {lat['cycles_dfma']:.2f} SM cycles; reciprocal (MUFU.RCP64H + 3 DFMA) + DADD: "
              f"{lat['cycles_rcp_add']:.2f} cycles\n")
        print("| layout | warps per sub-partition | trajectories | ms | us per step | 1e9 steps/s |")
        print("|---|---|---|---|---|---|")
        for path, name, per_warp in ((P.IA_PATH_COOP_ONLY, "cooperative (3 lanes)", 10), (P.IA_PATH_BULK_ONLY, "bulk (1 lane)", 32)):
            for wps in (0.25, 0.5, 1, 1.5, 2, 3, 4):
                if per_warp == 32 and wps > 3:
                    continue
                n = int(n_sm * 4 * wps) * per_warp
                y = torch.tensor(np.tile(ic[j, :12], (n, 1)), device="cuda")
                ph = torch.full((n,), float(ic[j, 12]), dtype=torch.float64, device="cuda")
                launch = I.Launch(mode=I.MODE_EXPLICIT, n=n, path=path)
                r, s, _ = ctx.alloc(n)
                ctx.run(launch, y, ph, r, s)                       # warm-up
                torch.cuda.synchronize()
                s.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                ctx.run(launch, y, ph, r, s)
                e1.record()
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1)
                sm = P.view_summary(s)
                total = int(sm["steps_acc"]) + int(sm["steps_rej"])
                print(f"| {name} | {wps:g} | {n} | {ms:.2f} | {1e3 * ms / steps:.3f} | {total / ms / 1e6:.2f} |")


if __name__ == "__main__":
    main()
