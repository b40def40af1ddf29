"""Runs the cells of BASELINE.json's configs through the library, one launch per cell, and prints one JSON line per
cell: ensemble results (complex-formation probability, mean ion energy gain, collision-count histogram, survival) and
device times of the two kernels from the library's own CUDA events.

    python -m paper_2509_15117_b200.sweep --configs 0,2,3:0:10,4,thermal [--scale 1.0]

A config may carry a slice of its cells (3:0:10 = cells 0..9 of config 3: the D_e = 0.1 K and 1 K rows).

--scale shrinks every cell (trajectories per cell = max(1024, scale * the config's own size)).  Marshalling and
printing only: every number comes out of ia_run's summary.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

os.environ.setdefault("CUDA_DEVICE_MAX_CONNECTIONS", "32")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

FLOP_PER_STEP = 886.0   # algorithmic FP64 flops per attempted step
KB_EH_PER_K = 3.1668115634564e-6


def cells_of(which: str, scale: float):
    import dataclasses

    import ia_inputs as I

    def shrink(c):
        n = max(1024, int(round(scale * c.launch.n)))
        if c.launch.mode == I.MODE_GRID:
            return c
        return dataclasses.replace(c, launch=dataclasses.replace(c.launch, n=min(n, c.launch.n)))
    if which == "0":
        return [I.config0()]
    if which == "1":
        side = max(32, int(round(512 * np.sqrt(scale))))
        return [I.config1(side)]
    if which == "2":
        return [shrink(c) for c in I.config2()]
    if which == "3":
        return [shrink(c) for c in I.config3()]
    if which == "4":
        return [shrink(c) for c in I.config4()]
    if which == "thermal":
        return [shrink(I.thermal(sp, T, De)) for De in (1.0, 100.0) for sp in I.SPECIES_ORDER for T in I.THERMAL_T_UK]
    raise SystemExit(f"unknown config {which}")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="0,2,3,4")
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--device", type=int, default=0)
    args = ap.parse_args()
    import torch

    import paper_2509_15117_b200 as P
    from paper_2509_15117_b200 import observables as Ob

    if not torch.cuda.is_available():
        raise SystemExit("sweep needs a CUDA device: the propagator has no CPU fallback")
    torch.cuda.set_device(args.device)
    peak = P.ia_fp64_peak(args.device, 300.0)["tflops"]
    for item in args.configs.split(","):
        which, _, sl = item.strip().partition(":")
        lo, _, hi = sl.partition(":")
        cells = cells_of(which, args.scale)
        for cell in cells[int(lo or 0):int(hi) if hi else len(cells)]:
            n = cell.launch.n
            with P.Context(cell.params, device=args.device) as ctx:
                rec, summ, _ = ctx.alloc(n)
                ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                ev0.record()
                ctx.run(cell.launch, records=rec, summary=summ)
                ev1.record()
                torch.cuda.synchronize()
                t = ctx.timing(0)
                T_rf = ctx.derived["T_rf"]
            s = P.view_summary(summ)
            wall = ev0.elapsed_time(ev1) * 1e-3
            steps = int(s["steps_acc"]) + int(s["steps_rej"]) + int(s["steps_loc"])
            n_esc = int(s["n_status"][0])
            tt, S = Ob.survival_curve(s, T_rf)
            line = {
                "cell": cell.name, "n": n, "seconds": wall, "trajectories_per_s": n / wall, "rk_steps_per_s": steps / wall,
                "rk_steps": steps, "steps_per_trajectory": steps / n,
                "bulk_ms": t["bulk_ms"], "chain_ms": t["coop_ms"],
                "bulk_frac_of_dfma_peak": FLOP_PER_STEP * (steps - int(s["steps_coop"])) / (t["bulk_ms"] * 1e-3) / 1e12 / peak,
                "bulk_lane_efficiency": (steps - int(s["steps_coop"])) / max(int(s["slots_bulk"]), 1),
                "p_complex": int(s["n_complex"]) / n, "n_status": [int(x) for x in s["n_status"]],
                "mean_ke_ion_uK": (float(s["sum_ke"]) / max(n_esc, 1)) / KB_EH_PER_K * 1e6,
                "hist_ncoll": [int(x) for x in s["hist_ncoll"][:12]],
                "survival_at_rf_periods": {f"{2.0 ** k:g}": float(S[4 * k + 7]) for k in (2, 4, 6, 8, 10)},
                "survival_slope_beyond_40_rf": Ob.power_law_exponent(tt, S, 40.0 * T_rf),
                "n_handoff": int(s["n_handoff"]), "warn": int(s["warn"]),
            }
            print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
