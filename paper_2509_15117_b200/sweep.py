"""Runs the cells of BASELINE.json's configs through the library, one launch per cell, and prints one JSON line per
cell: ensemble results (complex-formation probability, mean ion energy gain, collision-count histogram, survival) and
device times of the two kernels from the library's own CUDA events.

    python -m paper_2509_15117_b200.sweep --configs 0,2,3:0:10,4,thermal,fig4 [--scale 1.0] [--concurrent] [--lengths]

A config may carry a slice of its cells (3:0:10 = cells 0..9 of config 3: the D_e = 0.1 K and 1 K rows).

--scale shrinks every cell (trajectories per cell = max(1024, scale * the config's own size)).  Marshalling and
printing only: every number comes out of ia_run's summary.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

FLOP_PER_STEP = 867.0   # FP64 flops per attempted step: 345 FMA + 144 products + 33 sums
KB_EH_PER_K = 3.1668115634564e-6


def cells_of(which: str, scale: float):
    import dataclasses

    import ia_inputs as I

    def shrink(c):
        """--scale: trajectories per cell = scale x the cell's own size (at least 1024); a scale above 1 only for the
        cells that are not pieces of one index stream (thermal bars at Fig. 3's 10^7: --scale 9.5367)"""
        n = max(1024, int(round(scale * c.launch.n)))
        if c.launch.mode == I.MODE_GRID:
            return c
        if scale > 1.0 and which == "4":
            raise SystemExit("--scale > 1 would make config 4's batches overlap")
        return dataclasses.replace(c, launch=dataclasses.replace(c.launch, n=n))
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
    if which == "fig4":
        # Fig. 4's radius r0 = 20 000 a0 at 10 uK for the four species of the figure with a
        # random rf phase, and Rb with the phase fixed at 0 and at pi
        cells = [I.fig4(sp, 10.0, n=2 ** 20) for sp in ("Li7", "Na23", "K39", "Rb87")]
        cells += [I.fig4("Rb87", 10.0, n=2 ** 20, phase_mode=0, phase0=ph) for ph in (0.0, float(np.pi))]
        return [shrink(c) for c in cells]
    if which == "thermal":
        return [shrink(I.thermal(sp, T, De)) for De in (1.0, 100.0) for sp in I.SPECIES_ORDER for T in I.THERMAL_T_UK]
    raise SystemExit(f"unknown config {which}")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="0,2,3,4")
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--t-max-rf", type=float, default=0.0,
                    help="override every cell's time limit (rf periods): bounds the straggler chain; complexes still "
                         "bound then are counted as such (status 1)")
    ap.add_argument("--lengths", action="store_true",
                    help="also print, per cell, the distribution of trajectory lengths (attempted steps) read from the "
                         "records: share of trajectories and of the work beyond 2^k steps")
    ap.add_argument("--concurrent", action="store_true",
                    help="enqueue every group of cells (one ctx each) on a stream of its own before waiting for any: "
                         "the straggler chains of cells with different parameters then overlap")
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
        cells = cells[int(lo or 0):int(hi) if hi else len(cells)]
        if args.t_max_rf > 0.0:
            import dataclasses
            cells = [dataclasses.replace(c, params=dataclasses.replace(c.params, t_max_rf=args.t_max_rf)) for c in cells]
        # consecutive cells of one (species, trap, D_e, tolerances) cell -- config 4's batches of one Philox stream, the
        # five temperatures of a thermal species -- share a ctx and run as one pipeline (ia_set_pipeline): the bulk
        # kernel of a cell first resumes what the cell before left unfinished; one straggler chain at the end
        groups = []
        for cell in cells:
            if groups and groups[-1][0].params == cell.params and len(groups[-1]) < 64:
                groups[-1].append(cell)
            else:
                groups.append([cell])
        def enqueue(group, stream):
            """one ctx per group; every run and the join enqueued on `stream`, nothing waited for"""
            ctx = P.Context(group[0].params, device=args.device)
            ctx.set_pipeline(len(group) if len(group) > 1 else 0)
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(stream):
                bufs = [ctx.alloc(c.launch.n) for c in group]   # zero-filled on the stream the kernels run on
                ev0.record()
                for c, (rec, summ, _) in zip(group, bufs):
                    ctx.run(c.launch, records=rec, summary=summ)
                ctx.join()
                ev1.record()
            return ctx, bufs, ev0, ev1

        def report(group, ctx, bufs, ev0, ev1, close=True):
            ev1.synchronize()
            times = [ctx.timing(len(group) - 1 - k) for k in range(len(group))]
            T_rf = ctx.derived["T_rf"]
            if close:       # ia_destroy frees device memory, which waits for the whole device: not while others run
                ctx.close()
            wall = ev0.elapsed_time(ev1) * 1e-3
            n_all = steps_all = 0
            for cell, (rec, summ, _), t in zip(group, bufs, times):
                n = cell.launch.n
                s = P.view_summary(summ)
                steps = int(s["steps_acc"]) + int(s["steps_rej"]) + int(s["steps_loc"])
                n_all += n
                steps_all += steps
                n_esc = int(s["n_status"][0])
                tt, S = Ob.survival_curve(s, T_rf)
                own = wall if len(group) == 1 else float("nan")   # the cells of a pipeline share its wall time
                line = {
                    "cell": cell.name, "n": n, "seconds": own, "trajectories_per_s": n / own, "rk_steps_per_s": steps / own,
                    "rk_steps": steps, "steps_per_trajectory": steps / n,
                    "bulk_ms": t["bulk_ms"], "chain_ms": t["coop_ms"],
                    # steps_kernel: what this cell's bulk kernel executed (its own trajectories and carried ones)
                    "bulk_frac_of_dfma_peak": FLOP_PER_STEP * int(s["steps_kernel"]) / (t["bulk_ms"] * 1e-3) / 1e12 / peak,
                    "bulk_lane_efficiency": int(s["steps_kernel"]) / max(int(s["slots_bulk"]), 1),
                    "p_complex": int(s["n_complex"]) / n, "n_status": [int(x) for x in s["n_status"]],
                    "mean_ke_ion_uK": (float(s["sum_ke"]) / max(n_esc, 1)) / KB_EH_PER_K * 1e6,
                    "hist_ncoll": [int(x) for x in s["hist_ncoll"][:12]],
                    "survival_at_rf_periods": {f"{2.0 ** k:g}": float(S[4 * k + 7]) for k in (2, 4, 6, 8, 10)},
                    "survival_slope_beyond_40_rf": Ob.power_law_exponent(tt, S, 40.0 * T_rf),
                    "n_handoff": int(s["n_handoff"]), "warn": int(s["warn"]),
                }
                print(json.dumps(line), flush=True)
                if args.lengths:
                    r = P.view_records(rec, n)
                    st = r["steps_acc"].astype(np.int64) + r["steps_rej"] + r["n_loc"]
                    tot = float(st.sum())
                    rows = {}
                    for k in range(9, 25):
                        m = st >= (1 << k)
                        rows[f"2^{k}"] = {"trajectories": float(m.mean()), "work": float(st[m].sum() / tot),
                                          "work_beyond": float((st[m] - (1 << k)).sum() / tot)}
                    tm = r["status"] == 1
                    print(json.dumps({"cell": cell.name, "lengths": {
                        "mean": tot / n, "median": float(np.median(st)), "max": int(st.max()), "beyond": rows,
                        "at_t_max": int(tm.sum()), "at_t_max_steps_min_mean_max":
                            [int(st[tm].min()), float(st[tm].mean()), int(st[tm].max())] if tm.any() else None}}), flush=True)
            if len(group) > 1:
                print(json.dumps({"pipeline": f"{group[0].name} .. {group[-1].name}", "cells": len(group), "n": n_all,
                                  "seconds": wall, "trajectories_per_s": n_all / wall, "rk_steps": steps_all,
                                  "rk_steps_per_s": steps_all / wall, "chain_ms": times[0]["coop_ms"],
                                  "bulk_ms_total": sum(t["bulk_ms"] for t in times)}), flush=True)

        if args.concurrent:
            # Cells with different parameters cannot share a pipeline, but their straggler chains can share the GPU: a
            # chain ends as a few hundred warps that wait on their own dependent chains, so the chains of all groups --
            # each on a stream of its own -- overlap one another and the bulk kernels of the groups enqueued later
            t0 = torch.cuda.Event(enable_timing=True)
            t1 = torch.cuda.Event(enable_timing=True)
            t0.record()
            inflight = []
            for g in groups:
                inflight.append((g, *enqueue(g, torch.cuda.Stream())))
                print(f"enqueued {g[0].name} ({len(inflight)} of {len(groups)})", file=sys.stderr, flush=True)
            for g, ctx, bufs, ev0, ev1 in inflight:
                report(g, ctx, bufs, ev0, ev1, close=False)
            t1.record()
            torch.cuda.synchronize()
            for _, ctx, _, _, _ in inflight:
                ctx.close()
            print(json.dumps({"concurrent_groups": len(groups), "config": which, "seconds": t0.elapsed_time(t1) * 1e-3,
                              "n": sum(c.launch.n for g in groups for c in g)}), flush=True)
        else:
            for group in groups:
                report(group, *enqueue(group, torch.cuda.current_stream()))


if __name__ == "__main__":
    main()
