#!/usr/bin/env python
"""bench.py -- throughput of the batched ion+atom propagator on BASELINE.json configs[1]
(Yb+ + 87Rb fractal angle map, 512x512 octant grid = 262,144 trajectories, E = 1.5 uK, t_max 1e4 T_rf).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n-side 512]

One "step" = one pass of the whole hot path (generator -> adaptive DP5(4) propagation -> events ->
exit localisation -> observables -> record write -> ensemble reduction) over the whole grid.
Prints ONE JSON line on rank 0.  `value` = trajectories/s with everything resident on the device;
`e2e` = the same metric through ia_run_host with HOST buffers (explicit initial conditions copied in,
records and summary copied out, inside the timed region).  `roofline` is against the FP64 FMA peak
measured live by the library's DFMA microbenchmark (MEASURED_PEAKS.json carries no FP64 figure).
`--impl reference` times the CPU oracle (test infrastructure; the only other place that may run it).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

# One hardware work queue per stream: with the default of 8, the straggler streams of a deep pipeline would share
# queues and their kernels would serialise behind one another (must be set before CUDA is initialised).
os.environ.setdefault("CUDA_DEVICE_MAX_CONNECTIONS", "32")

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import ia_inputs as I  # noqa: E402

METRIC = "trajectories/s"
# Algorithmic FP64 flops per ATTEMPTED RK step (FMA = 2), counted from the formulas of the
# Nystrom-collapsed DP5(4) step in DESIGN.md section "Roofline": coefficient products 35, five cosines 135,
# stage sums 300, six accelerations 234, d.w 8, error sums 120, norm cross-products 22,
# controller / time keeping 32.
FLOP_PER_STEP = 886.0
ORACLE_SAMPLE_EVERY = 8   # cpu_baseline: every 8th grid point in theta and phi (64x64 = 4,096 trajectories)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=16)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n-side", type=int, default=512)
    ap.add_argument("--workload", default="config1",
                    help="config1 (default, the bench line) | config0 | config2.<cell 0-24> | config3.<cell 0-19> | "
                         "config4 (one batch): the other BASELINE.json configs, for profiling and inspection")
    ap.add_argument("--n", type=int, default=0, help="trajectories per pass for the Philox workloads (default: "
                                                     "the config's own cell / batch size)")
    ap.add_argument("--t-max-rf", type=float, default=0.0,
                    help="override the time limit (rf periods) -- profiling runs only; the bench line uses the config's own")
    ap.add_argument("--handoff", type=int, default=-1,
                    help="hand-over threshold of the bulk kernel in lanes (0 = bulk kernel only; default: the library's)")
    ap.add_argument("--path", type=int, default=0, help="ia_path: 0 production kernel pair, 1 bulk only, 2 cooperative only")
    ap.add_argument("--pipeline", type=int, default=64,
                    help="ia_set_pipeline depth: passes per generation, i.e. how many passes share one straggler kernel "
                         "(it runs on the library's stream while the next generation's bulk kernels run); "
                         "0 = strictly one pass after another, both kernels of a pass back to back")
    ap.add_argument("--chain", default="", help="levels,budget of the straggler chain (ia_set_chain); default: the library's")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def pick_workload(args):
    """BASELINE.json configs -> one cell (params + launch).  config1 is the bench workload."""
    cell = _pick_workload(args)
    if args.t_max_rf > 0.0:
        import dataclasses
        cell = dataclasses.replace(cell, name=f"{cell.name}_tmax{args.t_max_rf:g}",
                                   params=dataclasses.replace(cell.params, t_max_rf=args.t_max_rf))
    return cell


def _pick_workload(args):
    w = args.workload
    if w == "config1":
        return I.config1(args.n_side)
    if w == "config0":
        return I.config0()
    name, _, idx = w.partition(".")
    if name == "config2":
        return I.config2(n_per_cell=args.n or 2 ** 20)[int(idx or 0)]
    if name == "config3":
        return I.config3(n_per_cell=args.n or 2 ** 22)[int(idx or 0)]
    if name == "config4":
        n = args.n or 2 ** 24
        return I.config4(n_total=n, batch=n)[0]
    raise SystemExit(f"unknown --workload {w}")


# ---- clocks ---------------------------------------------------------------------------------------

class ClockSampler:
    """nvidia-smi sampling during the timed region (the recipe's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index: int):
        self.dev = device_index
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.dev)], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.tmp.flush()
        self.tmp.seek(0)
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.tmp.read().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.tmp.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---- the oracle legs (cpu_baseline and --impl reference) -----------------------------------------

def oracle_sample(cell, n_side: int):
    """Times the oracle, as it stands, on a bounded sample of the same workload: the decimated sub-grid
    of a GRID launch, the first 4,096 indices of a Philox launch."""
    from oracle import ia_oracle as O
    cores = os.cpu_count() or 1
    if cell.launch.mode != I.MODE_GRID or cell.launch.n_theta != n_side:
        idx = np.arange(min(cell.launch.n, 4096), dtype=np.uint64)
        t0 = time.perf_counter()
        out = O.run_generated(cell.params, cell.launch, indices=idx, nthreads=cores)
        dt = time.perf_counter() - t0
        steps = int(out["steps_acc"].astype(np.int64).sum() + out["steps_rej"].astype(np.int64).sum())
        return {"n": len(idx), "seconds": dt, "steps": steps, "cores": cores,
                "sample": f"first {len(idx)} trajectories of {cell.name} ({steps} RK steps), one trajectory per "
                          f"task over {cores} std::threads"}
    idx = I.subgrid_indices(n_side, ORACLE_SAMPLE_EVERY) if n_side >= ORACLE_SAMPLE_EVERY else np.arange(n_side * n_side)
    t0 = time.perf_counter()
    out = O.run_generated(cell.params, cell.launch, indices=idx, nthreads=cores)
    dt = time.perf_counter() - t0
    steps = int(out["steps_acc"].astype(np.int64).sum() + out["steps_rej"].astype(np.int64).sum())
    return {"n": len(idx), "seconds": dt, "steps": steps, "cores": cores,
            "sample": f"every {ORACLE_SAMPLE_EVERY}th grid point in theta and phi of the {n_side}x{n_side} grid "
                      f"({len(idx)} trajectories, {steps} RK steps), one trajectory per task over {cores} std::threads"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cell = pick_workload(args)
    times, last = [], None
    for it in range(args.warmup + args.steps):
        last = oracle_sample(cell, args.n_side)
        if it >= args.warmup:
            times.append(last["seconds"])
    total = float(sum(times))
    value = last["n"] * args.steps / total
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "trajectories/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cell.name, "trajectories_per_step": last["n"], "note": "CPU oracle on a bounded sample"},
            "rk_steps_per_s": last["steps"] * args.steps / total,
            "cpu_baseline": {"value": value, "unit": "trajectories/s", "cores": last["cores"], "kind": "oracle",
                             "sample": last["sample"]},
            "e2e": {"value": value, "unit": "trajectories/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---- our arm ----------------------------------------------------------------------------------------

def run_ours(args):
    import dataclasses

    import torch
    import torch.distributed as dist

    import paper_2509_15117_b200 as P
    from paper_2509_15117_b200 import dist as D

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the propagator has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    K, W = args.steps, max(args.warmup, 3)

    # Workload: configs[1].  Trajectories are independent, so N GPUs run N grids of the same shape (weak
    # scaling, no data-path collective): rank r maps the octant at rf phase 2 pi r / N.
    cell = pick_workload(args)
    if cell.launch.mode == I.MODE_GRID:
        launch = dataclasses.replace(cell.launch, phase0=2.0 * np.pi * rank / world)
    else:   # Philox workloads: rank r continues the same stream at index r * n
        launch = dataclasses.replace(cell.launch, first_index=cell.launch.first_index + rank * cell.launch.n)
    n = launch.n

    def barrier():
        if world > 1:
            dist.barrier(device_ids=[local])
        torch.cuda.synchronize(dev)

    peak = P.ia_fp64_peak(local, 300.0)          # the roofline denominator, measured on this GPU now
    ctx = P.Context(cell.params, device=local)
    if args.handoff >= 0:
        ctx.set_handoff(args.handoff)
    levels = P.IA_STRAGGLER_LEVELS
    if args.chain:
        levels, budget = (int(x) for x in args.chain.split(","))
        ctx.set_chain(levels, budget)
    depth = max(0, min(args.pipeline, 64, K))
    ctx.set_pipeline(depth)
    launch = dataclasses.replace(launch, path=args.path)
    info = ctx.kernel_info
    nbuf = min(K, 2 * max(depth, 1))             # passes in flight (two generations) never share an output buffer
    recs_d = [torch.empty(n * P.RECORD_BYTES, dtype=torch.uint8, device=dev) for _ in range(nbuf)]
    summaries = torch.zeros((W + K, P.SUMMARY_BYTES), dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    for w in range(W):
        ctx.run(launch, records=recs_d[w % nbuf], summary=summaries[w])
        flush.fill_(w)
    ctx.join()
    barrier()
    clocks = ClockSampler(local)
    clocks.start()
    ev0.record()
    for k in range(K):
        # one step = one pass over the grid: its bulk kernel here; its stragglers are finished by the straggler
        # kernel of its generation (depth 0: right behind the bulk kernel; depth > 0: one launch for `depth` passes,
        # on the library's stream, while the next generation's bulk kernels run)
        ctx.run(launch, records=recs_d[k % nbuf], summary=summaries[W + k])
        flush.fill_(k)                                             # L2 flush between timed iterations
    ctx.join()                                                     # the stream waits for every straggler kernel
    ev1.record()
    barrier()
    clk = clocks.stop()
    total_s = D.all_reduce_max(ev0.elapsed_time(ev1) * 1e-3, dev)
    kernel_times = []                              # the library's own CUDA events around each kernel
    for back in range(K):
        try:
            kernel_times.append(ctx.timing(back))
        except P.IaError:                          # older than the two generations the library keeps on record
            break
    n_coop_launches = K if depth == 0 else -(-K // depth)
    summ = P.view_summary(summaries[W + K - 1])
    bulk_ms = float(np.mean([t["bulk_ms"] for t in kernel_times]))
    coop_ms = float(np.mean([t["coop_ms"] for t in kernel_times]))
    attempted = int(summ["steps_acc"]) + int(summ["steps_rej"]) + int(summ["steps_loc"])
    steps_coop = int(summ["steps_coop"])
    recs = P.view_records(recs_d[(K - 1) % nbuf], n)
    longest = int((recs["steps_acc"].astype(np.int64) + recs["steps_rej"]).max())
    tot = D.all_reduce_summary(summ, dev)
    attempted_all = tot["steps_acc"] + tot["steps_rej"] + tot["steps_loc"]
    value = world * n * K / total_s
    step_avg_ms = 1e3 * total_s / K

    # end to end through the host entry points: explicit initial conditions in pinned host memory -> device,
    # records + summary -> pinned host memory, all inside the timed region (ia_submit_host x K, ia_wait)
    e2e = None
    if not args.no_e2e:
        ic = ctx.generate(launch)                                   # untimed: the inputs of the e2e leg
        y0 = torch.from_numpy(np.ascontiguousarray(ic[:, :12])).pin_memory()
        ph = torch.from_numpy(np.ascontiguousarray(ic[:, 12])).pin_memory()
        rec_h = [torch.empty(n * P.RECORD_BYTES, dtype=torch.uint8).pin_memory() for _ in range(nbuf)]
        sum_h = [torch.zeros(P.SUMMARY_BYTES, dtype=torch.uint8).pin_memory() for _ in range(nbuf)]
        lx = I.Launch(mode=I.MODE_EXPLICIT, n=n)
        cl = P.make_launch(lx, y0, ph)
        P.ia_run_host(ctx.handle, cl, rec_h[0], sum_h[0])           # warm-up (staging allocation)
        barrier()
        t0 = time.perf_counter()
        for k in range(K):
            P.ia_submit_host(ctx.handle, cl, rec_h[k % nbuf], sum_h[k % nbuf])
        ctx.wait()                                                  # blocks until every copy back has landed
        e2e_s = D.all_reduce_max(time.perf_counter() - t0, dev)
        done = int(sum_h[(K - 1) % nbuf].numpy().view(P.SUMMARY_DTYPE)[0]["n_done"])
        assert done == n, (done, n)
        e2e = {"value": world * n * K / e2e_s, "unit": "trajectories/s",
               "h2d_bytes_per_step": int(y0.numel() * 8 + ph.numel() * 8),
               "d2h_bytes_per_step": int(rec_h[0].numel() + sum_h[0].numel()), "ms_per_step": 1e3 * e2e_s / K}
    ctx.close()
    if world > 1:
        dist.barrier(device_ids=[local])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # roofline of the kernel that does the arithmetic: the bulk kernel (one lane per trajectory) over its own
    # launch duration; the steps the straggler kernel took are not counted for it
    achieved_tflops = FLOP_PER_STEP * (attempted - steps_coop) / (bulk_ms * 1e-3) / 1e12
    line = {
        "metric": METRIC, "value": value, "unit": "trajectories/s", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": 1e3 * total_s / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cell.name, "trajectories_per_step_per_gpu": n, "parallelism": f"dp{world}",
                   "l2": "flushed between timed iterations (256 MiB write); the kernel reads no input arrays",
                   "pipeline_depth": depth,
                   "rtol": cell.params.rtol, "atol": cell.params.atol, "t_max_rf": cell.params.t_max_rf},
        "rk_steps_per_s": attempted_all * K / total_s,
        "rk_steps_per_pass": attempted_all,
        "p_complex": tot["n_complex"] / max(tot["n_done"], 1), "n_status": tot["n_status"],
        "roofline": {"bound": "alu", "achieved": achieved_tflops, "peak": peak["tflops"], "unit": "TFLOP/s",
                     "frac": achieved_tflops / peak["tflops"],
                     # dram__bytes_read.sum + dram__bytes_write.sum of one K1 launch on this workload from the ncu --set full
                     # capture in profiles/r01e_end_of_round.md (the 16.8 MB of records are still in L2 when the kernel ends)
                     "traffic": 111104 if cell.name.startswith("config1_") and args.n_side == 512 and args.t_max_rf == 0.0 else None,
                     "peak_source": "ia_fp64_peak (DFMA chains on all SMs, measured in this run); nominal 37.2",
                     "flop_per_attempted_step": FLOP_PER_STEP, "kernel": "ia_persistent_kernel<1> (bulk)",
                     "kernel_ms": bulk_ms, "steps_in_kernel": attempted - steps_coop,
                     "share_of_step_time": bulk_ms / step_avg_ms, "share_of_step_flops": 1.0 - steps_coop / max(attempted, 1),
                     # share of the kernel's lane-steps (32 per warp and attempt) that advanced a trajectory
                     "lane_efficiency": (attempted - steps_coop) / max(int(summ["slots_bulk"]), 1),
                     "ms_until_work_counter_empty": (int(summ["t_first_idle_ns"]) - int(summ["t_start_ns"])) * 1e-6},
        # the straggler kernel is bound by the serial latency of the longest trajectories, not by throughput
        "tail": {"kernel": f"ia_persistent_kernel<3> (cooperative, 3 lanes per trajectory), chain of {levels} launches",
                 "kernel_ms": coop_ms,
                 "launches": n_coop_launches, "passes_per_launch": K / n_coop_launches,
                 "share_of_step_time": coop_ms * n_coop_launches / K / step_avg_ms,
                 "trajectories_handed_over_per_pass": int(summ["n_handoff"]),
                 "steps_in_kernel_per_pass": steps_coop, "longest_trajectory_steps": longest,
                 "us_per_step_serial_bound": 1e3 * coop_ms / max(longest, 1),
                 "note": "a trajectory is a serial chain: the launch cannot end before its longest one (DESIGN.md 'Tail')"},
        "kernel_info": info, "clocks": clk, "e2e": e2e, "gpu_launches": K + n_coop_launches * levels,
    }
    if not args.no_cpu_baseline and world == 1:
        s = oracle_sample(cell, args.n_side)
        line["cpu_baseline"] = {"value": s["n"] / s["seconds"], "unit": "trajectories/s", "cores": s["cores"],
                                "kind": "oracle", "sample": s["sample"], "rk_steps_per_s": s["steps"] / s["seconds"]}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
