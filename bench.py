#!/usr/bin/env python
"""bench.py -- throughput of the batched ion+atom propagator on BASELINE.json configs[4], the largest
single-GPU configuration (the paper's ">3x10^8 trajectories"): Yb+ + 87Rb, E log-uniform in
[1,100] uK, full sphere, uniform rf phase, ONE Philox stream in batches of 2^24 trajectories.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload config4|config1|...]

One "step" = one batch of the stream through the whole hot path (generator -> adaptive DP5(4) propagation ->
events -> exit localisation -> observables -> 64-byte record -> ensemble reduction); first_index advances from
step to step.  The steps run as a pipeline (ia_set_pipeline): the bulk kernel of a step first resumes the
trajectories the step before left unfinished, so the power-law tail of trajectory lengths lives in
full warps while new trajectories keep arriving.  The timed region is K consecutive steps of the running stream,
entered after W warm-up steps (the first of them alone and timed separately: `latency_one_step_alone_ms`) and left
when the K-th bulk kernel ends; `value` = trajectories FINISHED inside it per second, device-resident.  The
straggler chain that ends the stream afterwards is timed on its own (`tail`); `whole_stream` = every trajectory of
the stream over the time from its first launch to the end of that chain.  `e2e` = a further stream of the same
shape through ia_submit_host with page-locked HOST buffers (launch descriptor in, 1 GiB of records per step copied
back), timed from the first submit until ia_wait returns: straggler chain, late records and summaries included
(`e2e.streaming`: the same leg stopped at ia_sync, i.e. the steady-state rate).  `roofline` is against the FP64 FMA
peak measured live by the library's DFMA microbenchmark (MEASURED_PEAKS.json carries no FP64 figure), with the
fraction of the pipe's nominal rate at the measured SM clock beside it.  Prints ONE JSON line on rank 0.
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

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import ia_inputs as I  # noqa: E402

METRIC = "trajectories/s"
# FP64 flops per ATTEMPTED RK step (FMA = 2) of the Nystrom-collapsed DP5(4) step as the kernels compute it
# (DESIGN.md section "Roofline"): 345 FMA + 144 products + 33 sums = 867.  It is the count of the formulas AND the
# count ncu reads off the bulk kernel (sass__inst_executed_per_opcode per warp and step: DFMA 345.0, DMUL 143.6,
# DADD 33.0; compares are not counted).  Round 1's step needed 886: the error norm and the controller have shed 19.
FLOP_PER_STEP = 867.0
# DRAM traffic of the bulk kernel (dram__bytes_read.sum + dram__bytes_write.sum under `ncu --set full`): 125.03 MB for a
# launch of 2^21 fresh trajectories = 59.6 B per trajectory, against 64 B of record written per trajectory (the kernel
# reads no input arrays; part of the last records is still in L2 when the kernel ends).  The bench line scales it to its
# own launch size.  Irrelevant to the bound (FP64 issue).
TRAFFIC_BYTES_PER_TRAJECTORY = 125030912 / 2097152
TRAFFIC_SOURCE = ("profiles/r03_k1_raw.csv: 22.24 MB read + 102.79 MB written by one bulk-kernel launch of 2^21 trajectories, "
                  "scaled per trajectory to this run's launch size")
ORACLE_SAMPLE_EVERY = 8   # oracle legs on a GRID workload: every 8th grid point in theta and phi (64x64 = 4,096)
ORACLE_SAMPLE_PHILOX = 8192   # ... on a Philox stream: its first 8,192 indices (reference arm, per step)
ORACLE_SAMPLE_BASELINE = 32768  # ... and for the one-shot cpu_baseline of our arm
E2E_STEPS_MAX = 12        # steps of the end-to-end leg (1 GiB of page-locked host memory each on config 4)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=16)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n-side", type=int, default=512)
    ap.add_argument("--workload", default="config4",
                    help="config4 (default, the bench line: one batch of 2^24 per step) | config1 | config0 | "
                         "config2.<cell 0-24> | config3.<cell 0-19>: the other BASELINE.json configs, for profiling "
                         "and inspection (a GRID workload repeats the same grid every step)")
    ap.add_argument("--n", type=int, default=0, help="trajectories per step for the Philox workloads (default: "
                                                     "the config's own cell / batch size)")
    ap.add_argument("--t-max-rf", type=float, default=0.0,
                    help="override the time limit (rf periods) -- profiling runs only; the bench line uses the config's own")
    ap.add_argument("--handoff", type=int, default=-1,
                    help="hand-over threshold of the bulk kernel in lanes (0 = bulk kernel only; default: the library's)")
    ap.add_argument("--path", type=int, default=0, help="ia_path: 0 production kernel pair, 1 bulk only, 2 cooperative only")
    ap.add_argument("--pipeline", type=int, default=64,
                    help="ia_set_pipeline depth (steps between two forced straggler chains); 0 = every step on its "
                         "own, bulk kernel and straggler chain back to back")
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

def oracle_sample(cell, n_side: int, n_philox: int = ORACLE_SAMPLE_PHILOX):
    """Times the oracle, as it stands, on a bounded sample of the same workload: the decimated sub-grid
    of a GRID launch, the first n_philox indices of a Philox launch."""
    from oracle import ia_oracle as O
    cores = os.cpu_count() or 1
    if cell.launch.mode != I.MODE_GRID or cell.launch.n_theta != n_side:
        idx = np.arange(min(cell.launch.n, n_philox), dtype=np.uint64)
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
    if world != args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus} but WORLD_SIZE={world}: start it through torch.distributed.run "
                         f"(a plain `python bench.py --gpus N` does that itself)")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the propagator has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    K, W = args.steps, max(args.warmup, 3)
    Ke = 0 if args.no_e2e else min(K, E2E_STEPS_MAX)

    # Workload.  Trajectories are independent, so N GPUs run N streams of the same shape (weak scaling, no
    # data-path collective): rank r takes its own index range of the Philox stream (a GRID workload: the same
    # grid at rf phase 2 pi r / N).
    cell = pick_workload(args)
    n = cell.launch.n
    stream_like = cell.launch.mode != I.MODE_GRID

    def launch_of(step: int):
        if stream_like:
            return dataclasses.replace(cell.launch, path=args.path,
                                       first_index=cell.launch.first_index + (rank * 4096 + step) * n)
        return dataclasses.replace(cell.launch, path=args.path, phase0=2.0 * np.pi * rank / world)

    def barrier():
        if world > 1:
            dist.barrier(device_ids=[local])
        torch.cuda.synchronize(dev)

    # the roofline denominator, measured on this GPU now: 2 s of DFMA chains on every SM, SM clock sampled meanwhile
    peak_clocks = ClockSampler(local)
    peak_clocks.start()
    time.sleep(0.3)
    peak = P.ia_fp64_peak(local, 2000.0)
    peak_clk = peak_clocks.stop()
    ctx = P.Context(cell.params, device=local)
    if args.handoff >= 0:
        ctx.set_handoff(args.handoff)
    levels = 1                                   # the library's default (ia_set_chain): one cooperative launch ends the chain
    if args.chain:
        levels, budget = (int(x) for x in args.chain.split(","))
        ctx.set_chain(levels, budget)
    depth = max(0, min(args.pipeline, 64))
    # the library ends a pipeline by itself after `depth` runs (ia_set_pipeline): keep the end-to-end leg (a stream of
    # its own) within one, and say so if the timed region itself is longer (a straggler chain then falls into it)
    if depth > 0:
        Ke = min(Ke, depth)
    chain_in_region = depth > 0 and W - 1 + K > depth
    info = ctx.kernel_info
    # every step of the device leg keeps its own record buffer until the stream is drained (a trajectory in flight
    # writes into the buffer of the step it belongs to)
    recs_d = [torch.empty(n * P.RECORD_BYTES, dtype=torch.uint8, device=dev) for _ in range(W + K)]
    summaries = torch.zeros((W + K, P.SUMMARY_BYTES), dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    mk = lambda: torch.cuda.Event(enable_timing=True)
    ev_a0, ev_a1, ev0, ev1 = mk(), mk(), mk(), mk()

    def view_all():
        return summaries.cpu().numpy().view(P.SUMMARY_DTYPE).reshape(-1)

    # warm-up step 0 on its own: bulk kernel + its straggler chain = the latency of one step alone
    ctx.set_pipeline(0)
    ev_a0.record()
    ctx.run(launch_of(0), records=recs_d[0], summary=summaries[0])
    ev_a1.record()
    torch.cuda.synchronize(dev)
    alone_ms = ev_a0.elapsed_time(ev_a1)
    alone_t = ctx.timing(0)
    # the stream proper: warm-up steps 1..W-1 fill the pipeline, then the timed region, no join in between
    ctx.set_pipeline(depth)
    ev_s0, ev_s1 = mk(), mk()
    ev_s0.record()                                # the stream starts here: W-1 warm-up + K timed steps, then its chain
    for w in range(1, W):
        ctx.run(launch_of(w), records=recs_d[w], summary=summaries[w])
        flush.fill_(w)
    barrier()
    done0 = int(view_all()["n_done"].sum())
    clocks = ClockSampler(local)
    clocks.start()
    ev0.record()
    for k in range(K):
        ctx.run(launch_of(W + k), records=recs_d[W + k], summary=summaries[W + k])
        flush.fill_(k)                                             # L2 flush between timed iterations
    if depth == 0:
        ctx.join()
    ev1.record()
    barrier()
    clk = clocks.stop()
    region_s = D.all_reduce_max(ev0.elapsed_time(ev1) * 1e-3, dev)
    mid = view_all()
    finished = int(D.all_reduce_sum(int(mid["n_done"].sum()) - done0, dev))     # trajectories finished inside the region
    steps_region = int(mid["steps_kernel"][W:].sum())     # attempted steps the K timed bulk kernels executed (this rank)
    slots_region = int(mid["slots_bulk"][W:].sum())
    steps_region_all = int(D.all_reduce_sum(steps_region, dev))

    # the end of the device-resident stream: one straggler chain for what the last bulk kernel left
    t0 = time.perf_counter()
    ctx.join()
    ev_s1.record()
    torch.cuda.synchronize(dev)
    drain_s = D.all_reduce_max(time.perf_counter() - t0, dev)
    stream_s = D.all_reduce_max(ev_s0.elapsed_time(ev_s1) * 1e-3, dev)   # first launch of the stream -> end of its chain
    chain_t = ctx.timing(0)
    kernel_ms = [ctx.timing(K - 1 - k)["bulk_ms"] for k in range(K)]   # the K timed bulk kernels

    # End to end, a stream of its own through the host entry points with page-locked host buffers: launch descriptor
    # in, records copied back behind every bulk kernel, and the clock stops when ia_wait returns -- after the straggler
    # chain, with the late records stored and every summary back on the host.
    e2e = None
    if Ke > 0:
        rec_h = []
        for _ in range(Ke):          # 1 GiB of page-locked memory per step on config 4: take what the host gives
            try:
                rec_h.append(torch.empty(n * P.RECORD_BYTES, dtype=torch.uint8).pin_memory())
            except RuntimeError:
                break
        Ke = len(rec_h)
    if Ke > 0:
        import ctypes
        sum_h = [torch.zeros(P.SUMMARY_BYTES, dtype=torch.uint8).pin_memory() for _ in range(Ke)]
        cls = [P.make_launch(launch_of(W + K + k)) for k in range(Ke)]
        barrier()
        t0 = time.perf_counter()
        for k in range(Ke):
            P.ia_submit_host(ctx.handle, cls[k], rec_h[k], sum_h[k])
        ctx.sync()                                                  # every bulk kernel and its copy back has landed
        sync_s = time.perf_counter() - t0
        ctx.wait()                                                  # chain, late records, summaries: everything is home
        e2e_s = D.all_reduce_max(time.perf_counter() - t0, dev)
        sync_s = D.all_reduce_max(sync_s, dev)
        done_h = sum(int(x.numpy().view(P.SUMMARY_DTYPE)[0]["n_done"]) for x in sum_h)
        assert done_h == Ke * n, (done_h, Ke * n)
        for r in rec_h:
            assert int((r.numpy().view(P.RECORD_DTYPE)["status"] > 4).sum()) == 0
        e2e_chain = ctx.timing(0)["coop_ms"]
        e2e = {"value": world * n * Ke / e2e_s, "unit": "trajectories/s", "steps": Ke,
               "h2d_bytes_per_step": ctypes.sizeof(P.ia_launch),
               "d2h_bytes_per_step": int(rec_h[0].numel()) + P.SUMMARY_BYTES, "ms_per_step": 1e3 * e2e_s / Ke,
               "seconds": e2e_s, "chain_ms": e2e_chain,
               "streaming": {"value": world * n * Ke / sync_s, "seconds": sync_s,
                             "note": "the same leg stopped at ia_sync: bulk kernels and their copies back done, the "
                                     "trajectories still in flight (<= one per lane of the grid) and the summaries not yet home"},
               "note": "a stream of its own: ia_submit_host x steps, then ia_wait; generator mode, so the input of a step is "
                       "its launch descriptor; records of a step are copied to page-locked host memory behind its bulk kernel; "
                       "the clock stops when ia_wait returns, i.e. after the straggler chain, the late records and the summaries"}
    fin = view_all()
    assert int(fin["n_done"].sum()) == (W + K) * n, (int(fin["n_done"].sum()), (W + K) * n)
    bulk_ms = float(np.mean(kernel_ms))
    tot = D.all_reduce_summary(D.sum_summaries(fin[W:]), dev)
    attempted = tot["steps_acc"] + tot["steps_rej"] + tot["steps_loc"]
    recs = P.view_records(recs_d[W + K - 1], n)
    longest = int((recs["steps_acc"].astype(np.int64) + recs["steps_rej"]).max())
    ctx.close()
    if world > 1:
        dist.barrier(device_ids=[local])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = finished / region_s
    achieved_tflops = FLOP_PER_STEP * steps_region / (sum(kernel_ms) * 1e-3) / 1e12
    whole_tflops = FLOP_PER_STEP * steps_region / region_s / 1e12
    # the FP64 pipe's own rate: 64 FMA per SM and clock (B200_PROFILING / B300_MICROARCH unit counts) at the SM clock
    # nvidia-smi reported during the timed region; the DFMA microbenchmark reaches about 92 % of it
    sm_mhz = clk.get("sm_mhz") or clk.get("sm_max_mhz") or peak_clk.get("sm_mhz") or 1965.0
    nominal_tflops = info["bulk"]["n_sm"] * 64 * 2 * sm_mhz * 1e6 / 1e12
    n_stream = (W - 1 + K) * n
    line = {
        "metric": METRIC, "value": value, "unit": "trajectories/s", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": 1e3 * region_s / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{cell.name}_stream_{n}" if stream_like else cell.name,
                   "trajectories_per_step_per_gpu": n, "parallelism": f"dp{world}",
                   "timed_region": "K consecutive steps of a running pipeline (ia_set_pipeline): entered after W warm-up steps "
                                   "without a join, left when the K-th bulk kernel ends; value = trajectories finished inside it; "
                                   "the straggler chain that ends the stream is timed separately (tail) and counted in whole_stream",
                   "l2": "flushed between timed iterations (256 MiB write); the kernel reads no input arrays",
                   "pipeline_depth": depth, "chain_inside_timed_region": bool(chain_in_region),
                   "rtol": cell.params.rtol, "atol": cell.params.atol, "t_max_rf": cell.params.t_max_rf},
        "trajectories_started_per_s": world * n * K / region_s,
        "rk_steps_per_s": steps_region_all / region_s,
        "rk_steps_per_step": steps_region / K,
        "latency_one_step_alone_ms": alone_ms,
        "one_step_alone": {"bulk_ms": alone_t["bulk_ms"], "chain_ms": alone_t["coop_ms"],
                           "trajectories_per_s": n / (alone_ms * 1e-3)},
        "p_complex": tot["n_complex"] / max(tot["n_done"], 1), "n_status": tot["n_status"],
        "roofline": {"bound": "alu", "achieved": achieved_tflops, "peak": nominal_tflops, "unit": "TFLOP/s",
                     "frac": achieved_tflops / nominal_tflops,
                     "peak_source": "FP64 pipe at its nominal rate: SMs x 64 FMA/clk x 2 x the median SM clock nvidia-smi "
                                    "reported in the timed region (unit counts: /opt/skills/guides; DESIGN.md 'Roofline'); ncu "
                                    "counts the pipe against the same rate (profiles/r03_ncu.md)",
                     "peak_measured_dfma": peak["tflops"], "frac_of_measured_dfma": achieved_tflops / peak["tflops"],
                     "peak_measured_dfma_source": "ia_fp64_peak: 2 s of independent DFMA chains on every SM in this run; it "
                                                  "keeps the pipe 92.2 % busy (ncu, profiles/r03_k4_raw.csv)",
                     "peak_elapsed_ms": peak["elapsed_ms"], "peak_clocks": peak_clk,
                     "traffic": TRAFFIC_BYTES_PER_TRAJECTORY * n, "traffic_source": TRAFFIC_SOURCE,
                     "progress_metric": "rk_steps_per_s (flops are executed flops: frac rises if a step does more arithmetic)",
                     "flop_per_attempted_step": FLOP_PER_STEP, "kernel": "ia_persistent_kernel<1, IA_SRC_BOTH> (bulk)",
                     "kernel_ms": bulk_ms, "steps_in_kernel": steps_region / K,
                     "share_of_step_time": sum(kernel_ms) * 1e-3 / region_s,
                     # share of the kernel's lane-steps (32 per warp and attempt) that advanced a trajectory
                     "lane_efficiency": steps_region / max(slots_region, 1)},
        # every attempted step executed inside the timed region over the whole region
        "whole_step": {"achieved": whole_tflops, "peak": nominal_tflops, "unit": "TFLOP/s",
                       "frac": whole_tflops / nominal_tflops,
                       "frac_of_measured_dfma": whole_tflops / peak["tflops"],
                       "rk_steps": steps_region, "seconds": region_s},
        # the whole device-resident stream, chain included: every trajectory of the W-1 warm-up and K timed steps over the
        # time from the first launch of the stream to the end of its straggler chain
        "whole_stream": {"value": world * n_stream / stream_s, "unit": "trajectories/s", "trajectories_per_gpu": n_stream,
                         "seconds": stream_s, "steps": W - 1 + K},
        # the end of the stream: a trajectory is a serial chain, so the chain lasts as long as the longest one left
        "tail": {"kernel": f"chain of {2 + levels} launches: ia_persistent_kernel<1, IA_SRC_BOTH> over a full grid (stage A), the "
                           f"same with one warp per SM sub-partition (stage B), ia_persistent_kernel<3, IA_SRC_QUEUE> "
                           f"(cooperative, 3 lanes per trajectory, one warp per sub-partition) x {levels} (stage C)",
                 "launches": 2 + levels,
                 "chain_ms": chain_t["coop_ms"], "drain_wall_ms": 1e3 * drain_s,
                 "share_of_step_time": 0.0,
                 "share_of_stream_time": chain_t["coop_ms"] * 1e-3 / (region_s + chain_t["coop_ms"] * 1e-3),
                 "longest_trajectory_steps_last_step": longest,
                 "note": "outside the timed region; paid once per stream, whatever its length (DESIGN.md 'Tail')"},
        "attempted_steps_of_timed_batches": attempted,
        "kernel_info": info, "clocks": clk, "e2e": e2e, "gpu_launches": K,   # the K bulk kernels of the timed region (the chain and the e2e leg are outside it)
    }
    if not args.no_cpu_baseline and world == 1:
        s = oracle_sample(cell, args.n_side, ORACLE_SAMPLE_BASELINE)
        line["cpu_baseline"] = {"value": s["n"] / s["seconds"], "unit": "trajectories/s", "cores": s["cores"],
                                "kind": "oracle", "sample": s["sample"], "rk_steps_per_s": s["steps"] / s["seconds"]}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves, the way the driver does."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd)


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
