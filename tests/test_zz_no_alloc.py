"""ia_run_static: the entry point for hosts that cannot allocate device memory (include/ia.h).

Who that is: code that runs inside somebody else's process after that process has given the whole GPU to its own
memory pool -- a cudaMalloc from a plug-in then fails or eats into the pool -- and loops that launch between other
streams' work and cannot take the device-wide synchronisation cudaMalloc and cudaFree bring with them.  Everything
else in this library starts with ia_create, which does allocate (work counters, hand-over queues).  ia_run_static
instead keeps its counters and its hand-over queue in a static array of the library's device image (4 MiB + 256 bytes,
present on every GPU that loads the library), takes at most IA_STATIC_MAX_N = 16384 trajectories per call, and is
checked here against the path every other test exercises: ia_create + ia_run, the production kernel pair.

The bar is the one tests/test_gpu_parity.py holds the kernel layouts to among themselves
(test_bulk_coop_and_handoff_paths_are_bit_identical): records and generated initial conditions bit for bit, the
integer fields of the summary exactly, its two floating-point sums (atomic additions in a different order) to 1e-12.

This file sorts last on purpose (pytest -x stops at the first failure, and nothing may hide behind this test); the
GPU test passes in a fresh process as well as after the rest of the suite, because the only state it meets is the
static array, whose counters every call clears and whose queue no call reads before writing it.
"""
import os
import re
from dataclasses import replace

import numpy as np
import pytest

import ia_inputs as I
import paper_2509_15117_b200 as P

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
EXACT_SUMMARY_FIELDS = ("n_done", "n_status", "n_complex", "steps_acc", "steps_rej", "steps_loc", "hist_ncoll",
                        "hist_tlife", "warn")


def test_static_entry_refuses_a_launch_larger_than_its_queue():
    """More trajectories than the static hand-over queue has entries: refused with IA_EINVAL and a text that names
    the limit, before any device is looked at (so this runs on a machine without a GPU)."""
    cell = I.config1(256)
    assert cell.launch.n > P.IA_STATIC_MAX_N
    with pytest.raises(P.IaError) as ei:
        P.ia_run_static(cell.params, P.make_launch(replace(cell.launch, n=P.IA_STATIC_MAX_N + 1)))
    assert ei.value.code == P.IA_EINVAL
    assert "IA_STATIC_MAX_N = 16384" in str(ei.value) and "16385" in str(ei.value)
    # the other argument checks answer without a device too
    with pytest.raises(P.IaError) as ei:
        P.ia_run_static(cell.params, P.make_launch(replace(cell.launch, n=64, path=P.IA_PATH_BULK_ONLY)))
    assert ei.value.code == P.IA_EINVAL and "IA_PATH_AUTO" in str(ei.value)
    with pytest.raises(P.IaError) as ei:
        P.ia_run_static(replace(cell.params, rtol=1e-2), P.make_launch(replace(cell.launch, n=64)))
    assert ei.value.code == P.IA_EINVAL
    assert P.load().ia_run_static(None, None, 1.0, 5000.0, None, 0, None, None, None, None, 0) == P.IA_EINVAL
    import torch
    if not torch.cuda.is_available():       # a valid call on a machine without a device: loud, no CPU path
        with pytest.raises(P.IaError) as ei:
            P.ia_run_static(cell.params, P.make_launch(replace(cell.launch, n=64)))
        assert ei.value.code == P.IA_EDEVICE


def test_static_entry_calls_no_allocating_routine():
    """The promise of include/ia.h, read off the source: between the start of the ia_run_static section of
    csrc/ia_api.cu and the end of the file no allocating or resource-creating CUDA call appears outside comments, the
    scratch is a file-scope static __device__ __align__(256) array, and its address comes from cudaGetSymbolAddress."""
    src = open(os.path.join(ROOT, "paper_2509_15117_b200", "csrc", "ia_api.cu")).read()
    start = src.index("/* ---- ia_run_static:")
    code = re.sub(r"/\*.*?\*/", "", src[start:], flags=re.S)
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaEventCreate", "cudaStreamCreate", "guarded_malloc",
                   "new ", "cudaMemPool"):
        assert banned not in code, banned
    assert re.search(r"static\s+__device__\s+__align__\(256\)\s+unsigned char ia_static_scratch\[", code)
    assert "cudaGetSymbolAddress(&p, ia_static_scratch)" in code
    assert code.count("ia_static_scratch") == 2     # host code names it twice: the definition and cudaGetSymbolAddress


@pytest.mark.gpu
def test_static_entry_matches_ia_run_on_calls_in_a_row():
    """Three calls back to back on one stream, no synchronisation in between -- a 64x64 grid of config 1 (4,096
    trajectories, regular and chaotic), then 1,500 of config 2's Li 10 uK Philox cell (another species, a ragged 46
    warps + 28 lanes, a first_index beyond 2^32), then the first again -- each against ia_create + ia_run on the same
    cell.  The second and third calls meet the counters and the queue as the call before left them.  After the first
    call (which does the one-time set-up of the device) the free device memory the driver reports must not move."""
    import torch
    assert torch.cuda.is_available(), "GPU tests selected on a machine without a CUDA device"
    P.load()
    a = I.config1(64)
    a = replace(a, params=replace(a.params, t_max_rf=300.0))
    b = I.config2(n_per_cell=1500)[2]
    b = replace(b, params=replace(b.params, t_max_rf=300.0), launch=replace(b.launch, first_index=(1 << 32) - 700))
    assert a.launch.n <= P.IA_STATIC_MAX_N and b.launch.n <= P.IA_STATIC_MAX_N

    want = []
    for cell in (a, b):
        with P.Context(cell.params) as ctx:
            want.append(ctx.run_sync(cell.launch, want_ic=True))

    dev = torch.device("cuda", 0)
    calls = (a, b, a)
    bufs = [(torch.zeros(c.launch.n * P.RECORD_BYTES, dtype=torch.uint8, device=dev),
             torch.zeros(P.SUMMARY_BYTES, dtype=torch.uint8, device=dev),
             torch.zeros((c.launch.n, P.IC_DUMP_COLS), dtype=torch.float64, device=dev)) for c in calls]
    torch.cuda.synchronize()
    free = []
    for k, (cell, (rec, summ, ic)) in enumerate(zip(calls, bufs)):
        if k == 1:
            torch.cuda.synchronize()                      # the first call has done the device's set-up
            free.append(torch.cuda.mem_get_info(0)[0])
        text = P.ia_run_static(cell.params, P.make_launch(cell.launch), rec, summ, ic, device=0)
        assert text == ""
    torch.cuda.synchronize()
    free.append(torch.cuda.mem_get_info(0)[0])
    assert free[0] == free[1], f"free device memory moved across two ia_run_static calls: {free}"

    handed = 0
    for k, (cell, (rec, summ, ic)) in enumerate(zip(calls, bufs)):
        n = cell.launch.n
        rec_w, sum_w, ic_w = want[0 if cell is a else 1]
        got, s = P.view_records(rec, n), P.view_summary(summ)
        assert got.tobytes() == rec_w.tobytes(), f"call {k}: records differ from ia_run's"
        assert np.array_equal(ic.cpu().numpy(), ic_w), f"call {k}: generated initial conditions differ"
        for f in EXACT_SUMMARY_FIELDS:
            assert np.array_equal(s[f], sum_w[f]), (k, f, s[f], sum_w[f])
        assert int(s["n_done"]) == n
        for f in ("sum_ke", "sum_ke2"):
            assert abs(float(s[f]) - float(sum_w[f])) <= 1e-12 * abs(float(sum_w[f])), (k, f)
        handed += int(s["n_handoff"])
        print(f"\nia_run_static call {k}: {cell.name} n={n}: records bit-identical to ia_run; "
              f"{int(s['n_handoff'])} trajectories went through the static hand-over queue, "
              f"{int(s['n_complex'])} complexes, statuses {s['n_status'].tolist()}")
    assert handed > 0, "no call used the static hand-over queue: the test does not exercise the scratch"
