"""paper_2509_15117_b200 -- thin Python binding of libia_b200.so (include/ia.h).

Argument marshalling only: every step of the hot path (initial-condition generation, the adaptive
Dormand-Prince 5(4) propagation of PAPER.md:13-20,26, events, exit localisation, observables,
ensemble reduction) runs in the sm_100a CUDA kernels behind the C-ABI.  PyTorch is used for device
memory and streams.  There is NO CPU fallback: without the built library (or without a
compute-capability-10.x device) the calls raise.

The functions carry the names of the C entry points (``ia_create``, ``ia_run``, ``ia_run_host``,
``ia_generate``, ``ia_step_map``, ``ia_trace``, ``ia_fp64_peak``, ``ia_destroy`` ...); ``Context``
is a small convenience wrapper that owns one ``ia_ctx`` handle.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional

import numpy as np

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libia_b200.so"

IA_OK, IA_EINVAL, IA_ENOMEM, IA_ECUDA, IA_EDEVICE = 0, -1, -2, -3, -4
IA_IC_EXPLICIT, IA_IC_GRID, IA_IC_PHILOX, IA_IC_THERMAL = 0, 1, 2, 3
IA_PATH_AUTO, IA_PATH_BULK_ONLY, IA_PATH_COOP_ONLY = 0, 1, 2
IA_ARITH_NOFMA, IA_ARITH_FMA, IA_ARITH_FMA_COOP = 0, 1, 2
IA_HIST_BINS = 32
IA_LIFE_BINS = 64
IA_STRAGGLER_LEVELS = 12
IA_STATIC_MAX_N = 16384   # most trajectories one ia_run_static call takes (include/ia.h)

# every symbol include/ia.h declares (tests/test_cabi.py checks the library exports each of them)
EXPORTS = ("ia_create", "ia_run", "ia_run_host", "ia_generate", "ia_step_map", "ia_trace", "ia_get_derived",
           "ia_get_kernel_info", "ia_set_handoff", "ia_set_chain", "ia_get_last_timing", "ia_get_timing", "ia_set_pipeline", "ia_join",
           "ia_submit_host", "ia_sync", "ia_wait", "ia_debug_check", "ia_fp64_peak", "ia_fp64_latency", "ia_run_static", "ia_destroy", "ia_strerror", "ia_last_error")


class IaError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"libia_b200: {text} (code {code})")
        self.code = code


# ---- C structs of include/ia.h -------------------------------------------------------------------

class ia_species(C.Structure):
    _fields_ = [("m_ion_u", C.c_double), ("m_atom_u", C.c_double), ("alpha_au", C.c_double)]


class ia_trap(C.Structure):
    _fields_ = [("a", C.c_double * 3), ("q", C.c_double * 3), ("omega_rf_au", C.c_double)]


class ia_tol(C.Structure):
    _fields_ = [("rtol", C.c_double), ("atol", C.c_double), ("t_max_rf", C.c_double), ("h_max_rf", C.c_double),
                ("r_coll_a0", C.c_double), ("max_steps", C.c_uint64)]


class ia_launch(C.Structure):
    _fields_ = [("mode", C.c_int32), ("domain", C.c_int32), ("phase_mode", C.c_int32),
                ("n_theta", C.c_uint32), ("n_phi", C.c_uint32), ("path", C.c_int32), ("n", C.c_uint64),
                ("y0", C.c_void_p), ("phase", C.c_void_p), ("phase0", C.c_double),
                ("E_min_uK", C.c_double), ("E_max_uK", C.c_double), ("seed", C.c_uint64),
                ("cell", C.c_uint32), ("first_index", C.c_uint64),
                ("T_atom_uK", C.c_double), ("T_ion_uK", C.c_double)]


class ia_outputs(C.Structure):
    _fields_ = [("records", C.c_void_p), ("summary", C.c_void_p), ("ic_dump", C.c_void_p)]


RECORD_DTYPE = np.dtype([("ke_ion", "<f8"), ("t_dwell", "<f8"), ("t_life", "<f8"), ("va_f", "<f8", (3,)),
                         ("n_coll", "<u4"), ("n_tp", "<u4"), ("steps_acc", "<u4"), ("steps_rej", "<u2"),
                         ("status", "u1"), ("n_loc", "u1")])
SUMMARY_DTYPE = np.dtype([("n_done", "<u8"), ("n_status", "<u8", (5,)), ("n_complex", "<u8"),
                          ("steps_acc", "<u8"), ("steps_rej", "<u8"), ("steps_loc", "<u8"),
                          ("sum_ke", "<f8"), ("sum_ke2", "<f8"), ("hist_ncoll", "<u8", (IA_HIST_BINS,)),
                          ("t_first_idle_ns", "<u8"), ("t_start_ns", "<u8"), ("t_end_ns", "<u8"),
                          ("warn", "<u8"), ("n_handoff", "<u8"), ("steps_coop", "<u8"), ("t_bulk_end_ns", "<u8"),
                          ("slots_bulk", "<u8"), ("steps_kernel", "<u8"), ("reserved", "<u8", (11,)), ("hist_tlife", "<u8", (IA_LIFE_BINS,))])
RECORD_BYTES, SUMMARY_BYTES, IC_DUMP_COLS = 64, 1024, 14
assert RECORD_DTYPE.itemsize == RECORD_BYTES and SUMMARY_DTYPE.itemsize == SUMMARY_BYTES

_lib: Optional[C.CDLL] = None


def load() -> C.CDLL:
    """Loads libia_b200.so (building it with nvcc first if the sources are newer).  Raises when the
    library cannot be had -- there is no other implementation to fall back to."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    try:
        _build.build()
    except Exception as exc:  # no nvcc on this machine: a previously built library is still fine
        if not LIB_PATH.exists():
            raise RuntimeError(f"libia_b200.so is missing and could not be built ({exc}); "
                               "there is no CPU fallback") from exc
    L = C.CDLL(str(LIB_PATH))
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
    L.ia_create.argtypes = [C.POINTER(vp), C.POINTER(ia_species), C.POINTER(ia_trap), C.c_double, C.c_double,
                            C.POINTER(ia_tol), C.c_int]
    L.ia_run.argtypes = [vp, C.POINTER(ia_launch), C.POINTER(ia_outputs), vp]
    L.ia_run_host.argtypes = [vp, C.POINTER(ia_launch), C.POINTER(ia_outputs)]
    L.ia_generate.argtypes = [vp, C.POINTER(ia_launch), vp, vp]
    L.ia_step_map.argtypes = [vp, C.c_uint64, vp, vp, vp, vp, vp, vp, C.c_int, vp]
    L.ia_trace.argtypes = [vp, dp, C.c_double, C.c_double, C.c_uint32, vp, C.c_int, vp]
    L.ia_get_derived.argtypes = [vp, dp]
    L.ia_get_kernel_info.argtypes = [vp, C.c_int, ip, ip, ip, ip]
    L.ia_set_handoff.argtypes = [vp, C.c_int]
    L.ia_get_last_timing.argtypes = [vp, dp, dp]
    L.ia_set_chain.argtypes = [vp, C.c_int, C.c_uint32]
    L.ia_get_timing.argtypes = [vp, C.c_int, dp, dp]
    L.ia_set_pipeline.argtypes = [vp, C.c_int]
    L.ia_join.argtypes = [vp, vp]
    L.ia_submit_host.argtypes = [vp, C.POINTER(ia_launch), C.POINTER(ia_outputs)]
    L.ia_wait.argtypes = [vp]
    L.ia_sync.argtypes = [vp]
    L.ia_debug_check.argtypes = [vp]
    L.ia_fp64_peak.argtypes = [C.c_int, C.c_double, dp, dp]
    L.ia_fp64_latency.argtypes = [C.c_int, dp, dp]
    L.ia_run_static.argtypes = [C.POINTER(ia_species), C.POINTER(ia_trap), C.c_double, C.c_double, C.POINTER(ia_tol),
                                C.c_int, C.POINTER(ia_launch), C.POINTER(ia_outputs), vp, C.c_char_p, C.c_size_t]
    L.ia_destroy.argtypes = [vp]
    L.ia_strerror.argtypes = [C.c_int]
    L.ia_strerror.restype = C.c_char_p
    L.ia_last_error.argtypes = [vp]
    L.ia_last_error.restype = C.c_char_p
    _lib = L  # every other entry point returns int, ctypes' default restype
    return L


def ia_strerror(code: int) -> str:
    return load().ia_strerror(int(code)).decode()


def ia_last_error(handle) -> str:
    return load().ia_last_error(handle).decode()


def _check(rc: int, handle=None):
    if rc != IA_OK:
        text = ia_strerror(rc)
        if handle:
            detail = ia_last_error(handle)
            if detail:
                text += ": " + detail
        raise IaError(rc, text)


# ---- marshalling helpers --------------------------------------------------------------------------

def _ptr(t) -> Optional[int]:
    """Device (or host) address of a torch tensor / numpy array / int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _stream_handle(stream) -> Optional[int]:
    """cudaStream_t of a torch.cuda.Stream, an int handle, or torch's current stream when None."""
    if isinstance(stream, int):
        return stream or None
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream or None


def make_launch(launch, y0=None, phase=None) -> ia_launch:
    """launch: any object with the attribute names of ia_inputs.Launch (mode, n, n_theta, ...)."""
    L = ia_launch()
    L.mode, L.domain, L.phase_mode = int(launch.mode), int(launch.domain), int(launch.phase_mode)
    L.n_theta, L.n_phi, L.n = int(launch.n_theta), int(launch.n_phi), int(launch.n)
    L.path = int(getattr(launch, "path", 0))
    L.y0, L.phase = _ptr(y0), _ptr(phase)
    L.phase0, L.E_min_uK, L.E_max_uK = float(launch.phase0), float(launch.E_min_uK), float(launch.E_max_uK)
    L.seed, L.cell, L.first_index = int(launch.seed), int(launch.cell), int(launch.first_index)
    L.T_atom_uK, L.T_ion_uK = float(getattr(launch, "T_atom_uK", 0.0)), float(getattr(launch, "T_ion_uK", 0.0))
    return L


# ---- the C entry points, same names ----------------------------------------------------------------

def ia_create(params, device: int = 0) -> int:
    """params: any object with the attribute names of ia_inputs.Params.  Returns the ia_ctx handle."""
    sp = ia_species(params.m_ion_u, params.m_atom_u, params.alpha_au)
    tr = ia_trap((C.c_double * 3)(*params.a), (C.c_double * 3)(*params.q), params.omega_rf_au)
    tol = ia_tol(params.rtol, params.atol, params.t_max_rf, params.h_max_rf, params.r_coll_a0, int(params.max_steps))
    h = C.c_void_p()
    _check(load().ia_create(C.byref(h), C.byref(sp), C.byref(tr), float(params.De_K), float(params.r0_a0),
                            C.byref(tol), int(device)))
    return h.value


def ia_destroy(handle) -> None:
    _check(load().ia_destroy(handle))


def ia_run(handle, launch: ia_launch, records=None, summary=None, ic_dump=None, stream=None) -> None:
    """Asynchronous: enqueues on `stream` (default: torch's current stream).  All buffers are device
    tensors: records uint8 [n*64], summary uint8 [1024] (accumulated into), ic_dump float64 [n,14]."""
    out = ia_outputs(_ptr(records), _ptr(summary), _ptr(ic_dump))
    _check(load().ia_run(handle, C.byref(launch), C.byref(out), _stream_handle(stream)), handle)


def ia_run_host(handle, launch: ia_launch, records=None, summary=None, ic_dump=None) -> None:
    """Host buffers (numpy arrays or pinned CPU tensors); synchronous."""
    out = ia_outputs(_ptr(records), _ptr(summary), _ptr(ic_dump))
    _check(load().ia_run_host(handle, C.byref(launch), C.byref(out)), handle)


def ia_generate(handle, launch: ia_launch, ic_dump, stream=None) -> None:
    _check(load().ia_generate(handle, C.byref(launch), _ptr(ic_dump), _stream_handle(stream)), handle)


def ia_step_map(handle, n, t_frac, phase, y, h, ynew, err=None, variant: int = IA_ARITH_FMA, stream=None) -> None:
    _check(load().ia_step_map(handle, int(n), _ptr(t_frac), _ptr(phase), _ptr(y), _ptr(h), _ptr(ynew), _ptr(err),
                              int(variant), _stream_handle(stream)), handle)


def ia_trace(handle, y0_host: np.ndarray, phase: float, h: float, nsteps: int, states, variant: int = IA_ARITH_FMA,
             stream=None) -> None:
    y0 = np.ascontiguousarray(y0_host, dtype=np.float64)
    assert y0.shape == (12,)
    _check(load().ia_trace(handle, y0.ctypes.data_as(C.POINTER(C.c_double)), float(phase), float(h), int(nsteps),
                           _ptr(states), int(variant), _stream_handle(stream)), handle)


_DERIVED_NAMES = ("m_i", "m_a", "C4", "C8", "De", "r_e", "Omega", "T_rf", "thr", "h_max", "h_min", "t_max", "r0",
                  "r_coll", "rtol", "atol")


def ia_get_derived(handle) -> dict:
    out = (C.c_double * 16)()
    _check(load().ia_get_derived(handle, out), handle)
    return dict(zip(_DERIVED_NAMES, list(out)))


def ia_get_kernel_info(handle, kernel: int = 0) -> dict:
    """kernel: 0 = bulk persistent kernel (one lane per trajectory), 1 = cooperative (three lanes)."""
    v = [C.c_int() for _ in range(4)]
    _check(load().ia_get_kernel_info(handle, int(kernel), *[C.byref(x) for x in v]), handle)
    return {"warps_per_sm": v[0].value, "n_sm": v[1].value, "regs_per_thread": v[2].value,
            "local_bytes_per_thread": v[3].value}


def ia_set_handoff(handle, lanes: int) -> None:
    _check(load().ia_set_handoff(handle, int(lanes)), handle)


def ia_set_chain(handle, levels: int, budget: int = 8192) -> None:
    """Straggler chain: `levels` launches of the cooperative kernel, level j lasting budget << j iterations."""
    _check(load().ia_set_chain(handle, int(levels), int(budget)), handle)


def ia_get_timing(handle, runs_back: int = 0) -> dict:
    """Device times (ms) of the two kernels of a recent run on this ctx (0 = the last); synchronises with it."""
    a, b = C.c_double(), C.c_double()
    _check(load().ia_get_timing(handle, int(runs_back), C.byref(a), C.byref(b)), handle)
    return {"bulk_ms": a.value, "coop_ms": b.value}


def ia_get_last_timing(handle) -> dict:
    a, b = C.c_double(), C.c_double()
    _check(load().ia_get_last_timing(handle, C.byref(a), C.byref(b)), handle)
    return {"bulk_ms": a.value, "coop_ms": b.value}


def ia_set_pipeline(handle, depth: int) -> None:
    """depth > 0: the bulk kernel of a run resumes what the run before left unfinished; ia_join ends the pipeline."""
    _check(load().ia_set_pipeline(handle, int(depth)), handle)


def ia_join(handle, stream=None) -> None:
    """Enqueues the straggler chain of the open pipeline on `stream` (default: torch's current stream)."""
    _check(load().ia_join(handle, _stream_handle(stream)), handle)


def ia_submit_host(handle, launch: ia_launch, records=None, summary=None, ic_dump=None) -> None:
    """Asynchronous ia_run_host: pinned host buffers, valid after ia_wait."""
    out = ia_outputs(_ptr(records), _ptr(summary), _ptr(ic_dump))
    _check(load().ia_submit_host(handle, C.byref(launch), C.byref(out)), handle)


def ia_wait(handle) -> None:
    _check(load().ia_wait(handle), handle)


def ia_sync(handle) -> None:
    """Blocks until every kernel and copy enqueued so far has finished; the pipeline stays open."""
    _check(load().ia_sync(handle), handle)


def ia_debug_check(handle) -> None:
    """Verifies the guard zones around every ctx-owned device buffer and the kernels' fault word; raises on a finding."""
    _check(load().ia_debug_check(handle), handle)


def ia_run_static(params, launch: ia_launch, records=None, summary=None, ic_dump=None, device: int = 0,
                  stream=None) -> str:
    """The production kernel pair without a ctx and without any device allocation inside the library, for hosts
    that cannot call cudaMalloc (a plug-in next to an application whose pool already owns the GPU's memory; a loop
    that cannot take cudaMalloc's device-wide synchronisation): the counters and the hand-over queue live in a
    static 4 MiB array of the library's device image.  At most IA_STATIC_MAX_N trajectories per call; calls that
    may overlap on the GPU race (keep them on one stream).  The first call on a device also looks up that array's
    address and loads the kernels: make it at start-up.  Same buffers as ia_run (device tensors, the summary is
    accumulated into), same results bit for bit.  Asynchronous; returns the warning text ("" if none)."""
    sp = ia_species(params.m_ion_u, params.m_atom_u, params.alpha_au)
    tr = ia_trap((C.c_double * 3)(*params.a), (C.c_double * 3)(*params.q), params.omega_rf_au)
    tol = ia_tol(params.rtol, params.atol, params.t_max_rf, params.h_max_rf, params.r_coll_a0, int(params.max_steps))
    out = ia_outputs(_ptr(records), _ptr(summary), _ptr(ic_dump))
    err = C.create_string_buffer(512)
    L = load()
    # torch's current stream is looked up only where there is a device: without one the library itself answers
    # (IA_EINVAL for a bad argument, IA_EDEVICE otherwise)
    st = stream or None
    if not isinstance(stream, int):
        import torch
        st = _stream_handle(stream) if (stream is not None or torch.cuda.is_available()) else None
    rc = L.ia_run_static(C.byref(sp), C.byref(tr), float(params.De_K), float(params.r0_a0), C.byref(tol), int(device),
                         C.byref(launch), C.byref(out), st, err, len(err))
    if rc != IA_OK:
        raise IaError(rc, ia_strerror(rc) + ": " + err.value.decode())
    return err.value.decode()


def ia_fp64_peak(device: int = 0, target_ms: float = 200.0) -> dict:
    """DFMA peak microbenchmark: {'tflops': 2*DFMA/s/1e12, 'elapsed_ms': ...}."""
    t, ms = C.c_double(), C.c_double()
    _check(load().ia_fp64_peak(int(device), float(target_ms), C.byref(t), C.byref(ms)))
    return {"tflops": t.value, "elapsed_ms": ms.value}


def ia_fp64_latency(device: int = 0) -> dict:
    """SM cycles per dependent DFMA and per reciprocal (MUFU.RCP64H + 3 DFMA) + DADD, one warp alone."""
    a, b = C.c_double(), C.c_double()
    _check(load().ia_fp64_latency(int(device), C.byref(a), C.byref(b)))
    return {"cycles_dfma": a.value, "cycles_rcp_add": b.value}


# ---- convenience wrapper ---------------------------------------------------------------------------

class Context:
    """Owns one ia_ctx (one (species, trap, De, r0, tolerances) cell) and allocates output tensors
    with torch.  Nothing here computes: it allocates, calls the C-ABI and views the bytes."""

    def __init__(self, params, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise IaError(IA_EDEVICE, "no CUDA device: the propagator has no CPU fallback")
        self.device = int(device)
        self.params = params
        self.handle = ia_create(params, self.device)

    def close(self):
        if getattr(self, "handle", None):
            ia_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def derived(self) -> dict:
        return ia_get_derived(self.handle)

    @property
    def kernel_info(self) -> dict:
        return {"bulk": ia_get_kernel_info(self.handle, 0), "coop": ia_get_kernel_info(self.handle, 1)}

    def set_handoff(self, lanes: int) -> None:
        ia_set_handoff(self.handle, lanes)

    @property
    def last_timing(self) -> dict:
        return ia_get_last_timing(self.handle)

    def timing(self, runs_back: int = 0) -> dict:
        return ia_get_timing(self.handle, runs_back)

    def set_chain(self, levels: int, budget: int = 8192) -> None:
        ia_set_chain(self.handle, levels, budget)

    def set_pipeline(self, depth: int) -> None:
        ia_set_pipeline(self.handle, depth)

    def join(self, stream=None) -> None:
        ia_join(self.handle, stream)

    def wait(self) -> None:
        ia_wait(self.handle)

    def sync(self) -> None:
        ia_sync(self.handle)

    def debug_check(self) -> None:
        ia_debug_check(self.handle)

    def alloc(self, n: int, ic_dump: bool = False):
        """(records uint8[n*64], summary uint8[1024] zeroed, ic_dump float64[n,14] or None) on the device."""
        import torch
        dev = torch.device("cuda", self.device)
        rec = torch.empty(max(n, 1) * RECORD_BYTES, dtype=torch.uint8, device=dev)
        summ = torch.zeros(SUMMARY_BYTES, dtype=torch.uint8, device=dev)
        ic = torch.empty((max(n, 1), IC_DUMP_COLS), dtype=torch.float64, device=dev) if ic_dump else None
        return rec, summ, ic

    def run(self, launch, y0=None, phase=None, records=None, summary=None, ic_dump=None, stream=None) -> None:
        """Asynchronous device-resident run (ia_run).  y0/phase: device float64 tensors for EXPLICIT."""
        ia_run(self.handle, make_launch(launch, y0, phase), records, summary, ic_dump, stream)

    def run_sync(self, launch, y0=None, phase=None, want_ic: bool = False):
        """Device-resident run, synchronised, results viewed as numpy structured arrays:
        (records[n], summary scalar, ic_dump[n,14] or None)."""
        import torch
        if y0 is not None and not hasattr(y0, "data_ptr"):
            y0 = torch.as_tensor(np.ascontiguousarray(y0, dtype=np.float64)).to(f"cuda:{self.device}")
        if phase is not None and not hasattr(phase, "data_ptr"):
            phase = torch.as_tensor(np.ascontiguousarray(phase, dtype=np.float64)).to(f"cuda:{self.device}")
        rec, summ, ic = self.alloc(int(launch.n), want_ic)
        self.run(launch, y0, phase, rec, summ, ic)
        torch.cuda.synchronize(self.device)
        return (view_records(rec, int(launch.n)), view_summary(summ),
                ic.cpu().numpy()[: int(launch.n)] if ic is not None else None)

    def run_host(self, launch, y0: Optional[np.ndarray] = None, phase: Optional[np.ndarray] = None,
                 records: Optional[np.ndarray] = None, summary: Optional[np.ndarray] = None,
                 ic_dump: Optional[np.ndarray] = None):
        """End-to-end entry with host buffers (ia_run_host): copies in, runs, copies back, synchronises."""
        n = int(launch.n)
        if records is None:
            records = np.zeros(n, dtype=RECORD_DTYPE)
        if summary is None:
            summary = np.zeros(1, dtype=SUMMARY_DTYPE)
        ia_run_host(self.handle, make_launch(launch, y0, phase), records, summary, ic_dump)
        return records, summary[0]

    def generate(self, launch) -> np.ndarray:
        import torch
        n = int(launch.n)
        ic = torch.empty((max(n, 1), IC_DUMP_COLS), dtype=torch.float64, device=f"cuda:{self.device}")
        ia_generate(self.handle, make_launch(launch), ic)
        torch.cuda.synchronize(self.device)
        return ic.cpu().numpy()[:n]

    def step_map(self, t_frac, phase, y, h, variant: int = IA_ARITH_FMA):
        """n single uncontrolled steps: returns (ynew[n,12], err[n]) as numpy."""
        import torch
        dev = f"cuda:{self.device}"
        y = np.ascontiguousarray(y, dtype=np.float64).reshape(-1, 12)
        n = len(y)
        bc = lambda a: np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.float64), (n,)))
        d = [torch.as_tensor(a).to(dev) for a in (bc(t_frac), bc(phase), y, bc(h))]
        ynew = torch.empty((max(n, 1), 12), dtype=torch.float64, device=dev)
        err = torch.empty(max(n, 1), dtype=torch.float64, device=dev)
        ia_step_map(self.handle, n, d[0], d[1], d[2], d[3], ynew, err, variant)
        torch.cuda.synchronize(self.device)
        return ynew.cpu().numpy()[:n], err.cpu().numpy()[:n]

    def trace(self, y0, phase: float, h: float, nsteps: int, variant: int = IA_ARITH_FMA) -> np.ndarray:
        """nsteps uncontrolled steps of size h: (t, y) rows [nsteps+1, 13] as numpy."""
        import torch
        st = torch.empty((nsteps + 1, 13), dtype=torch.float64, device=f"cuda:{self.device}")
        ia_trace(self.handle, np.asarray(y0, dtype=np.float64), phase, h, nsteps, st, variant)
        torch.cuda.synchronize(self.device)
        return st.cpu().numpy()


def view_records(rec_tensor, n: int) -> np.ndarray:
    return rec_tensor.cpu().numpy()[: n * RECORD_BYTES].view(RECORD_DTYPE).copy()


def view_summary(summ_tensor) -> np.void:
    return summ_tensor.cpu().numpy().view(SUMMARY_DTYPE)[0].copy()
