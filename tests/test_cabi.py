"""The C-ABI library of include/ia.h: it builds, loads, exports every declared symbol, and its
argument checks answer without a GPU (no compute call is made here).  CPU-only."""
import ctypes as C
import os
import re

import pytest

import ia_inputs as I
import paper_2509_15117_b200 as P

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    """Every function include/ia.h declares (a name followed by '(' at the start of a declaration)."""
    text = open(os.path.join(ROOT, "include", "ia.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ia_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_all_exported():
    names = declared_symbols()
    assert set(names) == set(P.EXPORTS), (names, P.EXPORTS)
    L = P.load()
    for n in names:
        assert hasattr(L, n), f"libia_b200.so does not export {n}"


def test_struct_sizes_match_the_header():
    # the byte layouts include/ia.h promises: 64-byte records, 1024-byte summary
    assert P.RECORD_DTYPE.itemsize == 64 and P.SUMMARY_DTYPE.itemsize == 1024
    assert C.sizeof(P.ia_species) == 24 and C.sizeof(P.ia_trap) == 56 and C.sizeof(P.ia_tol) == 48
    assert C.sizeof(P.ia_launch) == 112 and C.sizeof(P.ia_outputs) == 24
    assert P.RECORD_DTYPE.fields["va_f"][1] == 24 and P.RECORD_DTYPE.fields["status"][1] == 62
    assert P.SUMMARY_DTYPE.fields["hist_ncoll"][1] == 96 and P.SUMMARY_DTYPE.fields["warn"][1] == 376
    assert P.SUMMARY_DTYPE.fields["hist_tlife"][1] == 512


def test_strerror_and_null_arguments():
    L = P.load()
    assert P.ia_strerror(0) == "ok"
    assert "fallback" in P.ia_strerror(P.IA_EDEVICE)          # the library says there is no CPU path
    assert P.ia_strerror(-99) == "unknown error code"
    assert L.ia_create(None, None, None, 1.0, 5000.0, None, 0) == P.IA_EINVAL
    assert L.ia_run(None, None, None, None) == P.IA_EINVAL
    assert L.ia_run_host(None, None, None) == P.IA_EINVAL
    assert L.ia_generate(None, None, None, None) == P.IA_EINVAL
    assert L.ia_step_map(None, 0, None, None, None, None, None, None, 0, None) == P.IA_EINVAL
    assert L.ia_trace(None, None, 0.0, 1.0, 1, None, 0, None) == P.IA_EINVAL
    assert L.ia_destroy(None) == P.IA_EINVAL
    assert L.ia_get_derived(None, None) == P.IA_EINVAL
    assert L.ia_get_kernel_info(None, 0, None, None, None, None) == P.IA_EINVAL
    assert L.ia_set_handoff(None, 8) == P.IA_EINVAL
    assert L.ia_get_last_timing(None, None, None) == P.IA_EINVAL
    assert L.ia_fp64_peak(0, 10.0, None, None) == P.IA_EINVAL
    assert P.ia_last_error(None) == ""


@pytest.mark.parametrize("field,value", [("m_atom_u", -1.0), ("alpha_au", 0.0), ("rtol", 1e-2), ("rtol", 1e-15),
                                         ("h_max_rf", 0.5), ("De_K", float("nan")), ("r0_a0", 0.0)])
def test_create_rejects_bad_parameters_before_touching_a_device(field, value):
    from dataclasses import replace
    p = replace(I.config1(8).params, **{field: value})
    with pytest.raises(P.IaError) as ei:
        P.ia_create(p, 0)
    assert ei.value.code == P.IA_EINVAL


def test_no_cpu_fallback_without_a_device():
    """On a box without a compute-capability-10.x device the product path fails loudly."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(P.IaError) as ei:
        P.ia_create(I.config0().params, 0)
    assert ei.value.code == P.IA_EDEVICE
    with pytest.raises(P.IaError):
        P.Context(I.config0().params)
    with pytest.raises(P.IaError):
        P.ia_fp64_peak(0, 10.0)


def test_product_path_does_not_import_the_oracle():
    """Nothing under paper_2509_15117_b200/ (nor ia_inputs) may import, read or link oracle/."""
    for base in ("paper_2509_15117_b200", "ia_inputs", "include"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, base)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                    src = open(os.path.join(dirpath, f)).read()
                    assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), (dirpath, f)
                    assert "ia_oracle" not in src, (dirpath, f)
