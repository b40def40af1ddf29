"""Builds libia_b200.so (the C-ABI library of include/ia.h) in-tree with nvcc for sm_100a.

    python -m paper_2509_15117_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  ia_kernels.cu is compiled with -fmad=false: the compiler never
contracts on its own, every fused operation is an explicit fma() in the source (csrc/ia_dev.cuh), so the
one-lane and three-lane layouts -- and the "fmad off" verification variant BASELINE.json's north_star
asks for -- differ only where the source says so.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
ROOT = HERE.parent
LIB = HERE / "libia_b200.so"

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v", *ARCH]
UNITS = [  # (source, extra flags)
    ("ia_kernels.cu", ["-fmad=false"]),
    ("ia_peak.cu", []),
    ("ia_api.cu", []),
]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and Path(cand).exists():
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built (there is no CPU fallback)")


def sources() -> list:
    return sorted(CSRC.glob("*.cu")) + sorted(CSRC.glob("*.cuh")) + [ROOT / "include" / "ia.h"]


def stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(s.stat().st_mtime > t for s in sources())


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not stale():
        return LIB
    cc = nvcc()
    objdir = HERE / "build"
    objdir.mkdir(exist_ok=True)
    objs = []
    log = []
    for src, extra in UNITS:
        obj = objdir / (Path(src).stem + ".o")
        cmd = [cc, *COMMON, *extra, "-c", str(CSRC / src), "-o", str(obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        log.append("$ " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + log[-1])
        objs.append(str(obj))
    tmp = LIB.with_suffix(f".{os.getpid()}.tmp")
    cmd = [cc, "-shared", *ARCH, "-o", str(tmp), *objs]
    r = subprocess.run(cmd, capture_output=True, text=True)
    log.append("$ " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + log[-1])
    os.replace(tmp, LIB)
    (objdir / "build.log").write_text("\n".join(log))
    if verbose:
        print("\n".join(log))
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="--verbose" in sys.argv)
    print(LIB)
