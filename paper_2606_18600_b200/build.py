"""Build libshuntstage.so in-tree with nvcc for sm_100a (no torch extension machinery: the boundary is a C-ABI)."""
from __future__ import annotations

import os
import subprocess
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libshuntstage.so"
SOURCES = ["gemm_tcgen05.cu", "attn_decode.cu", "attn_prefill.cu", "elementwise.cu", "stage.cu", "op_static.cu"]
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
         "--use_fast_math=false"]


def _stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + list(CSRC.glob("*.h")) + \
        [HERE.parent / "include" / "shuntstage.h"]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    flags = [f for f in FLAGS if not f.startswith("--use_fast_math")] + os.environ.get("SS_NVCC_EXTRA", "").split()
    objs = []
    procs = []
    (HERE / "build").mkdir(exist_ok=True)
    for src in SOURCES:
        obj = HERE / "build" / (src + ".o")
        cmd = [nvcc, *flags, "-c", str(CSRC / src), "-o", str(obj)]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(str(obj))
    for cmd, p in procs:
        out, _ = p.communicate()
        if verbose and out:
            print(out)
        if p.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd) + "\n" + (out or ""))
    link = [nvcc, "-shared", "-o", str(LIB), *objs]  # static cudart: no runtime library-path dependency
    subprocess.run(link, check=True)
    return LIB


PLACE_LIB = HERE / "libshuntplace.so"


def build_placement(force: bool = False) -> Path:
    """libshuntplace.so: the host-only estimator + placement optimizer (csrc/placement.cpp), plain g++."""
    src = CSRC / "placement.cpp"
    hdr = HERE.parent / "include" / "shuntplace.h"
    if not force and PLACE_LIB.exists() and PLACE_LIB.stat().st_mtime >= max(src.stat().st_mtime, hdr.stat().st_mtime):
        return PLACE_LIB
    cmd = [os.environ.get("CXX", "g++"), "-O2", "-std=c++17", "-fPIC", "-shared", "-Wall", str(src), "-o", str(PLACE_LIB)]
    subprocess.run(cmd, check=True)
    return PLACE_LIB


if __name__ == "__main__":
    print(build_placement(force=True))
    print(build(force=True, verbose=True))
