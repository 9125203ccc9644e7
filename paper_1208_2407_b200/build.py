"""Build libts.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1208_2407_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
INCLUDE = PKG.parent / "include"
LIB = PKG / "libts.so"
# (source, object stem, extra flags); ts_stream.cu is compiled once per dtype so that its kernel
# instantiations build in parallel
SOURCES = ["ts_api.cu", "ts_generic.cu", "ts_fused.cu", "ts_stream.cu", "ts_tiny.cu", "ts_axis.cu",
           "ts_noalloc.cu"]
UNITS = [("ts_api.cu", "ts_api", []), ("ts_generic.cu", "ts_generic", []),
         ("ts_fused.cu", "ts_fused", []), ("ts_tiny.cu", "ts_tiny", []),
         ("ts_axis.cu", "ts_axis", []), ("ts_noalloc.cu", "ts_noalloc", []),
         ("ts_stream.cu", "ts_stream_f32", ["-DTS_STREAM_TU=32"]),
         ("ts_stream.cu", "ts_stream_f64", ["-DTS_STREAM_TU=64"])]
HEADERS = [CSRC / "ts_internal.h", CSRC / "ts_rows.cuh", CSRC / "ts_tma.cuh", INCLUDE / "ts.h"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or Path(cand).exists()):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = [CSRC / s for s in SOURCES] + HEADERS + [Path(__file__)]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    nvcc = _nvcc()
    flags = list(NVCC_FLAGS)
    if verbose:
        flags += ["-Xptxas", "-v"]
    objs = []
    procs = []
    for s, stem, extra in UNITS:
        obj = CSRC / (stem + ".o")
        cmd = [nvcc, *flags, *extra, "-I", str(INCLUDE), "-I", str(CSRC), "-c", str(CSRC / s),
               "-o", str(obj)]
        procs.append((cmd, subprocess.Popen(cmd)))
        objs.append(str(obj))
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [nvcc, "-shared", "-o", str(tmp), *objs, "-gencode", "arch=compute_100a,code=sm_100a"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
