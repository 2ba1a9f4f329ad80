"""Build libbg.so (the CUDA library behind include/bg.h) in-tree with nvcc for sm_100a.

Every translation unit is compiled to an object file under csrc/build/ (in parallel, only when it or a header is
newer than its object) and the objects are linked into libbg.so."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(_HERE, "libbg.so")
SOURCES = ["bg_api.cu", "bg_generic.cu", "bg_cobg_generic.cu", "bg_cdbg_prog.cu", "bg_cdbg_prog_dd.cu", "bg_program.cpp",
           "bg_cobg_shared.cu", "bg_cdbg_dd.cu", "bg_generate.cu", "bg_colour_probe.cu", "bg_static.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]
NVCC_FLAGS += os.environ.get("BG_NVCC_EXTRA", "").split()      # e.g. extra -D switches of an experiment
if os.environ.get("BG_BOUNDS_CHECK"):      # debug build: every interpreter state access is range-checked (traps)
    NVCC_FLAGS.insert(0, "-DBG_BOUNDS_CHECK")


def _header_mtime() -> float:
    t = 0.0
    for d in (CSRC, os.path.join(os.path.dirname(_HERE), "include")):
        for f in os.listdir(d):
            if f.endswith((".h", ".cuh")):
                t = max(t, os.path.getmtime(os.path.join(d, f)))
    return t


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    hdr = _header_mtime()
    jobs = []
    objs = []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(OBJ, os.path.splitext(s)[0] + ".o")
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(hdr, os.path.getmtime(src)):
            cmd = ["nvcc", *NVCC_FLAGS, "-c", src, "-o", obj]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            jobs.append(cmd)
    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as pool:
            for rc in pool.map(subprocess.call, jobs):
                if rc != 0:
                    raise subprocess.CalledProcessError(rc, "nvcc")
    if jobs or not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        subprocess.check_call(["nvcc", *NVCC_FLAGS, "-shared", "-o", LIB, *objs])
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="-f" in sys.argv, verbose="-v" in sys.argv))
