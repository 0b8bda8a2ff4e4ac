"""Builds libdg.so (the C-ABI CUDA library) in-tree for sm_100a with nvcc.

    python -m paper_1602_07997_b200.build [--force] [--jobs J]

One object per (model, degree) pair from csrc/stage_inst.cu, plus csrc/dg_api.cu and
csrc/host_setup.cpp; objects live in csrc/build/ (git-ignored), the library next to this file.
"""
from __future__ import annotations

import argparse
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libdg.so")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "--use_fast_math=false"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _newer(target: str, deps: list[str]) -> bool:
    if not os.path.exists(target):
        return False
    t = os.path.getmtime(target)
    return all(os.path.getmtime(d) <= t for d in deps)


def _run(cmd: list[str]) -> None:
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("build failed: " + " ".join(cmd) + "\n" + r.stdout + r.stderr)


def build(force: bool = False, jobs: int | None = None, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()
    flags = [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")]
    if os.environ.get("DG_PROF"):          # development: role timeline counters in the variant-4 kernel
        flags.append("-DDG_PROF")
    hdrs = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".hpp", ".h")))
    hdrs += [os.path.join(HERE, "..", "include", "dg.h"), os.path.abspath(__file__)]
    tasks = []
    objs = []
    for model in (0, 1):
        for N in range(1, 11):
            o = os.path.join(OBJ, f"stage_{model}_{N}.o")
            objs.append(o)
            src = os.path.join(CSRC, "stage_inst.cu")
            if force or not _newer(o, [src] + hdrs):
                tasks.append([nvcc, *ARCH, *flags, f"-DDG_MODEL={model}", f"-DDG_N={N}", "-c", src, "-o", o])
    for name in ("dg_api.cu", "host_setup.cpp", "partition.cpp"):
        src = os.path.join(CSRC, name)
        o = os.path.join(OBJ, name.rsplit(".", 1)[0] + ".o")
        objs.append(o)
        if force or not _newer(o, [src] + hdrs):
            tasks.append([nvcc, *ARCH, *flags, "-c", src, "-o", o])
    if tasks:
        if verbose:
            print(f"[build] compiling {len(tasks)} objects", file=sys.stderr)
        with ThreadPoolExecutor(max_workers=jobs or os.cpu_count() or 4) as ex:
            list(ex.map(_run, tasks))
    if tasks or not os.path.exists(LIB):
        _run([nvcc, *ARCH, "-shared", "-o", LIB, *objs, "-lcudart"])
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--jobs", type=int, default=None)
    a = ap.parse_args()
    print(build(a.force, a.jobs, verbose=True))
