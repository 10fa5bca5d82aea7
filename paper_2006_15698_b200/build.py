"""Build libdg_b200.so (the C-ABI library of include/dg_b200.h) in-tree with nvcc for sm_100a.

One translation unit per N = p+1 (csrc/dg_kernels.cu with -DDG_N=<N>) plus the boundary
(csrc/dg_api.cu) and the allocation-free wavespeed call (csrc/dg_noalloc.cu), compiled in parallel, linked into paper_2006_15698_b200/libdg_b200.so.
ptxas resource usage (-Xptxas -v) of every TU is kept in build/ptxas_N<N>.log.

Usage:  python -m paper_2006_15698_b200.build [--force] [--all-variants]
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
BUILD = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libdg_b200.so")
NS = [2, 3, 4, 5, 6, 7, 8]

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v", "-fmad=true",
]


INCLUDE = os.path.join(os.path.dirname(HERE), "include")
# what each translation unit includes (a change to the public header does not touch the seven kernel objects)
DEPS_KERNELS = [os.path.join(CSRC, f) for f in ("dg_kernels.cu", "dg_internal.h")]
DEPS_API = [os.path.join(CSRC, f) for f in ("dg_api.cu", "dg_internal.h")] + [
    os.path.join(INCLUDE, f) for f in ("dg_b200.h", "dg_b200_test.h")]
DEPS_NOALLOC = [os.path.join(CSRC, "dg_noalloc.cu"), os.path.join(INCLUDE, "dg_b200.h")]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(args):
    obj, cmd, log = args
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {obj}:\n{r.stdout}\n{r.stderr}")
    return obj


def build(force=False, verbose=False, all_variants=False):
    """Compile what is stale; return the path of the shared library.  all_variants=True also compiles the stage-kernel
    variants that only dg_set_variant can reach (-DDG_ALL_VARIANTS; for bench.py --sweep-variants): 48 instead of 30
    variants, a 41 MB instead of a 25 MB library.  Switching between the two needs force=True."""
    os.makedirs(BUILD, exist_ok=True)
    jobs, objs = [], []
    for n in NS:
        obj = os.path.join(BUILD, f"dg_kernels_N{n}.o")
        objs.append(obj)
        if force or _stale(obj, DEPS_KERNELS):
            cmd = ["nvcc"] + NVCC_FLAGS + (["-DDG_ALL_VARIANTS"] if all_variants else []) + [f"-DDG_N={n}", "-c", os.path.join(CSRC, "dg_kernels.cu"), "-o", obj]
            jobs.append((obj, cmd, os.path.join(BUILD, f"ptxas_N{n}.log")))
    obj = os.path.join(BUILD, "dg_api.o")
    objs.append(obj)
    if force or _stale(obj, DEPS_API):
        cmd = ["nvcc"] + NVCC_FLAGS + ["-c", os.path.join(CSRC, "dg_api.cu"), "-o", obj]
        jobs.append((obj, cmd, os.path.join(BUILD, "ptxas_api.log")))
    # dg_max_wavespeed_noalloc: its own translation unit (holds the static __device__ scratch array)
    obj = os.path.join(BUILD, "dg_noalloc.o")
    objs.append(obj)
    if force or _stale(obj, DEPS_NOALLOC):
        cmd = ["nvcc"] + NVCC_FLAGS + ["-c", os.path.join(CSRC, "dg_noalloc.cu"), "-o", obj]
        jobs.append((obj, cmd, os.path.join(BUILD, "ptxas_noalloc.log")))
    if jobs:
        if verbose:
            print(f"compiling {len(jobs)} translation units for sm_100a ...", flush=True)
        with ThreadPoolExecutor(max_workers=min(8, len(jobs))) as ex:
            list(ex.map(_compile, jobs))
    if jobs or force or _stale(LIB, objs):
        cmd = ["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs
        if verbose:
            print(" ".join(cmd), flush=True)
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv or "--all-variants" in sys.argv, verbose=True,
                all_variants="--all-variants" in sys.argv))
