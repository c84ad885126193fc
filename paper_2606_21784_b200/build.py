"""Build libkineticsim.so (the product) and libkineticsim_bench.so (ablation + roofline
microbenchmarks, linked against the product) for sm_100a, in-tree, with nvcc.
`python -m paper_2606_21784_b200.build [--force] [-v]`."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libkineticsim.so")
BENCH_LIB = os.path.join(HERE, "libkineticsim_bench.so")
SOURCES = ["ks_api.cu"]
BENCH_SOURCES = ["ks_microbench.cu"]
HEADERS = ["ks_device.cuh", "ks_kernel.cuh", "ks_cluster.cuh", "ks_decoupled.cuh", "ks_trace.cuh", os.path.join("..", "..", "include", "kineticsim.h"),
           os.path.join("..", "..", "include", "kineticsim_bench.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC,-fvisibility=hidden", "-shared", "-cudart", "static"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def is_stale() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(BENCH_LIB):
        return True
    t = min(os.path.getmtime(LIB), os.path.getmtime(BENCH_LIB))
    deps = [os.path.join(CSRC, f) for f in SOURCES + BENCH_SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(out: str, sources, extra, verbose: bool) -> None:
    tmp = out + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp] + [os.path.join(CSRC, f) for f in sources] + extra
    subprocess.check_call(cmd)
    os.replace(tmp, out)


DEBUG_LIB = os.path.join(HERE, "libkineticsim_dbg.so")


DEBUG_INJECT_LIB = os.path.join(HERE, "libkineticsim_dbg_inject.so")


def build_debug_checks(verbose: bool = False, inject_race: bool = False) -> str:
    """The same library compiled with -DKS_DEBUG_CHECKS (ks_device.cuh): device-side bounds and
    phase-structure checks that trap on failure.  Loaded instead of the product library by setting
    KINETICSIM_LIB to its path (tests/test_gpu_parity.py::test_debug_checks_build).
    inject_race: the negative control -- additionally drops barrier B1 of the persistent kernel
    (-DKS_DEBUG_INJECT_RACE), which the checks must catch."""
    out = DEBUG_INJECT_LIB if inject_race else DEBUG_LIB
    tmp = out + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + ["-DKS_DEBUG_CHECKS"] + (["-DKS_DEBUG_INJECT_RACE"] if inject_race else []) + \
          (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + [os.path.join(CSRC, f) for f in SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, out)
    return out


def debug_is_stale(path: str) -> bool:
    if not os.path.exists(path):
        return True
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > os.path.getmtime(path) for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    _compile(LIB, SOURCES, [], verbose)
    # the bench library resolves ks_run from the product library beside it ($ORIGIN)
    _compile(BENCH_LIB, BENCH_SOURCES, ["-L" + HERE, "-l:libkineticsim.so", "-Xlinker", "-rpath=$ORIGIN"], verbose)
    return LIB


def build_all(force: bool = True) -> None:
    """Product + bench libraries and the two KS_DEBUG_CHECKS builds, the three independent nvcc runs
    side by side (each is one translation unit of ~75 s)."""
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(3) as ex:
        jobs = [ex.submit(build, force), ex.submit(build_debug_checks), ex.submit(build_debug_checks, False, True)]
        for j in jobs:
            j.result()


if __name__ == "__main__":
    if "--debug-checks" in sys.argv:
        print(build_debug_checks(verbose="-v" in sys.argv))
        print(build_debug_checks(verbose="-v" in sys.argv, inject_race=True))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
