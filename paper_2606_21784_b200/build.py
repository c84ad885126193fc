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


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    _compile(LIB, SOURCES, [], verbose)
    # the bench library resolves ks_run from the product library beside it ($ORIGIN)
    _compile(BENCH_LIB, BENCH_SOURCES, ["-L" + HERE, "-l:libkineticsim.so", "-Xlinker", "-rpath=$ORIGIN"], verbose)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
