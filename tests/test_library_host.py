"""Host-side checks of the C-ABI library that need no GPU: it builds for sm_100a, loads, exports
every symbol the headers declare (and nothing else), validates arguments before touching CUDA,
fails loudly without a device, and its fp64 derivation agrees with the oracle's on equal integers."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

from paper_2606_21784_b200 import binding, build
from paper_2606_21784_b200.workloads import CONFIGS, zi_params

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def _declared(header):
    src = open(os.path.join(ROOT, "include", header)).read()
    return re.findall(r"KS_API\s+[\w\s\*]+?\b(ks_\w+)\s*\(", src)


def _exported(path):
    out = subprocess.check_output(["nm", "-D", "--defined-only", path]).decode()
    return {l.split()[-1] for l in out.splitlines() if " T " in l and l.split()[-1].startswith("ks_")}


def test_headers_declare_what_the_binding_lists():
    assert sorted(_declared("kineticsim.h")) == sorted(binding.EXPORTS)
    assert sorted(_declared("kineticsim_bench.h")) == sorted(binding.BENCH_EXPORTS)


def test_libraries_export_every_declared_symbol(lib):
    """The product library exports exactly include/kineticsim.h, the bench library exactly
    include/kineticsim_bench.h (ablation + microbenchmarks live OUTSIDE the product)."""
    assert _exported(binding.LIB_PATH) == set(_declared("kineticsim.h"))
    assert _exported(binding.BENCH_LIB_PATH) == set(_declared("kineticsim_bench.h"))
    for n in _declared("kineticsim.h"):
        assert getattr(lib, n) is not None
    bench = binding.load_bench()
    for n in _declared("kineticsim_bench.h"):
        assert getattr(bench, n) is not None


def test_product_library_never_allocates_device_memory():
    """include/kineticsim.h: the state buffer is the caller's; the product library holds no
    cudaMalloc / cudaFree call (the bench library may, and says so)."""
    for f in ("ks_api.cu", "ks_kernel.cuh", "ks_device.cuh", "ks_cluster.cuh", "ks_decoupled.cuh", "ks_trace.cuh"):
        src = open(os.path.join(ROOT, "paper_2606_21784_b200", "csrc", f)).read()
        assert not re.search(r"\bcudaMalloc\w*\s*\(|\bcudaFree\s*\(", src), f
    out = subprocess.check_output(["nm", "-D", "--undefined-only", binding.LIB_PATH]).decode()
    assert "cudaMalloc" not in out


def test_library_is_sm100a_with_shared_atomics():
    """The cubin inside the library targets sm_100a and the persistent kernel uses ATOMS (shared
    atomics) and REDUX (warp reductions) -- i.e. the hot path is in the kernel, not on the host."""
    out = subprocess.check_output(["cuobjdump", "-sass", binding.LIB_PATH]).decode()
    assert "sm_100a" in out
    body = out.split("ks_persistent_kernel")[1]
    assert "ATOMS" in body and "REDUX" in body and "IMAD.WIDE.U32" in body


def test_hot_loops_execute_the_multiplies_bench_reports():
    """bench.py turns events/s into executed multiplies/s with EXEC_MULTS_PER_EVENT; count them in
    the SASS of the built library so that the constants cannot go stale: per unrolled hot loop (4
    events, or 2 PACKED4 blocks of 4 agents), IMAD.WIDE.U32 + IMAD.HI.U32 per event."""
    import bench
    from ks_testlib import sass_innermost_loops
    sass = subprocess.check_output(["cuobjdump", "-sass", binding.LIB_PATH]).decode()
    per = bench.EXEC_MULTS_PER_CLASS

    def hot(kernel, min_atoms):
        return [l for l in sass_innermost_loops(sass, kernel) if l["atoms"] >= min_atoms]

    zi = hot("ks_persistent_kernelILi0ELi0ELb0EEE", 4)                 # no-clamp and clamp noise loops
    assert len(zi) == 2 and {l["mults"] / 4 for l in zi} == {per["noise"]} == {bench.EXEC_MULTS_PER_EVENT["zi"]}
    assert all(l["atoms"] == 4 for l in zi)
    mix = hot("ks_persistent_kernelILi1ELi0ELb0EEE", 4)                # noise / maker / momentum x no-clamp / clamp
    assert len(mix) == 6
    assert {l["mults"] / 4 for l in mix} == {per["noise"], per["maker"], per["momentum"]}
    assert min(l["mults"] for l in mix if l["atoms"] == 8) / 4 == per["maker"]          # the no-clamp maker loop
    pk = hot("ks_persistent_kernelILi0ELi0ELb1EEE", 8)                 # 2 blocks x 4 agents per iteration
    assert len(pk) == 2 and {l["mults"] / 8 for l in pk} == {bench.EXEC_MULTS_PER_EVENT["zi_packed4"]}
    assert bench.EXEC_MULTS_PER_EVENT["zi_packed4"] == per["packed_block"] / 4 + 2
    pm = hot("ks_persistent_kernelILi1ELi0ELb1EEE", 8)                 # three block classes x no-clamp / clamp
    assert len(pm) == 6 and sum(l["mults"] for l in pm) / (6 * 8) == pytest.approx(bench.EXEC_MULTS_PER_EVENT["mix3_packed4"])
    # the decoupled kernel with two steps per pass: the step-independent rounds are shared (18 per event);
    # the single-step loops of the run's last, partial group keep 19
    dp = [l for l in hot("ks_decoupled_kernelILb0ELi1ELi4ELi160ELi7ELi2ELb0EEE", 4) if l["atoms"] == 4]
    assert {l["mults"] / 4 for l in dp} == {per["noise_pair"], per["noise"]}
    # the three-type population under the decoupled kernel: noise 18, maker 13 (one bin, one atomic),
    # momentum 18 per event in the pair loops; 19 / 14 / 19 in the single-step loops of a partial group
    dm = hot("ks_decoupled_kernelILb0ELi1ELi4ELi160ELi7ELi2ELb1EEE", 4)
    assert {l["mults"] / 4 for l in dm} == {per["noise_pair"], per["maker_pair"], per["momentum_pair"], per["noise"], per["maker"], per["momentum"]}
    assert min(l["mults"] for l in dm) / 4 == per["maker_pair"]
    pa = hot("ks_persistent_kernelILi2ELi0ELb0EEE", 4)                 # model 4: three classes x no-clamp / clamp
    assert len(pa) == 6
    assert {l["mults"] / 4 for l in pa} == {per["paper_noise"], per["paper_momentum"], per["paper_maker"]}


def test_state_bytes(lib):
    assert binding.ks_state_bytes(1, 64) == 1 * (8 * 64 + 128) + 256
    assert binding.ks_state_bytes(65536, 512) == 65536 * (8 * 512 + 128) + 256
    for M, L in [(0, 64), (1, 48), (1, 16), (-3, 64), (1, 65536)]:
        assert binding.ks_state_bytes(M, L) == 0


def test_argument_validation_precedes_cuda(lib):
    h = C.c_void_p(None)
    P = binding._params(zi_params(8, 10))
    fake = 0x1000   # never dereferenced: every call below must fail before any CUDA work
    assert lib.ks_create(C.byref(h), 1, 64, 256, C.byref(P), 0, None, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_create(None, 1, 64, 256, C.byref(P), 0, fake, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_create(C.byref(h), 1, 48, 256, C.byref(P), 0, fake, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_create(C.byref(h), 0, 64, 256, C.byref(P), 0, fake, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_create(C.byref(h), 1, 64, -1, C.byref(P), 0, fake, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_create(C.byref(h), 1, 64, 256, C.byref(P), 0, fake + 4, None) == binding.KS_ERR_INVALID_ARG
    bad = binding._params(zi_params(8, 0))
    assert lib.ks_create(C.byref(h), 1, 64, 256, C.byref(bad), 0, fake, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_create(C.byref(h), 1, 65536, 256, C.byref(P), 0, fake, None) == binding.KS_ERR_UNSUPPORTED
    assert h.value is None
    assert lib.ks_run(None, 1, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_read_books(None, None, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_set_option(None, 0, 0) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_error_state(None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_attach(C.byref(h), 1, 48, 256, C.byref(P), 0, 0, fake, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_attach(C.byref(h), 1, 64, 256, C.byref(P), 0, 0, None, None) == binding.KS_ERR_INVALID_ARG
    assert b"NULL" in lib.ks_last_error()
    lib.ks_destroy(None)


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p(None)
    P = binding._params(zi_params(8, 10))
    assert lib.ks_create(C.byref(h), 1, 64, 256, C.byref(P), 0, 0x1000, None) == binding.KS_ERR_CUDA
    assert h.value is None and len(lib.ks_last_error()) > 0
    ops, sec = C.c_double(0), C.c_double(0)
    assert binding.load_bench().ks_bench_int_pipe(0, 256, 1, 1, 0, 1, None, C.byref(ops), C.byref(sec)) == binding.KS_ERR_CUDA


def test_derive_stats_matches_oracle_on_equal_integers(lib, oracle):
    c = CONFIGS["C1"]
    _, recs = oracle.run_markets(c.params, c.L, c.A, c.seed, [0, 1, 2], 80)
    recs = np.vstack([recs, oracle.init_state(1, 64)[1]])       # a record with zero steps -> NaNs
    got = binding.ks_derive_stats(recs)
    exp = np.stack([oracle.derived(r) for r in recs])
    assert np.array_equal(np.isnan(got), np.isnan(exp)) and np.isnan(got[-1]).all()
    m = ~np.isnan(exp)
    assert np.all(np.abs(got[m] - exp[m]) <= 1e-12 * np.abs(exp[m]))


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", "/nonexistent/libkineticsim.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.load()
