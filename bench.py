#!/usr/bin/env python
"""bench.py -- agent events/s of the call-auction hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]
                    [--scaling weak|strong] [--rng literal|packed4] [--no-extras]
    python bench.py --case NAME [--S n] [--M m] [--mode persistent|stepwise|traced|state_io]   # one run, for ncu

A "step" is one pass of the whole hot path over one batch: ks_create (state init) + ONE ks_run of
all S steps of the workload (a0-a7).  Workload: BASELINE.json configs[3] ("throughput scale", C4:
M=65536, L=512, A=4096, S=1000, seed 3), the largest config and the one the metric's roofline
clause is quoted on.  N > 1: one process per GPU (the driver launches torchrun; a plain
`python bench.py --gpus N` re-executes itself under torch.distributed.run), markets sharded by
market_base, no data-path collective.  Prints ONE JSON line (rank 0).  DESIGN.md 7 explains every
field.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_21784_b200.workloads import (CONFIGS, KS_MODEL_PAPER, KS_MODEL_ZI, packed4, paper_params,  # noqa: E402
                                             sampled_markets, shard_markets, zi_params)

# Roofline of the headline kernel: the fmaheavy pipe that executes the 32x32->64
# multiplies.  Algorithmic multiplies per agent event: 20 of Philox4x32-10 + the
# mulhi draws of the rule (noise/momentum: offset and quantity; maker: spread only).
ALG_MULTS_PER_EVENT = {"zi": 22.0, "mix3": (22.0 + 21.0 + 22.0) / 3.0,
                       # PACKED4 (A22): a Philox block per 4 agents + the rule's multiply-extract draws
                       "zi_packed4": 20.0 / 4 + 2.0, "mix3_packed4": 20.0 / 4 + (2.0 + 1.0 + 2.0) / 3.0,
                       # model 4 (A24): 20 of Philox + offset and quantity (momentum / maker: quantity only)
                       "paper": 0.70 * 22.0 + 0.30 * 21.0}
# Multiplies the kernel actually issues per event (IMAD.WIDE.U32 + IMAD.HI.U32 per ATOMS in the
# hot loops).  tests/test_library_host.py counts them in the SASS of the built library, so these
# constants cannot go stale silently.
EXEC_MULTS_PER_CLASS = {"noise": 19.0, "maker": 14.0, "momentum": 19.0,                 # literal contract (a%3 classes)
                        "noise_pair": 18.0,      # decoupled kernel, two steps per pass: rounds 0-2's step-independent products shared
                        "maker_pair": 13.0, "momentum_pair": 18.0,
                        "paper_noise": 19.0, "paper_momentum": 18.0, "paper_maker": 16.0,   # model 4 (all four words)
                        "packed_block": 17.0}                                               # one Philox block of 4 agents
EXEC_MULTS_PER_EVENT = {"zi": 19.0, "mix3": (19.0 + 14.0 + 19.0) / 3.0,
                        "zi_packed4": 17.0 / 4 + 2.0, "mix3_packed4": 17.0 / 4 + (2.0 + 1.0 + 2.0) / 3.0,
                        # model 4 at the mix bench.py times (case model4_C4shape: 70 % noise, 15 % momentum, 15 % makers)
                        "paper": 0.70 * 19.0 + 0.15 * 18.0 + 0.15 * 16.0}
# derived peak: a 32-lane IMAD.WIDE/IMAD.HI occupies an SMSP's fmaheavy pipe for 4 cycles -> 8 lanes/clk/SMSP
WIDE_MUL_LANES_PER_SM_PER_CLK = 4 * 8
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the headline kernel from the
# `ncu --set full` capture summarised under profiles/ (None until measured for that config).
PROFILED_DRAM_BYTES_PER_LAUNCH = {"C4": 26893824 + 238403072,            # profiles/r2d_c4_full.md
                                  "C4_packed4": 22112512 + 253766400}    # profiles/r2c_c4_packed4_full.md


def exec_mults(params: dict, plan: str) -> float:
    """Executed multiplies per event of the kernel the library's plan names (ks_plan_string)."""
    mk = model_key(params)
    if mk == "zi" and "steps_per_pass=2" in plan:
        return EXEC_MULTS_PER_CLASS["noise_pair"]
    if mk == "mix3" and "steps_per_pass=2" in plan:
        return (EXEC_MULTS_PER_CLASS["noise_pair"] + EXEC_MULTS_PER_CLASS["maker_pair"] + EXEC_MULTS_PER_CLASS["momentum_pair"]) / 3.0
    return EXEC_MULTS_PER_EVENT[mk]


def model_key(params: dict) -> str:
    if params["model"] == KS_MODEL_PAPER:
        return "paper"
    return ("zi" if (params["model"] & 1) == KS_MODEL_ZI else "mix3") + ("_packed4" if params["model"] >= 2 else "")


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.1):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.stop_flag = threading.Event()
        self.sm, self.reasons, self.sm_max, self.err = [], set(), None, None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.sm_max = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {
                nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
                nv.nvmlClocksThrottleReasonApplicationsClocksSetting: "applications_clocks_setting",
            }
            while not self.stop_flag.is_set():
                self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                self.stop_flag.wait(self.period)
        except Exception as e:  # NVML missing: report it, do not fail the bench
            self.err = repr(e)

    def result(self):
        self.stop_flag.set()
        self.join(timeout=2)
        med = float(np.median(self.sm)) if self.sm else None
        out = {"sm_mhz": med, "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons), "samples": len(self.sm)}
        if self.err:
            out["error"] = self.err
        return out


def physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ---------------------------------------------------------------------------------------------
# Multi-GPU launch logic: one process per GPU.  Pure function of the arguments
# and the environment so that tests/test_bench_launch.py can check it without a GPU.
# ---------------------------------------------------------------------------------------------
def launch_plan(gpus: int, env: dict, n_visible, argv, impl: str = "ours"):
    """-> ("run", rank, local_rank, world) when this process is a rank (or the single-GPU run),
          ("spawn", cmd) when `--gpus N > 1` was given WITHOUT torchrun: re-execute under
          torch.distributed.run with N ranks on 127.0.0.1,
          ("error", message) when the request cannot be honoured -- bench.py then exits non-zero
          instead of printing a line whose n_gpus differs from --gpus."""
    if gpus < 1:
        return ("error", "--gpus must be >= 1")
    if "WORLD_SIZE" in env:
        world = int(env["WORLD_SIZE"])
        rank, local_rank = int(env.get("RANK", "0")), int(env.get("LOCAL_RANK", env.get("RANK", "0")))
        if world != gpus:
            return ("error", "WORLD_SIZE=%d but --gpus %d: launch torchrun with --nproc-per-node %d" % (world, gpus, gpus))
        if not 0 <= rank < world:
            return ("error", "RANK=%d outside [0, %d)" % (rank, world))
        if impl == "ours" and n_visible is not None and local_rank >= n_visible:
            return ("error", "LOCAL_RANK=%d but only %d CUDA device(s) are visible" % (local_rank, n_visible))
        return ("run", rank, local_rank, world)
    if gpus == 1 or impl == "reference":       # the reference arm is CPU-only: rank 0 alone does the work
        return ("run", 0, 0, 1 if impl == "ours" else gpus)
    if n_visible is not None and n_visible < gpus:
        return ("error", "--gpus %d but only %d CUDA device(s) are visible" % (gpus, n_visible))
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    return ("spawn", cmd)


def rank_markets(cfg_M: int, rank: int, world: int, scaling: str):
    """(market_base, markets of this rank, markets of the whole job).  weak: every GPU runs the
    config's M markets, rank r keyed from r*M; strong: the config's M markets are cut into
    contiguous shards (workloads.shard_markets)."""
    if scaling == "strong":
        base, count = shard_markets(cfg_M, rank, world)
        return base, count, cfg_M
    return rank * cfg_M, cfg_M, world * cfg_M


def time_oracle(cfg, n_markets: int, S: int):
    """The oracle as it stands, one thread, on the first n sampled markets of cfg for S steps."""
    from oracle import ks_oracle
    ids = sampled_markets(cfg.M, cfg.seed, 64)[:n_markets]
    t0 = time.perf_counter()
    ks_oracle.run_markets(cfg.params, cfg.L, cfg.A, cfg.seed, ids, S)
    dt = time.perf_counter() - t0
    return len(ids) * cfg.A * S / dt, dt, len(ids)


def workload_config(cfg, n_gpus, scaling="weak"):
    if scaling == "strong":
        par = "strong: the %d markets cut into %d contiguous shards (workloads.shard_markets), market_base = shard start, no collective" % (cfg.M, n_gpus)
    else:
        par = "weak: %d markets on each of %d GPU(s), market_base = rank*M, no collective" % (cfg.M, n_gpus)
    kind = "paper agent model (model 4)" if cfg.params["model"] == KS_MODEL_PAPER else \
        ("zero-intelligence" if (cfg.params["model"] & 1) == KS_MODEL_ZI else "noise/maker/momentum by a%3") + \
        (", PACKED4 draw contract (NOT the BASELINE.json one; DESIGN.md A22)" if cfg.params["model"] >= 2 else "")
    return {"workload": "%s: BASELINE.json configs[%d] -- M=%d markets%s, L=%d ticks, A=%d agents, S=%d steps, seed=%d, %s"
                        % (cfg.name, int(cfg.name[1]) - 1, cfg.M, "/GPU" if scaling == "weak" else " in all", cfg.L, cfg.A, cfg.S,
                           cfg.seed, kind),
            "M": cfg.M, "L": cfg.L, "A": cfg.A, "S": cfg.S, "seed": cfg.seed, "parallelism": par,
            "l2": ("state buffer %.0f MB per GPU exceeds the 126 MB L2; every timed step (ks_create + ks_run) rewrites all of it"
                   if cfg.M * (8 * cfg.L + 128) > 126e6 else
                   "state buffer %.1f MB per GPU fits the L2, but a fresh ks_run never READS it (ks_create zeroes it, the kernel "
                   "skips the load of an all-zero book): there is no input to keep warm")
                  % (cfg.M * (8 * cfg.L + 128) / 1e6)}


def run_reference(args, cfg, rank: int):
    """--impl reference: this tier's reference arm is the CPU oracle (no GPU, rank 0 only)."""
    if rank != 0:
        return
    from oracle import ks_oracle
    ks_oracle.lib()
    n_mk, S = 4, cfg.S                   # bounded sample per step: 4 sampled markets x all S steps
    if cfg.M < n_mk:
        n_mk = cfg.M
    for _ in range(args.warmup):
        time_oracle(cfg, 1, max(1, S // 10))
    tot_ev, tot_t = 0.0, 0.0
    for _ in range(args.steps):
        ev_s, dt, n = time_oracle(cfg, n_mk, S)
        tot_ev += n * cfg.A * S
        tot_t += dt
    value = tot_ev / tot_t
    sample = "%d sampled markets x S=%d steps of %s per step (%.3g events/step), 1 thread" % (n_mk, S, cfg.name, n_mk * cfg.A * S)
    line = {
        "impl": "reference", "metric": "agent_events_per_s", "value": value, "unit": "events/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
        "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": workload_config(cfg, args.gpus, args.scaling),
        "cpu_baseline": {"value": value, "unit": "events/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
# One named case, timed with CUDA events (extras of the default line and the `--case` mode that
# the ncu / compute-sanitizer commands under profiles/ run).
# ---------------------------------------------------------------------------------------------
def case_config(name: str):
    """Named cases: C1..C5, C4_packed4, C5_packed4, model4_C4shape (the paper's own agent model on
    the C4 shape, alpha_mom = alpha_maker = 0.15, P_mkt = 0.02), table4 / latency (the paper's own
    shapes with zero-intelligence agents: context), cluster (L = 32768 on a 2-CTA cluster)."""
    from paper_2606_21784_b200.workloads import Config, mix3_params
    if name in CONFIGS:
        return CONFIGS[name]
    if name.endswith("_packed4") and name[:-8] in CONFIGS:
        c = CONFIGS[name[:-8]]
        return dataclasses.replace(c, name=name, params=packed4(c.params))
    if name == "model4_C4shape":
        c = CONFIGS["C4"]
        return dataclasses.replace(c, name=name, params=paper_params(c.A, 0.15, 0.15, delta=32, qmax=100, half_spread=2, p_mkt=0.02))
    if name == "table4":
        return Config(name, 8192, 128, 256, 500, 5, zi_params(8, 10))
    if name == "latency":
        return Config(name, 4096, 128, 256, 500, 5, zi_params(8, 10))
    if name == "cluster":
        return Config(name, 64, 32768, 4096, 200, 6, mix3_params())
    raise SystemExit("bench.py: unknown case %r" % name)


def time_case(ks, torch, dev, c, *, reps=3, mode="persistent", S=None, M=None, opts=(), warm=1):
    """Median device time (ms) of ks_run(S) on config c (ks_create outside the events)."""
    M = M or c.M
    S = S or c.S
    st = torch.empty(ks.ks_state_bytes(M, c.L), dtype=torch.uint8, device=dev)
    tr = torch.empty((M, S, 2), dtype=torch.int32, device=dev) if mode == "traced" else None
    ts = []
    for i in range(warm + reps):
        sim = ks.KsSim(M, c.L, c.A, c.params, c.seed, state=st)
        try:
            for o, v in opts:
                sim.ks_set_option(o, v)
            plan = sim.ks_plan_string()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            if mode == "stepwise":
                sim.ks_run_stepwise(S)
            elif mode == "traced":
                sim.ks_run_traced(S, tr)
            else:
                sim.ks_run(S)
            b.record()
            torch.cuda.synchronize()
            sim.ks_error_state()
            ts.append(a.elapsed_time(b))
        finally:
            sim.ks_destroy()
    ms = float(np.median(ts[warm:]))
    return {"ms": ms, "events_per_s": float(M) * c.A * S / (ms * 1e-3), "M": M, "L": c.L, "A": c.A, "S": S, "reps": reps,
            "plan": plan}


def time_state_io(ks, torch, dev, c, hbm_peak_gbs, reps=5, warm_steps=8, threads=0):
    """a0 + a7 alone (north_star: "HBM peak for the book load and store"; Eq.6): the
    config's own resting books after `warm_steps` real steps, resident in HBM; then a handle with NO
    agents attached to that state (ks_attach) runs ONE step -- the launch loads every book and
    record, clears an already uncrossed book (nothing trades) and stores them again.
    Bytes = 2 * M * (8L + 128).  Median device time of `reps` launches, CUDA events."""
    M, L = c.M, c.L
    st = torch.empty(ks.ks_state_bytes(M, L), dtype=torch.uint8, device=dev)
    sim = ks.KsSim(M, L, c.A, c.params, c.seed, state=st)
    sim.ks_run(warm_steps)
    torch.cuda.synchronize()
    sim.ks_error_state()
    sim.ks_destroy()
    ts, plan = [], ""
    for i in range(1 + reps):
        sim = ks.KsSim(M, L, 0, c.params, c.seed, state=st, attach=True)      # synchronises
        try:
            if threads:
                sim.ks_set_option(ks.KS_OPT_BLOCK_THREADS, threads)
            plan = sim.ks_plan_string()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); sim.ks_run(1); b.record()
            torch.cuda.synchronize()
            sim.ks_error_state()
            ts.append(a.elapsed_time(b))
        finally:
            sim.ks_destroy()
    ms = float(np.median(ts[1:]))
    nbytes = 2 * M * (8 * L + 128)
    return {"ms": ms, "bytes": nbytes, "GBps": nbytes / (ms * 1e-3) / 1e9, "frac_of_hbm": nbytes / (ms * 1e-3) / 1e9 / hbm_peak_gbs,
            "plan": plan}


def time_e2e_small(ks, torch, dev, c, reps=20):
    """End to end through the C ABI with HOST buffers for a latency-regime config: opening books H2D
    from pinned memory, ks_run(S), books + records D2H into pinned memory.  Host clock around the
    calls and the final synchronize (what a caller waits), CUDA events beside it; medians."""
    M, L = c.M, c.L
    st = torch.empty(ks.ks_state_bytes(M, L), dtype=torch.uint8, device=dev)
    h_open = torch.zeros((M, 2, L), dtype=torch.int32).pin_memory()
    h_books = torch.empty((M, 2, L), dtype=torch.int32).pin_memory()
    h_recs = torch.empty((M, 16), dtype=torch.int64).pin_memory()
    host_ms, dev_ms = [], []
    for i in range(3 + reps):
        sim = ks.KsSim(M, L, c.A, c.params, c.seed, state=st)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        a.record()
        sim.ks_write_books(h_open); sim.ks_run(c.S); sim.ks_read_books(h_books); sim.ks_read_stats(h_recs)
        b.record()
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        sim.ks_destroy()
        if i >= 3:
            host_ms.append((t1 - t0) * 1e3)
            dev_ms.append(a.elapsed_time(b))
    hm, dm = float(np.median(host_ms)), float(np.median(dev_ms))
    ev = float(M) * c.A * c.S
    return {"host_ms": hm, "device_ms": dm, "events_per_s_host_clock": ev / (hm * 1e-3), "us_per_step_host_clock": hm * 1e3 / c.S,
            "h2d_bytes": int(h_open.numel() * 4), "d2h_bytes": int(h_books.numel() * 4 + h_recs.numel() * 8)}


def run_case(args):
    """--case: ONE timed run of a named case (after one warm-up), a small JSON line."""
    import torch
    from paper_2606_21784_b200 import binding as ks
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    ks.load()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    c = case_config(args.case)
    opts = []
    if args.threads:
        opts.append((ks.KS_OPT_BLOCK_THREADS, args.threads))
    if args.atomic_mode:
        opts.append((ks.KS_OPT_ATOMIC_MODE, args.atomic_mode))
    if args.pipeline:
        opts.append((ks.KS_OPT_PIPELINE, args.pipeline))
    if args.rel_columns:
        opts.append((ks.KS_OPT_REL_COLUMNS, args.rel_columns))
    n0 = ks.ks_launch_count()
    if args.mode == "state_io":
        # the state phase alone (a0 + a7): the launch bench.py's state_io key times
        r = time_state_io(ks, torch, dev, c, 1.0, reps=1, threads=args.threads)
        r.update({"case": c.name, "mode": args.mode, "gpu_launches": ks.ks_launch_count() - n0})
        del r["frac_of_hbm"]
        print(json.dumps(r), flush=True)
        return
    r = time_case(ks, torch, dev, c, reps=1, mode=args.mode, S=args.S, M=args.M, opts=opts)
    if args.trace_stats:
        M, S = r["M"], r["S"]
        tr = torch.zeros((M, S, 2), dtype=torch.int32, device=dev)
        sim = ks.KsSim(M, c.L, c.A, c.params, c.seed)
        sim.ks_run_traced(S, tr)
        ks.ks_trace_stats(tr, M, S, 20)
        torch.cuda.synchronize()
        sim.ks_destroy()
    r.update({"case": c.name, "mode": args.mode, "gpu_launches": ks.ks_launch_count() - n0,
              "hbm_bytes_persistent": float(r["M"]) * (8 * c.L + 128)})
    print(json.dumps(r), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4", choices=sorted(CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = the config's M markets on EVERY GPU (default); strong = the config's M markets "
                         "cut into N contiguous shards (SURVEY.md S8(e))")
    ap.add_argument("--threads", type=int, default=0, help="KS_OPT_BLOCK_THREADS (0 = automatic)")
    ap.add_argument("--atomic-mode", type=int, default=0)
    ap.add_argument("--pipeline", type=int, default=0, help="KS_OPT_PIPELINE (--case only)")
    ap.add_argument("--rel-columns", type=int, default=0, help="KS_OPT_REL_COLUMNS (--case only)")
    ap.add_argument("--rng", default="literal", choices=["literal", "packed4"],
                    help="draw contract: literal = BASELINE.json (one Philox block per agent); packed4 = the "
                         "separately named PACKED4 contract (DESIGN.md A22), reported beside it, never instead of it")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-microbench", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the other configs / contracts / ablation keys")
    ap.add_argument("--all-configs", action="store_true", help="(kept for compatibility: the extras are on by default)")
    ap.add_argument("--case", default=None, help="run ONE named case once and print a small JSON line (ncu / sanitizer helper)")
    ap.add_argument("--mode", default="persistent", choices=["persistent", "stepwise", "traced", "state_io"])
    ap.add_argument("--trace-stats", action="store_true", help="--case: also launch ks_run_traced + ks_trace_stats once")
    ap.add_argument("--S", type=int, default=None, help="--case: override the number of steps")
    ap.add_argument("--M", type=int, default=None, help="--case: override the number of markets")
    args = ap.parse_args()
    if args.case:
        run_case(args)
        return
    cfg = CONFIGS[args.config]
    if args.rng == "packed4":
        cfg = dataclasses.replace(cfg, params=packed4(cfg.params))

    n_visible = None
    if args.impl == "ours":
        import torch
        n_visible = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if n_visible == 0:
            raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    plan = launch_plan(args.gpus, os.environ, n_visible, sys.argv[1:], args.impl)
    if plan[0] == "error":
        print("bench.py: " + plan[1], file=sys.stderr)
        sys.exit(2)
    if plan[0] == "spawn":
        sys.exit(subprocess.call(plan[1]))
    _, rank, local_rank, world = plan

    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    import torch.distributed as dist
    from paper_2606_21784_b200 import binding as ks

    ks.load()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
        if dist.get_world_size() != args.gpus:
            print("bench.py: process group has %d ranks, --gpus %d" % (dist.get_world_size(), args.gpus), file=sys.stderr)
            sys.exit(2)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    L, A, S = cfg.L, cfg.A, cfg.S
    base, M, M_job = rank_markets(cfg.M, rank, world, args.scaling)
    state = torch.empty(ks.ks_state_bytes(M, L), dtype=torch.uint8, device=dev)

    plans = []

    def one_step(ev_pairs=None):
        sim = ks.KsSim(M, L, A, cfg.params, cfg.seed, market_base=base, state=state)
        if args.threads:
            sim.ks_set_option(ks.KS_OPT_BLOCK_THREADS, args.threads)
        if args.atomic_mode:
            sim.ks_set_option(ks.KS_OPT_ATOMIC_MODE, args.atomic_mode)
        if args.pipeline:
            sim.ks_set_option(ks.KS_OPT_PIPELINE, args.pipeline)
        plans.append(sim.ks_plan_string())
        if ev_pairs is not None:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            sim.ks_run(S)
            e1.record()
            ev_pairs.append((e0, e1))
        else:
            sim.ks_run(S)
        return sim

    # ---- warm-up, then K timed steps (device-resident), CUDA events on the launching stream
    for _ in range(args.warmup):
        one_step().ks_destroy()
    barrier()
    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()
    launches0 = ks.ks_launch_count()
    pairs, sims = [], []
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_start.record()
    for _ in range(args.steps):
        sims.append(one_step(pairs))
    t_end.record()
    barrier()
    launches = ks.ks_launch_count() - launches0
    clocks = sampler.result()
    total_ms = t_start.elapsed_time(t_end)
    kern_ms = [a.elapsed_time(b) for a, b in pairs]
    for s_ in sims:
        s_.ks_error_state()
        s_.ks_destroy()
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    events_per_step = float(M) * A * S                    # this rank
    job_events_per_step = float(M_job) * A * S            # all ranks
    value = job_events_per_step * args.steps / (total_ms * 1e-3)

    # ---- end to end through the C ABI with HOST buffers: opening book H2D from pinned memory,
    #      ks_run, books + records D2H into pinned memory, all inside the timed region
    h_open = torch.zeros((M, 2, L), dtype=torch.int32).pin_memory()
    h_books = torch.empty((M, 2, L), dtype=torch.int32).pin_memory()
    h_recs = torch.empty((M, 16), dtype=torch.int64).pin_memory()

    def e2e_step():
        sim = ks.KsSim(M, L, A, cfg.params, cfg.seed, market_base=base, state=state)
        if args.threads:
            sim.ks_set_option(ks.KS_OPT_BLOCK_THREADS, args.threads)
        sim.ks_write_books(h_open)
        sim.ks_run(S)
        sim.ks_read_books(h_books)
        sim.ks_read_stats(h_recs)
        return sim

    e2e_step().ks_destroy()
    barrier()
    e_start, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_e2e = max(1, min(args.steps, 3))
    e_start.record()
    esims = [e2e_step() for _ in range(n_e2e)]
    e_end.record()
    barrier()
    e2e_ms = e_start.elapsed_time(e_end)
    for s_ in esims:
        s_.ks_destroy()
    if world > 1:
        t = torch.tensor([e2e_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_ms = float(t.item())
    e2e_value = job_events_per_step * n_e2e / (e2e_ms * 1e-3)
    # the e2e result is the same simulation: check it against the device-resident run's records
    chk = torch.empty((M, 16), dtype=torch.int64).pin_memory()
    sim = one_step(); sim.ks_read_stats(chk); torch.cuda.synchronize(); sim.ks_destroy()
    assert torch.equal(chk, h_recs), "e2e run and device-resident run disagree"

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- microbenchmarks in the same process (same clocks): the measured multiply-pipe peak, the
    #      BASELINE.json smem-atomic roofline and the generation-only (integer ALU) ceiling
    model = model_key(cfg.params)
    avg_kern_s = float(np.mean(kern_ms)) * 1e-3
    kev = events_per_step / avg_kern_s
    peaks = {}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peaks = json.load(f)
    except Exception:
        pass
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    peak_derived = sms * WIDE_MUL_LANES_PER_SM_PER_CLK * sm_max_mhz * 1e6 / 1e12
    micro, mulwide_peak = None, None
    if not args.no_microbench:
        delta = cfg.params["noise_delta"]
        Lb = min(L, 8192)
        thr = 256
        peak_ops, _ = ks.ks_bench_smem_atomic(0, delta, Lb, thr, 8, 2000)
        pat_ops, _ = ks.ks_bench_smem_atomic(1, delta, Lb, thr, 8, 2000)
        agg_ops, _ = ks.ks_bench_smem_atomic(2, delta, Lb, thr, 8, 500)
        one_ops, _ = ks.ks_bench_smem_atomic(3, delta, Lb, thr, 8, 500)
        gen_M = min(M, sms * 16 * 4)
        gen_S = max(1, min(S, int(2e10 / (gen_M * A))))
        gen_ev, _ = ks.ks_bench_generate_only(cfg.params, gen_M, L, A, gen_S, args.threads or 32)
        wide, _ = ks.ks_bench_int_pipe(0)
        lop, _ = ks.ks_bench_int_pipe(1)
        mix, _ = ks.ks_bench_int_pipe(2)
        mix2, _ = ks.ks_bench_int_pipe(3)
        mix3, _ = ks.ks_bench_int_pipe(4)
        mulwide, _ = ks.ks_bench_int_pipe(5)
        mulwide_peak = mulwide / 1e12
        cyc = lambda ops_s, per: sms * 4 * sm_max_mhz * 1e6 * 32 * per / ops_s      # SMSP cycles per IMAD.WIDE
        atomics_per_event = {"zi": 1.0, "zi_packed4": 1.0, "paper": 1.0}.get(model, 4.0 / 3.0)
        micro = {
            "mul_wide_u32_thread_ops_per_s": mulwide,
            "smem_atomic_peak_lane_ops_per_s": peak_ops, "smem_atomic_pattern_lane_ops_per_s": pat_ops,
            "smem_atomic_pattern_warp_aggregated_lane_ops_per_s": agg_ops, "smem_atomic_same_address_lane_ops_per_s": one_ops,
            "generate_only_events_per_s": gen_ev, "imad_wide_accumulate_thread_ops_per_s": wide, "lop3_thread_ops_per_s": lop,
            "imad_wide_lop3_mix_thread_ops_per_s": mix,
            "smsp_cycles_per_imad_wide": {"mul_wide_alone": cyc(mulwide, 1), "accumulate_alone": cyc(wide, 1),
                                          "with_1_lop3": cyc(mix, 2), "with_2_lop3": cyc(mix2, 3), "with_3_lop3": cyc(mix3, 4)},
            "frac_of_smem_atomic_peak": kev * atomics_per_event / peak_ops,
            "frac_of_smem_atomic_pattern": kev * atomics_per_event / pat_ops,
            "frac_of_generate_only": kev / gen_ev,
        }

    # ---- roofline of the dominant kernel (ks_persistent_kernel): bound by the 32x32->64 multiply pipe
    peak = mulwide_peak if mulwide_peak else peak_derived
    achieved = ALG_MULTS_PER_EVENT[model] * kev / 1e12
    exec_per_event = exec_mults(cfg.params, plans[-1])
    executed = exec_per_event * kev / 1e12
    roofline = {"bound": "alu", "kernel": plans[-1], "achieved": executed, "peak": peak,
                "unit": "T 32x32->64-bit integer multiplies/s", "frac": executed / peak,
                "achieved_algorithmic": achieved, "frac_algorithmic": achieved / peak,
                "traffic": PROFILED_DRAM_BYTES_PER_LAUNCH.get(cfg.name if args.rng == "literal" else cfg.name + "_packed4"),
                "peak_source": ("measured in this process: ks_bench_int_pipe(5), a pure mul.wide.u32 stream "
                                "(include/kineticsim_bench.h)") if mulwide_peak else
                               "derived (microbenchmarks skipped): see peak_derived_source",
                "peak_derived": peak_derived, "frac_of_derived_peak": executed / peak_derived,
                "frac_algorithmic_of_derived_peak": achieved / peak_derived,
                "peak_derived_source": "%d SMs x 4 SMSPs x 8 lanes/clk (IMAD.WIDE = 2 passes of the 16-lane fmaheavy pipe) x %.0f MHz (%s)"
                                       % (sms, sm_max_mhz, "MEASURED_PEAKS.json sm_max_mhz" if peaks else "NVML max clock"),
                "alg_mults_per_event": ALG_MULTS_PER_EVENT[model], "executed_mults_per_event": exec_per_event,
                "avg_launch_ms": avg_kern_s * 1e3,
                "frac_note": "achieved/frac count the multiplies the kernel EXECUTES per event (counted in the SASS by "
                             "tests/test_library_host.py): a utilisation of the multiply pipe, <= 1 (ncu: "
                             "sm__pipe_fmaheavy_cycles_active, profiles/).  achieved_algorithmic/frac_algorithmic count SURVEY.md "
                             "S8(d)'s ALGORITHMIC 22 per event; the kernel executes fewer (19, or 18 when two steps share a pass: "
                             "hoisted / strength-reduced / shared rounds, w3 skipped), so that figure can pass 1.0",
                "hbm": None}
    if micro:
        # BASELINE.json's metric names the smem-atomic roofline: keep its two fractions beside the headline
        roofline["frac_of_smem_atomic_peak"] = micro["frac_of_smem_atomic_peak"]
        roofline["frac_of_smem_atomic_pattern"] = micro["frac_of_smem_atomic_pattern"]

    line = {
        "metric": "agent_events_per_s", "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": args.scaling,
        "vs_baseline": None, "dtype": "int32", "data": "synthetic", "config": workload_config(cfg, world, args.scaling),
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": int(h_open.numel() * 4),
                "d2h_bytes_per_step": int(h_books.numel() * 4 + h_recs.numel() * 8), "steps": n_e2e,
                "ms_per_step": e2e_ms / n_e2e},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "kernel_events_per_s": kev,
        "paper_context": {"events_per_s": 5.47e10, "where": "RTX 5090, M=8192 A=1024 L=128 S=500, PAPER.md:313 (other GPU, other agent model)"},
    }
    # ---- a0/a7 against HBM: the state phase alone (A = 0, S = 1 after ks_write_books) on the C4 and C5 shapes
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    state_io = {name: time_state_io(ks, torch, dev, CONFIGS[name], hbm_peak) for name in ("C4", "C5")}
    # the same with the block size of the plan the config itself runs under (C4: 96, C5: 160 threads)
    state_io["C4_T96"] = time_state_io(ks, torch, dev, CONFIGS["C4"], hbm_peak, threads=96)
    state_io["C5_T160"] = time_state_io(ks, torch, dev, CONFIGS["C5"], hbm_peak, threads=160)
    state_io["peak_GBps"] = hbm_peak
    state_io["peak_source"] = "MEASURED_PEAKS.json hbm_gbs (measured)" if peaks else "fallback (B200_PROFILING.md)"
    state_io["what"] = ("ks_run(S=1) of a handle with A=0 attached to the config's own resting books (8 real steps): book + record load, "
                        "one clearing of an uncrossed book, book + record store; 2*M*(8L+128) bytes, median device time of 5")
    roofline["hbm"] = {"algorithmic_bytes": state_io["C4"]["bytes"], "achieved_GBps": state_io["C4"]["GBps"], "peak_GBps": hbm_peak,
                       "frac": state_io["C4"]["frac_of_hbm"], "peak_source": state_io["peak_source"],
                       "what": "the state phase (a0 + a7) of the C4 shape timed alone, see state_io; inside the 608 ms launch "
                               "it is 0.02 % of the time"}

    detail, tail = {}, {}
    if micro:
        detail["microbench"] = micro
        tail["microbench"] = {"mul_wide_u32_T_per_s": micro["mul_wide_u32_thread_ops_per_s"] / 1e12,
                              "smem_atomic_peak_T_per_s": micro["smem_atomic_peak_lane_ops_per_s"] / 1e12,
                              "smem_atomic_pattern_T_per_s": micro["smem_atomic_pattern_lane_ops_per_s"] / 1e12,
                              "generate_only_events_per_s": micro["generate_only_events_per_s"]}
    if not args.no_extras:
        d_, t_ = extras(ks, torch, dev, peak, cfg, micro)
        detail.update(d_)
        tail.update(t_)
    line["detail"] = detail

    if not args.no_cpu_baseline:
        n_mk = min(cfg.M, 64)
        ev_s, dt, n = time_oracle(cfg, n_mk, S)
        line["cpu_baseline"] = {"value": ev_s, "unit": "events/s", "cores": 1, "kind": "oracle",
                                "sample": "%d seeded sampled markets x S=%d steps of %s (%.3g events, %.1f s), 1 thread of %d host cores"
                                          % (n, S, cfg.name, n * A * S, dt, os.cpu_count() or 0)}
    # compact per-config numbers LAST: the driver's record keeps the tail of the line
    line["state_io"] = state_io
    line.update(tail)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum and the L1 global load + store bytes, summed over the
# launches of one run, from the ncu captures of `bench.py --case C2 --S 1000 [--mode stepwise]`
# (profiles/r2d_traffic.md): measured counters, not algorithmic bytes.
PROFILED_TRAFFIC_C2 = {"persistent": {"dram_bytes": 215040 + 0, "global_load_store_bytes": 131072 + 2228224},
                       "launch_per_step": {"dram_bytes": 2301881088 + 0, "global_load_store_bytes": 2226e6 + 2228e6},
                       "source": "profiles/r2d_traffic.md (ncu; the L2 is invalidated between launches under ncu)"}


def compact(r):
    """{ms, events_per_s, frac_executed, plan} of a timed case, plan shortened."""
    return {"ms": round(r["ms"], 4), "events_per_s": float("%.4g" % r["events_per_s"]), "frac_executed": round(r["frac_executed"], 4),
            "plan": r["plan"].replace("ks_", "").replace("_kernel", "").replace("steps_per_pass", "spp")}


def extras(ks, torch, dev, peak_tmults, headline_cfg, micro):
    """The other BASELINE configs, the other contracts and the ablation, timed in the same process
    (each a few ms to a few hundred ms of GPU time): every number DESIGN.md quotes is in the
    driver-run line.  frac_executed = executed multiplies/s over the same measured peak as the
    headline's roofline.  -> (detail, tail): the full records, and the compact ones that go LAST in
    the JSON line."""
    out, tail = {}, {}

    def with_frac(r, c):
        r["executed_mults_per_event"] = exec_mults(c.params, r["plan"])
        r["frac_executed"] = r["executed_mults_per_event"] * r["events_per_s"] / 1e12 / peak_tmults
        r["us_per_step"] = r["ms"] * 1e3 / r["S"]
        return r

    allc = {}
    for name in sorted(CONFIGS):
        if name == headline_cfg.name and headline_cfg.params == CONFIGS[name].params:
            continue
        c = CONFIGS[name]
        allc[name] = with_frac(time_case(ks, torch, dev, c, reps=5 if c.events < 5e10 else 3), c)
    out["all_configs"] = allc
    tail["all_configs"] = {k: compact(v) for k, v in allc.items()}
    for name in ("C1", "C3"):
        if name in allc:
            tail["all_configs"][name]["us_per_step"] = round(allc[name]["us_per_step"], 4)
    for key, case in (("packed4_C4", "C4_packed4"), ("model4_C4shape", "model4_C4shape")):
        c = case_config(case)
        out[key] = with_frac(time_case(ks, torch, dev, c, reps=3), c)
        tail[key] = compact(out[key])
    out["packed4_C4"]["note"] = "PACKED4 draw contract (DESIGN.md A22): NOT the BASELINE.json contract, reported beside it"
    out["model4_C4shape"]["note"] = ("the paper's own agent model (DESIGN.md A24) on the C4 shape, alpha_mom = alpha_maker = 0.15, "
                                     "Delta = 32, q <= 100, P_mkt = 0.02 (parameter values ours: the paper gives none)")
    if micro:
        # PACKED4 is where the smem-atomic roofline BASELINE.json names can be approached: its fractions too
        tail["packed4_C4"]["frac_of_smem_atomic_peak"] = round(out["packed4_C4"]["events_per_s"] / micro["smem_atomic_peak_lane_ops_per_s"], 4)
        tail["packed4_C4"]["frac_of_smem_atomic_pattern"] = round(out["packed4_C4"]["events_per_s"] / micro["smem_atomic_pattern_lane_ops_per_s"], 4)

    # end to end (host buffers, host clock) for the latency-regime configs
    tail["e2e_small"] = {name: {k: (round(v, 4) if isinstance(v, float) and v < 1e6 else v) for k, v in
                                time_e2e_small(ks, torch, dev, CONFIGS[name]).items()} for name in ("C1", "C3")}

    # a8 ablation on C2: one launch per step, book through HBM every step
    c = CONFIGS["C2"]
    pers = allc.get("C2") or time_case(ks, torch, dev, c, reps=5)
    sw = time_case(ks, torch, dev, c, reps=2, mode="stepwise")
    out["ablation_launch_per_step_C2"] = {
        "ms": sw["ms"], "events_per_s": sw["events_per_s"], "launches": c.S, "persistent_ms": pers["ms"],
        "slowdown_vs_persistent": sw["ms"] / pers["ms"],
        "algorithmic_hbm_bytes": float(c.S) * c.M * 2 * (8 * c.L + 128), "persistent_algorithmic_hbm_bytes": float(c.M) * (8 * c.L + 128),
        "measured_traffic": PROFILED_TRAFFIC_C2}
    tail["ablation_launch_per_step_C2"] = {"ms": round(sw["ms"], 4), "persistent_ms": round(pers["ms"], 4), "launches": c.S,
                                           "us_per_launch": round(sw["ms"] * 1e3 / c.S, 3),
                                           "slowdown_vs_persistent": round(sw["ms"] / pers["ms"], 3)}

    # context runs in the paper's own shapes: Table IV's fixed workload and the
    # latency configuration with zero-intelligence agents -- NOT the paper's
    # agent model or GPU
    ctx = {}
    for name in ("table4", "latency"):
        c = case_config(name)
        ctx["%s_M%d_A%d_L%d_S%d" % (name, c.M, c.A, c.L, c.S)] = with_frac(time_case(ks, torch, dev, c, reps=5), c)
    ctx["paper"] = "KineticSim on RTX 5090: 20.2 ms, 5.2e10 events/s (Table IV); 22.1 us median per step at M=4096 (PAPER.md:438)"
    out["paper_shape_context"] = ctx

    # SIV-J sweep shape: alpha_mom = 0 .. 0.70 in steps of 0.05, alpha_maker =
    # 0.15, M = 64 markets x S = 1000 steps each, the paper's own agent model (model 4), traced,
    # statistics on the device.  A = 200 (12.8e6 events / 64 / 1000: PAPER.md:458); L, Delta, q_max,
    # P_mkt are not given -- workloads.paper_params defaults.  Context, not a parity case.
    Ms, Ls, As, Ss, K = 64, 128, 200, 1000, 20
    st = torch.empty(ks.ks_state_bytes(Ms, Ls), dtype=torch.uint8, device=dev)
    tr = torch.empty((Ms, Ss, 2), dtype=torch.int32, device=dev)
    res = torch.empty((Ms, 4 + 2 * K), dtype=torch.float64, device=dev)
    alphas = [round(0.05 * i, 2) for i in range(15)]
    rows = []

    def sweep(record):
        for al in alphas:
            sim = ks.KsSim(Ms, Ls, As, paper_params(As, al), 5, state=st)
            sim.ks_run_traced(Ss, tr)
            ks.ks_trace_stats(tr, Ms, Ss, K, res)
            if record and al in (0.0, 0.15, 0.7):
                o = res.cpu().numpy()
                rows.append({"alpha_mom": al, "volatility": float(np.nanmean(o[:, 0])), "excess_kurtosis": float(np.nanmean(o[:, 1])),
                             "volume_per_step": float(np.nanmean(o[:, 2])), "acf_r_lag1": float(np.nanmean(o[:, 4])),
                             "acf_abs_r_lag1": float(np.nanmean(o[:, 4 + K]))})
            sim.ks_destroy()

    sweep(False)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(); sweep(False); b.record(); torch.cuda.synchronize()
    sweep(True)
    out["sivj_sweep"] = {"configs": len(alphas), "M": Ms, "L": Ls, "A": As, "S": Ss, "agent_events": len(alphas) * Ms * As * Ss,
                         "ms_total_device": a.elapsed_time(b), "paper": "< 250 ms for 12.8e6 events (RTX 5090, PAPER.md:458)",
                         "mean_over_markets": rows}
    return out, tail


if __name__ == "__main__":
    main()
