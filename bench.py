#!/usr/bin/env python
"""bench.py -- agent events/s of the call-auction hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch: ks_create (state init) + ONE ks_run of
all S steps of the workload (a0-a7), on M markets per GPU.  Workload: BASELINE.json configs[3]
("throughput scale", C4: M=65536, L=512, A=4096, S=1000, seed 3), the largest config and the one
the metric's roofline clause is quoted on.  For N > 1 each rank runs its own M markets with
market_base = rank*M (weak scaling, no data-path collective: markets are independent).
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import dataclasses  # noqa: E402

from paper_2606_21784_b200.workloads import CONFIGS, KS_MODEL_ZI, packed4, paper_params, sampled_markets  # noqa: E402

# Roofline of ks_persistent_kernel: the fmaheavy pipe that executes the 32x32->64
# multiplies.  Algorithmic multiplies per agent event: 20 of Philox4x32-10 + the
# mulhi draws of the rule (noise/momentum: offset and quantity; maker: spread only).
ALG_MULTS_PER_EVENT = {"zi": 22.0, "mix3": (22.0 + 21.0 + 22.0) / 3.0,
                       # PACKED4 (A22): a Philox block per 4 agents + the rule's multiply-extract draws
                       "zi_packed4": 20.0 / 4 + 2.0, "mix3_packed4": 20.0 / 4 + (2.0 + 1.0 + 2.0) / 3.0}
# Multiplies the kernel actually issues per event (IMAD.WIDE.U32 + IMAD.HI.U32 in the hot loop,
# from cuobjdump -sass): hoisting of (market, step)-uniform products, round 0's M0*agent carried as
# a running 64-bit sum, w3 never computed.
EXEC_MULTS_PER_EVENT = {"zi": 19.0, "mix3": (19.0 + 17.0 + 19.0) / 3.0,
                        "zi_packed4": 17.0 / 4 + 2.0, "mix3_packed4": 17.0 / 4 + (2.0 + 1.0 + 2.0) / 3.0}
# a 32-lane IMAD.WIDE/IMAD.HI occupies an SMSP's fmaheavy pipe for 4 cycles -> 8 lanes/clk/SMSP
WIDE_MUL_LANES_PER_SM_PER_CLK = 4 * 8


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


def time_oracle(cfg, n_markets: int, S: int):
    """The oracle as it stands, one thread, on the first n sampled markets of cfg for S steps."""
    from oracle import ks_oracle
    ids = sampled_markets(cfg.M, cfg.seed, 64)[:n_markets]
    t0 = time.perf_counter()
    ks_oracle.run_markets(cfg.params, cfg.L, cfg.A, cfg.seed, ids, S)
    dt = time.perf_counter() - t0
    return len(ids) * cfg.A * S / dt, dt, len(ids)


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
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": workload_config(cfg, args.gpus),
        "cpu_baseline": {"value": value, "unit": "events/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(cfg, n_gpus):
    return {"workload": "%s: BASELINE.json configs[%d] -- M=%d markets/GPU, L=%d ticks, A=%d agents, S=%d steps, seed=%d, %s"
                        % (cfg.name, int(cfg.name[1]) - 1, cfg.M, cfg.L, cfg.A, cfg.S, cfg.seed,
                           ("zero-intelligence" if (cfg.params["model"] & 1) == KS_MODEL_ZI else "noise/maker/momentum by a%3")
                           + (", PACKED4 draw contract (NOT the BASELINE.json one; DESIGN.md A22)" if cfg.params["model"] >= 2 else "")),
            "M_per_gpu": cfg.M, "L": cfg.L, "A": cfg.A, "S": cfg.S, "seed": cfg.seed,
            "parallelism": "markets sharded across %d GPU(s), market_base = rank*M, no collective" % n_gpus,
            "l2": "state buffer %.0f MB per GPU exceeds the 126 MB L2; written once per step" % (cfg.M * (8 * cfg.L + 128) / 1e6)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4", choices=sorted(CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--threads", type=int, default=0, help="KS_OPT_BLOCK_THREADS (0 = automatic)")
    ap.add_argument("--atomic-mode", type=int, default=0)
    ap.add_argument("--rng", default="literal", choices=["literal", "packed4"],
                    help="draw contract: literal = BASELINE.json (one Philox block per agent); packed4 = the "
                         "separately named PACKED4 contract (DESIGN.md A22), reported beside it, never instead of it")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-microbench", action="store_true")
    ap.add_argument("--all-configs", action="store_true", help="also time C1..C5 (extra keys)")
    args = ap.parse_args()
    cfg = CONFIGS[args.config]
    if args.rng == "packed4":
        cfg = dataclasses.replace(cfg, params=packed4(cfg.params))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_2606_21784_b200 import binding as ks

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    ks.load()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    assert world == args.gpus or world == 1, "launch with torchrun --nproc-per-node N for --gpus N"

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    M, L, A, S = cfg.M, cfg.L, cfg.A, cfg.S
    base = rank * M
    state = torch.empty(ks.ks_state_bytes(M, L), dtype=torch.uint8, device=dev)

    def one_step(ev_pairs=None):
        sim = ks.KsSim(M, L, A, cfg.params, cfg.seed, market_base=base, state=state)
        if args.threads:
            sim.ks_set_option(ks.KS_OPT_BLOCK_THREADS, args.threads)
        if args.atomic_mode:
            sim.ks_set_option(ks.KS_OPT_ATOMIC_MODE, args.atomic_mode)
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
        s_.ks_destroy()
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    events_per_step = float(M) * A * S
    value = world * events_per_step * args.steps / (total_ms * 1e-3)

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
    e2e_value = world * events_per_step * n_e2e / (e2e_ms * 1e-3)
    # the e2e result is the same simulation: check it against the device-resident run's records
    chk = torch.empty((M, 16), dtype=torch.int64).pin_memory()
    sim = one_step(); sim.ks_read_stats(chk); torch.cuda.synchronize(); sim.ks_destroy()
    assert torch.equal(chk, h_recs), "e2e run and device-resident run disagree"

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (ks_persistent_kernel): ALU / issue bound
    model = ("zi" if (cfg.params["model"] & 1) == KS_MODEL_ZI else "mix3") + ("_packed4" if cfg.params["model"] >= 2 else "")
    avg_kern_s = float(np.mean(kern_ms)) * 1e-3
    peaks = {}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peaks = json.load(f)
    except Exception:
        pass
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    peak = sms * WIDE_MUL_LANES_PER_SM_PER_CLK * sm_max_mhz * 1e6 / 1e12
    achieved = ALG_MULTS_PER_EVENT[model] * events_per_step / avg_kern_s / 1e12
    executed = EXEC_MULTS_PER_EVENT[model] * events_per_step / avg_kern_s / 1e12
    roofline = {"bound": "alu", "kernel": "ks_persistent_kernel", "achieved": achieved, "peak": peak,
                "unit": "T 32x32->64-bit integer multiplies/s", "frac": achieved / peak,
                "traffic": PROFILED_DRAM_BYTES_PER_LAUNCH.get(cfg.name if args.rng == "literal" else cfg.name + "_packed4"),
                "alg_mults_per_event": ALG_MULTS_PER_EVENT[model], "avg_launch_ms": avg_kern_s * 1e3,
                "executed_mults_per_event": EXEC_MULTS_PER_EVENT[model], "fmaheavy_pipe_frac_from_executed": executed / peak,
                "frac_note": "achieved counts the ALGORITHMIC multiplies (SURVEY.md S8(d)); the kernel executes fewer "
                             "(hoisted / strength-reduced rounds, w3 skipped), so frac can reach or pass 1.0 -- the pipe's own "
                             "utilisation is fmaheavy_pipe_frac_from_executed (ncu: 95.8 % with the address multiply-adds, "
                             "profiles/r1h_persistent_full.md)",
                "peak_source": "derived (DESIGN.md 7.2): %d SMs x 4 SMSPs x 8 lanes/clk (IMAD.WIDE = 2 passes of the 16-lane fmaheavy pipe) x %.0f MHz (%s)"
                               % (sms, sm_max_mhz, "MEASURED_PEAKS.json sm_max_mhz" if peaks else "NVML max clock"),
                "hbm": {"algorithmic_bytes": M * (8 * L + 128), "achieved_GBps": M * (8 * L + 128) / avg_kern_s / 1e9,
                        "peak_GBps": peaks.get("hbm_gbs", 6650.0),
                        "peak_source": "MEASURED_PEAKS.json (measured)" if peaks else "fallback (B200_PROFILING.md)"}}

    line = {
        "metric": "agent_events_per_s", "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32", "data": "synthetic", "config": workload_config(cfg, world),
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": int(h_open.numel() * 4),
                "d2h_bytes_per_step": int(h_books.numel() * 4 + h_recs.numel() * 8), "steps": n_e2e,
                "ms_per_step": e2e_ms / n_e2e},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "kernel_events_per_s": events_per_step / avg_kern_s,
        "paper_context": {"events_per_s": 5.47e10, "where": "RTX 5090, M=8192 A=1024 L=128 S=500, PAPER.md:313 (other GPU, other agent model)"},
    }

    # ---- microbenchmarks in the same process (same clocks): the BASELINE.json smem-atomic
    #      roofline and the generation-only (integer ALU) ceiling
    if not args.no_microbench and world == 1:
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
        cyc = lambda ops_s, per: sms * 4 * sm_max_mhz * 1e6 * 32 * per / ops_s      # SMSP cycles per IMAD.WIDE
        atomics_per_event = 1.0 if model.startswith("zi") else 4.0 / 3.0
        kev = events_per_step / avg_kern_s
        line["microbench"] = {
            "smem_atomic_peak_lane_ops_per_s": peak_ops, "smem_atomic_pattern_lane_ops_per_s": pat_ops,
            "smem_atomic_pattern_warp_aggregated_lane_ops_per_s": agg_ops, "smem_atomic_same_address_lane_ops_per_s": one_ops,
            "generate_only_events_per_s": gen_ev, "imad_wide_thread_ops_per_s": wide, "lop3_thread_ops_per_s": lop,
            "imad_wide_lop3_mix_thread_ops_per_s": mix,
            "smsp_cycles_per_imad_wide": {"alone": cyc(wide, 1), "with_1_lop3": cyc(mix, 2), "with_2_lop3": cyc(mix2, 3),
                                          "with_3_lop3": cyc(mix3, 4)},
            "frac_of_smem_atomic_peak": kev * atomics_per_event / peak_ops,
            "frac_of_smem_atomic_pattern": kev * atomics_per_event / pat_ops,
            "frac_of_generate_only": kev / gen_ev,
        }

    if args.all_configs and world == 1:
        extra = {}
        for name in sorted(CONFIGS):
            c = CONFIGS[name]
            st = torch.empty(ks.ks_state_bytes(c.M, c.L), dtype=torch.uint8, device=dev)
            ts = []
            for i in range(4):
                sim = ks.KsSim(c.M, c.L, c.A, c.params, c.seed, state=st)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); sim.ks_run(c.S); b.record(); torch.cuda.synchronize()
                ts.append(a.elapsed_time(b)); sim.ks_destroy()
            extra[name] = {"ms_median_of_3": float(np.median(ts[1:])), "events_per_s": c.events / (float(np.median(ts[1:])) * 1e-3)}
        line["all_configs"] = extra
        # a8 ablation on C2: one launch per step, book through HBM every step
        c = CONFIGS["C2"]
        st = torch.empty(ks.ks_state_bytes(c.M, c.L), dtype=torch.uint8, device=dev)
        ts = []
        for i in range(3):
            sim = ks.KsSim(c.M, c.L, c.A, c.params, c.seed, state=st)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); sim.ks_run_stepwise(c.S); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b)); sim.ks_destroy()
        ms = float(np.median(ts[1:]))
        hbm_bytes = float(c.S) * c.M * 2 * (8 * c.L + 128)          # load + store of book and record, every step
        line["ablation_launch_per_step_C2"] = {
            "ms": ms, "events_per_s": c.events / (ms * 1e-3), "launches": c.S,
            "slowdown_vs_persistent": ms / extra["C2"]["ms_median_of_3"],
            "algorithmic_hbm_bytes": hbm_bytes, "hbm_GBps": hbm_bytes / (ms * 1e-3) / 1e9,
            "persistent_hbm_bytes": float(c.M) * (8 * c.L + 128)}

    if args.all_configs and world == 1:
        # context runs in the paper's own shapes: Table IV's fixed workload M=8192,
        # A=256, L=128, S=500 and the latency configuration M=4096, A=256 with
        # zero-intelligence agents Delta=8, q<=10, seed 5 -- NOT the paper's agent model or GPU
        from paper_2606_21784_b200.workloads import zi_params
        ctx = {}
        for name, Mp in (("table4_M8192_A256_L128_S500", 8192), ("latency_M4096_A256_L128_S500", 4096)):
            st = torch.empty(ks.ks_state_bytes(Mp, 128), dtype=torch.uint8, device=dev)
            ts = []
            for i in range(6):
                sim = ks.KsSim(Mp, 128, 256, zi_params(8, 10), 5, state=st)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); sim.ks_run(500); b.record(); torch.cuda.synchronize()
                ts.append(a.elapsed_time(b)); sim.ks_destroy()
            ms = float(np.median(ts[1:]))
            ctx[name] = {"ms_median_of_5": ms, "events_per_s": Mp * 256 * 500 / (ms * 1e-3), "us_per_step": ms * 1e3 / 500}
        ctx["paper"] = "KineticSim on RTX 5090: 20.2 ms, 5.2e10 events/s (Table IV); 22.1 us median per step at M=4096 (PAPER.md:438)"
        line["paper_shape_context"] = ctx

    if args.all_configs and world == 1:
        # SIV-J sweep shape: alpha_mom = 0 .. 0.70 in steps of 0.05, alpha_maker
        # = 0.15, M = 64 markets x S = 1000 steps each, the paper's own agent model (model 4), traced,
        # statistics on the device.  A = 200 (12.8e6 events / 64 / 1000: PAPER.md:458); L, Delta,
        # q_max, P_mkt are not given -- workloads.paper_params defaults.  Context, not a parity case.
        Ms, Ls, As, Ss, K = 64, 128, 200, 1000, 20
        st = torch.empty(ks.ks_state_bytes(Ms, Ls), dtype=torch.uint8, device=dev)
        tr = torch.empty((Ms, Ss, 2), dtype=torch.int32, device=dev)
        out = torch.empty((Ms, 4 + 2 * K), dtype=torch.float64, device=dev)
        alphas = [round(0.05 * i, 2) for i in range(15)]
        rows = []

        def sweep(record):
            for al in alphas:
                sim = ks.KsSim(Ms, Ls, As, paper_params(As, al), 5, state=st)
                sim.ks_run_traced(Ss, tr)
                ks.ks_trace_stats(tr, Ms, Ss, K, out)
                if record:
                    o = out.cpu().numpy()
                    rows.append({"alpha_mom": al, "volatility": float(np.nanmean(o[:, 0])), "excess_kurtosis": float(np.nanmean(o[:, 1])),
                                 "volume_per_step": float(np.nanmean(o[:, 2])), "acf_r_lag1": float(np.nanmean(o[:, 4])),
                                 "acf_abs_r_lag1": float(np.nanmean(o[:, 4 + K]))})
                sim.ks_destroy()

        sweep(False)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); sweep(False); b.record(); torch.cuda.synchronize()
        sweep(True)
        line["sivj_sweep"] = {"configs": len(alphas), "M": Ms, "L": Ls, "A": As, "S": Ss, "agent_events": len(alphas) * Ms * As * Ss,
                              "ms_total_device": a.elapsed_time(b), "paper": "< 250 ms for 12.8e6 events (RTX 5090, PAPER.md:458)",
                              "mean_over_markets": rows}

    if not args.no_cpu_baseline and world == 1:
        n_mk = min(cfg.M, 64)
        ev_s, dt, n = time_oracle(cfg, n_mk, S)
        line["cpu_baseline"] = {"value": ev_s, "unit": "events/s", "cores": 1, "kind": "oracle",
                                "sample": "%d seeded sampled markets x S=%d steps of %s (%.3g events, %.1f s), 1 thread of %d host cores"
                                          % (n, S, cfg.name, n * A * S, dt, os.cpu_count() or 0)}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum of one ks_persistent_kernel launch from the
# `ncu --set full` capture summarised under profiles/ (None until measured for that config).
PROFILED_DRAM_BYTES_PER_LAUNCH = {"C4": 25261312 + 237688320,            # profiles/r1h_persistent_full.md
                                  "C4_packed4": 23691008 + 254493952}    # profiles/r1g_packed_persistent_full.md

if __name__ == "__main__":
    main()
