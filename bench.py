#!/usr/bin/env python
"""bench.py -- headline benchmark of libpimc on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--sweeps-per-step S]

Metric (BASELINE.json): Metropolis site-updates/s and sweeps/s, Hodgkin-Huxley, M = 32768, fp64, states + 7
parameters (configs[3]); one "step" = one pimc_sweep call of S full sweeps (even + odd half-sweep, 7 sequential
parameter moves, moment accumulation) over the seeded synthetic workload, i.e. one pass of every §8(a) row.
Rank 0 prints ONE JSON line.  N > 1 runs N independent replicas (the path does not shard: "replicas only").
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
sys.path.insert(0, ROOT)

from workloads import make_workload  # noqa: E402

METRIC = "Metropolis site-updates/sec and sweeps/sec (HH, M=32768, fp64) vs FP64 roofline"
UNIT = "site-updates/s"

# ---- work model (one slot = one FP64-pipe lane operation = 2 FLOP at peak) -----------------------------
# (1) ORACLE-COUNTED algorithmic work: what a straightforward evaluation of the paper's formulas needs per joint site update and
#     per parameter-move model evaluation.  Written by `python -m oracle.count_work` (an instrumented restatement of the oracle's
#     arithmetic, validated bit for bit against it; libm calls costed by a stated table) into oracle/work_constants.json;
#     tests/test_work_model.py keeps these literals equal to that file.
W_SITE_ORACLE = 869.0
W_EVAL_ORACLE = 666.0
# (2) EXECUTED FP64-pipe thread instructions of the production kernels per OWNED unit, counted by ncu (source page, DFMA + DMUL +
#     DADD + DSETP, predicated-on threads; profiles/r02_work_counts.md).  They include the redundant halo updates and the
#     producers' random-number arithmetic, so executed x rate / peak is the lane-level FP64 pipe utilisation: it cannot
#     flatter.  The kernels execute FEWER operations than (1) (one shared exponential per RK4 stage instead of three tanh, one
#     reciprocal series instead of two divides per gate, cached first-stage gate rates in parameter moves), so the useful
#     fraction credits min((1), (2) / redundancy).
EXEC_FP64_COMPUTED = {   # engine -> (per COMPUTED site update, per COMPUTED parameter-move evaluation); HH tanh kinetics, fp64, RK4 map, joint updates
    "tile": (519.4, 252.2),      # tile_sweep_kernel, profiles/r02_head_verification.md: 594.2 and 288.5 per OWNED unit at cfg3 / (254 / 222)
                                 # (303.1 per evaluation until the warp sums of the block reductions moved to the FP64 tensor cores)
    "tilemc": (502.4, 255.4),    # tilemc_sweep_kernel (many-chain tile-resident engine), profiles/r02_tilemc.md: 545 and 277 per OWNED unit at cfg4 / (256 / 236)
    "global": (521.0, 285.0),    # sweep_kernel (one CTA per chain, no halos, stage-1 rates cached in global memory), profiles/r02_cfg4.md: launch total minus
                                 # 521 per site update, over the evaluations
}
# ncu sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed of the same kernels, same launches
NCU_PIPE_FP64_ACTIVE = {3: {"full_sweep": 0.310, "a2_only": 0.431, "a4_only": 0.272, "source": "profiles/r02_head_verification.md"},
                        4: {"full_sweep": 0.527, "a2_only": 0.518, "a4_only": 0.513, "source": "profiles/r02_tilemc.md (TILE_MC engine; GLOBAL engine: 0.453, profiles/r02_cfg4.md)"}}
# trapezoid discretisation / component-wise updates: estimated slots (no oracle count yet), used for the non-headline variants only
W_SITE_SLOTS_TRAP = 380.0
W_SITE_SLOTS_COMP = 2300.0
W_EVAL_SLOTS_TRAP = 140.0
# FP64 peak derived from unit counts and clocks: 148 SMs x 64 FP64 lanes/clk/SM x 1.965 GHz, 2 FLOP per lane-FMA.
FP64_LANES_PER_SM_CLK = 64
SM_COUNT = 148
SM_MAX_HZ = 1.965e9
PEAK_TFLOPS_DERIVED = SM_COUNT * FP64_LANES_PER_SM_CLK * SM_MAX_HZ * 2 / 1e12
NCU_DRAM_BYTES_PER_LAUNCH = 5918464.0   # cfg3 full sweep launch: 5.904 MB read + 14 KB written (profiles/r02_work_counts.md)


def rank_info():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index, period=0.05):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons, self.stop_flag = index, period, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap", nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_rate(w, budget_s, chain=0, disc=0, mode=0):
    """Time the CPU oracle, as it stands, on a bounded sample of the same workload.  Returns (site-updates/s, sweeps, seconds)."""
    from oracle import OracleChain
    o = OracleChain.from_workload(w, chain=chain)
    if disc:
        o.set_discretisation(disc)
    if mode:
        o.set_update_mode(mode)
    t0 = time.perf_counter()
    o.sweep(2, seed=w.chain_seed)                       # warm-up + first estimate
    per = (time.perf_counter() - t0) / 2
    n = max(2, int(budget_s / max(per, 1e-6)))
    t0 = time.perf_counter()
    o.sweep(n, seed=w.chain_seed)
    dt = time.perf_counter() - t0
    return (w.M + 1) * n / dt, n, dt


def oracle_rate_all_cores(w, budget_s, per_sweep_s):
    """The oracle on every host core at once, one independent chain per core ("an all-cores rate with one
    independent chain per core").  ctypes releases the GIL inside orc_sweep, so plain threads run in parallel."""
    from oracle import OracleChain
    cores = os.cpu_count() or 1
    chains = [OracleChain.from_workload(w, chain=0) for _ in range(cores)]
    n = max(1, int(budget_s / max(per_sweep_s, 1e-6)))
    ths = [threading.Thread(target=lambda o=o, k=k: o.sweep(n, seed=w.chain_seed + 1000 + k)) for k, o in enumerate(chains)]
    t0 = time.perf_counter()
    for t in ths:
        t.start()
    for t in ths:
        t.join()
    dt = time.perf_counter() - t0
    return (w.M + 1) * n * cores / dt, cores, n, dt


ENGINE_NAMES = {1: "GLOBAL", 2: "TILE", 3: "TILE_MC"}
OTHER_CONFIGS = [   # (config, dtype, sweeps per step, chains or None): every BASELINE.json config besides the headline one, its fp32
    # variant, and FOUR independent chains of the headline shape in one launch (north_star: "HH chains at M=32768 sustaining >= 50 % of
    # the FP64 pipe for the checkerboard sweep": a single chain offers M/2 independent updates per half-sweep, several chains fill the SMs)
    (0, 64, 2000, None), (1, 64, 1000, None), (2, 64, 1000, None), (4, 64, 100, None), (3, 32, 1000, None), (3, 64, 100, 4),
    # the paper's own trapezoid discretisation (Eq. 7): the headline shape, and the paper-shaped workload (config 5, not a BASELINE config)
    (3, 64, 1000, None, "trapezoid"), (5, 64, 1000, None, "trapezoid"), (4, 64, 50, None, "trapezoid"),
]


def measure_other_config(P, torch, flush, cfg, dtype, S, steps, cpu_budget, w=None, n_chains=None, disc="rk4"):
    """One extra line of the "other_configs" block: the same timed protocol as the headline (3 warm-up steps, L2 flushed before
    every step, CUDA events on the launching stream), full sweeps with accumulation every sweep, oracle on one core beside it."""
    w = w or (make_workload(cfg, n_chains=n_chains) if n_chains else make_workload(cfg))
    h = P.Pimc.from_workload(w, dtype=dtype)
    if disc == "trapezoid":
        h.set_discretisation(P.DISC_TRAPEZOID)
    h.set_accum(True, 1)
    h.reset_moments()
    stream = torch.cuda.current_stream()
    seed = w.chain_seed

    def one():
        flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream); h.sweep(S, seed); e1.record(stream)
        return e0, e1
    for _ in range(3):
        one()
    torch.cuda.synchronize()
    n0 = h.launch_count
    evs = [one() for _ in range(steps)]
    torch.cuda.synchronize()
    ms = float(np.mean([a.elapsed_time(b) for a, b in evs]))
    gpu_launches = h.launch_count - n0
    units = float(w.n_chains) * (w.M + 1) * S
    a2 = None
    if w.n_chains > 1:          # many-chain workloads: the checkerboard sweep (row A2) on its own as well
        def one_a2():
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); h.sweep_states_only(S, seed); e1.record(stream)
            return e0, e1
        one_a2(); torch.cuda.synchronize()
        ev2 = [one_a2() for _ in range(steps)]
        torch.cuda.synchronize()
        a2 = units / (float(np.mean([a.elapsed_time(b) for a, b in ev2])) * 1e-3)
    fault = h.fault()
    out = {"workload": w.name + ("_trapezoid" if disc == "trapezoid" else ""), "dtype": "f64" if dtype == 64 else "f32", "value": units / (ms * 1e-3), "unit": UNIT,
           "chain_sweeps_per_s": w.n_chains * S / (ms * 1e-3), "ms_per_step": ms, "sweeps_per_step": S, "steps": steps,
           "params_moved": int(np.count_nonzero(w.w_param)), "engine": ENGINE_NAMES[h.get_engine()["engine"]],
           "launch": h.get_launch(), "gpu_launches": int(gpu_launches), "fault": int(fault)}
    if a2 is not None:
        out["a2_only_site_updates_per_s"] = a2
        eng = h.get_engine()
        if eng["engine"] == P.ENGINE_TILE_MC and dtype == 64 and w.model == 1:     # executed FP64 lane operations of the checkerboard sweep over the derived peak
            out["a2_only_frac"] = 2.0 * a2 * EXEC_FP64_COMPUTED["tilemc"][0] * (256.0 / h.get_launch()["tile_sites"]) / 1e12 / PEAK_TFLOPS_DERIVED
    if cpu_budget > 0 and dtype == 64:
        r, n, dt = oracle_rate(w, cpu_budget, disc=1 if disc == "trapezoid" else 0)
        out["oracle_1core"] = {"value": r, "unit": UNIT, "sample": f"{n} full sweeps of chain 0 in {dt:.1f} s"}
    del h
    return out


def run_reference(args):
    """--impl reference: the oracle (as it stands) on the host cores, bounded sample per step.  Rank 0 only."""
    rank, _, world = rank_info()
    if rank != 0:
        return
    from oracle import OracleChain
    w = make_workload(args.config, kinetics=args.kinetics)
    trap = args.disc == "trapezoid"
    o = OracleChain.from_workload(w, chain=0)
    if trap:
        o.set_discretisation(1)
    t0 = time.perf_counter(); o.sweep(1, seed=1); per = time.perf_counter() - t0
    n_per_step = max(1, int(min(args.ref_budget / (args.steps + args.warmup), 60.0) / per))
    for _ in range(args.warmup):
        o.sweep(n_per_step, seed=1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.sweep(n_per_step, seed=1)
    dt = time.perf_counter() - t0
    value = (w.M + 1) * n_per_step * args.steps / dt
    sample = f"{n_per_step} full sweeps per step of chain 0 of {w.name} (states + 7 parameter moves), serial fp64 C++ -O2"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": w.name + ("_trapezoid" if trap else ""), "discretisation": args.disc, "M": w.M, "n_chains": 1, "sweeps_per_step": n_per_step},
        "sweeps_per_s": n_per_step * args.steps / dt,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def reduce_over_ranks(local_seconds, local_units, world, dist=None):
    """Whole-job throughput = units processed by all ranks / max over ranks of the timed seconds."""
    if world == 1 or dist is None:
        return local_seconds, local_units
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([local_seconds], dtype=torch.float64, device=dev)
    u = torch.tensor([local_units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def run_ours(args):
    import torch
    import paper_1103_4887_b200 as P
    rank, local_rank, world = rank_info()
    dist = None
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (libpimc has no CPU fallback)")
    dev_index = torch.cuda.current_device()

    # replicas only: every rank runs the same shape with its own data realisation and Philox key
    w = make_workload(args.config, seed=None if rank == 0 else 11034887 + args.config + 7919 * rank, kinetics=args.kinetics)
    seed = w.chain_seed + rank
    S = args.sweeps_per_step
    h = P.Pimc.from_workload(w, dtype=args.dtype)
    trap = args.disc == "trapezoid"
    if trap:
        h.set_discretisation(P.DISC_TRAPEZOID)
    w_site, w_eval = (W_SITE_SLOTS_TRAP, W_EVAL_SLOTS_TRAP) if trap else (W_SITE_ORACLE, W_EVAL_ORACLE)
    comp = args.update == "componentwise"
    if comp:
        h.set_update_mode(P.UPDATE_COMPONENTWISE)
        w_site = W_SITE_SLOTS_COMP if not trap else 4 * 205.0 + 300.0
    headline = args.config == 3 and args.kinetics == "tanh" and not trap and not comp
    peak_tflops = PEAK_TFLOPS_DERIVED * (1.0 if args.dtype == 64 else 2.0)   # fp32: 128 FP32 lanes/clk/SM
    if args.exchange_hold is not None:
        h.set_exchange(args.exchange_hold)
    h.set_accum(True, 1)
    h.reset_moments()
    shape = h.get_launch()
    eng = h.get_engine()
    # executed-instruction counts exist for the HH tanh / fp64 / RK4-map / joint-update kernels; redundancy = computed / owned sites
    # of an interior tile (tile-resident engine with more than one tile per chain: h halo sites on each side are updated redundantly)
    exec_counts, red = None, None
    if w.model == 1 and args.dtype == 64 and not trap and not comp:
        tile_engine = eng["engine"] in (P.ENGINE_TILE, P.ENGINE_TILE_MC)
        red = (shape["tile_sites"] + 2.0 * eng["halo"]) / shape["tile_sites"] if (tile_engine and shape["ctas_per_chain"] > 1) else 1.0
        if eng["engine"] == P.ENGINE_TILE_MC:
            red = 256.0 / shape["tile_sites"]       # every thread of a group computes its site pair in branch-free blocks, masked or not
        per = EXEC_FP64_COMPUTED[{P.ENGINE_TILE: "tile", P.ENGINE_TILE_MC: "tilemc"}.get(eng["engine"], "global")]
        exec_counts = (per[0] * red, per[1] * red)
    units_per_step = float(w.n_chains) * (w.M + 1) * S
    n_active = int(np.count_nonzero(w.w_param))
    evals_per_step = float(w.n_chains) * w.M * S * n_active

    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    stream = torch.cuda.current_stream()

    def one_step(fn, n=S):
        flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream); fn(n, seed); e1.record(stream)
        return e0, e1

    for _ in range(args.warmup):
        one_step(h.sweep)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(dev_index)
    sampler.start()
    launches0 = h.launch_count
    t_wall0 = time.perf_counter()
    evs = [one_step(h.sweep) for _ in range(args.steps)]
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t_wall = time.perf_counter() - t_wall0
    sampler.stop_flag = True
    sampler.join()
    launches = h.launch_count - launches0
    step_ms = [a.elapsed_time(b) for a, b in evs]
    local_s = sum(step_ms) * 1e-3
    tot_s, tot_units = reduce_over_ranks(local_s, units_per_step * args.steps, world, dist)
    value = tot_units / tot_s
    ms_per_step = tot_s / args.steps * 1e3

    # rows A2 and A4 on their own (same launch shape, same data), for the breakdown the north_star asks for; same statistic
    # (mean over the timed launches) as the headline
    def rate(fn, units, reps=3):
        fn(max(1, S // 10), seed); torch.cuda.synchronize()
        ms = []
        for _ in range(reps):
            a, b = one_step(fn); torch.cuda.synchronize(); ms.append(a.elapsed_time(b))
        return units / (float(np.mean(ms)) * 1e-3), float(np.mean(ms))
    a2_rate, a2_ms = rate(h.sweep_states_only, units_per_step)
    a4_rate, a4_ms = (rate(h.sweep_params_only, evals_per_step) if n_active else (0.0, 0.0))

    # roofline of the dominant (only) kernel of the step: the persistent sweep kernel.
    #   frac              = EXECUTED FP64 lane operations (ncu-counted per owned unit, redundant halo work included) / time / peak:
    #                       the lane-level FP64 pipe utilisation; ~ ncu's sm__pipe_fp64_cycles_active (warp level) x active lanes
    #   frac_owned        = the same without the redundant halo updates (/ computed-per-owned sites)
    #   frac_oracle_work  = oracle-counted algorithmic work / time / peak (a plain evaluation of the paper's formulas would need
    #                       this many operations; the kernels need fewer, so this one may exceed the pipe utilisation)
    step_s = float(np.mean(step_ms)) * 1e-3
    tfl = lambda slots, seconds: 2.0 * slots / seconds / 1e12
    oracle_tflops = tfl(units_per_step * w_site + evals_per_step * w_eval, step_s)
    if exec_counts:
        achieved_tflops = tfl(units_per_step * exec_counts[0] + evals_per_step * exec_counts[1], step_s)
        a2_frac, a4_frac = tfl(a2_rate * exec_counts[0], 1.0) / peak_tflops, tfl(a4_rate * exec_counts[1], 1.0) / peak_tflops
        useful_site, useful_eval = min(w_site, exec_counts[0] / red), min(w_eval, exec_counts[1] / red)
        frac_useful = tfl(units_per_step * useful_site + evals_per_step * useful_eval, step_s) / peak_tflops
    else:           # variants without an ncu count: the (estimated or oracle-counted) work model only
        achieved_tflops = oracle_tflops
        a2_frac, a4_frac = tfl(a2_rate * w_site, 1.0) / peak_tflops, tfl(a4_rate * w_eval, 1.0) / peak_tflops
        frac_useful = None
    measured_peak = P.fp64_peak(150) * 2 / 1e12 if rank == 0 else None
    tile = bool(shape.get("smem_bytes", 0))
    model_name = {0: "LinearModel", 1: "HHModelK<0>", 2: "HHModelK<1>"}[w.model]
    rtype = "double" if args.dtype == 64 else "float"
    kernel = (f"pimc::tilemc_sweep_kernel<{model_name},{rtype},NGRP={shape['threads_per_cta'] // 128}>" if eng["engine"] == P.ENGINE_TILE_MC else
              f"pimc::tile_sweep_kernel<{model_name},{rtype},MAXT={256 if shape['threads_per_cta'] <= 256 else 512},TRAP={int(trap)},COMP={int(comp)},KG={int(n_active > 0 and not trap)},TR=0>"
              if tile else f"pimc::sweep_kernel<{model_name},{rtype}>")
    roofline = {"bound": "alu", "achieved": achieved_tflops, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved_tflops / peak_tflops,
                "frac_definition": ("executed FP64 lane operations (ncu-counted per owned unit, redundant halo updates and RNG included) x units / CUDA-event time / peak"
                                    if exec_counts else "work-model slots x units / CUDA-event time / peak (no ncu count for this variant)"),
                "frac_owned": (achieved_tflops / peak_tflops / red) if red else None,
                "frac_useful": frac_useful,
                "frac_oracle_work": oracle_tflops / peak_tflops,
                "halo_redundancy": red,
                "pipe_fp64_active_ncu": NCU_PIPE_FP64_ACTIVE.get(args.config) if exec_counts else None,
                "target": ("north_star: >= 50 % of the FP64 pipe for the checkerboard sweep (A2), judged on ncu's sm__pipe_fp64_cycles_active: ONE chain of M = 32768 "
                           "(config 3, this line's workload when --config 3): 42.7 %, NOT reached (M/2 independent updates per half-sweep are one warp per scheduler); "
                           "several chains per launch on the TILE_MC engine: 54.3 % for four chains of M = 32768, 51.8 % for config 4: reached (profiles/r02_tilemc.md)"),
                "traffic": NCU_DRAM_BYTES_PER_LAUNCH if (headline and args.dtype == 64) else None,
                "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of one launch, ncu --set full, profiles/r02_work_counts.md (tile loaded once, written back once: independent of the sweeps per launch)",
                "peak_source": ("derived: 148 SM x 64 FP64 lanes/clk x 1.965 GHz x 2 FLOP (DESIGN.md); no FP64 figure in MEASURED_PEAKS.json" if args.dtype == 64 else "derived: 148 SM x 128 FP32 lanes/clk x 1.965 GHz x 2 FLOP (DESIGN.md)"),
                "peak_measured_dfma_tflops": measured_peak,
                "frac_of_measured_dfma": (achieved_tflops / measured_peak) if measured_peak else None,
                "kernel": kernel,
                "work_model": {"oracle_slots_per_site_update": w_site, "oracle_slots_per_param_eval": w_eval,
                               "executed_fp64_per_owned_site_update": exec_counts[0] if exec_counts else None,
                               "executed_fp64_per_owned_param_eval": exec_counts[1] if exec_counts else None,
                               "site_updates_per_launch": units_per_step, "param_evals_per_launch": evals_per_step},
                "a2_only": {"site_updates_per_s": a2_rate, "ms_per_launch": a2_ms, "frac": a2_frac,
                            "frac_oracle_work": tfl(a2_rate * w_site, 1.0) / peak_tflops},
                "a4_only": {"param_evals_per_s": a4_rate, "ms_per_launch": a4_ms, "frac": a4_frac,
                            "frac_oracle_work": tfl(a4_rate * w_eval, 1.0) / peak_tflops,
                            "note": ("trapezoid rule on the tile engine: the parameter moves are decided from one reduction of sufficient statistics per sweep "
                                     "(DESIGN.md 6.1b); param_evals_per_s counts the evaluations the paper's K2/K3 would have made, none is executed") if (trap and tile and w.model != 0) else None}}

    # end to end through the C ABI on HOST buffers: H2D of y, I, x0, p0 + sweeps + D2H of the moments inside the timed region
    e2e = None
    if (rank == 0 or world > 1) and not trap and not comp:     # pimc_run_host is the RK4-map, joint-update convenience call
        scratch = P.run_host_scratch(w, dtype=args.dtype)                   # device scratch owned by the caller: no cudaMalloc in the timed calls
        P.run_host(w, 0, max(1, S // 10), seed, dtype=args.dtype, scratch=scratch)         # warm-up
        reps = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(reps):
            out = P.run_host(w, 0, S, seed, dtype=args.dtype, scratch=scratch)
        dt_e2e = time.perf_counter() - t0
        s_e2e, u_e2e = reduce_over_ranks(dt_e2e, units_per_step * reps, world, dist)
        e2e = {"value": u_e2e / s_e2e, "unit": UNIT, "h2d_bytes_per_step": out["h2d_bytes"], "d2h_bytes_per_step": out["d2h_bytes"],
               "ms_per_step": s_e2e / reps * 1e3, "call": "pimc_run_host_ws on HOST buffers (H2D of y, I, x0, p0 + pimc_init + cache build + pimc_sweep + pimc_moments + D2H + fault check + sync; device scratch provided by the caller)"}

    if rank == 0:
        cpu_rate, cpu_n, cpu_s = oracle_rate(w, args.cpu_budget, disc=1 if trap else 0, mode=1 if comp else 0)
        cpu = {"value": cpu_rate, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{cpu_n} full sweeps of chain 0 of {w.name} in {cpu_s:.1f} s (serial fp64 C++ -O2, {os.cpu_count()} cores present)"}
        other = None
        if headline and args.dtype == 64 and world == 1 and not args.no_other_configs:
            # the rest of BASELINE.json's workloads (north_star: "Report throughput on the synthetic workloads below at 1 GPU"),
            # after the timed region of the headline; and the oracle on all host cores (one independent chain per core)
            other = []
            for cfg, dt_, S_, nch, *rest in OTHER_CONFIGS:
                other.append(measure_other_config(P, torch, flush, cfg, dt_, S_, 3, min(args.cpu_budget, 2.0) if not nch else 0.0,
                                                  w=w if (cfg == 3 and not nch) else None, n_chains=nch, disc=rest[0] if rest else "rk4"))
            ar, cores, an, adt = oracle_rate_all_cores(w, min(args.cpu_budget, 8.0), cpu_s / max(cpu_n, 1))
            cpu["all_cores"] = {"value": ar, "unit": UNIT, "cores": cores,
                                "sample": f"{cores} independent chains of {w.name}, one per core (threads), {an} full sweeps each in {adt:.1f} s"}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64" if args.dtype == 64 else "f32",
            "data": "synthetic",
            "config": {"workload": w.name + ("_trapezoid" if trap else ""), "discretisation": args.disc, "update": args.update, "M": w.M, "n_chains": w.n_chains, "sweeps_per_step": S, "params_moved": n_active,
                       "accumulate_every": 1, "launch": shape, "engine": ENGINE_NAMES[eng["engine"]], "l2": "flushed between timed steps (256 MiB fill)",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "sweeps_per_s": value / (w.M + 1),
            "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu, "other_configs": other,
            "wall_s_timed_region": t_wall, "speedup_vs_oracle_1core": value / cpu_rate,
        }
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--kinetics", default="tanh", choices=["tanh", "classic"], help="HH gate kinetics: the paper's tanh forms (default) or the classic alpha/beta rate functions (model 2)")
    ap.add_argument("--update", default="joint", choices=["joint", "componentwise"], help="site update: joint D-vector proposal (default) or one component at a time (both engines)")
    ap.add_argument("--disc", default="rk4", choices=["rk4", "trapezoid"], help="model-error discretisation: the north_star's RK4 map or the paper's trapezoid rule")
    ap.add_argument("--dtype", type=int, default=64, choices=[64, 32], help="arithmetic type of the path (config 3 is also quoted in fp32)")
    ap.add_argument("--sweeps-per-step", type=int, default=1000)
    ap.add_argument("--no-other-configs", action="store_true", help="skip the other_configs block (cfg0, 1, 2, 4 and cfg3-fp32 after the headline)")
    ap.add_argument("--exchange-hold", type=int, default=None, help="SM clock ticks between publishing a Delta-A partial and the first poll (pimc_set_exchange; default: the library's)")
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle time for cpu_baseline")
    ap.add_argument("--ref-budget", type=float, default=120.0, help="seconds of oracle time for --impl reference")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        run_reference(args)
    else:
        from paper_1103_4887_b200 import build
        rank, _, world = rank_info()
        if rank == 0:
            build.build()
        run_ours(args)


if __name__ == "__main__":
    main()
