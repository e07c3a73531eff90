#!/usr/bin/env python
"""bench.py — throughput of the Beagle scoring hot path on B200 (BASELINE.json metric: GP ops/s =
tokens x fitness cases per second; % of the FP32 issue roofline).

A step = one pass of the whole hot path (offsets, per-program scan + length-sorted schedule, case
staging, fetch, interpret, reduce + tax, store: SURVEY.md §8(a) a1-a8) over one synthetic colony.
Default workload: BASELINE.json configs[2] ("paper-scale generation": P = 1,048,576, N = 512, d = 5),
the configuration north_star's target is quoted on. `--config 1..5` selects another one.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

N > 1 (torchrun, one rank per GPU): the path shards by individuals with no exchange, so
every rank scores its own colony of the same shape (weak scaling) and the value is the sum of units
over ranks divided by the slowest rank's device time. Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "gp_ops_per_sec"
UNIT = "GPops/s"            # 1 GP op = 1 token evaluated on 1 fitness case
FP32_LANES_PER_SM = 128     # 4 schedulers x 32 lanes (B200_PROFILING.md / DESIGN.md §8)


def fp32_issue_peak(sm_mhz: float, sm_count: int) -> float:
    """FP32 lane-instructions per second: the 'alu' roofline of DESIGN.md §8 (1 GP op = 1 lane-instr).
    sm_count comes from the device (cudaGetDeviceProperties), not from a constant."""
    return sm_count * FP32_LANES_PER_SM * sm_mhz * 1e6


# SURVEY.md §8(d) "Algorithmic work per unit": issue slots / MUFU-pipe instructions / shared-memory words per token x case,
# by opcode class, for the cheapest correct implementation the survey names. The f1 commands added with the same logic:
# SIGN, SQUARE one instruction, CUBE two, DUP / SWAP / DEL one move at most.
MIX_WEIGHTS = {  # name: (issue, mufu, smem words)
    "LOAD": (1, 0, 1), "CONST": (1, 0, 0), "ADD": (1, 0, 0), "SUB": (1, 0, 0), "MUL": (1, 0, 0),
    "DIV": (4, 1, 0), "SQRT": (3, 1, 0), "EXP": (3, 1, 0), "LOG": (4, 1, 0), "SIN": (2, 1, 0), "COS": (2, 1, 0),
    "SIGN": (1, 0, 0), "SQUARE": (1, 0, 0), "CUBE": (2, 0, 0), "DUP": (1, 0, 0), "SWAP": (1, 0, 0), "DEL": (0, 0, 0),
}


def mix_ceilings(token_hist):
    """Fractions of the FP32 issue roofline that the realised token mix allows: the issue ceiling
    1 / mean issue slots per GP op; the MUFU ceiling (16 lanes per clock and SM against 128: a MUFU instruction on every
    token would allow 1/8); the shared-memory ceiling (32 words per clock and SM against 128 GP ops). The binding one is the
    smallest. Commands without a weight (POW, library functions, variables: blockwise kernel) are left out and reported."""
    tot = sum(v for k, v in token_hist.items() if k in MIX_WEIGHTS)
    other = sum(v for k, v in token_hist.items() if k not in MIX_WEIGHTS)
    if tot == 0:
        return None
    issue = sum(MIX_WEIGHTS[k][0] * v for k, v in token_hist.items() if k in MIX_WEIGHTS) / tot
    mufu = sum(MIX_WEIGHTS[k][1] * v for k, v in token_hist.items() if k in MIX_WEIGHTS) / tot
    smem = sum(MIX_WEIGHTS[k][2] * v for k, v in token_hist.items() if k in MIX_WEIGHTS) / tot
    c = {"issue_slots_per_gp_op": issue, "mufu_per_gp_op": mufu, "smem_words_per_gp_op": smem,
         "issue_ceiling": 1.0 / issue if issue else None, "mufu_ceiling": 1.0 / (8.0 * mufu) if mufu else None,
         "smem_ceiling": 1.0 / (4.0 * smem) if smem else None, "tokens_without_weight": other}
    c["ceiling"] = min(v for v in (c["issue_ceiling"], c["mufu_ceiling"], c["smem_ceiling"]) if v)
    return c


def dram_traffic_table():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the ncu --set full captures
    summarised in profiles/r2_dram_traffic.csv (columns: config,fitness,kernel,dram_read_bytes,dram_write_bytes)."""
    t = {}
    try:
        with open(os.path.join(ROOT, "profiles", "r2_dram_traffic.csv")) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) >= 5 and c[0].isdigit():
                    t[(int(c[0]), c[1], c[2])] = int(c[3]) + int(c[4])
    except OSError:
        pass
    return t


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


# ------------------------------------------------------------------------------------------------
# distributed plumbing (host logic; covered by the world_size-2 gloo test)
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def dist_init(backend: str):
    import torch.distributed as dist
    rank, local_rank, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def dist_barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def dist_reduce(values, op: str, world, device="cpu"):
    """all-reduce a list of floats with 'max' or 'sum' (fp64). Identity at world == 1."""
    if world <= 1:
        return list(values)
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return t.tolist()


def rank_seed_offset(rank: int) -> int:
    """Each rank draws its own colony of the same shape (weak scaling)."""
    return 0x10000 * rank


def job_throughput(units_per_rank_step, steps, ms_local, world, device="cpu"):
    """Whole-job units/s: sum of units over ranks / max device time over ranks."""
    (ms_max,) = dist_reduce([ms_local], "max", world, device)
    (units,) = dist_reduce([float(units_per_rank_step) * steps], "sum", world, device)
    return units / (ms_max * 1e-3), ms_max


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.p = None
        self.gpu_index = gpu_index
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill(); out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        note = None
        if not sm:          # the timed region was shorter than one sampling period: one query right after it
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.gpu_index}", f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=10).stdout
                f = [x.strip() for x in out.strip().splitlines()[0].split(",")]
                sm.append(float(f[0])); mx.append(float(f[1]))
                for n, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
                note = "timed region shorter than the sampling period: one query right after it"
            except Exception:
                pass
        r = {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
             "samples": len(sm), "reasons": sorted(reasons)}
        if note:
            r["note"] = note
        return r


# ------------------------------------------------------------------------------------------------
def oracle_rate(col, n_ind, threads=None):
    """Time the oracle, as it stands, on the first n_ind individuals; returns (GPops/s, seconds, ops, threads)."""
    import numpy as np
    from oracle import binding
    threads = threads or os.cpu_count() or 1
    n_ind = min(n_ind, col.P)
    T = int(np.sum(col.lengths[:n_ind]))
    N = col.X.shape[0]
    t0 = time.perf_counter()
    binding.evaluate_parallel(col.genomes[:T], col.lengths[:n_ind], col.consts, col.X, col.y, col.tax, threads=threads)
    dt = time.perf_counter() - t0
    return T * N / dt, dt, T * N, threads


def cpu_baseline(col, target_seconds=12.0):
    """The oracle on all host cores, on a bounded leading sample of the same colony (~10-30 s of work)."""
    from oracle import binding
    binding.build()
    rate0, dt0, _, threads = oracle_rate(col, 2048)
    n = int(min(col.P, max(2048, 2048 * target_seconds / max(dt0, 1e-3))))
    rate, dt, ops, threads = oracle_rate(col, n)
    # SURVEY.md §8(d) "CPU baseline (i)": the same function on ONE thread (the oracle is single-threaded; the fan-out
    # above is wall-time plumbing), on a sample sized for a few seconds
    n1 = int(min(col.P, max(512, n / max(threads, 1) / 3)))
    rate1, dt1, ops1, _ = oracle_rate(col, n1, threads=1)
    return {"value": rate / 1e9, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"first {n} individuals of the workload ({ops / 1e9:.3f} GPops, fp64 + error bound, "
                      f"{dt:.1f} s wall on {threads} threads)",
            "one_thread": {"value": rate1 / 1e9, "unit": UNIT, "cores": 1,
                           "sample": f"first {n1} individuals ({ops1 / 1e9:.3f} GPops, {dt1:.1f} s)"}}


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    from paper_2607_06731_b200 import colonies
    from oracle import binding
    binding.build()
    cfg = colonies.CONFIGS[args.config]
    n_ind = min(cfg.P, args.ref_sample)
    col = colonies.make_colony(args.config, n_ind)
    threads = os.cpu_count() or 1
    for _ in range(args.warmup):
        oracle_rate(col, n_ind, threads)
    t_total, ops_total = 0.0, 0
    for _ in range(args.steps):
        _, dt, ops, _ = oracle_rate(col, n_ind, threads)
        t_total += dt; ops_total += ops
    value = ops_total / t_total / 1e9
    sample = f"each step = the first {n_ind} individuals of config {args.config} ({ops_total / args.steps / 1e9:.3f} GPops)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "gpu_launches": 0,
            "config": {"workload": workload_name(cfg), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


def workload_name(cfg):
    return (f"BASELINE.json configs[{cfg.number - 1}] '{cfg.name}': P={cfg.P}, N={cfg.N}, d={cfg.d}, "
            f"L<={cfg.lcap}, seeded synthetic colony (DESIGN.md §5)")


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    from paper_2607_06731_b200 import api, colonies

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    rank, local_rank, world = dist_init("nccl")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    api.lib()                                   # fails loudly if the CUDA library is missing

    cfg = colonies.CONFIGS[args.config]
    P = cfg.P if args.population is None else args.population
    tokens, lengths, consts = colonies.generate_programs(cfg, P, seed_offset=rank_seed_offset(rank), gcl_mix=args.gcl_mix)
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    Xh, yh, _ = colonies.make_dataset(cfg)
    N, d = Xh.shape
    T = int(tokens.shape[0])
    units = T * N                               # GP ops per step on this rank
    stream = torch.cuda.current_stream()
    sp = stream.cuda_stream

    X = torch.from_numpy(Xh).to(dev); y = torch.from_numpy(yh).to(dev)
    out = torch.empty(P, dtype=torch.float32, device=dev)
    resident = not (cfg.budget_bytes and args.population is None)   # config 5 does not fit its budget
    api.beagle_reserve(P if resident else 1, T)
    if resident:
        g = torch.from_numpy(tokens).to(dev); l = torch.from_numpy(lengths).to(dev)
        c = torch.from_numpy(consts).to(dev)

    # pinned host copies for the end-to-end leg (and for config 5's only leg)
    hg = torch.from_numpy(tokens).pin_memory(); hl = torch.from_numpy(lengths).pin_memory()
    hc = torch.from_numpy(consts).pin_memory()
    hout = torch.empty(P, dtype=torch.float32).pin_memory()
    budget = cfg.budget_bytes or args.e2e_budget
    api.beagle_reserve_chunked(budget)

    # --fit correlation: the paper's own objective (Eq. 1-2) on the same colony; M as the paper's
    # logs imply it, the tax at the paper's default rate M N / 85 per command
    fit_kind = {"mse": api.FIT_MSE, "correlation": api.FIT_CORRELATION, "std": api.FIT_STD, "std_hyper": api.FIT_STD_HYPER}[args.fit]
    fit_M = 10000.0
    tax = fit_M * N / 85.0 if fit_kind != api.FIT_MSE else cfg.tax

    def step_resident():
        if fit_kind == api.FIT_MSE:
            api.beagle_eval(g, l, P, c, len(consts), X, y, N, d, tax, out, sp)
        else:
            api.beagle_eval_fit(g, l, P, c, len(consts), X, y, N, d, fit_kind, fit_M, tax, out, sp)

    def step_e2e():
        if fit_kind == api.FIT_MSE:
            api.beagle_eval_chunked(hg, hl, P, hc, len(consts), X, y, N, d, tax, out, budget, sp)
        else:
            api.beagle_eval_chunked_fit(hg, hl, P, hc, len(consts), X, y, N, d, fit_kind, fit_M, tax, out, budget, sp)
        hout.copy_(out, non_blocking=True)
        stream.synchronize()

    step = step_resident if resident else step_e2e

    # ---- device-resident leg: W warm-up steps, then exactly K timed steps -------------------------
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize(); dist_barrier(world)
    clocks = ClockSampler(local_rank) if rank == 0 else None
    api.beagle_set_profiling(4)                 # CUDA events around k_eval on every 4th step of the timed region
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    launches = 0
    for _ in range(args.steps):
        step()
        launches += api.beagle_last_launch_count()
    ev1.record(stream)
    torch.cuda.synchronize(); dist_barrier(world)
    ms_local = ev0.elapsed_time(ev1)
    n_prof, eval_ms = api.beagle_profiled_eval_kernel_ms()
    _, prepass_ms = api.beagle_profiled_prepass_ms()
    api.beagle_set_profiling(False)
    counts = api.beagle_debug_counts(sp) if resident else None
    clk = clocks.stop() if clocks else None
    value, ms_max = job_throughput(units, args.steps, ms_local, world, dev)

    # ---- SURVEY.md §8(d) protocol beside the contract's K-step mean: 20 calls, CUDA events around each, median and best
    per_call = []
    if resident:
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(20)]
        for a, b in evs:
            a.record(stream); step(); b.record(stream)
        torch.cuda.synchronize()
        per_call = sorted(a.elapsed_time(b) for a, b in evs)

    # ---- end-to-end leg: pinned host buffers -> C-ABI -> result back on the host, every step -------
    for _ in range(min(args.warmup, 3)):
        step_e2e()
    torch.cuda.synchronize(); dist_barrier(world)
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        step_e2e()
    torch.cuda.synchronize()
    e2e_ms_local = (time.perf_counter() - t0) * 1e3
    dist_barrier(world)
    e2e_value, _ = job_throughput(units, e2e_steps, e2e_ms_local, world, dev)
    h2d = 4 * T + 4 * P + 4 * len(consts)
    d2h = 4 * P

    if rank != 0:
        return 0
    peaks = measured_peaks()
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    peak = fp32_issue_peak(sm_max, sm_count)
    stats = colonies.colony_stats(tokens, lengths)
    mix = mix_ceilings(stats["token_hist"])
    traffic = dram_traffic_table()
    pre_bytes = 4 * T + 4 * len(consts) + 4 * P + 16 * P          # tokens, constants, lengths, start records: read once
    n_cmd = T - stats["token_hist"]["CONST"] - stats["token_hist"]["LOAD"]     # one 8-byte micro-op record per command token
    pre_bytes_out = 8 * (n_cmd + 3 * P) + 16 * P + 16 * P + 4 * P + 8 * P    # records (+ 3 per program), start records, meta, depth, offsets
    kernel_rate = units / (eval_ms * 1e-3) if (resident and n_prof > 0 and eval_ms > 0) else None
    fit = hout.numpy()
    line = {
        "metric": METRIC, "value": value / 1e9, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg) + ("" if args.population is None else f" [first {P}]"),
                   "fitness": args.fit, "gcl_mix": args.gcl_mix,
                   "tokens": T, "gp_ops_per_step": units, "timed": "beagle_eval, inputs resident in HBM" if resident
                   else "beagle_eval_chunked from pinned host memory (the colony exceeds its device budget)",
                   "l2": f"token stream {4 * T / 1e6:.0f} MB per step vs 126 MB L2 (inputs larger than L2)"
                   if 4 * T > 126e6 else f"token stream {4 * T / 1e6:.1f} MB fits L2; no flush (ALU-bound path)",
                   "parallelism": f"dp{world} (independent colonies, no collective)"},
        "pct_of_fp32_issue_roofline": 100.0 * value / world / peak,
        "pct_of_mix_weighted_ceiling": None if not mix else 100.0 * value / world / peak / mix["ceiling"],
        "mix": mix,
        "step_ms_median_of_20": per_call[len(per_call) // 2] if per_call else None,
        "step_ms_best_of_20": per_call[0] if per_call else None,
        "prepass_counts": counts,
        "clocks": clk,
        "e2e": {"value": e2e_value / 1e9, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "via": f"beagle_eval_chunked(pinned host genomes, budget {budget >> 20} MiB) + D2H of fitness"},
        "gpu_launches": launches,
        "roofline": {"bound": "alu", "kernel": "k_eval_* (the interpreter launches of one step)",
                     "achieved": None if kernel_rate is None else kernel_rate / 1e12,
                     "peak": peak / 1e12, "unit": "T lane-instr/s (1 GP op = 1 FP32 lane-instruction)",
                     "frac": None if kernel_rate is None else kernel_rate / peak,
                     "peak_basis": f"{sm_count} SMs (device properties) x 128 FP32 lanes x {sm_max:.0f} MHz (MEASURED_PEAKS.json sm_max_mhz; DESIGN.md §8)",
                     "kernel_ms": eval_ms if n_prof else None, "kernel_launches_timed": n_prof, "kernel_share_of_step": (eval_ms / (ms_local / args.steps)) if n_prof else None,
                     "hbm_gbs_on_genome_stream": None if kernel_rate is None else (4 * T + 12 * P) / (eval_ms * 1e-3) / 1e9,
                     "traffic": traffic.get((args.config, args.fit, "k_eval")) if args.gcl_mix == "hot" else None},
        # the pre-pass (scan, sort, compile) against the HBM roofline: the token stream is read here
        "roofline_prepass": None if not (resident and n_prof > 0 and prepass_ms > 0) else {
            "bound": "hbm", "kernel": "k_len_pass1/2, k_scatter, k_compile, k_compile_general",
            "achieved": (pre_bytes + pre_bytes_out) / (prepass_ms * 1e-3) / 1e9, "peak": float(peaks.get("hbm_gbs", 6650.0)),
            "unit": "GB/s", "frac": (pre_bytes + pre_bytes_out) / (prepass_ms * 1e-3) / 1e9 / float(peaks.get("hbm_gbs", 6650.0)),
            "peak_basis": "MEASURED_PEAKS.json hbm_gbs (copy bandwidth)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)",
            "algorithmic_bytes": pre_bytes + pre_bytes_out, "prepass_ms": prepass_ms,
            "genome_stream_gbs": 4 * T / (prepass_ms * 1e-3) / 1e9,
            "traffic": traffic.get((args.config, args.fit, "k_compile")) if args.gcl_mix == "hot" else None},
        "result_check": {"finite": int(np.isfinite(fit).sum()), "nan": int(np.isnan(fit).sum()),
                         "inf": int(np.isinf(fit).sum())},
    }
    # the step that follows scoring: Monte-Carlo ranking of the fitness vector left on the device; timed on its
    # own after the main measurement (not part of `value`), against the HBM roofline: 4 bytes in + 1 byte out per individual
    if rank == 0:
        rs = torch.from_numpy(np.random.default_rng(7).integers(0, P, 100).astype(np.int64)).to(dev)
        dec = torch.empty(P, dtype=torch.uint8, device=dev); hist = torch.empty(10, dtype=torch.int64, device=dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(3):
            api.beagle_rank(out, P, rs, 100, fit_kind != api.FIT_MSE, dec, hist, sp)
        e0.record(stream)
        for _ in range(20):
            api.beagle_rank(out, P, rs, 100, fit_kind != api.FIT_MSE, dec, hist, sp)
        e1.record(stream); stream.synchronize()
        rms = e0.elapsed_time(e1) / 20
        births = float((hist.cpu().numpy() * np.array(api.TABLE2)).sum())
        line["ranking"] = {"ms": rms, "hbm_gbs": 5.0 * P / (rms * 1e-3) / 1e9, "expected_births_over_P": births / P,
                           "note": "beagle_rank (memset + k_rank) on the resident fitness vector; fits L2, launch-bound at this P"}
    if not args.no_cpu_baseline and world == 1:
        n_ind = min(P, 1 << 16)
        col = colonies.Colony(cfg, tokens[: int(lengths[:n_ind].sum())], lengths[:n_ind], consts, Xh, yh, cfg.tax)
        line["cpu_baseline"] = cpu_baseline(col, args.cpu_seconds)
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--population", type=int, default=None, help="first P individuals only (debugging; not a bench value)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--gcl-mix", default="hot", choices=["hot", "f1"],
                    help="hot: the eleven commands of BASELINE.json's configs; f1: the same trees with SIGN SQUARE CUBE and "
                         "DUP SWAP DEL woven in (SURVEY f1; not BASELINE.json's metric)")
    ap.add_argument("--fit", default="mse", choices=["mse", "correlation", "std", "std_hyper"],
                    help="fitness function; mse is BASELINE.json's metric, correlation the paper's default objective (f2)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--e2e-budget", type=int, default=64 << 20, help="device genome budget of the end-to-end leg, bytes")
    ap.add_argument("--ref-sample", type=int, default=8192, help="individuals per step of --impl reference")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: note: fewer than 3 warm-up steps is not a valid bench value", file=sys.stderr)
    _, _, world = dist_env()
    if world != args.gpus and world > 1:
        print(f"bench.py: WORLD_SIZE={world} but --gpus {args.gpus}; using WORLD_SIZE", file=sys.stderr)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
