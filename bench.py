#!/usr/bin/env python
"""bench.py -- throughput of the GAME hot path (arXiv:1211.5481) on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3] [--impl ours|reference]

A *step* is one whole generation of the hot path over the synthetic knowledge base: fused fitness
evaluation of the population + the GA generation kernel (a6-a10), enqueued on one
stream with no host synchronisation between steps (a11).  Metric (BASELINE.json): chromosome-pattern
fitness evaluations per second = P * M * K / t.  Workload: BASELINE.json configs[3] ("c3", the config the
roofline headline is quoted on; it fits one GPU); --workload c0|c1|c2|c3 selects another.

Legs of one run (N = 1): value (inputs resident in HBM), e2e (game_generation_host: pinned host buffers,
H2D of the knowledge base + population and D2H of fitness + next population inside the timed region),
roofline (the fused fitness kernel's executed tensor flops / its CUDA-event duration, against the measured
fp16/bf16 peak of MEASURED_PEAKS.json), cpu_baseline (the oracle, as it stands, one host thread, on a bounded
sample).  N > 1: replicas only (the path is single-GPU by BASELINE.json north_star):
every rank runs the same workload on its own GPU, timing is the max over ranks, value the sum of units.
--impl reference times the CPU oracle on bounded samples of the same workload (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import workloads as wl

METRIC = "chromosome_pattern_fitness_evals_per_s"
UNIT = "evals/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the fused fitness kernel, from the `ncu --set full`
# captures summarised in profiles/ (a bench run cannot measure DRAM traffic itself: numbers taken under a profiler are not
# bench values).  Each entry names the capture it comes from and the sha-256 prefix of csrc/fitness_umma.cuh at capture
# time: when the kernel source has changed since, the figure is withheld (traffic = null) rather than repeated.
NCU_TRAFFIC = {
    "c1": {"bytes": 4666880, "source": "profiles/r02_README.md (4.67 MB read + 0 written; algorithmic 4.40 MB)", "kernel_sha": "0fd22f973aa0"},
    "c2": {"bytes": 70417408, "source": "profiles/r03_README.md (68.75 MB read + 1.67 MB written; algorithmic 68.0 MB)", "kernel_sha": "b20770215ef3"},
    "c3": {"bytes": 545894400, "source": "profiles/r03_README.md (536.24 MB read + 9.66 MB written; algorithmic 528.0 MB)", "kernel_sha": "b20770215ef3"},
}
TENSOR_FLOP_PER_CLK_PER_SM = 8192          # dense fp16/bf16 tcgen05 rate (2.25 PFLOP/s nominal = 8192 x 148 SMs x 1.86 GHz)


def kernel_sha() -> str:
    import hashlib
    with open(os.path.join(ROOT, "paper_1211_5481_b200", "csrc", "fitness_umma.cuh"), "rb") as f:
        return hashlib.sha256(f.read()).hexdigest()[:12]


def traffic_entry(name):
    e = NCU_TRAFFIC.get(name)
    if e is None:
        return None, "no ncu --set full capture of this workload"
    if e["kernel_sha"] != kernel_sha():
        return None, f"withheld: {e['source']} is a capture of another version of the kernel ({e['kernel_sha']} != {kernel_sha()})"
    return e["bytes"], f"{e['source']} (ncu --set full), not measured in this run"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c3", choices=sorted(wl.CONFIGS) + ["c4", "n1", "n1s", "n1grid"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scheme", default="auto", choices=["auto", "ffma", "f16x3"])
    ap.add_argument("--multi", default="replicas", choices=["replicas", "shard"],
                    help="N > 1: independent replicas (default), or ONE population over pattern shards with an all-reduce of M sums per generation")
    ap.add_argument("--fused", action="store_true",
                    help="small problems: time game_evolve_fused (the whole generation loop as one persistent kernel)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sweep", action="store_true",
                    help="default c3 line: leave out the `sweep` key (c0, c1, c2 and the configs[4] grid in the same process)")
    return ap.parse_args()


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return dict(FALLBACK_PEAKS), "fallback"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled every 100 ms while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.thread, self.index = [], None, None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        busy = [v for v in sm if mx and v > 0.3 * mx] or sm
        return {"sm_mhz": float(np.median(busy)) if busy else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_sample(cfg, X, t, W, p_sample: int, seed: int, gen: int):
    """One generation of the oracle (as it stands, one thread) on the first p_sample patterns."""
    import oracle
    t0 = time.perf_counter()
    F = oracle.eval_fitness(cfg.d, cfg.family, X[:p_sample], t[:p_sample], W)
    Wn = oracle.step(W, F.astype(np.float32), cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma, seed, gen)
    return time.perf_counter() - t0, Wn


def run_reference(args, cfg, rank, world):
    """--impl reference: the CPU oracle on bounded samples of the workload; rank 0 only."""
    if rank != 0:
        return
    import oracle
    oracle.build()
    p_sample = min(cfg.P, 1024 if cfg.G > 100 else 8192)
    small = wl.scaled(cfg, P=max(p_sample, 1))
    X, t, _ = wl.make_kb(small)
    W = oracle.init_population(cfg.M, cfg.G, cfg.seed)
    total = 0.0
    for i in range(args.warmup + args.steps):
        dt, W = oracle_sample(cfg, X, t, W, p_sample, cfg.seed, i)
        if i >= args.warmup:
            total += dt
    value = p_sample * cfg.M * args.steps / total
    sample = f"each step: first {p_sample} patterns x all {cfg.M} chromosomes of {cfg.name}, oracle eval + GA step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(cfg, "oracle (CPU, fp64, 1 thread)", args.gpus),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def max_over_ranks(ms: float, dist, device) -> float:
    """Multi-GPU timing rule: the job takes as long as its slowest rank."""
    if dist is None:
        return ms
    import torch
    tt = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def job_value(P: int, M: int, steps: int, world: int, ms: float) -> float:
    """Whole-job throughput: units all ranks processed / max-over-ranks time (replicas: weak scaling)."""
    return P * M * steps * world / (ms * 1e-3)


def config_dict(cfg, scheme_name, n_gpus):
    return {"workload": (f"{cfg.name}: BASELINE.json configs[{cfg.name[1:]}]" if cfg.name.startswith("c") else
                         f"{cfg.name}: the paper's own experiment shape (PAPER.md:120-136), synthetic stand-in, ranking selection" + (", shared coefficients (eq. 2)" if cfg.shared else "")), "P": cfg.P, "N": cfg.N, "d": cfg.d,
            "G": cfg.G, "M": cfg.M, "expansion": "chebyshev" if cfg.expansion == 0 else "trig",
            "activation": ["identity", "sigmoid", "tanh"][cfg.activation], "elite": cfg.elite,
            "tournament": cfg.tournament, "p_cross": cfg.p_cross, "p_mut": cfg.p_mut, "sigma": cfg.sigma,
            "scheme": scheme_name, "step": "one generation = fused fitness eval + GA step kernel",
            "parallelism": "single GPU" if n_gpus == 1 else f"{n_gpus} ranks: independent replicas by default; --multi shard = one population, patterns sharded, all-reduce of M sums per generation",
            "l2": "inputs larger than L2 (X = %.0f MB)" % (cfg.P * cfg.N * 4 / 1e6) if cfg.P * cfg.N * 4 > 126e6
                  else "L2 flushed between timed steps is not possible inside a no-sync generation loop; inputs fit L2"}


def roofline_of(cfg, game, scheme, fused, kernel_ms, kernel_n, loop_ms, steps, peaks, peaks_src, clocks):
    """Roofline object of the dominant kernel.  `peak` is the measured figure the contract names (sustained bf16 = fp16
    rate for a kernel timed inside a long step loop); because a run under the power cap can exceed a cuBLAS-derived
    figure, the fractions against the burst figure and against the clock-scaled hardware rate are printed beside it."""
    if fused:      # one persistent kernel = the whole timed region: fp32 FFMA arithmetic, 2 P M G flop per generation
        flops_per_launch = 2.0 * cfg.P * cfg.M * cfg.G * steps
        kernel_ms, kernel_n = loop_ms, 1
    elif scheme == game.SCHEME_F16X3:
        flops_per_launch = 6.0 * cfg.P * cfg.M * (cfg.G - 1)     # 3 MMAs per gene; the bias gene rides on the epilogue
    else:
        flops_per_launch = 2.0 * cfg.P * cfg.M * cfg.G
    avg_s = kernel_ms * 1e-3 / max(kernel_n, 1)
    achieved = flops_per_launch / avg_s / 1e12 if avg_s > 0 else 0.0
    tensor = scheme == game.SCHEME_F16X3 and not fused
    sm_mhz = (clocks or {}).get("sm_mhz") or float(peaks.get("sm_max_mhz", 1965.0))
    if tensor:
        peak = float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
        burst = float(peaks["bf16_tflops"])
        clock_peak = TENSOR_FLOP_PER_CLK_PER_SM * 148 * sm_mhz * 1e6 / 1e12
        peak_note = (f"{peaks_src} bf16_tflops_sustained (fp16 and bf16 share the kind::f16 rate; kernel timed inside a step loop)")
        bound = "tensor"
        extra = {"frac_of_burst": achieved / burst, "peak_burst": burst,
                 "frac_of_clock_scaled_peak": achieved / clock_peak, "peak_clock_scaled": clock_peak,
                 "peak_clock_scaled_note": f"{TENSOR_FLOP_PER_CLK_PER_SM} flop/clk/SM x 148 SMs x the SM clock sampled in the step loop ({sm_mhz:.0f} MHz): the ceiling at this clock",
                 "useful_tflops": achieved / 3.0}
    else:
        peak = 148 * 128 * 2 * 1.965e9 / 1e12
        peak_note = "derived fp32 FFMA peak: 148 SM x 128 lanes x 2 flop x 1.965 GHz"
        bound = "alu"
        extra = {}
    traffic, traffic_source = traffic_entry(cfg.name) if tensor else (None, "not captured")
    mufu_per_eval = 0.0 if (cfg.activation == wl.ACT_IDENTITY or fused) else 1.25
    fr = {"tensor": achieved / peak if tensor else 0.0,
          "mufu": mufu_per_eval * cfg.P * cfg.M / avg_s / (148 * 16 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6) if avg_s > 0 else 0.0,
          "hbm": 4 * (cfg.P * (cfg.N + 1)) / avg_s / 1e9 / float(peaks["hbm_gbs"]) if avg_s > 0 else 0.0}
    out = {"bound": bound, "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
           "traffic": traffic, "traffic_source": traffic_source,
           "kernel": "ga_fused_kernel" if fused else ("fitness_umma_kernel" if tensor else "fitness_ffma_kernel"),
           "kernel_ms_avg": avg_s * 1e3, "kernel_launches_timed": kernel_n,
           "kernel_share_of_step": (avg_s * 1e3) / (loop_ms / steps) if loop_ms > 0 else None,
           "flops_per_launch": flops_per_launch, "peak_source": peak_note,
           "hbm_algorithmic_bytes_per_launch": 4 * (cfg.P * (cfg.N + 1)),
           "mufu_frac_at_max_clock": fr["mufu"], "hbm_frac_of_measured": fr["hbm"],
           "binding_unit": max(fr, key=fr.get) if tensor else "alu"}
    out.update(extra)
    return out


def sweep_points(args, game, torch, peaks, peaks_src):
    """The other BASELINE.json configurations in the same process: c0, c1, c2 as generation loops (device-resident,
    uninstrumented loop + an instrumented pass for the kernel time) and the configs[4] fitness-kernel grid."""
    pts = []
    # timed windows of 50-150 ms: with 400 steps c0 was timed over 5 ms and c1 over 20 ms, right after the host-side
    # generation of their knowledge bases, and c1 came out at 50 or 60 us per generation from run to run
    for name, steps, warmup in (("c0", 4000, 400), ("c1", 2000, 200), ("c2", 200, 20)):
        cfg = wl.CONFIGS[name]
        X, t, _ = wl.make_kb(cfg)
        G = game.Game(cfg.P, cfg.N, cfg.d, cfg.M, cfg.expansion, cfg.activation)
        G.set_ga_params(cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma)
        G.load_kb(X, t)
        G.init_population(cfg.seed)
        game.game_evolve(G.ctx, cfg.seed, 0, warmup)
        torch.cuda.synchronize()
        sampler = ClockSampler(0)
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = G.launch_count()
        e0.record()
        game.game_evolve(G.ctx, cfg.seed, warmup, steps)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        launches = G.launch_count() - l0
        clocks = sampler.stop()
        game.game_time_fitness_kernel(G.ctx, True)
        game.game_evolve(G.ctx, cfg.seed, warmup + steps, min(steps, 50))
        torch.cuda.synchronize()
        kms, kn = game.game_fitness_kernel_ms(G.ctx)
        game.game_time_fitness_kernel(G.ctx, False)
        rf = roofline_of(cfg, game, G.scheme(), False, kms, kn, ms, steps, peaks, peaks_src, clocks)
        pts.append({"workload": f"{name}: BASELINE.json configs[{name[1:]}]", "P": cfg.P, "G": cfg.G, "M": cfg.M, "steps": steps,
                    "evals_per_s": cfg.P * cfg.M * steps / (ms * 1e-3), "generations_per_s": steps / (ms * 1e-3),
                    "ms_per_step": ms / steps, "gpu_launches": int(launches), "kernel_ms": rf["kernel_ms_avg"],
                    # everything of a generation that is not the fused fitness kernel: finalisation, GA step, launch gaps and,
                    # for regression outputs (c2), the calibration launches, which kernel_ms does not include
                    "other_ms_per_step": ms / steps - rf["kernel_ms_avg"],
                    "calibration": "3 launches per evaluation, outside kernel_ms" if cfg.activation != wl.ACT_SIGMOID else "none",
                    "tensor_tflops": rf["achieved"], "tensor_frac_of_sustained": rf["frac"], "tensor_frac_of_burst": rf.get("frac_of_burst"),
                    "mufu_frac_at_max_clock": rf["mufu_frac_at_max_clock"], "hbm_frac": rf["hbm_frac_of_measured"],
                    "binding_unit": "launch latency" if name in ("c0", "c1") else rf["binding_unit"], "clocks": clocks,
                    "l2": "X fits L2 (not flushed: the loop has no host sync)"})
        G.close()
    # configs[4]: fitness kernel only, M x P grid
    big = wl.c4(max(wl.C4_M), max(wl.C4_P))
    X, t, _ = wl.make_kb(big)
    Xd, td = torch.from_numpy(X).cuda(), torch.from_numpy(t).cuda()
    for M in wl.C4_M:
        W = torch.from_numpy(wl.uniform_population(M, big.G, seed=4)).cuda()
        for P in wl.C4_P:
            pts.append(c4_point(game, torch, big, M, P, Xd, td, W, max(args.warmup, 3), 5, peaks))
    return pts


def c4_point(game, torch, big, M, P, Xd, td, W, warmup, steps, peaks):
    G = game.Game(P, big.N, big.d, M, big.expansion, big.activation)
    G.X.copy_(Xd[:P]); G.t.copy_(td[:P]); G.set_population(W)
    for _ in range(warmup):
        game.game_eval_fitness(G.ctx)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    game.game_time_fitness_kernel(G.ctx, True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = G.launch_count()
    e0.record()
    for _ in range(steps):
        game.game_eval_fitness(G.ctx)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    kms, kn = game.game_fitness_kernel_ms(G.ctx)
    game.game_time_fitness_kernel(G.ctx, False)
    clocks = sampler.stop()
    launches = G.launch_count() - launches0      # the library's own count (fitness + finalize per evaluation)
    tf = 6.0 * P * M * (big.G - 1) / (kms / kn * 1e-3) / 1e12
    fr = {"tensor": tf / float(peaks["bf16_tflops"]),
          # epilogue: 1.25 MUFU per evaluation (ex2 each, one rcp per four), 16 MUFU lanes per SM per clock
          "mufu": 1.25 * P * M / (kms / kn * 1e-3) / (148 * 16 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6),
          "hbm": 4.0 * P * (big.N + 1) / (kms / kn * 1e-3) / 1e9 / float(peaks["hbm_gbs"])}
    G.close()
    return {"workload": "c4: BASELINE.json configs[4] (fitness kernel only)", "M": M, "P": P, "G": big.G, "ms_per_eval": ms,
            "evals_per_s": P * M / (ms * 1e-3), "kernel_ms": kms / kn, "gpu_launches": int(launches),
            "tensor_tflops": tf, "tensor_frac_of_burst": fr["tensor"], "tensor_frac": fr["tensor"],
            "mufu_frac_at_max_clock": fr["mufu"], "hbm_frac": fr["hbm"], "binding_unit": max(fr, key=fr.get),
            "sm_mhz": clocks.get("sm_mhz"), "l2": "X larger than L2" if P * big.N * 4 > 126e6 else "X fits L2 (not flushed)"}


def run_ours(args, cfg, rank, world, local_rank):
    import torch
    import paper_1211_5481_b200 as game
    from paper_1211_5481_b200 import build as game_build

    if rank == 0:
        game_build.build()
    dist = None
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
        dist.barrier()
    dev = f"cuda:{local_rank}"
    torch.cuda.set_device(local_rank)
    scheme = {"auto": game.SCHEME_AUTO, "ffma": game.SCHEME_FFMA, "f16x3": game.SCHEME_F16X3}[args.scheme]
    X, t, _ = wl.make_kb(cfg, seed=cfg.seed + 1000 * rank)           # every replica its own knowledge base
    G = game.Game(cfg.P, cfg.N, cfg.d, cfg.M, cfg.expansion, cfg.activation, device=dev, scheme=scheme, shared=cfg.shared)
    G.set_ga_params(cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma)
    scheme_name = {game.SCHEME_FFMA: "FFMA fp32", game.SCHEME_F16X3: "F16X3 (3 x tcgen05 kind::f16, 2-term fp16 split, fp32 accumulate)"}[G.scheme()]
    G.load_kb(X, t)
    if cfg.name in ("n1", "n1s"):             # the paper's settings: ranking selection
        game.game_set_selection(G.ctx, game.SEL_RANKING)
    seed = cfg.seed
    G.init_population(seed)
    G.sync()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    shard = dist is not None and args.multi == "shard"
    if shard:
        ident = [game.game_comm_unique_id() if rank == 0 else None]
        dist.broadcast_object_list(ident, src=0)
        game.game_comm_init(G.ctx, ident[0], rank, world)

    def generations(first_gen, n):
        if args.fused:
            game.game_evolve_fused(G.ctx, seed, first_gen, n, None)   # one persistent kernel for all n generations
            return
        if not shard:
            game.game_evolve(G.ctx, seed, first_gen, n)      # n x (fused fitness eval, GA step): launches only
            return
        # one population, patterns sharded over the ranks: the whole loop runs inside the library -- per generation the
        # evaluation kernels, ONE ncclAllReduce of M doubles on the library's stream, finalisation, GA step; no Python
        game.game_evolve_sharded(G.ctx, seed, first_gen, n, cfg.P * world, None)

    # ---------------- device-resident leg: NO instrumentation inside the timed region (the generation loop is replayed from
    # a CUDA graph / runs under programmatic dependent launch; per-kernel events would sit inside the chain they overlap)
    generations(0, args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    launches0 = G.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    generations(args.warmup, args.steps)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = G.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    ms = max_over_ranks(ms, dist, dev)
    units = cfg.P * cfg.M * args.steps * world
    value = job_value(cfg.P, cfg.M, args.steps, world, ms)
    # ---------------- the dominant kernel's own duration: a second, instrumented pass over the same steps (CUDA events on
    # the library's stream around every launch of the fused fitness kernel; plain launches, no graph)
    kernel_ms, kernel_n = 0.0, 0
    if not args.fused and not shard:
        n_k = min(args.steps, 50)
        game.game_time_fitness_kernel(G.ctx, True)
        generations(args.warmup + args.steps, n_k)
        barrier()
        kernel_ms, kernel_n = game.game_fitness_kernel_ms(G.ctx)
        game.game_time_fitness_kernel(G.ctx, False)

    # ---------------- end-to-end leg: host buffers through game_generation_host
    e2e = None
    if not args.no_e2e:
        Xh, th = torch.from_numpy(X).pin_memory(), torch.from_numpy(t).pin_memory()
        Wh = [torch.empty((cfg.M, cfg.G), dtype=torch.float32).pin_memory() for _ in range(2)]
        Fh = torch.empty(cfg.M, dtype=torch.float32).pin_memory()
        Wh[0].copy_(G.current().cpu())

        def host_generations(first_gen, n, k0):
            for i in range(n):
                a, b = Wh[(k0 + i) & 1], Wh[(k0 + i + 1) & 1]
                game.game_generation_host(G.ctx, Xh.data_ptr(), th.data_ptr(), a.data_ptr(), Fh.data_ptr(), b.data_ptr(),
                                          seed, first_gen + i)
        w = max(1, min(args.warmup, 3))
        host_generations(10_000, w, 0)
        barrier()
        t0 = time.perf_counter()
        e0.record()
        host_generations(10_000 + w, args.steps, w)
        e1.record()
        barrier()
        ms_e2e = max(e0.elapsed_time(e1), 0.0)
        wall_ms = (time.perf_counter() - t0) * 1e3
        ms_e2e = max(ms_e2e, 0.0) if ms_e2e > 0 else wall_ms
        ms_e2e = max_over_ranks(ms_e2e, dist, dev)
        e2e = {"value": units / (ms_e2e * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": 4 * (cfg.P * cfg.N + cfg.P + cfg.M * cfg.G) * world,
               "d2h_bytes_per_step": 4 * (cfg.M + cfg.M * cfg.G) * world, "ms_per_step": ms_e2e / args.steps,
               "api": "game_generation_host (pinned host buffers; H2D X,t,W + eval + step + D2H F,W' per step)"}

    # ---------------- out-of-core leg: the same evaluation with the knowledge base in pinned
    # host memory and only a 64 MB ring of device buffers, game_eval_fitness_streamed
    out_of_core = None
    if not args.no_e2e and world == 1 and cfg.name == "c3" and G.scheme() == game.SCHEME_F16X3:
        n_slots = 3
        quantum = 256 * 74
        slot_rows = max(quantum, (64 << 20) // (4 * (cfg.N + 1)) // n_slots // quantum * quantum)
        Xr = torch.empty((n_slots * slot_rows, cfg.N), dtype=torch.float32, device=dev)
        tr = torch.empty((n_slots * slot_rows,), dtype=torch.float32, device=dev)
        F_res = None
        game.game_eval_fitness(G.ctx); G.sync(); F_res = G.get_fitness()

        def streamed(n):
            for _ in range(n):
                game.game_eval_fitness_streamed(G.ctx, Xh.data_ptr(), th.data_ptr(), Xr.data_ptr(), tr.data_ptr(), slot_rows, n_slots)
        streamed(2)
        barrier()
        n_ev = max(3, min(args.steps, 10))
        e0.record()
        streamed(n_ev)
        e1.record()
        barrier()
        ms_oc = e0.elapsed_time(e1) / n_ev
        out_of_core = {"api": "game_eval_fitness_streamed (fitness evaluation only; knowledge base in pinned host memory)",
                       "ring_bytes": int(Xr.numel() * 4 + tr.numel() * 4), "slots": n_slots, "slot_rows": int(slot_rows),
                       "kb_bytes": 4 * cfg.P * (cfg.N + 1), "ms_per_eval": ms_oc, "evals_per_s": cfg.P * cfg.M / (ms_oc * 1e-3),
                       "h2d_gb_per_s": 4 * cfg.P * (cfg.N + 1) / (ms_oc * 1e-3) / 1e9,
                       "bit_identical_to_resident": bool(np.array_equal(G.get_fitness().view(np.uint32), F_res.view(np.uint32)))}
        del Xr, tr

    if rank != 0:
        G.close()
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---------------- roofline of the dominant kernel (fused fitness)
    peaks, peaks_src = load_peaks()
    fused = args.fused
    roofline = roofline_of(cfg, game, G.scheme(), fused, kernel_ms, kernel_n, ms, args.steps, peaks, peaks_src, clocks)
    bound = roofline["bound"]

    # ---------------- CPU baseline: the oracle as it stands, one thread, bounded sample
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        p_sample = int(min(cfg.P, max(256, 8e7 * 321 / cfg.G / cfg.M)))        # ~10-30 s of CPU work
        W0 = oracle.init_population(cfg.M, cfg.G, seed)
        dt, _ = oracle_sample(cfg, X, t, W0, p_sample, seed, 0)
        cpu = {"value": p_sample * cfg.M / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
               "precision": "fp64, ONE thread, plain loops (the parity oracle as it stands; not a tuned or multi-core CPU baseline)",
               "host_cores_available": os.cpu_count(),
               "sample": f"one generation (oracle eval + GA step) on the first {p_sample} patterns x all {cfg.M} chromosomes of {cfg.name}"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f16x3->f32" if bound == "tensor" else "f32", "data": "synthetic",
            "config": config_dict(cfg, scheme_name, world), "generations_per_s": args.steps / (ms * 1e-3),
            "e2e": e2e, "gpu_launches": int(launches), "graph_replays": int(game.game_graph_replays(G.ctx)),
            "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu}
    if out_of_core is not None:
        line["out_of_core"] = out_of_core
    G.close()
    # ---------------- the other BASELINE.json configurations, same process, same box (default c3 line, one GPU only)
    if world == 1 and cfg.name == "c3" and not args.no_sweep and not args.fused:
        del X, t
        line["sweep"] = sweep_points(args, game, torch, peaks, peaks_src)
        line["sweep_note"] = ("c0/c1/c2: generation loops (game_evolve, device-resident, no instrumentation in the timed loop; kernel_ms "
                              "from a separate instrumented pass); c4: game_eval_fitness only, every point timed alone against the burst peak; "
                              "peaks: " + peaks_src + " MEASURED_PEAKS.json; c0 / c1 / c2 are timed over 50-150 ms right after the power-capped c3 leg: "
                              "their `clocks` say at which SM clock (c0 alone on a cool GPU: 72-74 k generations/s at 1965 MHz)")
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_c4_sweep(args):
    """BASELINE.json configs[4]: fitness-kernel sweep (no GA step), M x P grid at N=20, d=6 (G=121).  One JSON line:
    `value` is the largest point; `sweep` lists evals/s and the tensor / HBM roofline fractions of every point."""
    import torch
    import paper_1211_5481_b200 as game
    from paper_1211_5481_b200 import build as game_build

    game_build.build()
    peaks, peaks_src = load_peaks()
    big = wl.c4(max(wl.C4_M), max(wl.C4_P))
    X, t, _ = wl.make_kb(big)
    Xd, td = torch.from_numpy(X).cuda(), torch.from_numpy(t).cuda()
    sweep, launches = [], 0
    for M in wl.C4_M:
        W = torch.from_numpy(wl.uniform_population(M, big.G, seed=4)).cuda()
        for P in wl.C4_P:
            pt = c4_point(game, torch, big, M, P, Xd, td, W, max(args.warmup, 3), args.steps, peaks)
            launches += pt["gpu_launches"]
            sweep.append(pt)
    mhz = [p_["sm_mhz"] for p_ in sweep if p_.get("sm_mhz")]
    clocks = {"sm_mhz": float(np.median(mhz)) if mhz else None, "sm_max_mhz": float(peaks.get("sm_max_mhz", 1965.0)),
              "reasons": ["per-point clocks in sweep[].sm_mhz"]}
    last = sweep[-1]
    line = {"metric": METRIC, "value": last["evals_per_s"], "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": last["ms_per_eval"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f16x3->f32", "data": "synthetic",
            "config": {"workload": "c4: BASELINE.json configs[4] fitness-kernel sweep (no GA step); value = largest point",
                       "N": big.N, "d": big.d, "G": big.G, "M": list(wl.C4_M), "P": list(wl.C4_P),
                       "peak": f"{peaks_src} bf16_tflops (burst: every point is timed alone)"},
            "e2e": None, "gpu_launches": launches, "clocks": clocks, "sweep": sweep,
            "roofline": {"bound": "tensor", "achieved": last["tensor_tflops"], "peak": float(peaks["bf16_tflops"]), "unit": "TFLOP/s",
                         "frac": last["tensor_frac"], "traffic": None}, "cpu_baseline": None}
    print(json.dumps(line), flush=True)


def run_n1_grid(args):
    """the paper's own experiment grid as generations/s -- P = 2100 synthetic patterns,
    N in {7, 9} feature columns, polytrigo degree in {1, 2, 4, 8}, RANKING and ROULETTE selection,
    crossover 0.9, mutation 0.2, elitism 2, B N + 1 chromosomes (B = 2), per-feature coefficients (BASELINE.json's form) and
    the paper's shared coefficients; both execution paths: the launch chain replayed from a CUDA graph (game_evolve) and the
    persistent whole-GA kernel (game_evolve_fused)."""
    import torch
    import paper_1211_5481_b200 as game
    from paper_1211_5481_b200 import build as game_build
    from dataclasses import replace

    game_build.build()
    rows = []
    steps, warmup = max(args.steps, 2000), 200
    for N in (7, 9):
        for d in (1, 2, 4, 8):
            for shared in (False, True):
                cfg = replace(wl.PAPER_SHAPE, name="n1grid", N=N, d=d, M=2 * N + 1, shared=shared, w_star_std=0.1 if shared else 0.3)
                X, t, _ = wl.make_kb(cfg)
                for sel_name, sel in (("ranking", game.SEL_RANKING), ("roulette", game.SEL_ROULETTE)):
                    G = game.Game(cfg.P, cfg.N, cfg.d, cfg.M, cfg.expansion, cfg.activation, shared=shared)
                    G.set_ga_params(cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma)
                    game.game_set_selection(G.ctx, sel)
                    G.load_kb(X, t)
                    res = {}
                    for path in ("graph", "fused"):
                        G.init_population(cfg.seed)
                        fn = (lambda g0, n: game.game_evolve(G.ctx, cfg.seed, g0, n)) if path == "graph" else \
                             (lambda g0, n: game.game_evolve_fused(G.ctx, cfg.seed, g0, n, None))
                        fn(0, warmup)
                        torch.cuda.synchronize()
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record(); fn(warmup, steps); e1.record()
                        torch.cuda.synchronize()
                        res[path] = steps / (e0.elapsed_time(e1) * 1e-3)
                    rows.append({"N": N, "degree": d, "G": cfg.G, "M": cfg.M, "coefficients": "shared" if shared else "per-feature",
                                 "selection": sel_name, "generations_per_s_graph": res["graph"], "generations_per_s_fused": res["fused"],
                                 "us_per_40000_iterations_fused": 40000 / res["fused"] * 1e6})
                    G.close()
    best = max(r["generations_per_s_fused"] for r in rows)
    line = {"metric": "generations_per_s", "value": best, "unit": "generations/s", "n_gpus": 1, "steps": steps, "warmup": warmup,
            "ms_per_step": 1e3 / best, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": {"workload": "n1grid: the paper's experiment grid (PAPER.md:128-136), synthetic stand-in, P = 2100"},
            "e2e": None, "gpu_launches": None, "grid": rows, "roofline": None, "cpu_baseline": None}
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus > 1 and world == 1 and args.impl == "ours":
        import socket
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if args.workload == "c4":
        if int(os.environ.get("RANK", "0")) == 0:
            run_c4_sweep(args)
        return
    if args.workload == "n1grid":
        if int(os.environ.get("RANK", "0")) == 0:
            run_n1_grid(args)
        return
    cfg = {"n1": wl.PAPER_SHAPE, "n1s": wl.PAPER_SHAPE_SHARED}.get(args.workload) or wl.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, cfg, rank, world)
    else:
        run_ours(args, cfg, rank, world, local_rank)


if __name__ == "__main__":
    main()
