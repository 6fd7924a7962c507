#!/usr/bin/env python
"""bench.py -- GAME hot path on B200: chromosome x pattern fitness evaluations / second.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]
                  [--path auto|fp32|tensor|split] [--shard] [--no-cpu-baseline]

A *step* is one generation of the whole hot path (fused fitness of every chromosome
on every pattern, rank, stop test, elitism, selection, crossover, mutation) on the config's synthetic
workload.  `game_evolve(K)` runs K such steps plus the final re-evaluation of the returned population
(DESIGN G18); the timed region is exactly that call, so `value` counts (K+1)*N*P evaluations and
`ms_per_step` = time / K (the final evaluation is charged to the steps).  Prints ONE JSON line.
The default workload is config 5, the largest (the one north_star quotes its roofline target on); --config picks the
others.  At N > 1 every rank runs its own replica (weak scaling); --shard splits ONE problem's patterns over the ranks
instead (one all-reduce of P doubles per generation, strong scaling).

--impl reference times the fp64 CPU oracle (oracle/, as it stands) on the box's host cores on a bounded
sample of the same workload -- a deliberately slow baseline, not a target.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "chromosome x pattern fitness evaluations per second"
UNIT = "evals/s"


def read_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"],
                    bf16_tflops_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    sm_max_mhz=d.get("sm_max_mhz", 1965.0), source="measured")
    # fallback stated in B200_PROFILING.md
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, sm_max_mhz=1965.0, source="fallback")


def ncu_traffic(w, path_name):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
    `ncu --set full` capture summarised in profiles/r01_traffic.csv (null when that config was not captured)."""
    p = os.path.join(ROOT, "profiles", "r01_traffic.csv")
    if not os.path.exists(p):
        return None
    key = "%s/%s" % (w.name, path_name)
    for line in open(p).read().splitlines()[1:]:
        f = line.split(",")
        if f[0] == key:
            return float(f[1])
    return None


class ClockSampler(threading.Thread):
    """SM clock + throttle reasons DURING the timed region (profiling recipe's clocks line): NVML every 10 ms
    (nvidia-smi every 100 ms when the NVML binding is missing)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index=0):
        super().__init__(daemon=True)
        self.index = index
        self.samples = []          # (sm_mhz, sm_max_mhz, power_w, [4 flags])
        self.stop_flag = False
        self.source = "nvml"
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.masks = [pynvml.nvmlClocksEventReasonHwSlowdown, pynvml.nvmlClocksEventReasonHwThermalSlowdown,
                          pynvml.nvmlClocksEventReasonSwThermalSlowdown, pynvml.nvmlClocksEventReasonSwPowerCap]
        except Exception:
            self.nv = None
            self.source = "nvidia-smi"

    def sample(self):
        if self.nv is not None:
            nv = self.nv
            r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
            return (float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)), self.sm_max,
                    nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0, [bool(r & m) for m in self.masks])
        out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                              "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
        f = [x.strip() for x in out.strip().split(",")]
        return (float(f[0]), float(f[1]), float(f[2]), [x.lower().startswith("active") for x in f[3:7]])

    def run(self):
        while not self.stop_flag:
            try:
                self.samples.append(self.sample())
            except Exception:
                pass
            time.sleep(0.01 if self.nv is not None else 0.1)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["clock sampling unavailable"]}
        sm = sorted(s[0] for s in self.samples)
        reasons = [n for i, n in enumerate(self.NAMES) if any(s[3][i] for s in self.samples)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_min_mhz": sm[0], "sm_max_mhz": self.samples[0][1], "reasons": reasons,
                "power_w_max": max(s[2] for s in self.samples), "samples": len(self.samples), "source": self.source}


def workload_dict(w, path_name):
    return {"workload": "%s: N=%d F=%d %s d=%d K=%d P=%d" % (w.name, w.N, w.F, "trig" if w.family == 0 else "cheb",
                                                              w.degree, w.K, w.P),
            "N": w.N, "F": w.F, "K": w.K, "P": w.P, "error": ["mse", "tmse", "rmse"][w.err], "activation": "sigmoid",
            "ga": "tournament %d, crossover %.2f, mutation %.2f, elitism %d, init normal" % (
                w.tournament_size, w.p_crossover, w.p_mutation, w.elitism),
            "fitness_path": path_name,
            "l2": "inputs larger than L2 (expansion matrix re-read every step)" if w.N * w.K * 2 > 126e6
                  else "L2 flushed between timed repeats is not needed: one timed region of K back-to-back steps; working set noted",
            "parallelism": "single GPU (replicas at N>1)"}


def pick_threads(w, oracle, X, t):
    """Use all host cores unless a quick probe shows one thread is faster (CPU-quota'd containers)."""
    from paper_1304_0597_b200 import workloads as wl
    allc = oracle.set_threads(0)
    if allc == 1:
        return 1
    Ns = min(w.N, 4096)
    pop = wl.uniform_population(allc, w.K, w.seed)
    best, best_dt = allc, None
    for th in (allc, 1):
        oracle.set_threads(th)
        t0 = time.perf_counter()
        oracle.fitness(w.family, w.degree, X[:Ns], t[:Ns], pop, act=w.act, err=w.err, R=w.R)
        dt = time.perf_counter() - t0
        if best_dt is None or dt < best_dt:
            best, best_dt = th, dt
    return oracle.set_threads(best)


def cpu_sample(w, oracle, X, t, seconds_target=40.0):
    """Time the oracle as it stands on a bounded sample: all N patterns x a few chromosomes."""
    from paper_1304_0597_b200 import workloads as wl
    cores = pick_threads(w, oracle, X, t)
    pop = wl.uniform_population(max(2 * cores, 4), w.K, w.seed)
    t0 = time.perf_counter()
    oracle.fitness(w.family, w.degree, X, t, pop[:cores], act=w.act, err=w.err, R=w.R)
    probe = time.perf_counter() - t0
    ps = int(min(cores * 128, max(cores, cores * round(seconds_target / max(probe, 1e-3)))))
    pop = wl.uniform_population(ps, w.K, w.seed)
    t0 = time.perf_counter()
    oracle.fitness(w.family, w.degree, X, t, pop, act=w.act, err=w.err, R=w.R)
    dt = time.perf_counter() - t0
    return {"value": w.N * ps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "fp64 oracle fitness (expansion + contraction + error) of %d chromosomes on all N=%d patterns, %.1f s"
                      % (ps, w.N, dt)}, ps, dt


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_1304_0597_b200 import workloads as wl
    X, t, _ = wl.make(w, lambda X, c: oracle.forward(w.family, w.degree, X, c))
    cores = pick_threads(w, oracle, X, t)
    ps = max(cores, 8)
    pop = wl.uniform_population(ps, w.K, w.seed)

    def step():
        oracle.fitness(w.family, w.degree, X, t, pop, act=w.act, err=w.err, R=w.R)
    for _ in range(args.warmup if args.warmup < 2 else 1):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    val = w.N * ps * args.steps / dt
    sample = "each step = fp64 oracle fitness of %d chromosomes on all N=%d patterns (bounded sample of the P=%d population)" % (
        ps, w.N, w.P)
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": workload_dict(w, "cpu-oracle"),
                      "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
                      "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                      "gpu_launches": 0}))


def run_ours(args, w):
    import torch
    import torch.distributed as dist

    import paper_1304_0597_b200 as g
    from paper_1304_0597_b200 import workloads as wl

    from paper_1304_0597_b200 import replicas
    world, rank, local = replicas.env_world()
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = read_peaks()

    # default: replicas -- every rank runs the same-shaped problem with its own seed (weak scaling, no data-path
    # collective).  --shard: ONE problem, its patterns split over the ranks, one all-reduce of P doubles per generation
    # (strong scaling; paper_1304_0597_b200/sharded.py).
    from paper_1304_0597_b200 import sharded
    wr = w if args.shard else replicas.replica_workload(w, rank)
    lo, hi = sharded.shard_rows(w.N, world, rank) if args.shard else (0, w.N)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        # planted targets need a forward pass of the planted chromosome: the library's own game_predict
        holder = {}

        def fwd(X, c0):
            ctx0 = g.Game(wr.family, wr.degree, wr.F, stream=stream)
            ctx0.load(torch.from_numpy(X).cuda(), torch.zeros(X.shape[0], device="cuda"))
            z, y = ctx0.predict(torch.from_numpy(c0).cuda())
            stream.synchronize()
            out = (z.cpu().numpy(), y.cpu().numpy())
            ctx0.destroy()
            return out
        X, t, _ = wl.make(wr, fwd)
        ctx = g.Game(wr.family, wr.degree, wr.F, stream=stream)
        ctx.set_error(wr.err, wr.R)
        if args.path != "auto":
            ctx.set_path({"fp32": g.GAME_PATH_FP32, "tensor": g.GAME_PATH_TENSOR, "split": g.GAME_PATH_TENSOR_SPLIT}[args.path])
        Xp, tp = torch.from_numpy(X[lo:hi]).pin_memory(), torch.from_numpy(t[lo:hi]).pin_memory()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        ctx.load_host(Xp.numpy(), tp.numpy())
        e1.record(stream)
        stream.synchronize()
        load_ms = e0.elapsed_time(e1)
        path = ctx.resolved_path(wr.P)
        path_name = {g.GAME_PATH_FP32: "fp32-ffma", g.GAME_PATH_TENSOR: "tensor-tcgen05-f16",
                     g.GAME_PATH_TENSOR_SPLIT: "tensor-tcgen05-f16x3-split"}[path]
        gp = g.ga_params(P=wr.P, tournament_size=wr.tournament_size, elitism=wr.elitism, init_mode=wr.init_mode,
                         p_crossover=wr.p_crossover, p_mutation=wr.p_mutation, stop_error=-1.0)

        def barrier():
            if world > 1:
                dist.barrier()
            torch.cuda.synchronize()

        if args.shard:
            sg = sharded.ShardedGame(ctx, w.N, world)

            class _Res:
                pass

            def evolve(k):
                done, last = sg.evolve(k, wr.seed, gp)
                r = _Res()
                r.generations_run, r.best_error = done, last.best_error
                return r
        else:
            def evolve(k):
                return ctx.evolve(k, wr.seed, gp)
        evolve(max(args.warmup, 3))                             # W untimed warm-up steps (also creates the population)
        # The dominant kernel is bracketed by CUDA events inside the timed region -- except on the launch-latency
        # bound configs (1-2), where per-launch events would perturb the captured-graph loop being timed: there
        # the kernel is timed in a second, identical pass right after.
        separate_pass = float(w.N) * w.P * w.K < 2e10
        ctx.set_kernel_timing(not separate_pass)
        ctx.get_kernel_timing()
        sampler = ClockSampler(local)
        sampler.start()
        barrier()
        launches0 = ctx.launch_count()
        e0.record(stream)
        res = evolve(args.steps)                                # exactly K steps (+ the final re-evaluation)
        e1.record(stream)
        barrier()
        sampler.stop_flag = True
        ms = e0.elapsed_time(e1)
        launches = ctx.launch_count() - launches0
        kern_ms, kern_n = ctx.get_kernel_timing()
        kern_pass_ms = ms
        if separate_pass:
            ctx.set_kernel_timing(True)
            e0.record(stream)
            evolve(min(args.steps, 200))
            e1.record(stream)
            stream.synchronize()
            kern_pass_ms = e0.elapsed_time(e1)
            kern_ms, kern_n = ctx.get_kernel_timing()
        ctx.set_kernel_timing(False)
        sampler.join()
        assert res.generations_run == args.steps

        share = 1.0 / world if args.shard else 1.0             # sharded: the ranks split ONE job's evaluations
        value, ms_max = replicas.job_throughput(float(w.N) * w.P * (args.steps + 1) * share, world, ms, "cuda")

        # e2e: the same metric through the C ABI with HOST buffers: population in, fitness out, every step
        pop_host, _, _ = ctx.get_population_host()
        pop_pin = torch.from_numpy(pop_host).pin_memory()
        fit_pin = torch.empty(wr.P, dtype=torch.float32).pin_memory()
        for _ in range(2):
            ctx.fitness_host(pop_pin.numpy(), fit_pin.numpy())
        e2e_steps = max(3, min(args.steps, 10))
        barrier()
        e0.record(stream)
        for _ in range(e2e_steps):
            ctx.fitness_host(pop_pin.numpy(), fit_pin.numpy())
        e1.record(stream)
        barrier()
        e2e_value, _ = replicas.job_throughput(float(hi - lo) * w.P * e2e_steps, world, e0.elapsed_time(e1), "cuda")
        e2e = {"value": e2e_value, "unit": UNIT,
               "h2d_bytes_per_step": int(wr.P * wr.K * 4), "d2h_bytes_per_step": int(wr.P * 4),
               "what": "game_fitness_host: population from pinned host memory in, fitness back out, per step; "
                       "dataset resident (game_load_host took %.1f ms once, incl. H2D of X and the expansion)" % load_ms}

    if rank != 0:
        return
    # roofline of the dominant kernel (fused contraction + epilogue)
    flops = 2.0 * (hi - lo) * w.K * w.P           # what ONE launch of this rank's kernel computes
    avg_s = kern_ms * 1e-3 / max(kern_n, 1)
    if path in (g.GAME_PATH_TENSOR, g.GAME_PATH_TENSOR_SPLIT):
        # two candidate bounds for the fused kernel: the tensor pipe (2NKP flops) and, for shallow contractions, the
        # epilogue's special-function unit (one tanh per evaluation at 16 lanes/clk/SM, measured with a micro-benchmark:
        # 15.9).  The one with the larger floor time binds and is the one reported.
        peak = peaks["bf16_tflops_sustained"]      # fp16 in / fp32 accumulate: same rate as bf16; timed inside a long step
        mufu_peak = 148 * 16 * peaks["sm_max_mhz"] * 1e6
        # the split path executes 3 fp16 MMAs per algorithmic multiply-add and the 2-MUFU logistic (ex2 + rcp); `achieved`
        # stays ALGORITHMIC (2NKP flops, one activation per evaluation), so its fraction is bounded by 1/3 resp. 1/2
        split = path == g.GAME_PATH_TENSOR_SPLIT
        t_tensor, t_mufu = (3 if split else 1) * flops / (peak * 1e12), (2 if split else 1) * float(hi - lo) * w.P / mufu_peak
        tensor = {"bound": "tensor", "achieved": flops / avg_s / 1e12, "peak": peak, "unit": "TFLOP/s",
                  "peak_source": "MEASURED_PEAKS.json bf16_tflops_sustained (%s), fp16 = bf16 rate" % peaks["source"]}
        if t_mufu > t_tensor:
            roof = {"bound": "alu", "achieved": float(hi - lo) * w.P / avg_s / 1e9, "peak": mufu_peak / 1e9, "unit": "Gop/s",
                    "peak_source": "special-function unit: 148 SM x 16 tanh lanes/clk x sm_max_mhz (derived; binds because "
                                   "N*P/peak_mufu = %.0f us > 2NKP/peak_tensor = %.0f us)" % (t_mufu * 1e6, t_tensor * 1e6),
                    "tensor_frac": tensor["achieved"] / tensor["peak"], "tensor_tflops": tensor["achieved"]}
        else:
            roof = tensor
            roof["mufu_frac"] = (float(hi - lo) * w.P / avg_s) / mufu_peak
    else:
        peak = 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
        roof = {"bound": "alu", "achieved": flops / avg_s / 1e12, "peak": peak, "unit": "TFLOP/s",
                "peak_source": "148 SM x 128 FFMA lanes x 2 flop x sm_max_mhz (derived; a register-only FFMA micro-benchmark on B200 "
                               "reaches 72.5 TFLOP/s = 97 % of it; DESIGN.md section 7)"}
    if path == g.GAME_PATH_TENSOR_SPLIT:
        roof["executed_over_algorithmic"] = {"tensor_flops": 3, "mufu_ops": 2}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["traffic"] = ncu_traffic(w, path_name)
    roof["kernel_ms_avg"] = avg_s * 1e3
    roof["kernel_launches_timed"] = kern_n
    roof["kernel_share_of_step"] = kern_ms / kern_pass_ms
    roof["kernel_timing"] = "separate pass after the timed region (launch-bound config)" if separate_pass else "inside the timed region"

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        Xo, to, _ = wl.make(w, lambda X, c: oracle.forward(w.family, w.degree, X, c))
        cpu, _, _ = cpu_sample(w, oracle, Xo, to)

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
           "ms_per_step": ms_max / args.steps, "generations_per_sec": args.steps / (ms_max * 1e-3),
           "higher_is_better": True, "scaling": "strong" if args.shard else "weak", "vs_baseline": None,
           "dtype": {g.GAME_PATH_TENSOR: "f16 operands, f32 accumulate", g.GAME_PATH_TENSOR_SPLIT: "split f16 (hi+lo) operands, f32 accumulate",
                     g.GAME_PATH_FP32: "f32"}[path],
           "data": "synthetic", "config": dict(workload_dict(w, path_name), **({"parallelism": "patterns sharded over %d ranks, all-reduce of P doubles per generation" % world} if args.shard else {})), "clocks": sampler.summary(), "e2e": e2e,
           "gpu_launches": int(launches), "roofline": roof, "cpu_baseline": cpu,
           "best_error": float(res.best_error), "load_ms": load_ms}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config number (1-5); 5 = the largest, the one the north star's target is quoted on")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", default="auto", choices=["auto", "fp32", "tensor", "split"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--shard", action="store_true", help="N>1: split the patterns of ONE problem over the ranks (all-reduce of P doubles per generation) instead of running replicas")
    args = ap.parse_args()
    from paper_1304_0597_b200 import workloads as wl
    w = wl.config(args.config)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
