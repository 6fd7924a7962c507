"""The paper's scaling experiment (Table 3) re-run on this library, in the paper's layout.

    python -m paper_1304_0597_b200.table3 [--iterations 4000] [--sizes 0.15,16,128,512] [--degrees 1,2,4,8]

The paper trains its trigonometric model (eq. 9: 2d+1 genes, population 2*11+1 = 23, L105) for 4000 iterations on
its 2100 x 11 catalogue and on row-replicated copies of it up to 512 MB (L326), and reports device processing,
host processing and transfer times per (degree, size).  The catalogue is not available: the rows here are the
synthetic stand-in of `workloads.paper_literal` (same shape, same replication construction).  Sizes map to rows
as 0.15 MB <-> 2100 rows (the paper's own pairing).  On this library the whole loop runs on the device, so the
columns are: LOAD = game_load_host (HtoD of X and targets + expansion, once), TRAIN = game_evolve(iterations)
(fitness + rank + operators, no host round trips), TOT = both.  These shapes (K = 2d+1 <= 17 terms, P = 23) are bound by
HBM, so every row also gets its roofline: READ = the bytes the fitness kernel streams per generation (the fp32 expansion
matrix K x N built once by game_load -- L254's hoisting -- plus the N targets), ALG = the algorithmic bytes (X and the
targets: what a kernel regenerating the sums would read), GB/s = READ x generations / TRAIN, and that rate as a fraction
of the measured HBM copy bandwidth (MEASURED_PEAKS.json, else the profiling guide's 6650 GB/s fallback).  Rows whose
working set fits the 126 MB L2 can exceed the HBM figure; they are marked.  Prints a markdown table.
"""
import argparse
import sys
import time

import numpy as np


def rows_for(mb):
    return int(round(2100 * mb / 0.15)) if mb > 0.15 else 2100


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--iterations", type=int, default=4000)
    ap.add_argument("--sizes", default="0.15,16,128,512")
    ap.add_argument("--degrees", default="1,2,4,8")
    args = ap.parse_args()
    import torch

    import paper_1304_0597_b200 as g
    from paper_1304_0597_b200 import workloads as wl

    import json
    import os
    peaks = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
    hbm_gbs = json.load(open(peaks))["hbm_gbs"] if os.path.exists(peaks) else 6650.0
    print("HBM peak used: %.1f GB/s (%s)\n" % (hbm_gbs, "MEASURED_PEAKS.json" if os.path.exists(peaks) else "fallback of B200_PROFILING.md"))
    stream = torch.cuda.Stream()
    print("| degree | size (MB) | rows | LOAD (s) | TRAIN (s) | TOT (s) | generations/s | evals/s | best TMSE | READ MB/gen | ALG MB/gen | GB/s | frac of HBM | frac (ALG) |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    with torch.cuda.stream(stream):
        for d in [int(v) for v in args.degrees.split(",")]:
            for mb in [float(v) for v in args.sizes.split(",")]:
                w = wl.paper_literal(degree=d, N=rows_for(mb), generations=args.iterations)

                def fwd(X, c0):
                    c = g.Game(w.family, w.degree, w.F, stream=stream)
                    c.set_activation(w.act)
                    c.load(torch.from_numpy(X).cuda(), torch.zeros(X.shape[0], device="cuda"))
                    z, y = c.predict(torch.from_numpy(c0).cuda())
                    stream.synchronize()
                    out = (z.cpu().numpy(), y.cpu().numpy())
                    c.destroy()
                    return out
                X, t, _ = wl.make(w, fwd)
                ctx = g.Game(w.family, w.degree, w.F, stream=stream)
                ctx.set_activation(w.act)
                ctx.set_error(w.err, w.R)
                gp = g.ga_params(P=w.P, tournament_size=w.tournament_size, elitism=w.elitism, init_mode=w.init_mode,
                                 p_crossover=w.p_crossover, p_mutation=w.p_mutation, stop_error=-1.0)
                Xp, tp = torch.from_numpy(X).pin_memory(), torch.from_numpy(t).pin_memory()
                stream.synchronize()
                t0 = time.perf_counter()
                ctx.load_host(Xp.numpy(), tp.numpy())
                stream.synchronize()
                t1 = time.perf_counter()
                res = ctx.evolve(args.iterations, w.seed, gp)
                t2 = time.perf_counter()
                load, train = t1 - t0, t2 - t1
                read_b = 4.0 * w.N * (ctx.K + 1)                # fp32 expansion matrix (K x N) + targets, once per evaluation
                alg_b = 4.0 * w.N * (w.F + 1)                   # X + targets
                gbs = read_b * (args.iterations + 1) / train / 1e9
                print("| %d | %g | %d | %.4f | %.3f | %.3f | %.0f | %.3e | %.4f | %.1f | %.1f | %.0f | %.2f%s | %.2f |" % (
                    d, mb, w.N, load, train, load + train, args.iterations / train,
                    float(w.N) * w.P * (args.iterations + 1) / train, res.best_error, read_b / 1e6, alg_b / 1e6, gbs,
                    gbs / hbm_gbs, " (L2-resident)" if read_b < 126e6 else "",
                    alg_b * (args.iterations + 1) / train / 1e9 / hbm_gbs))
                sys.stdout.flush()
                ctx.destroy()
                del X, t, Xp, tp
                torch.cuda.empty_cache()


if __name__ == "__main__":
    main()
