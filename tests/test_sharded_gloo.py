"""Pattern-sharded run, host logic on CPU: world_size 2, gloo backend.

The loop, the row partition and the exchange step of paper_1304_0597_b200/sharded.py run here with the fp64 oracle
standing behind the evaluate / advance callables (tests may use the oracle; the product path puts the CUDA library
there -- tests/test_gpu_parity.py runs that on the GPU)."""
import os
import socket
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    import numpy as np, torch, torch.distributed as dist
    import oracle
    from paper_1304_0597_b200 import sharded, workloads as wl
    oracle.build()
    world, rank = int(os.environ["WORLD_SIZE"]), int(os.environ["RANK"])
    dist.init_process_group("gloo")
    w = wl.config(1).scaled(P=16, generations=5)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: oracle.forward(fam, d, X, c))
    lo, hi = sharded.shard_rows(w.N, world, rank)
    Xl, tl = X[lo:hi], t[lo:hi]
    gp = oracle.GaParams(P=w.P, tournament_size=3, elitism=2, elite_mode=0, selection=0, init_mode=1,
                         p_crossover=0.9, p_mutation=0.05, stop_error=-1.0)
    state = {"pop": oracle.init_population(1, w.seed, w.P, w.K), "gen": 0, "fit": None, "order": None, "sums": [], "since": 0}

    class Res:
        generations_run = 0
        stopped_on_error = 0

    def evaluate():                      # local totals: mean over the shard x shard size (MSE-type errors)
        f = oracle.fitness(fam, d, Xl, tl, state["pop"], act=w.act, err=0, R=0.0)
        return torch.from_numpy(np.asarray(f, dtype=np.float64) * (hi - lo))

    def advance(sums, apply):
        state["sums"].append(sums.numpy().copy())
        fit = (sums.numpy() / w.N).astype(np.float32)
        order = oracle.rank(fit)
        state["fit"], state["order"] = fit, order
        if apply:
            state["pop"] = oracle.ga_step(gp, w.seed, state["gen"], order, fit, state["pop"])
            state["gen"] += 1
            state["since"] += 1

    def sync():
        r = Res()
        r.generations_run, state["since"] = state["since"], 0
        return r

    done, res = sharded.run_generations(evaluate, advance, sync, world, w.generations, poll_every=2)
    assert done == w.generations and state["gen"] == w.generations and len(state["sums"]) == w.generations + 1
    # every rank holds the same population and fitness, bit for bit
    mine = torch.from_numpy(np.concatenate([state["pop"].view(np.uint32).ravel(), state["fit"].view(np.uint32)]).astype(np.int64))
    both = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(both, mine)
    assert all(torch.equal(both[0], b) for b in both)
    # the exchanged totals are the full-data totals
    full = np.asarray(oracle.fitness(fam, d, X, t, state["pop"], act=w.act, err=0, R=0.0), dtype=np.float64) * w.N
    assert np.allclose(state["sums"][-1], full, rtol=1e-12, atol=0)
    dist.barrier()
    dist.destroy_process_group()
    print("rank", rank, "ok")
""") % ROOT


def test_shard_rows_partition():
    from paper_1304_0597_b200 import sharded
    for N in (0, 1, 7, 2100, 1000003):
        for world in (1, 2, 3, 8):
            edges = [sharded.shard_rows(N, world, r) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == N
            assert all(edges[i][1] == edges[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in edges]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        sharded.shard_rows(10, 2, 2)


def test_chunk_ranges():
    from paper_1304_0597_b200 import sharded
    import numpy as np
    X = np.zeros((10, 2), np.float32)
    t = np.zeros(10, np.float32)
    cg = sharded.ChunkedGame(None, X, t, 4)
    assert cg.chunks() == [(0, 4), (4, 8), (8, 10)] and cg.N_total == 10
    assert sharded.ChunkedGame(None, X, t, 10).chunks() == [(0, 10)]
    assert sharded.ChunkedGame(None, X, t, 99).chunks() == [(0, 10)]
    with pytest.raises(ValueError):
        sharded.ChunkedGame(None, X, t, 0)


def test_single_rank_loop_calls():
    from paper_1304_0597_b200 import sharded
    calls, st = [], {"since": 0, "stopped": 0, "polls": 0}

    class R:
        def __init__(self, g, s):
            self.generations_run, self.stopped_on_error = g, s

    def adv(s, apply):                       # a device that stops at its 3rd evaluation: later advances are no-ops
        calls.append(apply)
        if len(calls) == 3:
            st["stopped"] = 1
        if apply and not st["stopped"]:
            st["since"] += 1

    def sync():
        st["polls"] += 1
        r = R(st["since"], st["stopped"])
        st["since"] = 0
        return r
    done, res = sharded.run_generations(lambda: 0, adv, sync, 1, 10, poll_every=4)
    # the stop is noticed at the first poll (after 4 enqueued generations): 2 applied, no final evaluation
    assert done == 2 and calls == [True] * 4 and res.stopped_on_error == 1 and st["polls"] == 1
    calls.clear()
    st.update(since=0, stopped=0, polls=0)
    done, _ = sharded.run_generations(lambda: 0, lambda s, a: (calls.append(a), st.__setitem__("since", st["since"] + a)), sync, 1,
                                      2, can_stop=False)
    assert done == 2 and calls == [True, True, False] and st["polls"] == 1              # no threshold: one sync at the end


def test_two_rank_sharded_run(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), OMP_NUM_THREADS="2")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=300)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, o
        assert "rank %d ok" % r in o
