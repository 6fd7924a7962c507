"""Pattern-sharded GA run over several GPUs, one process per GPU (the paper's future work (iii), L421).

Rank r holds rows ``shard_rows(N, world, r)`` of X and the targets.  One generation is

    sums_r = game_fitness_sums(population)          # a1-a5 on the local patterns, fp64 totals, no mean
    sums   = all_reduce(sums_r, SUM)                # THE exchange step: P doubles (80 B ... 64 KB)
    game_advance(sums, N_total, seed, params)       # mean, rank, stop test, GA operators -- replicated

The all-reduce leaves the same bits on every rank and the operators draw counter-based random numbers, so every
rank holds the same population afterwards without any further traffic.  This module is host logic only (which rows,
which calls, the reduction); every step of the method runs in the library's kernels.  The evaluate / advance steps
are passed in as callables so the same loop is exercised on CPU with ``gloo`` in the tests (tests/ may put the
oracle behind them; the product path always puts a ``Game`` context there, see ``ShardedGame``).
"""


def shard_rows(N, world, rank):
    """Contiguous, balanced row range [lo, hi) of rank `rank`: the first N % world ranks take one extra row."""
    if not (0 <= rank < world) or N < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(N, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def all_reduce_sum(t, world):
    """SUM-reduce a tensor of per-chromosome totals over the ranks, in place (no-op for one rank)."""
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t


def run_generations(evaluate, advance, sync, world, generations, final_evaluation=True, can_stop=True, poll_every=16):
    """The sharded loop.  evaluate() -> local fp64 totals (tensor of P); advance(totals, apply) ENQUEUES the rest of the
    generation and returns nothing; sync() waits and returns a result with .generations_run (applied since the previous
    sync) and .stopped_on_error.  Nothing waits on the host inside a generation: the stop flag lives on the device (once
    it fires, later advances leave the population alone) and is polled every `poll_every` generations, and only when a
    stop threshold is set at all.  Returns (generations applied, last result)."""
    done = 0
    for g in range(generations):
        advance(all_reduce_sum(evaluate(), world), True)
        if can_stop and g % poll_every == poll_every - 1:
            res = sync()
            done += res.generations_run
            if res.stopped_on_error:
                return done, res
    if final_evaluation:          # the returned fitness belongs to the returned population (DESIGN G18)
        advance(all_reduce_sum(evaluate(), world), False)
    res = sync()
    return done + res.generations_run, res


class ShardedGame:
    """A ``Game`` context per rank holding that rank's rows; `evolve` runs the loop above over the process group."""

    def __init__(self, game, N_total, world):
        self.game, self.N_total, self.world = game, int(N_total), int(world)
        game.set_global_patterns(self.N_total)      # AUTO picks the path from the global N: one tolerance class for all shards
        self._sums = None
        self._agreed = world == 1

    @classmethod
    def load(cls, family, degree, X, targets, world, rank, stream=None, configure=None):
        """X, targets: the FULL host arrays (numpy); this rank uploads only its rows."""
        import torch
        from .binding import Game
        lo, hi = shard_rows(X.shape[0], world, rank)
        if hi <= lo:
            raise ValueError("rank %d of %d would hold no pattern (N = %d)" % (rank, world, X.shape[0]))
        g = Game(family, degree, X.shape[1], stream=stream)
        if configure is not None:
            configure(g)
        g.set_global_patterns(X.shape[0])
        g.load(torch.from_numpy(X[lo:hi]).cuda(), torch.from_numpy(targets[lo:hi]).cuda())
        return cls(g, X.shape[0], world)

    def _check_same_path(self, P):
        """Every shard must evaluate on the same path (a shard whose |E| rules a tensor path out would otherwise mix
        tolerance classes into one sum)."""
        if self._agreed:
            return
        import torch
        import torch.distributed as dist
        p = torch.tensor([self.game.resolved_path(P), -self.game.resolved_path(P)], device="cuda")
        dist.all_reduce(p, op=dist.ReduceOp.MAX)
        if int(p[0]) != -int(p[1]) or int(p[0]) < 0:
            raise RuntimeError("the shards resolve to different fitness paths; set one explicitly with game_set_path")
        self._agreed = True

    def evolve(self, generations, seed, params):
        import torch
        g = self.game
        P = params.P
        # the exchange (NCCL all-reduce of P doubles) is enqueued on the context's stream like the kernels around it
        with torch.cuda.stream(g.stream):
            if g.population_size() == 0:
                # a12: every rank draws the same initial population (counter-based), no evaluation needed for it
                g.set_population(g.init_population(params.init_mode, seed, P))
            self._check_same_path(P)
            if self._sums is None or self._sums.shape[0] != P:
                self._sums = torch.empty(P, dtype=torch.float64, device="cuda")
            sums = self._sums
            return run_generations(lambda: g.fitness_sums(None, P, out=sums),
                                   lambda s, apply: g.advance(s, self.N_total, seed, params, apply, sync=False),
                                   g.sync, self.world, generations, can_stop=params.stop_error >= 0)


class ChunkedGame:
    """Out-of-core evaluation ("massive datasets ... GPU memory management", L417): the same
    decomposition in TIME instead of space.  The dataset stays in (pinned) host memory; every generation its row
    chunks pass through ONE context one after the other -- game_load(chunk) (upload + expansion), game_fitness_sums
    with its accumulate flag, so the fp64 totals add up inside the library -- before game_advance takes the mean over
    all N.  The population lives in the context and survives the loads.  Costs one upload and one expansion of the
    dataset per generation: for datasets that do not fit beside their expansion, not a fast path for those that do."""

    def __init__(self, game, X_host, t_host, rows_per_chunk):
        if rows_per_chunk < 1:
            raise ValueError("rows_per_chunk must be >= 1")
        self.game, self.X, self.t, self.rows = game, X_host, t_host, int(rows_per_chunk)
        self.N_total = X_host.shape[0]
        if game is not None:
            game.set_global_patterns(self.N_total)

    def chunks(self):
        return [(lo, min(lo + self.rows, self.N_total)) for lo in range(0, self.N_total, self.rows)]

    def totals(self, P):
        import torch
        sums = torch.empty(P, dtype=torch.float64, device="cuda")
        for i, (lo, hi) in enumerate(self.chunks()):
            self.game.load_host(self.X[lo:hi], self.t[lo:hi])
            self.game.fitness_sums(None, P, out=sums, accumulate=i > 0)
        return sums

    def evolve(self, generations, seed, params):
        g = self.game
        if g.population_size() == 0:
            g.set_population(g.init_population(params.init_mode, seed, params.P))      # a12
        return run_generations(lambda: self.totals(params.P),
                               lambda sums, apply: g.advance(sums, self.N_total, seed, params, apply, sync=False),
                               g.sync, 1, generations, can_stop=params.stop_error >= 0)
