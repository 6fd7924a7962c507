"""Seeded synthetic workloads shaped like the paper's globular-cluster data and the larger sweeps.

This module is the ONLY code shared by the CUDA path and the CPU oracle, and it holds none of
the method's arithmetic: it draws random numbers (numpy PCG64, fixed draw order) and applies
label noise.  Where a recipe needs a forward pass of a planted chromosome (configs 1, 2, 4, 5)
the caller supplies it as ``forward(X, genes) -> (z, y)`` -- the tests pass the oracle's, the
benchmark passes the library's ``game_predict``.

The paper's own data (NGC 1399 catalogue, 2100 patterns x 11 features + 0/1 target,
PAPER.md:L170-L187, L273) is not available; configs 1-2 take its shape and stand in for it,
configs 3-5 are BASELINE.json's larger sweeps.  Recipes: DESIGN.md section 4.
"""
from dataclasses import dataclass, field, replace

import numpy as np

TRIG, CHEB, TRIG_TIED, POLY_TIED = 0, 1, 2, 3
SIGMOID, IDENTITY = 0, 1
MSE, TMSE, RMSE = 0, 1, 2


@dataclass(frozen=True)
class Workload:
    name: str
    N: int
    F: int
    family: int
    degree: int
    P: int
    generations: int
    seed: int
    kind: str                 # "planted_binary" | "mixture" | "planted_regression"
    flip: float = 0.0         # label-flip probability (planted_binary)
    noise: float = 0.0        # target noise sd (planted_regression)
    act: int = SIGMOID
    err: int = TMSE
    R: float = 0.49           # the paper's TMSE threshold
    tournament_size: int = 3
    p_crossover: float = 0.9
    p_mutation: float = 0.05
    elitism: int = 2
    init_mode: int = 1        # normal in [-1, 1]
    extra: dict = field(default_factory=dict)

    @property
    def K(self):
        if self.family == TRIG_TIED:      # paper-literal eq. 7: (B*d)+1 genes with B = 2
            return 2 * self.degree + 1
        if self.family == POLY_TIED:
            return self.degree + 1
        return self.F * (2 * self.degree + 1 if self.family == TRIG else self.degree + 1)

    def scaled(self, N=None, P=None, generations=None):
        """Same recipe at a reduced size (parity cases the oracle finishes in seconds)."""
        return replace(self, N=self.N if N is None else N, P=self.P if P is None else P,
                       generations=self.generations if generations is None else generations,
                       name=self.name + "-scaled")


# BASELINE.json `configs`, in order.
CONFIGS = [
    Workload("cfg1-toy-gc", 2100, 11, TRIG, 4, 20, 100, 1, "planted_binary", flip=0.10),
    Workload("cfg2-gc-wide", 2100, 11, CHEB, 8, 1024, 2000, 2, "planted_binary", flip=0.10),
    Workload("cfg3-mid-catalogue", 100000, 16, CHEB, 6, 4096, 500, 3, "mixture"),
    Workload("cfg4-streaming", 1000000, 32, TRIG, 8, 256, 200, 4, "planted_binary", flip=0.05),
    Workload("cfg5-contraction", 250000, 64, CHEB, 12, 8192, 200, 5, "planted_regression",
             noise=0.05, err=MSE),
]


def paper_literal(degree=4, N=2100, generations=4000):
    """The paper's own experiment shape (L187, L273, L282-L291, eq. 6-7): 2100 patterns x 11 features, tied
    trigonometric model with 2d+1 genes, population 2*11+1 = 23, tournament 4, crossover 0.9, mutation 0.2,
    elitism 2, TMSE 0.49, normal initial population.  Identity output as eq. 9 prints it.  Larger N replicates
    the 2100 rows, as the paper's scaling runs do (L326)."""
    return Workload("paper-literal-d%d" % degree, N, 11, TRIG_TIED, degree, 23, generations, 1, "planted_binary",
                    flip=0.10, act=IDENTITY, tournament_size=4, p_mutation=0.2, extra={"base_rows": 2100})


def config(i):
    """1-based, as BASELINE.json / SURVEY.md number them."""
    return CONFIGS[i - 1]


def make(w, forward=None):
    """Return (X float32 [N,F], targets float32 [N], planted float32 [K] or None).

    Draw order per recipe is fixed; the same bytes go to the oracle and to the GPU library.
    """
    base = w.extra.get("base_rows")
    if base and w.N > base:             # the paper's scaling construction: replicate the catalogue's rows (L326)
        X, t, c0 = make(replace(w, N=base), forward)
        reps = -(-w.N // base)
        return np.tile(X, (reps, 1))[:w.N].copy(), np.tile(t, reps)[:w.N].copy(), c0
    rng = np.random.default_rng(w.seed)
    N, F, K = w.N, w.F, w.K
    if w.kind == "mixture":
        lab = rng.integers(0, 2, N)
        mean = np.where(lab == 1, 0.5, -0.5)[:, None]
        X = np.clip(rng.normal(mean, 0.3, (N, F)), -1.0, 1.0).astype(np.float32)
        return X, lab.astype(np.float32), None
    X = rng.uniform(-1.0, 1.0, (N, F)).astype(np.float32)
    if forward is None:
        raise ValueError("workload %s needs a forward(X, genes) -> (z, y) callable" % w.name)
    if w.kind == "planted_binary":
        c0 = rng.standard_normal(K).astype(np.float32)
        z, _ = forward(X, c0)
        t = (np.asarray(z, dtype=np.float64) > (0.0 if w.act == SIGMOID else 0.5))     # output above one half
        flips = rng.random(N) < w.flip
        t = np.where(flips, ~t, t)
        return X, t.astype(np.float32), c0
    if w.kind == "planted_regression":
        s = 2.0 / np.sqrt(K / 2.0)   # sd(z) ~ 2 so the sigmoid spans (0,1) instead of saturating
        c0 = (rng.standard_normal(K) * s).astype(np.float32)
        _, y = forward(X, c0)
        t = np.asarray(y, dtype=np.float64) + rng.normal(0.0, w.noise, N)
        return X, t.astype(np.float32), c0
    raise ValueError(w.kind)


def uniform_population(P, K, seed):
    """U[-1,1) genes for stand-alone fitness benchmarks and parity cases."""
    rng = np.random.default_rng(seed + 1000003)
    return rng.uniform(-1.0, 1.0, (P, K)).astype(np.float32)
