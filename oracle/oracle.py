"""ctypes marshalling for ``game_oracle.c`` -- no arithmetic of the method lives here.

Every function cites the C routine it calls; the C routine cites the paper.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "game_oracle.c")
# GAME_ORACLE_SANITIZE=1 (set by tests/test_oracle_sanitized.py for its child pytest): the same source built with
# -fsanitize=address,undefined -O1 -g into a separate library; the child process preloads the sanitizer runtimes
_SANITIZE = os.environ.get("GAME_ORACLE_SANITIZE") == "1"
_LIB = os.path.join(_HERE, "libgame_oracle_san.so" if _SANITIZE else "libgame_oracle.so")

TRIG, CHEB, TRIG_TIED, POLY_TIED = 0, 1, 2, 3
SIGMOID, IDENTITY = 0, 1
MSE, TMSE, RMSE = 0, 1, 2
TOURNAMENT, ROULETTE = 0, 1
INIT_UNIFORM_PM1, INIT_NORMAL_PM1, INIT_UNIFORM_01 = 0, 1, 2
ELITE_COPIES_OF_BEST, ELITE_TOP_E = 0, 1


class GaParams(C.Structure):
    _fields_ = [("P", C.c_int), ("tournament_size", C.c_int), ("elitism", C.c_int),
                ("elite_mode", C.c_int), ("selection", C.c_int), ("init_mode", C.c_int),
                ("p_crossover", C.c_float), ("p_mutation", C.c_float), ("stop_error", C.c_float)]


class Result(C.Structure):
    _fields_ = [("generations_run", C.c_int), ("stopped_on_error", C.c_int),
                ("best_error", C.c_float), ("best_index", C.c_int)]


def build(force=False):
    """Compile the oracle with gcc (-O2, OpenMP). Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
               "-fno-omit-frame-pointer"] if _SANITIZE else ["-O2"]
        subprocess.check_call(["gcc"] + opt + ["-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.oracle_set_threads.restype = C.c_int
        L.oracle_num_terms.restype = C.c_int
        L.oracle_idx.restype = C.c_uint32
        L.oracle_idx.argtypes = [C.c_uint32, C.c_uint32]
        L.oracle_thr.restype = C.c_uint32
        L.oracle_thr.argtypes = [C.c_float, C.POINTER(C.c_int)]
        L.oracle_upm1.restype = C.c_float
        L.oracle_upm1.argtypes = [C.c_uint32]
        L.oracle_u01.restype = C.c_float
        L.oracle_u01.argtypes = [C.c_uint32]
        L.oracle_init_gene.restype = C.c_float
        L.oracle_init_gene.argtypes = [C.c_int, C.c_uint64, C.c_int, C.c_int]
        L.oracle_fitness.restype = C.c_int
        L.oracle_evolve.restype = C.c_int
        _lib = L
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _p(a, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def set_threads(n):
    """oracle_set_threads: set / query the OpenMP thread count used by fitness()."""
    return int(lib().oracle_set_threads(C.c_int(int(n))))


def num_terms(family, degree, F):
    return int(lib().oracle_num_terms(C.c_int(family), C.c_int(degree), C.c_int(F)))


def expand(family, degree, X):
    """oracle_expand: E[N][K] float64 (a1)."""
    X = _f32(X)
    N, F = X.shape
    K = num_terms(family, degree, F)
    E = np.empty((N, K), dtype=np.float64)
    lib().oracle_expand(C.c_int(family), C.c_int(degree), C.c_int(F), _p(X, C.c_float),
                        C.c_longlong(N), _p(E, C.c_double))
    return E


def forward(family, degree, X, genes, act=SIGMOID):
    """oracle_forward: (z, y) float64 of one chromosome on every pattern (a1-a3)."""
    X = _f32(X)
    genes = _f32(genes)
    N, F = X.shape
    assert genes.shape == (num_terms(family, degree, F),)
    z = np.empty(N, dtype=np.float64)
    y = np.empty(N, dtype=np.float64)
    lib().oracle_forward(C.c_int(family), C.c_int(degree), C.c_int(F), C.c_int(act),
                         _p(X, C.c_float), C.c_longlong(N), _p(genes, C.c_float),
                         _p(z, C.c_double), _p(y, C.c_double))
    return z, y


def fitness(family, degree, X, t, pop, act=SIGMOID, err=MSE, R=0.0, delta=None):
    """oracle_fitness: fit[P] float64 (a1-a5); with ``delta`` also the near-threshold counts."""
    X = _f32(X)
    t = _f32(t)
    pop = _f32(pop)
    N, F = X.shape
    P, K = pop.shape
    assert K == num_terms(family, degree, F) and t.shape == (N,)
    fit = np.empty(P, dtype=np.float64)
    near = np.zeros(P, dtype=np.int64)
    rc = lib().oracle_fitness(C.c_int(family), C.c_int(degree), C.c_int(F), C.c_int(act),
                              C.c_int(err), C.c_double(R), _p(X, C.c_float), _p(t, C.c_float),
                              C.c_longlong(N), _p(pop, C.c_float), C.c_int(P), _p(fit, C.c_double),
                              _p(near, C.c_longlong), C.c_double(0.0 if delta is None else delta))
    if rc:
        raise RuntimeError("oracle_fitness failed: %d" % rc)
    return fit if delta is None else (fit, near)


def classify(family, degree, X, t, genes, act=SIGMOID, cut=0.5, delta=0.0):
    """oracle_classify: (counts[TP,FP,TN,FN], (accuracy, completeness, contamination), near) -- L301."""
    X = _f32(X)
    t = _f32(t)
    genes = _f32(genes)
    N, F = X.shape
    counts = np.zeros(4, dtype=np.int64)
    fom = np.zeros(3, dtype=np.float64)
    near = C.c_longlong(0)
    lib().oracle_classify(C.c_int(family), C.c_int(degree), C.c_int(F), C.c_int(act), _p(X, C.c_float),
                          _p(t, C.c_float), C.c_longlong(N), _p(genes, C.c_float), C.c_double(cut),
                          _p(counts, C.c_longlong), _p(fom, C.c_double), C.byref(near), C.c_double(delta))
    return counts, fom, int(near.value)


def philox4x32_10(key, ctr):
    """oracle_philox4x32_10: four uint32 words for (key[2], counter[4])."""
    k = np.asarray(key, dtype=np.uint32)
    c = np.asarray(ctr, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(k, C.c_uint32), _p(c, C.c_uint32), _p(out, C.c_uint32))
    return out


def idx(w, n):
    return int(lib().oracle_idx(int(w), int(n)))


def thr(p):
    always = C.c_int(0)
    v = lib().oracle_thr(C.c_float(p), C.byref(always))
    return int(v), bool(always.value)


def upm1(w):
    return float(lib().oracle_upm1(int(w)))


def u01(w):
    return float(lib().oracle_u01(int(w)))


def init_population(mode, seed, P, K):
    """oracle_init_population: P x K float32 genes (a12)."""
    pop = np.empty((P, K), dtype=np.float32)
    lib().oracle_init_population(C.c_int(mode), C.c_uint64(seed), C.c_int(P), C.c_int(K),
                                 _p(pop, C.c_float))
    return pop


def rank(fit):
    """oracle_rank: order[P] int32, ascending (error, index), NaN last (a6)."""
    fit = _f32(fit)
    order = np.empty(fit.shape[0], dtype=np.int32)
    lib().oracle_rank(_p(fit, C.c_float), C.c_int(fit.shape[0]), _p(order, C.c_int))
    return order


def roulette_weights(fit, order):
    fit = _f32(fit)
    order = np.ascontiguousarray(order, dtype=np.int32)
    w = np.empty(fit.shape[0], dtype=np.uint32)
    lib().oracle_roulette_weights(_p(fit, C.c_float), _p(order, C.c_int), C.c_int(fit.shape[0]),
                                  _p(w, C.c_uint32))
    return w


def ga_step(gp, seed, gen, order, fit, pop, debug=False):
    """oracle_ga_step: next population from (pop, order) for absolute generation ``gen`` (a8-a11)."""
    pop = _f32(pop)
    fit = _f32(fit)
    order = np.ascontiguousarray(order, dtype=np.int32)
    P, K = pop.shape
    assert P == gp.P
    nxt = np.empty_like(pop)
    npairs = (P - gp.elitism + 1) // 2
    par = np.zeros(2 * max(npairs, 1), dtype=np.int32)
    do = np.zeros(max(npairs, 1), dtype=np.int32)
    cut = np.zeros(max(npairs, 1), dtype=np.int32)
    lib().oracle_ga_step(C.byref(gp), C.c_uint64(seed), C.c_uint32(gen), C.c_int(K),
                         _p(order, C.c_int), _p(fit, C.c_float), _p(pop, C.c_float),
                         _p(nxt, C.c_float), _p(par, C.c_int), _p(do, C.c_int), _p(cut, C.c_int))
    if debug:
        return nxt, par[:2 * npairs].reshape(npairs, 2), do[:npairs], cut[:npairs]
    return nxt


def evolve(family, degree, X, t, gp, seed, generations, act=SIGMOID, err=MSE, R=0.0, pop=None,
           gen0=0, history=False):
    """oracle_evolve: the whole training loop on the CPU.

    Returns dict(pop, fit, order, gen, result[, best_hist])."""
    X = _f32(X)
    t = _f32(t)
    N, F = X.shape
    K = num_terms(family, degree, F)
    have = pop is not None
    popbuf = _f32(pop).copy() if have else np.empty((gp.P, K), dtype=np.float32)
    fit = np.empty(gp.P, dtype=np.float32)
    order = np.empty(gp.P, dtype=np.int32)
    gen = C.c_uint32(gen0)
    res = Result()
    hist = np.full(generations + 1, np.nan, dtype=np.float32)
    rc = lib().oracle_evolve(C.c_int(family), C.c_int(degree), C.c_int(F), C.c_int(act),
                             C.c_int(err), C.c_double(R), _p(X, C.c_float), _p(t, C.c_float),
                             C.c_longlong(N), C.byref(gp), C.c_uint64(seed), C.c_int(generations),
                             _p(popbuf, C.c_float), C.c_int(1 if have else 0), C.byref(gen),
                             _p(fit, C.c_float), _p(order, C.c_int), C.byref(res),
                             _p(hist, C.c_float))
    if rc:
        raise RuntimeError("oracle_evolve failed: %d" % rc)
    out = dict(pop=popbuf, fit=fit, order=order, gen=int(gen.value), result=res)
    if history:
        out["best_hist"] = hist
    return out
