"""Thin ctypes binding over libgame_b200.so -- argument marshalling only.

Every function has the name and meaning of the C entry point in ``include/game.h`` (product API) or
``include/game_bench.h`` (measurement aids); every step of
the path runs in the library's CUDA kernels.  Device arrays are ``torch`` CUDA tensors (torch is used
for device memory and streams only), host arrays are numpy.  There is no CPU fallback: if the
library is missing or no CUDA device is present the calls raise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgame_b200.so")

GAME_TRIG, GAME_CHEB, GAME_TRIG_TIED, GAME_POLY_TIED = 0, 1, 2, 3
GAME_ACT_SIGMOID, GAME_ACT_IDENTITY = 0, 1
GAME_ERR_MSE, GAME_ERR_TMSE, GAME_ERR_RMSE = 0, 1, 2
GAME_SEL_TOURNAMENT, GAME_SEL_ROULETTE = 0, 1
GAME_INIT_UNIFORM_PM1, GAME_INIT_NORMAL_PM1, GAME_INIT_UNIFORM_01 = 0, 1, 2
GAME_ELITE_COPIES_OF_BEST, GAME_ELITE_TOP_E = 0, 1
GAME_PATH_AUTO, GAME_PATH_FP32, GAME_PATH_TENSOR, GAME_PATH_TENSOR_SPLIT = 0, 1, 2, 3
GAME_EXPAND_AUTO, GAME_EXPAND_MATERIALIZED, GAME_EXPAND_REGENERATED = 0, 1, 2
(GAME_TUNE_PDL, GAME_TUNE_CTA_GROUP, GAME_TUNE_SIGMOID, GAME_TUNE_RESIDENT, GAME_TUNE_TEAMS, GAME_TUNE_HALF_TILES,
 GAME_TUNE_PERSISTENT, GAME_TUNE_RATIONAL_SHARE) = range(8)
GAME_PEAK_FFMA, GAME_PEAK_FFMA2, GAME_PEAK_TANH, GAME_PEAK_EX2, GAME_PEAK_TANH_MIX = range(5)
ERROR_NAMES = {1: "INVALID_ARG", 2: "NOT_LOADED", 3: "ALLOC", 4: "CUDA", 5: "UNSUPPORTED", 6: "NONFINITE_INPUT"}

# every symbol include/game.h and include/game_bench.h declare (tests check the library exports exactly these)
SYMBOLS = [
    "game_create", "game_destroy", "game_num_terms", "game_generation", "game_last_error",
    "game_set_stream", "game_set_activation", "game_set_error", "game_set_path", "game_resolved_path",
    "game_set_expansion", "game_resolved_expansion", "game_fitness_sums", "game_advance", "game_sync",
    "game_set_tuning", "game_set_global_patterns", "game_predict_new", "game_population_size",
    "game_load", "game_load_host", "game_fitness", "game_fitness_host", "game_predict", "game_classify",
    "game_set_population", "game_set_generation", "game_evolve", "game_get_population",
    "game_get_population_host", "game_rank", "game_ga_step", "game_init_population", "game_philox",
    "game_launch_count", "game_set_kernel_timing", "game_get_kernel_timing", "game_microbench",
    "game_rank_static", "game_rank_static_error",
]
GAME_RANK_STATIC_MAX_P = 65536


class game_ga_params(C.Structure):
    _fields_ = [("P", C.c_int), ("tournament_size", C.c_int), ("elitism", C.c_int),
                ("elite_mode", C.c_int), ("selection", C.c_int), ("init_mode", C.c_int),
                ("p_crossover", C.c_float), ("p_mutation", C.c_float), ("stop_error", C.c_float)]


class game_result(C.Structure):
    _fields_ = [("generations_run", C.c_int), ("stopped_on_error", C.c_int),
                ("best_error", C.c_float), ("best_index", C.c_int)]


class GameError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libgame_b200: %s (%d): %s" % (ERROR_NAMES.get(code, "?"), code, msg))
        self.code = code


_lib = None


def load_library():
    """dlopen the in-tree library; fails loudly when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            # a fresh checkout: compile the CUDA library once (nvcc, sm_100a); there is no CPU fallback to fall to
            try:
                from . import build
                build.build_library()
            except Exception as e:
                raise ImportError("%s not found and building it failed (%s): run `python -m paper_1304_0597_b200.build`"
                                  % (LIB_PATH, e))
        L = C.CDLL(LIB_PATH)
        vp, ll, i, u64 = C.c_void_p, C.c_longlong, C.c_int, C.c_uint64
        L.game_create.argtypes = [i, i, i, C.POINTER(vp)]
        L.game_destroy.argtypes = [vp]
        L.game_destroy.restype = None
        L.game_num_terms.argtypes = [vp]
        L.game_generation.argtypes = [vp]
        L.game_generation.restype = ll
        L.game_last_error.argtypes = [vp]
        L.game_last_error.restype = C.c_char_p
        L.game_launch_count.argtypes = [vp]
        L.game_launch_count.restype = ll
        L.game_set_stream.argtypes = [vp, vp]
        L.game_set_activation.argtypes = [vp, i]
        L.game_set_error.argtypes = [vp, i, C.c_float]
        L.game_set_path.argtypes = [vp, i]
        L.game_resolved_path.argtypes = [vp, i]
        L.game_fitness_sums.argtypes = [vp, vp, i, vp, i]
        L.game_advance.argtypes = [vp, vp, ll, u64, C.POINTER(game_ga_params), i, C.POINTER(game_result)]
        L.game_sync.argtypes = [vp, C.POINTER(game_result)]
        L.game_set_tuning.argtypes = [vp, i, i]
        L.game_set_global_patterns.argtypes = [vp, ll]
        L.game_predict_new.argtypes = [vp, vp, vp, ll, vp, vp]
        L.game_population_size.argtypes = [vp]
        L.game_set_expansion.argtypes = [vp, i]
        L.game_resolved_expansion.argtypes = [vp, i]
        L.game_load.argtypes = [vp, vp, vp, ll]
        L.game_load_host.argtypes = [vp, vp, vp, ll]
        L.game_fitness.argtypes = [vp, vp, i, vp]
        L.game_fitness_host.argtypes = [vp, vp, i, vp]
        L.game_predict.argtypes = [vp, vp, vp, vp]
        L.game_classify.argtypes = [vp, vp, C.c_float, vp, vp]
        L.game_set_population.argtypes = [vp, vp, i]
        L.game_set_generation.argtypes = [vp, ll]
        L.game_evolve.argtypes = [vp, i, u64, C.POINTER(game_ga_params), C.POINTER(game_result)]
        L.game_get_population.argtypes = [vp, vp, vp, vp]
        L.game_get_population_host.argtypes = [vp, vp, vp, vp]
        L.game_rank.argtypes = [vp, vp, i, vp]
        L.game_ga_step.argtypes = [vp, C.POINTER(game_ga_params), u64, ll, vp, vp, vp, vp]
        L.game_init_population.argtypes = [vp, i, u64, i, vp]
        L.game_philox.argtypes = [vp, u64, vp, i, vp]
        L.game_set_kernel_timing.argtypes = [vp, i]
        L.game_get_kernel_timing.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(ll)]
        L.game_microbench.argtypes = [vp, i, i, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.game_rank_static.argtypes = [vp, i, vp, vp]
        L.game_rank_static_error.restype = C.c_char_p
        L.game_rank_static_error.argtypes = []
        _lib = L
    return _lib


def _dev(t, dtype=None):
    """device pointer of a contiguous CUDA tensor (or None)"""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError("expected dtype %s, got %s" % (dtype, t.dtype))
    return C.c_void_p(t.data_ptr())


def _host(a, dtype):
    if a is None:
        return None
    if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags["C_CONTIGUOUS"]):
        raise ValueError("expected a C-contiguous numpy array of %s" % dtype)
    return C.c_void_p(a.ctypes.data)


def ga_params(P, tournament_size=3, elitism=2, elite_mode=GAME_ELITE_COPIES_OF_BEST,
              selection=GAME_SEL_TOURNAMENT, init_mode=GAME_INIT_NORMAL_PM1, p_crossover=0.9,
              p_mutation=0.05, stop_error=-1.0):
    return game_ga_params(P, tournament_size, elitism, elite_mode, selection, init_mode,
                          p_crossover, p_mutation, stop_error)


def rank_static(fit, order=None, stream=None):
    """``game_rank_static``: rank P errors (CUDA float32 tensor) into ``order`` (int32, order[0] = best) without allocating
    device memory inside the library -- for hosts whose GPU memory belongs to another allocator or that must stay off the
    driver's allocation path.  Pass a preallocated ``order`` to keep this wrapper from allocating either (it only makes
    one when none is given).  P <= GAME_RANK_STATIC_MAX_P; the library's one scratch array is shared, so calls that
    could overlap on the GPU must be ordered by the caller.  Enqueued on ``stream`` (default: torch's current stream)."""
    import torch
    L = load_library()
    if not torch.cuda.is_available():
        raise RuntimeError("libgame_b200 needs a CUDA device; there is no CPU fallback")
    if order is None:
        order = torch.empty(fit.shape[0], dtype=torch.int32, device=fit.device)
    s = stream if stream is not None else torch.cuda.current_stream(fit.device)
    with torch.cuda.device(fit.device):
        rc = L.game_rank_static(_dev(fit, torch.float32), fit.shape[0], _dev(order, torch.int32), C.c_void_p(s.cuda_stream))
    if rc:
        raise GameError(rc, L.game_rank_static_error().decode())
    return order


class Game:
    """One ``game_ctx``.  Method names are the C entry points minus the ``game_`` prefix."""

    def __init__(self, family, degree, F, stream=None):
        import torch
        self._torch = torch
        self._L = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("libgame_b200 needs a CUDA device; there is no CPU fallback")
        h = C.c_void_p()
        rc = self._L.game_create(family, degree, F, C.byref(h))
        if rc:
            raise GameError(rc, "game_create failed")
        self._h = h
        self.family, self.degree, self.F = family, degree, F
        self.K = self._L.game_num_terms(h)
        self.N = 0
        self.set_stream(stream if stream is not None else torch.cuda.current_stream())

    def _ck(self, rc):
        if rc:
            raise GameError(rc, self._L.game_last_error(self._h).decode())

    def destroy(self):
        if getattr(self, "_h", None):
            self._L.game_destroy(self._h)
            self._h = None

    __del__ = destroy

    def num_terms(self):
        return self._L.game_num_terms(self._h)

    def generation(self):
        return int(self._L.game_generation(self._h))

    def launch_count(self):
        return int(self._L.game_launch_count(self._h))

    def set_kernel_timing(self, enabled):
        self._ck(self._L.game_set_kernel_timing(self._h, 1 if enabled else 0))

    def get_kernel_timing(self):
        ms, n = C.c_double(0.0), C.c_longlong(0)
        self._ck(self._L.game_get_kernel_timing(self._h, C.byref(ms), C.byref(n)))
        return ms.value, int(n.value)

    def microbench(self, kind, param=0):
        """(ops per second over the whole GPU, milliseconds of the timed launch) of one GAME_PEAK_* micro-benchmark."""
        ops, ms = C.c_double(0.0), C.c_double(0.0)
        self._ck(self._L.game_microbench(self._h, kind, param, C.byref(ops), C.byref(ms)))
        return ops.value, ms.value

    def set_stream(self, stream):
        self.stream = stream
        self._ck(self._L.game_set_stream(self._h, C.c_void_p(stream.cuda_stream)))

    def set_activation(self, act):
        self._ck(self._L.game_set_activation(self._h, act))

    def set_error(self, err, R=0.0):
        self._ck(self._L.game_set_error(self._h, err, R))

    def set_path(self, path):
        self._ck(self._L.game_set_path(self._h, path))

    def fitness_sums(self, pop=None, P=0, out=None, accumulate=False):
        """Per-chromosome fp64 error totals over this context's patterns (pop None: the context's own population of P);
        accumulate: add them to `out` inside the library (out-of-core chunks)."""
        t = self._torch
        if pop is not None:
            P = pop.shape[0]
            assert pop.shape == (P, self.K)
        if out is None:
            if accumulate:
                raise ValueError("accumulate needs the buffer to add to")
            out = t.empty(P, dtype=t.float64, device="cuda")
        self._ck(self._L.game_fitness_sums(self._h, _dev(pop, t.float32), P, _dev(out, t.float64), 1 if accumulate else 0))
        return out

    def advance(self, sums, N_total, seed, params, apply_operators=True, sync=True):
        """sync=False: asynchronous (res == NULL in the C call); collect with sync()."""
        res = game_result() if sync else None
        self._ck(self._L.game_advance(self._h, _dev(sums, self._torch.float64), N_total, seed, C.byref(params),
                                      1 if apply_operators else 0, C.byref(res) if sync else None))
        return res

    def sync(self):
        res = game_result()
        self._ck(self._L.game_sync(self._h, C.byref(res)))
        return res

    def set_tuning(self, knob, value):
        self._ck(self._L.game_set_tuning(self._h, knob, value))

    def set_global_patterns(self, N_total):
        self._ck(self._L.game_set_global_patterns(self._h, N_total))

    def population_size(self):
        return int(self._L.game_population_size(self._h))

    def predict_new(self, genes, X_new, want_z=True, want_y=True):
        t = self._torch
        N = X_new.shape[0]
        assert X_new.shape == (N, self.F)
        z = t.empty(N, dtype=t.float32, device=genes.device) if want_z else None
        y = t.empty(N, dtype=t.float32, device=genes.device) if want_y else None
        self._ck(self._L.game_predict_new(self._h, _dev(genes, t.float32), _dev(X_new, t.float32), N, _dev(z), _dev(y)))
        return z, y

    def set_expansion(self, mode):
        self._ck(self._L.game_set_expansion(self._h, mode))

    def resolved_expansion(self, P):
        return self._L.game_resolved_expansion(self._h, P)

    def resolved_path(self, P):
        return self._L.game_resolved_path(self._h, P)

    def load(self, X, targets):
        t = self._torch
        N = X.shape[0]
        assert X.shape == (N, self.F) and targets.shape == (N,)
        self._ck(self._L.game_load(self._h, _dev(X, t.float32), _dev(targets, t.float32), N))
        self.N = N

    def load_host(self, X, targets):
        N = X.shape[0]
        assert X.shape == (N, self.F) and targets.shape == (N,)
        self._ck(self._L.game_load_host(self._h, _host(X, np.float32), _host(targets, np.float32), N))
        self.N = N

    def fitness(self, pop, out=None):
        t = self._torch
        P = pop.shape[0]
        assert pop.shape == (P, self.K)
        if out is None:
            out = t.empty(P, dtype=t.float32, device=pop.device)
        self._ck(self._L.game_fitness(self._h, _dev(pop, t.float32), P, _dev(out, t.float32)))
        return out

    def fitness_host(self, pop, out=None):
        P = pop.shape[0]
        assert pop.shape == (P, self.K)
        if out is None:
            out = np.empty(P, dtype=np.float32)
        self._ck(self._L.game_fitness_host(self._h, _host(pop, np.float32), P, _host(out, np.float32)))
        return out

    def predict(self, genes, want_z=True, want_y=True):
        t = self._torch
        z = t.empty(self.N, dtype=t.float32, device=genes.device) if want_z else None
        y = t.empty(self.N, dtype=t.float32, device=genes.device) if want_y else None
        self._ck(self._L.game_predict(self._h, _dev(genes, t.float32), _dev(z), _dev(y)))
        return z, y

    def classify(self, genes, cut=0.5):
        t = self._torch
        counts = t.empty(4, dtype=t.int64, device=genes.device)
        fom = t.empty(3, dtype=t.float64, device=genes.device)
        self._ck(self._L.game_classify(self._h, _dev(genes, t.float32), cut, _dev(counts), _dev(fom)))
        return counts, fom

    def set_population(self, pop):
        self._ck(self._L.game_set_population(self._h, _dev(pop, self._torch.float32), pop.shape[0]))
        self._P = pop.shape[0]

    def set_generation(self, g):
        self._ck(self._L.game_set_generation(self._h, g))

    def evolve(self, generations, seed, params):
        res = game_result()
        self._ck(self._L.game_evolve(self._h, generations, seed, C.byref(params), C.byref(res)))
        self._P = params.P
        return res

    def get_population(self, want_fit=True):
        t = self._torch
        P = self._P
        dev = "cuda"
        pop = t.empty((P, self.K), dtype=t.float32, device=dev)
        fit = t.empty(P, dtype=t.float32, device=dev) if want_fit else None
        order = t.empty(P, dtype=t.int32, device=dev) if want_fit else None
        self._ck(self._L.game_get_population(self._h, _dev(pop), _dev(fit), _dev(order)))
        return pop, fit, order

    def get_population_host(self, want_fit=True):
        P = self._P
        pop = np.empty((P, self.K), dtype=np.float32)
        fit = np.empty(P, dtype=np.float32) if want_fit else None
        order = np.empty(P, dtype=np.int32) if want_fit else None
        self._ck(self._L.game_get_population_host(self._h, _host(pop, np.float32), _host(fit, np.float32),
                                                  _host(order, np.int32)))
        return pop, fit, order

    def rank(self, fit):
        t = self._torch
        order = t.empty(fit.shape[0], dtype=t.int32, device=fit.device)
        self._ck(self._L.game_rank(self._h, _dev(fit, t.float32), fit.shape[0], _dev(order)))
        return order

    def ga_step(self, params, seed, generation, order, fit, pop):
        t = self._torch
        nxt = t.empty_like(pop)
        self._ck(self._L.game_ga_step(self._h, C.byref(params), seed, generation, _dev(order, t.int32),
                                      _dev(fit, t.float32), _dev(pop, t.float32), _dev(nxt)))
        return nxt

    def init_population(self, mode, seed, P):
        t = self._torch
        pop = t.empty((P, self.K), dtype=t.float32, device="cuda")
        self._ck(self._L.game_init_population(self._h, mode, seed, P, _dev(pop)))
        return pop

    def philox(self, seed, ctr):
        t = self._torch
        out = t.empty_like(ctr)
        self._ck(self._L.game_philox(self._h, seed, _dev(ctr, t.int32), ctr.shape[0], _dev(out)))
        return out
