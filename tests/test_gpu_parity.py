"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element.

Tolerances: fitness |gpu - ref| <= rtol*|ref| + atol with rtol=1e-5, atol=1e-7 on
the FP32 and TENSOR_SPLIT paths and rtol=1e-3, atol=1e-5 on the TENSOR path; TMSE is discontinuous at |r| = R, so its
bound is widened by near_p*(R+delta)^2/N where near_p counts the patterns within delta of the tube
(delta = 1e-5 / 5e-3).  GA decisions (rank, parents, cut points, mutation masks and values, initial
genes, Philox words) are bit-exact.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("no CUDA device", allow_module_level=True)

import paper_1304_0597_b200 as g  # noqa: E402
from paper_1304_0597_b200 import workloads as wl  # noqa: E402

TRIG, CHEB = 0, 1
SIGMOID, IDENTITY = 0, 1
MSE, TMSE, RMSE = 0, 1, 2
TOL = {g.GAME_PATH_FP32: (1e-5, 1e-7, 1e-5), g.GAME_PATH_TENSOR: (1e-3, 1e-5, 5e-3),
       g.GAME_PATH_TENSOR_SPLIT: (1e-5, 1e-7, 1e-5)}       # split-fp16 on the tensor cores: the FP32 path's class


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# What the TMSE slack is worth: per check, the largest slack / (rtol |ref| + atol) -- how much wider than
# the plain tolerance the bound was -- and the largest |gpu - ref| / (rtol |ref| + atol) -- whether the slack was needed at
# all (<= 1: the check passes WITHOUT it).  conftest.py writes the records to $GAME_PARITY_LOG at session end.
PARITY_LOG = []


def check_fitness(orc, gpu_fit, fam, d, X, t, pop, act, err, R, path, what=""):
    rtol, atol, delta = TOL[path]
    if err == TMSE:
        ref, near = orc.fitness(fam, d, X, t, pop, act=act, err=err, R=R, delta=delta)
        slack = near * (R + delta) ** 2 / X.shape[0]
    else:
        ref = orc.fitness(fam, d, X, t, pop, act=act, err=err, R=R)
        slack = 0.0
    got = np.asarray(gpu_fit, dtype=np.float64)
    plain = rtol * np.abs(ref) + atol
    bound = plain + slack
    PARITY_LOG.append(dict(what=what, path=int(path), err=int(err), act=int(act), N=int(X.shape[0]), K=int(pop.shape[1]),
                           rows=int(got.size), slack_over_tol=float(np.max(slack / plain)),
                           err_over_tol=float(np.max(np.abs(got - ref) / plain)),
                           err_over_bound=float(np.max(np.abs(got - ref) / bound)),
                           mean_signed_rel=float(np.mean((got - ref) / np.maximum(np.abs(ref), 1e-300)))))
    bad = np.abs(got - ref) > bound
    assert not bad.any(), "%s: %d/%d off; worst %g (bound %g) at p=%d" % (
        what, bad.sum(), bad.size, np.abs(got - ref).max(), bound[np.abs(got - ref).argmax()],
        int(np.abs(got - ref).argmax()))
    return ref


def make_ctx(fam, d, X, t, act=SIGMOID, err=MSE, R=0.0, path=g.GAME_PATH_AUTO):
    ctx = g.Game(fam, d, X.shape[1])
    ctx.set_activation(act)
    ctx.set_error(err, R)
    ctx.set_path(path)
    ctx.load(dev(X), dev(t))
    return ctx


def paths_available(ctx, P):
    out = [g.GAME_PATH_FP32]
    for path in (g.GAME_PATH_TENSOR, g.GAME_PATH_TENSOR_SPLIT):
        ctx.set_path(path)
        if ctx.resolved_path(P) == path:
            out.append(path)
    ctx.set_path(g.GAME_PATH_AUTO)
    return out


# ---- RNG and operators: bit-exact ----------------------------------------------------------------
def test_philox_words(orc):
    ctx = g.Game(TRIG, 1, 1)
    rng = np.random.default_rng(20)
    ctr = rng.integers(0, 2**32, (513, 4), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0
    ctr[1] = 0xFFFFFFFF
    for seed in (0, 1, 0xDEADBEEFCAFEF00D, 2**64 - 1):
        out = ctx.philox(seed, dev(ctr.view(np.int32))).cpu().numpy().view(np.uint32)
        for i in range(0, 513, 7):
            ref = orc.philox4x32_10([seed & 0xFFFFFFFF, seed >> 32], ctr[i])
            assert np.array_equal(out[i], ref), (seed, i)


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_init_population_bit_exact(orc, mode):
    ctx = g.Game(CHEB, 8, 11)          # K = 99
    for seed, P in ((1, 20), (0xABCDEF0123456789, 333)):
        got = ctx.init_population(mode, seed, P).cpu().numpy()
        ref = orc.init_population(mode, seed, P, ctx.K)
        assert np.array_equal(got.view(np.uint32), ref.view(np.uint32))


def test_rank_bit_exact(orc):
    ctx = g.Game(TRIG, 1, 1)
    rng = np.random.default_rng(21)
    for P in (1, 2, 20, 255, 256, 257, 2048, 2049, 5000, 8192):
        fit = rng.random(P).astype(np.float32)
        if P > 10:
            fit[rng.integers(0, P, P // 10)] = fit[0]          # ties
            fit[rng.integers(0, P, 3)] = np.nan
            fit[rng.integers(0, P, 2)] = np.inf
            fit[rng.integers(0, P, 2)] = -0.0
            fit[rng.integers(0, P, 2)] = 0.0
        got = ctx.rank(dev(fit)).cpu().numpy()
        assert np.array_equal(got, orc.rank(fit)), P


GA_CASES = [
    dict(P=20, K_fd=(TRIG, 4, 11), tournament_size=3, elitism=2),
    dict(P=21, K_fd=(CHEB, 8, 11), tournament_size=4, elitism=2, p_mutation=0.2),      # paper's parameters, odd children
    dict(P=64, K_fd=(CHEB, 1, 1), tournament_size=1, elitism=0, p_crossover=1.0),       # K = 2: only cut = 1
    dict(P=33, K_fd=(TRIG, 1, 1), tournament_size=9, elitism=5, elite_mode=1, p_crossover=0.5, p_mutation=1.0),
    dict(P=1024, K_fd=(CHEB, 8, 11), tournament_size=3, elitism=2),
    dict(P=50, K_fd=(TRIG, 8, 32), selection=1, elitism=1),                              # roulette, K = 544
    dict(P=4096, K_fd=(CHEB, 6, 16), selection=1, elitism=2, p_mutation=0.0),
    dict(P=300, K_fd=(CHEB, 12, 64), tournament_size=2, elitism=299),                    # almost all elites
]


@pytest.mark.parametrize("case", GA_CASES)
def test_ga_step_bit_exact(orc, case):
    case = dict(case)
    fam, d, F = case.pop("K_fd")
    ctx = g.Game(fam, d, F)
    K, P = ctx.K, case["P"]
    rng = np.random.default_rng(22)
    pop = rng.uniform(-1, 1, (P, K)).astype(np.float32)
    fit = rng.random(P).astype(np.float32)
    fit[rng.integers(0, P, 2)] = np.nan
    order = orc.rank(fit)
    gp_g = g.ga_params(**case)
    gp_o = orc.GaParams(P=P, tournament_size=gp_g.tournament_size, elitism=gp_g.elitism, elite_mode=gp_g.elite_mode,
                        selection=gp_g.selection, init_mode=gp_g.init_mode, p_crossover=gp_g.p_crossover,
                        p_mutation=gp_g.p_mutation, stop_error=-1.0)
    for seed, gen in ((5, 0), (2**63 + 11, 7), (5, 4000000000)):
        got = ctx.ga_step(gp_g, seed, gen, dev(order), dev(fit), dev(pop)).cpu().numpy()
        ref = orc.ga_step(gp_o, seed, gen, order, fit, pop)
        assert np.array_equal(got.view(np.uint32), ref.view(np.uint32)), (seed, gen)


# ---- fitness parity at sizes spanning several tiles and ragged tails -------------------------------
FIT_SHAPES = [
    # fam, d, F, N, P
    (TRIG, 4, 11, 2100, 20),       # config 1's shape
    (CHEB, 8, 11, 2100, 300),      # config 2's shape, ragged P
    (CHEB, 6, 16, 1000, 257),
    (TRIG, 8, 32, 777, 130),       # K = 544
    (CHEB, 12, 64, 515, 384),      # K = 832
    (TRIG, 1, 1, 1, 2),            # degenerate: one pattern, K = 3
    (CHEB, 1, 1, 129, 1),          # one chromosome
]


@pytest.mark.parametrize("shape", FIT_SHAPES)
@pytest.mark.parametrize("act,err,R", [(SIGMOID, MSE, 0.0), (SIGMOID, TMSE, 0.49), (SIGMOID, RMSE, 0.0),
                                       (IDENTITY, MSE, 0.0), (IDENTITY, TMSE, 0.3)])
def test_fitness_parity_small(orc, shape, act, err, R):
    fam, d, F, N, P = shape
    rng = np.random.default_rng(23)
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    t = rng.integers(0, 2, N).astype(np.float32)
    K = orc.num_terms(fam, d, F)
    scale = 1.0 if act == SIGMOID else 1.0 / np.sqrt(K)
    pop = (rng.uniform(-1, 1, (P, K)) * scale).astype(np.float32)
    ctx = make_ctx(fam, d, X, t, act, err, R)
    for path in paths_available(ctx, P):
        ctx.set_path(path)
        got = ctx.fitness(dev(pop)).cpu().numpy()
        check_fitness(orc, got, fam, d, X, t, pop, act, err, R, path, "path %d" % path)
        # P20: a chromosome's fitness does not depend on where it sits in the population
        perm = rng.permutation(P)
        got2 = ctx.fitness(dev(pop[perm])).cpu().numpy()
        assert np.array_equal(got2.view(np.uint32), got[perm].view(np.uint32))


def test_fitness_host_matches_device(orc):
    fam, d, F, N, P = CHEB, 8, 11, 2100, 64
    w = wl.config(2).scaled(P=P)
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    pop = wl.uniform_population(P, w.K, 2)
    ctx = g.Game(fam, d, F)
    ctx.set_error(TMSE, 0.49)
    ctx.load_host(X, t)
    a = ctx.fitness_host(pop)
    b = ctx.fitness(dev(pop)).cpu().numpy()
    assert np.array_equal(a.view(np.uint32), b.view(np.uint32))
    check_fitness(orc, a, fam, d, X, t, pop, SIGMOID, TMSE, 0.49, ctx.resolved_path(P))


@pytest.mark.parametrize("cfg,N,P", [(3, 20000, 20000), (3, 30000, 4096), (5, 6000, 5000), (2, None, 4100),
                                     (5, 12000, 3073)])      # four chunks of 1024 would leave a ONE-row tail: folded into the third
def test_fitness_host_chunked_upload(orc, cfg, N, P):
    """game_fitness_host uploads populations of >= 2048 chromosomes in two (>= 1 MB) or four (>= 8 MB) chunks on a copy stream, a chunk ahead of the
    kernels; a chromosome's fitness does not depend on its row (P20), so the result equals the device call bit for bit --
    also with a ragged last chunk, pinned or pageable host memory, and twice in a row (the staging area is reused).  Small
    datasets (config 2: a chunk would fall below one wave of tiles and change the tile shape) go up in one piece."""
    w = wl.config(cfg)
    w = w.scaled(N=N or w.N, P=P)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    pop = wl.uniform_population(P, w.K, cfg)
    ctx = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    b = ctx.fitness(dev(pop)).cpu().numpy()
    pinned = torch.from_numpy(pop).pin_memory().numpy()
    for src in (pop, pinned, pinned):
        a = ctx.fitness_host(src)
        assert np.array_equal(a.view(np.uint32), b.view(np.uint32))
    rows = np.array([0, 1023, 1024, P // 2, P - 1])
    check_fitness(orc, b[rows], fam, d, X, t, pop[rows], w.act, w.err, w.R, ctx.resolved_path(P), "host chunks")
    # a gene outside the fp16 range in the LAST chunk is still reported
    bad = pop.copy(); bad[P - 1, 0] = 1e6
    if ctx.resolved_path(P) != g.GAME_PATH_FP32:
        with pytest.raises(g.GameError) as e:
            ctx.fitness_host(bad)
        assert e.value.code == 5


def test_planted_and_replication(orc):
    # P8 / P10 on the GPU: the planted chromosome scores ~0; replicated rows leave the error unchanged
    fam, d, F, N = TRIG, 4, 11, 2100
    rng = np.random.default_rng(24)
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    c0 = rng.standard_normal(orc.num_terms(fam, d, F)).astype(np.float32)
    _, y = orc.forward(fam, d, X, c0)
    t = y.astype(np.float32)
    pop = np.stack([c0, -c0, c0 * 0.5]).astype(np.float32)
    ctx = make_ctx(fam, d, X, t, SIGMOID, MSE, path=g.GAME_PATH_FP32)
    f = ctx.fitness(dev(pop)).cpu().numpy()
    assert 0.0 <= f[0] <= 1e-7 and f[1] > 1e-3 and f[2] > 1e-5
    ctx4 = make_ctx(fam, d, np.tile(X, (4, 1)), np.tile(t, 4), SIGMOID, MSE, path=g.GAME_PATH_FP32)
    f4 = ctx4.fitness(dev(pop)).cpu().numpy()
    assert np.allclose(f4[1:], f[1:], rtol=2e-6)


def test_predict_parity(orc):
    fam, d, F, N = CHEB, 12, 64, 1000
    rng = np.random.default_rng(25)
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    c = (rng.standard_normal(orc.num_terms(fam, d, F)) * 0.1).astype(np.float32)
    ctx = make_ctx(fam, d, X, np.zeros(N, dtype=np.float32))
    z, y = ctx.predict(dev(c))
    zr, yr = orc.forward(fam, d, X, c)
    assert np.allclose(z.cpu().numpy(), zr, rtol=1e-5, atol=1e-5)
    assert np.allclose(y.cpu().numpy(), yr, rtol=1e-5, atol=1e-6)


def test_classify_figures_of_merit(orc):
    # L301: counts are integers decided by a float (y > cut).  The kernel decides in fp32, the oracle in fp64,
    # so patterns the oracle finds within delta of the cut may fall either way; everything else must agree.
    for cfg, scale in ((1, 1.0), (3, 0.05)):
        w = wl.config(cfg)
        fam, d = w.family, w.degree
        X, t, c0 = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
        rng = np.random.default_rng(26)
        genes = c0 if c0 is not None else (rng.standard_normal(w.K) * scale).astype(np.float32)
        ctx = make_ctx(fam, d, X, t)
        counts, fom = ctx.classify(dev(genes), 0.5)
        counts, fom = counts.cpu().numpy(), fom.cpu().numpy()
        ref_c, ref_f, near = orc.classify(fam, d, X, t, genes, cut=0.5, delta=1e-5)
        assert counts.sum() == w.N == ref_c.sum()
        assert np.abs(counts - ref_c).max() <= near, (counts, ref_c, near)
        # the ratios are exactly those of the kernel's own counts, and within near/N of the oracle's
        tp, fp, tn, fn = [float(v) for v in counts]
        assert fom[0] == (tp + tn) / w.N and fom[1] == tp / (tp + fn) and fom[2] == fp / (fp + tn)
        assert np.abs(fom - ref_f).max() <= (near + 1e-9) / min(tp + fn, fp + tn)
        if c0 is not None:      # planted labels with 10 % flips: accuracy ~ 0.9
            assert 0.85 < fom[0] < 0.95


def test_error_paths():
    ctx = g.Game(TRIG, 2, 3)
    pop = torch.zeros((4, ctx.K), device="cuda")
    with pytest.raises(g.GameError) as e:
        ctx.fitness(pop)
    assert e.value.code == 2                                   # NOT_LOADED
    X = torch.zeros((10, 3), device="cuda")
    X[3, 1] = float("nan")
    with pytest.raises(g.GameError) as e:
        ctx.load(X, torch.zeros(10, device="cuda"))
    assert e.value.code == 6                                   # NONFINITE_INPUT
    with pytest.raises(g.GameError) as e:
        ctx.set_error(TMSE, 1.5)
    assert e.value.code == 1
    ctx.load(torch.zeros((10, 3), device="cuda"), torch.zeros(10, device="cuda"))
    with pytest.raises(g.GameError) as e:
        ctx.evolve(1, 1, g.ga_params(P=1))
    assert e.value.code == 1


# ---- whole GA runs, generation by generation, GPU population injected into the oracle (c.4) --------
def trajectory(orc, w, generations, full_check_every=1, subset=None, selection=0, elite_mode=0, stream=None):
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    if stream is None:
        ctx = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    else:                                   # bench.py's launch configuration: the context on its own (capturable) stream
        ctx = g.Game(fam, d, X.shape[1], stream=stream)
        ctx.set_activation(w.act)
        ctx.set_error(w.err, w.R)
        ctx.load(dev(X), dev(t))
    path = ctx.resolved_path(w.P)
    gp_g = g.ga_params(P=w.P, tournament_size=w.tournament_size, elitism=w.elitism, init_mode=w.init_mode,
                       p_crossover=w.p_crossover, p_mutation=w.p_mutation, selection=selection, elite_mode=elite_mode)
    gp_o = orc.GaParams(P=w.P, tournament_size=w.tournament_size, elitism=w.elitism, elite_mode=elite_mode,
                        selection=selection, init_mode=w.init_mode, p_crossover=w.p_crossover, p_mutation=w.p_mutation, stop_error=-1.0)
    res = ctx.evolve(0, w.seed, gp_g)                         # init + fitness + rank
    pop, fit, order = ctx.get_population_host()
    assert np.array_equal(pop.view(np.uint32), orc.init_population(w.init_mode, w.seed, w.P, w.K).view(np.uint32))
    best_prev = None
    rng = np.random.default_rng(99)
    for gen in range(generations + 1):
        # (ii) fitness of the GPU's population within tolerance
        if gen % full_check_every == 0 or gen == generations:
            rows = (np.arange(w.P) if subset is None else subset(gen, rng) if callable(subset)
                    else np.sort(rng.choice(w.P, subset, replace=False)))
            check_fitness(orc, fit[rows], fam, d, X, t, pop[rows], w.act, w.err, w.R, path, "%s gen %d" % (w.name, gen))
        # (iii) the rank kernel sorted the GPU's own fitness bits exactly
        assert np.array_equal(order, orc.rank(fit)), gen
        assert res.best_index == order[0] and res.best_error == fit[order[0]]
        # P20: elitism never lets the best error worsen, exactly
        if best_prev is not None:
            assert fit[order[0]] <= best_prev, gen
        best_prev = fit[order[0]]
        if gen == generations:
            break
        # (iv) the operators, from the GPU's order, reproduce the GPU's next population bit for bit
        ref_next = orc.ga_step(gp_o, w.seed, gen, order, fit, pop)
        res = ctx.evolve(1, w.seed, gp_g)
        assert res.generations_run == 1 and ctx.generation() == gen + 1
        pop, fit, order = ctx.get_population_host()
        assert np.array_equal(pop.view(np.uint32), ref_next.view(np.uint32)), gen
    return ctx, pop, fit, order


def test_trajectory_config1_full(orc):
    trajectory(orc, wl.config(1), 100)


def test_trajectory_config2_scaled(orc):
    # config 2's data and GA parameters, full P, fewer generations (the oracle needs ~0.2 s each)
    trajectory(orc, wl.config(2), 24, full_check_every=4)


def test_trajectory_paper_parameters(orc):
    # the paper's own settings (L282-L291): tournament 4, mutation 0.2, P = 23 (eq. 6), TMSE 0.49
    w = wl.config(1)
    from dataclasses import replace
    trajectory(orc, replace(w, P=23, tournament_size=4, p_mutation=0.2), 20)


@pytest.mark.parametrize("cfg,init_mode,selection,elite_mode", [(3, 0, 1, 0), (3, 2, 1, 1), (2, 0, 1, 1), (2, 2, 0, 1)])
def test_trajectory_roulette_and_init_modes_at_scale(orc, cfg, init_mode, selection, elite_mode):
    # roulette selection (R4), init modes U[-1,1) / U[0,1) and top-e elitism on the larger
    # configs at full P; fitness on a chromosome subset where the oracle would need minutes for all of them
    from dataclasses import replace
    w = replace(wl.config(cfg), init_mode=init_mode)
    trajectory(orc, w, 3, subset=48 if cfg == 3 else None, selection=selection, elite_mode=elite_mode)


def block_rows(P, rng, extra=0):
    """One chromosome in EVERY block of 128 -- i.e. in both halves of every 256-chromosome CTA pair and in every single-CTA
    block of the tensor kernels -- at a random position inside the block, plus `extra` random rows, plus the first and last."""
    starts = np.arange(0, P, 128)
    rows = starts + rng.integers(0, np.minimum(128, P - starts))
    more = rng.choice(P, extra, replace=False) if extra else np.empty(0, dtype=np.int64)
    return np.unique(np.concatenate([rows, more, [0, P - 1]])).astype(np.int64)


def full_size_rows(cfg, P, rng, ends):
    """the FULL population where the oracle can afford it (configs 3 and 4: all 4096 / all 256
    chromosomes), every chromosome block otherwise (config 5: 64 blocks of 128 + 64 random rows), at the generations where
    `ends` is true (first and last); a random subset of 64 at the generations between."""
    if not ends:
        return np.sort(rng.choice(P, min(64, P), replace=False))
    return np.arange(P) if cfg in (3, 4) else block_rows(P, rng, extra=64)


@pytest.mark.parametrize("cfg,generations", [(3, 4), (4, 3), (5, 3)])
def test_trajectory_full_size_big_configs(orc, cfg, generations):
    """SURVEY 8(c) c.4 / 8(g).3 at FULL size on configs 3 (tournament), 4 and 5, in bench.py's launch configuration
    (context on its own stream, AUTO path): every generation (iii) the rank is the exact sort of the GPU's fitness bits and
    (iv) oracle.ga_step from the GPU's order reproduces the GPU's next population (P x K genes) bit for bit; (ii) the
    oracle's fitness against the GPU's for the WHOLE population (configs 3, 4) or a chromosome in every 128-chromosome block,
    both halves of every CTA pair (config 5), at generation 0 and at the last one, and for 64 random chromosomes at every
    generation between (full_size_rows).  PAPER.md L217-L220 (the loop), L286-L291 (the operators' parameters); the paper's
    own validation is this kind of whole-run cross-check between implementations (L299, L324)."""
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        w = wl.config(cfg)
        ctx, pop, fit, order = trajectory(orc, w, generations, full_check_every=1, stream=stream,
                                          subset=lambda gen, rng: full_size_rows(cfg, w.P, rng, gen in (0, generations)))
    assert ctx.generation() == generations


FULL_MODES = [(SIGMOID, MSE, 0.0), (SIGMOID, TMSE, 0.49), (SIGMOID, RMSE, 0.0), (IDENTITY, MSE, 0.0), (IDENTITY, RMSE, 0.0)]


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_full_size_all_error_and_activation_modes(orc, cfg):
    """fitness parity with MSE, TMSE, RMSE and with the identity activation on EVERY config at its full N and
    P, in the launch configuration bench.py times (AUTO path, full population in one call).  The oracle evaluates the
    whole population on configs 1-4 (config 4: in the paper's mode TMSE and in identity / RMSE; the other three modes on
    a chromosome of every block) and a chromosome of every 128-chromosome block plus 64 random ones on config 5."""
    w = wl.config(cfg)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    rng = np.random.default_rng(100 + cfg)
    pop_s = wl.uniform_population(w.P, w.K, w.seed)
    pop_i = (pop_s / np.sqrt(w.K)).astype(np.float32)            # identity output: keep z = O(1)
    all_rows, some_rows = np.arange(w.P), block_rows(w.P, rng, extra=min(64, w.P // 2))
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ctx = g.Game(fam, d, w.F, stream=stream)
        ctx.load(dev(X), dev(t))
        path = ctx.resolved_path(w.P)
        for act, err, R in FULL_MODES:
            ctx.set_activation(act)
            ctx.set_error(err, R)
            pop = pop_s if act == SIGMOID else pop_i
            got = ctx.fitness(dev(pop)).cpu().numpy()
            assert np.all(np.isfinite(got))
            rows = some_rows if cfg == 5 or (cfg == 4 and (act, err) not in ((SIGMOID, TMSE), (IDENTITY, RMSE))) else all_rows
            check_fitness(orc, got[rows], fam, d, X, t, pop[rows], act, err, R, path,
                          "%s full size act %d err %d" % (w.name, act, err))


def test_resume_and_single_call_agree(orc):
    # P22: evolve(a); evolve(b) == evolve(a+b), bit for bit; and == the step-by-step run
    w = wl.config(1)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    gp = g.ga_params(P=w.P)
    a = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    ra = a.evolve(30, w.seed, gp)
    b = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    b.evolve(12, w.seed, gp)
    rb = b.evolve(18, w.seed, gp)
    pa, fa, oa = a.get_population_host()
    pb, fb, ob = b.get_population_host()
    assert a.generation() == b.generation() == 30 and ra.generations_run == 30 and rb.generations_run == 18
    assert np.array_equal(pa.view(np.uint32), pb.view(np.uint32))
    assert np.array_equal(fa.view(np.uint32), fb.view(np.uint32)) and np.array_equal(oa, ob)
    assert ra.best_error == rb.best_error and ra.best_index == rb.best_index
    # checkpoint: export, import into a fresh context, continue
    c = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    p12 = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    p12.evolve(12, w.seed, gp)
    pop12, _, _ = p12.get_population()
    c.set_population(pop12)
    c.set_generation(12)
    c.evolve(18, w.seed, gp)
    pc, fc, oc = c.get_population_host()
    assert np.array_equal(pc.view(np.uint32), pa.view(np.uint32)) and np.array_equal(oc, oa)


def test_stop_criterion(orc):
    w = wl.config(1)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    gp = g.ga_params(P=w.P)
    a = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    hist = [a.evolve(0, w.seed, gp).best_error]              # hist[i] = best error after i generations
    for _ in range(80):
        hist.append(a.evolve(1, w.seed, gp).best_error)
    target = hist[40]
    first = next(i for i, h in enumerate(hist) if h <= target)           # generations needed
    b = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    gp_stop = g.ga_params(P=w.P, stop_error=float(target))
    r = b.evolve(80, w.seed, gp_stop)
    assert r.stopped_on_error == 1 and r.generations_run == first and b.generation() == first
    assert r.best_error <= target
    pop, fit, order = b.get_population_host()
    assert fit[order[0]] == r.best_error


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times: sampled outputs ---------
@pytest.mark.parametrize("cfg,nsample,want_path", [(3, 24, g.GAME_PATH_AUTO), (4, 8, g.GAME_PATH_AUTO), (5, 8, g.GAME_PATH_AUTO),
                                                  (3, 24, g.GAME_PATH_TENSOR_SPLIT), (5, 8, g.GAME_PATH_TENSOR_SPLIT),
                                                  (1, 15, g.GAME_PATH_AUTO), (2, 24, g.GAME_PATH_AUTO)])
def test_full_size_sampled(orc, cfg, nsample, want_path):
    w = wl.config(cfg)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    ctx = make_ctx(fam, d, X, t, w.act, w.err, w.R, want_path)
    path = ctx.resolved_path(w.P)
    assert path == (want_path if want_path != g.GAME_PATH_AUTO else (g.GAME_PATH_TENSOR if w.N >= 16384 else g.GAME_PATH_TENSOR_SPLIT))
    gp = g.ga_params(P=w.P)
    ctx.evolve(2, w.seed, gp)                                 # init + two real generations at full size
    pop, fit, order = ctx.get_population_host()
    assert np.array_equal(order, orc.rank(fit))
    rng = np.random.default_rng(cfg)
    rows = np.unique(np.concatenate([[0, 1, order[0], order[-1], w.P - 1], rng.choice(w.P, nsample, replace=False)]))
    check_fitness(orc, fit[rows], fam, d, X, t, pop[rows], w.act, w.err, w.R, path, "cfg %d" % cfg)
    # stand-alone fitness call on the same population gives the same bits as the loop's
    f2 = ctx.fitness(dev(pop)).cpu().numpy()
    assert np.array_equal(f2.view(np.uint32), fit.view(np.uint32))
    # properties that hold at any size: elites are copies of the previous winner -> rows 0,1 identical
    assert np.array_equal(pop[0], pop[1]) and fit[0] == fit[1]
    assert np.all(np.abs(pop) <= 1.0) and np.all(np.isfinite(fit)) and np.all(fit >= 0)


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_position_independence_and_split_crosscheck(orc, cfg):
    """Two whole-population checks at FULL size that need no oracle time:
    (P20) a chromosome's fitness does not depend on its row or on its neighbours -- the fitness of a randomly permuted
    population is the permuted fitness, bit for bit, for all P; a defect tied to a chromosome block, a CTA-pair half or a
    `partial` row offset would break it;  and the one-pass fp16 TENSOR result of every chromosome agrees with the
    TENSOR_SPLIT result (the 1e-5 class, a different kernel variant and operand layout) within the 1e-3 class."""
    w = wl.config(cfg)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    pop = wl.uniform_population(w.P, w.K, 31 + cfg)
    perm = np.random.default_rng(cfg).permutation(w.P)
    ctx = make_ctx(fam, d, X, t, SIGMOID, MSE)
    assert ctx.resolved_path(w.P) == g.GAME_PATH_TENSOR
    f = ctx.fitness(dev(pop)).cpu().numpy()
    fp = ctx.fitness(dev(pop[perm])).cpu().numpy()
    assert np.array_equal(fp.view(np.uint32), f[perm].view(np.uint32))
    ctx.set_path(g.GAME_PATH_TENSOR_SPLIT)
    assert ctx.resolved_path(w.P) == g.GAME_PATH_TENSOR_SPLIT
    fs = ctx.fitness(dev(pop)).cpu().numpy().astype(np.float64)
    rtol, atol, _ = TOL[g.GAME_PATH_TENSOR]
    bad = np.abs(f - fs) > rtol * np.abs(fs) + atol
    assert not bad.any(), (int(bad.sum()), float(np.abs(f - fs).max()))
    fsp = ctx.fitness(dev(pop[perm])).cpu().numpy()
    assert np.array_equal(fsp.view(np.uint32), fs.astype(np.float32)[perm].view(np.uint32))


# ---- the paper-literal tied-coefficient models ------------------------------------------
@pytest.mark.parametrize("fam,d", [(2, 1), (2, 8), (3, 1), (3, 6)])
def test_tied_families_fitness(orc, fam, d):
    rng = np.random.default_rng(27)
    N, F, P = 2100, 11, 23
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    t = rng.integers(0, 2, N).astype(np.float32)
    K = orc.num_terms(fam, d, F)
    pop = rng.uniform(-1, 1, (P, K)).astype(np.float32)
    for act, err, R in ((IDENTITY, MSE, 0.0), (IDENTITY, TMSE, 0.49), (SIGMOID, TMSE, 0.49), (SIGMOID, RMSE, 0.0)):
        ctx = make_ctx(fam, d, X, t, act, err, R)
        assert ctx.K == K and ctx.resolved_path(P) == g.GAME_PATH_FP32
        got = ctx.fitness(dev(pop)).cpu().numpy()
        check_fitness(orc, got, fam, d, X, t, pop, act, err, R, g.GAME_PATH_FP32, "tied fam %d d %d" % (fam, d))


def test_trajectory_paper_literal(orc):
    # the paper's own experiment shape and settings (eq. 6-7) on stand-in data, 40 generations
    trajectory(orc, wl.paper_literal(degree=4), 40)
    # and on row-replicated data (L326): same shape of run, 4x the rows
    trajectory(orc, wl.paper_literal(degree=2, N=8400), 6)


# ---- north_star (1): the expansion regenerated inside the fused kernel (game_set_expansion) -----------------------
REGEN_SHAPES = [
    # family, degree, F, N, P
    (TRIG, 8, 32, 1000, 256),      # config 4's K = 544 (9 k-blocks), ragged N over several tiles
    (CHEB, 12, 24, 700, 130),      # ragged P, T = 13 terms per feature
    (TRIG, 4, 11, 2100, 20),       # F not a multiple of 8 (scalar feature loads, padded feature lanes)
    (CHEB, 6, 16, 257, 256),       # one full tile + a one-pattern tail
    (TRIG, 1, 3, 5, 2),            # degenerate: K = 9, fewer patterns than one tile
    (CHEB, 32, 8, 300, 64),        # deepest recurrence the ABI allows
]


@pytest.mark.parametrize("shape", REGEN_SHAPES)
@pytest.mark.parametrize("act,err,R", [(SIGMOID, MSE, 0.0), (SIGMOID, TMSE, 0.49), (IDENTITY, MSE, 0.0)])
def test_fitness_parity_regenerated(orc, shape, act, err, R):
    fam, d, F, N, P = shape
    rng = np.random.default_rng(29)
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    t = rng.integers(0, 2, N).astype(np.float32)
    K = orc.num_terms(fam, d, F)
    scale = 1.0 if act == SIGMOID else 1.0 / np.sqrt(K)
    pop = (rng.uniform(-1, 1, (P, K)) * scale).astype(np.float32)
    ctx = make_ctx(fam, d, X, t, act, err, R, g.GAME_PATH_TENSOR)
    assert ctx.resolved_path(P) == g.GAME_PATH_TENSOR
    assert ctx.resolved_expansion(P) == g.GAME_EXPAND_MATERIALIZED          # AUTO: the measured choice
    ref_fit = ctx.fitness(dev(pop)).cpu().numpy()
    ctx.set_expansion(g.GAME_EXPAND_REGENERATED)
    assert ctx.resolved_expansion(P) == g.GAME_EXPAND_REGENERATED
    got = ctx.fitness(dev(pop)).cpu().numpy()
    check_fitness(orc, got, fam, d, X, t, pop, act, err, R, g.GAME_PATH_TENSOR, "regenerated")
    # the two sources round the same values to fp16 (fp64 vs fp32 arithmetic before the rounding): results agree
    # closely (TMSE is discontinuous at the tube, so it is held to the oracle bound above only)
    if err != TMSE:
        assert np.allclose(got, ref_fit, rtol=2e-4, atol=2e-6)
    perm = rng.permutation(P)                                              # P20 holds for this variant too
    got2 = ctx.fitness(dev(pop[perm])).cpu().numpy()
    assert np.array_equal(got2.view(np.uint32), got[perm].view(np.uint32))


def test_regenerated_expansion_limits():
    rng = np.random.default_rng(31)
    # more than one CTA pair of chromosomes: unavailable, and the call says so
    X = rng.uniform(-1, 1, (300, 8)).astype(np.float32)
    t = np.zeros(300, np.float32)
    ctx = make_ctx(CHEB, 3, X, t, path=g.GAME_PATH_TENSOR)
    ctx.set_expansion(g.GAME_EXPAND_REGENERATED)
    assert ctx.resolved_expansion(256) == g.GAME_EXPAND_REGENERATED and ctx.resolved_expansion(257) == -1
    with pytest.raises(g.GameError) as e:
        ctx.fitness(dev(np.zeros((257, ctx.num_terms()), np.float32)))
    assert e.value.code == 5
    # trigonometric family outside [-pi, pi]: the fast sincos is not offered
    X2 = (X * 4.0).astype(np.float32)
    ctx2 = make_ctx(TRIG, 3, X2, t, path=g.GAME_PATH_TENSOR)
    ctx2.set_expansion(g.GAME_EXPAND_REGENERATED)
    assert ctx2.resolved_expansion(64) == -1
    ctx2.set_expansion(g.GAME_EXPAND_AUTO)
    assert ctx2.resolved_expansion(64) == g.GAME_EXPAND_MATERIALIZED


def test_auto_regenerates_config4_full_size(orc):
    """AUTO's measured choice: config 4 -- 9 k-blocks, four feature groups, 3907 tiles -- runs the
    regenerated expansion; both sources are held to the oracle at full size, agree closely with each other, and the
    neighbouring shapes where the materialised matrix measured faster keep it."""
    w = wl.config(4)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    rng = np.random.default_rng(41)
    pop = rng.uniform(-1, 1, (w.P, w.K)).astype(np.float32)
    rows = np.unique(np.concatenate([[0, w.P - 1], rng.choice(w.P, 6, replace=False)]))
    ctx = make_ctx(fam, d, X, t, w.act, w.err, w.R, g.GAME_PATH_AUTO)
    assert ctx.resolved_path(w.P) == g.GAME_PATH_TENSOR
    assert ctx.resolved_expansion(w.P) == g.GAME_EXPAND_REGENERATED
    assert ctx.resolved_expansion(20) == g.GAME_EXPAND_MATERIALIZED          # small populations: no gain measured
    assert ctx.resolved_expansion(257) == g.GAME_EXPAND_MATERIALIZED         # more than one CTA pair of chromosomes
    got = {}
    for mode in (g.GAME_EXPAND_AUTO, g.GAME_EXPAND_MATERIALIZED):
        ctx.set_expansion(mode)
        got[mode] = ctx.fitness(dev(pop)).cpu().numpy()
        check_fitness(orc, got[mode][rows], fam, d, X, t, pop[rows], w.act, w.err, w.R, g.GAME_PATH_TENSOR, "cfg 4 expansion %d" % mode)
    # the generator's stores race with nothing: repeated launches give the same bits
    ctx.set_expansion(g.GAME_EXPAND_AUTO)
    for _ in range(6):
        again = ctx.fitness(dev(pop)).cpu().numpy()
        assert np.array_equal(again.view(np.uint32), got[g.GAME_EXPAND_AUTO].view(np.uint32))
    # MSE is continuous in z: there the two sources must agree far inside the tolerance class
    ctx.set_error(MSE, 0.0)
    for mode in (g.GAME_EXPAND_AUTO, g.GAME_EXPAND_MATERIALIZED):
        ctx.set_expansion(mode)
        got[mode] = ctx.fitness(dev(pop)).cpu().numpy()
    assert np.allclose(got[g.GAME_EXPAND_AUTO], got[g.GAME_EXPAND_MATERIALIZED], rtol=2e-4, atol=2e-6)
    ctx.destroy()
    # a fifth of the patterns (782 tiles per launch): the start-up is not amortised, AUTO streams the matrix
    ctx = make_ctx(fam, d, X[:200000], t[:200000], w.act, w.err, w.R, g.GAME_PATH_AUTO)
    assert ctx.resolved_expansion(w.P) == g.GAME_EXPAND_MATERIALIZED
    ctx.destroy()


def test_expansion_matrix_is_built_on_first_use(orc):
    """game_load defers the fp16 expansion matrix when max|E| is known without measuring (trig; Chebyshev on [-1, 1]):
    a context whose fitness calls regenerate the expansion in the kernel never allocates its 2 N Kpad bytes; the first
    call that streams the matrix builds it, with the same result as before."""
    import torch
    N, F, d, P = 300000, 32, 8, 64
    rng = np.random.default_rng(77)
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    t = rng.integers(0, 2, N).astype(np.float32)
    e16_bytes = ((N + 255) // 256) * 256 * 576 * 2
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    ctx = make_ctx(TRIG, d, X, t, SIGMOID, MSE, 0.0, g.GAME_PATH_TENSOR)
    pop = rng.uniform(-1, 1, (P, ctx.num_terms())).astype(np.float32)
    ctx.set_expansion(g.GAME_EXPAND_REGENERATED)
    a = ctx.fitness(dev(pop)).cpu().numpy()
    torch.cuda.synchronize()
    used_regen = free0 - torch.cuda.mem_get_info()[0]
    assert used_regen < e16_bytes // 2, (used_regen, e16_bytes)
    ctx.set_expansion(g.GAME_EXPAND_MATERIALIZED)
    b = ctx.fitness(dev(pop)).cpu().numpy()
    torch.cuda.synchronize()
    used_mat = free0 - torch.cuda.mem_get_info()[0]
    assert used_mat >= e16_bytes, (used_mat, e16_bytes)
    assert np.allclose(a, b, rtol=2e-4, atol=2e-6)
    rows = np.array([0, 17, P - 1])
    check_fitness(orc, b[rows], TRIG, d, X, t, pop[rows], SIGMOID, MSE, 0.0, g.GAME_PATH_TENSOR, "deferred E16")
    ctx.destroy()
    # Chebyshev features outside [-1, 1]: the maximum has to be measured, so the matrix is built at load (and the path decided)
    ctx = make_ctx(CHEB, 3, (X[:4096, :8] * 1.5).astype(np.float32), t[:4096], path=g.GAME_PATH_AUTO)
    assert ctx.resolved_path(P) in (g.GAME_PATH_TENSOR_SPLIT, g.GAME_PATH_FP32)          # max|T_3(1.5)| = 9 > 2: no one-pass fp16 path
    ctx.destroy()


def test_trajectory_regenerated(orc):
    """A GA run with the regenerated expansion: operators bit-exact, fitness within the tensor class."""
    w = wl.config(1).scaled(P=64, generations=6)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    ctx = make_ctx(fam, d, X, t, w.act, w.err, w.R, g.GAME_PATH_TENSOR)
    ctx.set_expansion(g.GAME_EXPAND_REGENERATED)
    gp = g.ga_params(P=w.P)
    gpo = orc.GaParams(P=w.P, tournament_size=3, elitism=2, elite_mode=0, selection=0, init_mode=1,
                       p_crossover=0.9, p_mutation=0.05, stop_error=-1.0)
    ctx.evolve(0, w.seed, gp)
    for gen in range(w.generations):
        pop, fit, order = ctx.get_population_host()
        check_fitness(orc, fit, fam, d, X, t, pop, w.act, w.err, w.R, g.GAME_PATH_TENSOR, "gen %d" % gen)
        assert np.array_equal(order, orc.rank(fit))
        nxt = orc.ga_step(gpo, w.seed, gen, order, fit, pop)
        ctx.evolve(1, w.seed, gp)
        pop2, _, _ = ctx.get_population_host()
        assert np.array_equal(pop2.view(np.uint32), nxt.view(np.uint32))


# ---- pattern-sharded evaluation (game_fitness_sums + game_advance) ------------------------------------
@pytest.mark.parametrize("cfg_P", [(1, 20), (2, 300), (3, 512)])
def test_sharded_one_rank_equals_evolve(orc, cfg_P):
    """One shard holding every pattern: the sharded loop reproduces game_evolve bit for bit."""
    from paper_1304_0597_b200 import sharded
    cfg, P = cfg_P
    w = wl.config(cfg).scaled(N=min(wl.config(cfg).N, 20000), P=P, generations=5)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    gp = g.ga_params(P=w.P)
    ref = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    ref.evolve(w.generations, w.seed, gp)
    pop_r, fit_r, ord_r = ref.get_population_host()

    def configure(c):
        c.set_activation(w.act)
        c.set_error(w.err, w.R)
    sg = sharded.ShardedGame.load(fam, d, X, t, 1, 0, configure=configure)
    done, res = sg.evolve(w.generations, w.seed, gp)
    assert done == w.generations and sg.game.generation() == w.generations
    pop_s, fit_s, ord_s = sg.game.get_population_host()
    assert np.array_equal(pop_s.view(np.uint32), pop_r.view(np.uint32))
    assert np.array_equal(fit_s.view(np.uint32), fit_r.view(np.uint32)) and np.array_equal(ord_s, ord_r)
    assert res.best_index == ord_r[0] and res.best_error == fit_r[ord_r[0]]


@pytest.mark.parametrize("path", [g.GAME_PATH_FP32, g.GAME_PATH_TENSOR])
@pytest.mark.parametrize("err,R", [(MSE, 0.0), (TMSE, 0.49), (RMSE, 0.0)])
def test_sharded_three_shards_one_gpu(orc, path, err, R):
    """Three uneven shards of the patterns, evaluated one after the other on this GPU (nothing waits on anything):
    the summed totals give the full-data fitness within the path's tolerance, and all shards end every generation
    with the same population, bit for bit -- which is also what the oracle's operators produce from that fitness."""
    from paper_1304_0597_b200 import sharded
    rng = np.random.default_rng(41)
    fam, d, F, N, P, world = CHEB, 5, 16, 40000, 256, 3
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    t = rng.integers(0, 2, N).astype(np.float32)
    seed = 77
    gp = g.ga_params(P=P)
    gpo = orc.GaParams(P=P, tournament_size=3, elitism=2, elite_mode=0, selection=0, init_mode=1, p_crossover=0.9,
                       p_mutation=0.05, stop_error=-1.0)

    def configure(c):
        c.set_error(err, R)
        c.set_path(path)
    shards = [sharded.ShardedGame.load(fam, d, X, t, world, r, configure=configure) for r in range(world)]
    for s in shards:
        s.game.evolve(0, seed, gp)                      # identical initial populations (counter-based)
    for gen in range(3):
        sums = sum(s.game.fitness_sums(None, P) for s in shards)          # what the all-reduce would deliver
        pop0 = shards[0].game.get_population_host(want_fit=False)[0]
        fit = (sums.cpu().numpy() / N)
        if err == RMSE:
            fit = np.sqrt(fit)
        check_fitness(orc, fit, fam, d, X, t, pop0, SIGMOID, err, R, path, "gen %d" % gen)
        results = [s.game.advance(sums, N, seed, gp, True) for s in shards]
        assert all(r.generations_run == 1 and r.best_index == results[0].best_index for r in results)
        fit32 = fit.astype(np.float32)
        nxt = orc.ga_step(gpo, seed, gen, orc.rank(fit32), fit32, pop0)
        for s in shards:
            p = s.game.get_population_host(want_fit=False)[0]
            assert np.array_equal(p.view(np.uint32), nxt.view(np.uint32))


def test_out_of_core_chunks(orc):
    """the dataset streamed through one context in row chunks every generation (ragged last chunk):
    fitness within the path's tolerance of the full-data oracle, operators bit-exact from the GPU's ranks."""
    from paper_1304_0597_b200 import sharded
    rng = np.random.default_rng(43)
    fam, d, F, N, P = TRIG, 3, 8, 10000, 64
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    t = rng.integers(0, 2, N).astype(np.float32)
    seed = 9
    gp = g.ga_params(P=P)
    gpo = orc.GaParams(P=P, tournament_size=3, elitism=2, elite_mode=0, selection=0, init_mode=1, p_crossover=0.9,
                       p_mutation=0.05, stop_error=-1.0)
    ctx = g.Game(fam, d, F)
    ctx.set_error(TMSE, 0.49)
    cg = sharded.ChunkedGame(ctx, X, t, 3000)
    assert cg.chunks() == [(0, 3000), (3000, 6000), (6000, 9000), (9000, 10000)]
    cg.evolve(0, seed, gp)
    for gen in range(3):
        pop = ctx.get_population_host(want_fit=False)[0]
        sums = cg.totals(P)
        path = ctx.resolved_path(P)
        fit = sums.cpu().numpy() / N
        check_fitness(orc, fit, fam, d, X, t, pop, SIGMOID, TMSE, 0.49, path, "gen %d" % gen)
        done, res = cg.evolve(1, seed, gp)
        assert done == 1 and ctx.generation() == gen + 1
        # evolve(1) recomputed the same totals (deterministic), so the operators started from `fit`
        fit32 = fit.astype(np.float32)
        nxt = orc.ga_step(gpo, seed, gen, orc.rank(fit32), fit32, pop)
        assert np.array_equal(ctx.get_population_host(want_fit=False)[0].view(np.uint32), nxt.view(np.uint32))


@pytest.mark.parametrize("fam,d,F,P", [(2, 8, 11, 23), (2, 1, 11, 23), (3, 6, 11, 32), (CHEB, 3, 2, 5), (TRIG, 2, 3, 17)])
@pytest.mark.parametrize("act,err,R", [(IDENTITY, TMSE, 0.49), (SIGMOID, MSE, 0.0)])
def test_thin_models_many_patterns(orc, fam, d, F, P, act, err, R):
    """Thin models on many patterns on the FP32 path (K <= 64 genes, P <= 32: the paper's Table 3 shapes), ragged N.
    (A dedicated two-patterns-per-thread kernel for these shapes was measured slower than fitness_small_kernel --
    2484 vs 2734 generations/s at 7e6 rows, degree 8 -- and dropped; the shapes stay covered here.)"""
    rng = np.random.default_rng(47)
    N = 70001
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    t = rng.integers(0, 2, N).astype(np.float32)
    K = orc.num_terms(fam, d, F)
    pop = (rng.uniform(-1, 1, (P, K)) / (np.sqrt(K) if act == IDENTITY else 1.0)).astype(np.float32)
    if fam in (2, 3):
        pop = (pop / F).astype(np.float32)               # tied terms are sums over F features
    ctx = make_ctx(fam, d, X, t, act, err, R, g.GAME_PATH_FP32)
    got = ctx.fitness(dev(pop)).cpu().numpy()
    check_fitness(orc, got, fam, d, X, t, pop, act, err, R, g.GAME_PATH_FP32, "thin")
    perm = rng.permutation(P)                             # P20: independent of the chromosome's position
    got2 = ctx.fitness(dev(pop[perm])).cpu().numpy()
    assert np.array_equal(got2.view(np.uint32), got[perm].view(np.uint32))


@pytest.mark.parametrize("cfg,N,P,path", [(1, None, None, g.GAME_PATH_AUTO), (2, None, 300, g.GAME_PATH_AUTO),
                                          (3, 20000, 512, g.GAME_PATH_AUTO), (4, 30000, 200, g.GAME_PATH_AUTO),
                                          (1, None, None, g.GAME_PATH_FP32)])
def test_graph_loop_equals_stepwise(orc, cfg, N, P, path):
    """game_evolve(G >= 8) on a capturable stream replays a CUDA graph of two generations (with the operators writing the
    next evaluation's fp16 genes); it must give, bit for bit, what G single-generation calls on the default stream give."""
    w = wl.config(cfg)
    w = w.scaled(N=N or w.N, P=P or w.P, generations=21)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    gp = g.ga_params(P=w.P)
    step = make_ctx(fam, d, X, t, w.act, w.err, w.R, path)
    for _ in range(w.generations):
        step.evolve(1, w.seed, gp)
    ps, fs, os_ = step.get_population_host()
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ctx = g.Game(fam, d, w.F, stream=stream)
        ctx.set_activation(w.act)
        ctx.set_error(w.err, w.R)
        ctx.set_path(path)
        ctx.load(dev(X), dev(t))
        res = ctx.evolve(w.generations, w.seed, gp)
        pg, fg, og = ctx.get_population_host()
    assert res.generations_run == w.generations
    assert np.array_equal(pg.view(np.uint32), ps.view(np.uint32))
    assert np.array_equal(fg.view(np.uint32), fs.view(np.uint32)) and np.array_equal(og, os_)


def test_split_path_beyond_unit_range(orc):
    """Features outside [-1, 1] make Chebyshev terms large (|T_3(1.6)| = 11.6): the one-pass fp16 path is withdrawn
    (max|E| > 2) but the split path keeps ~22 bits of every value and still meets the FP32 tolerance class."""
    rng = np.random.default_rng(53)
    fam, d, F, N, P = CHEB, 3, 6, 3000, 40
    X = rng.uniform(-1.6, 1.6, (N, F)).astype(np.float32)
    t = rng.integers(0, 2, N).astype(np.float32)
    K = orc.num_terms(fam, d, F)
    pop = (rng.uniform(-1, 1, (P, K)) / 8).astype(np.float32)
    ctx = make_ctx(fam, d, X, t, SIGMOID, MSE, 0.0)
    assert ctx.resolved_path(P) == g.GAME_PATH_TENSOR_SPLIT
    ctx.set_path(g.GAME_PATH_TENSOR)
    assert ctx.resolved_path(P) == -1
    ctx.set_path(g.GAME_PATH_AUTO)
    got = ctx.fitness(dev(pop)).cpu().numpy()
    check_fitness(orc, got, fam, d, X, t, pop, SIGMOID, MSE, 0.0, g.GAME_PATH_TENSOR_SPLIT, "split, |E| up to 11.6")
    ctx.set_activation(IDENTITY)
    got = ctx.fitness(dev(pop)).cpu().numpy()
    check_fitness(orc, got, fam, d, X, t, pop, IDENTITY, MSE, 0.0, g.GAME_PATH_TENSOR_SPLIT, "split identity")


# ---- round 2: boundary hardening -----------------------------------------------------------------
@pytest.mark.parametrize("fam,d,F", [(TRIG, 8, 32), (CHEB, 12, 64), (CHEB, 6, 16), (2, 8, 11), (3, 6, 11), (TRIG, 1, 1)])
def test_predict_new_equals_load_then_predict(orc, fam, d, F):
    """game_predict_new (SURVEY 8(f) NEXT-1's signature; a trained chromosome applied to new data) on
    caller-supplied patterns, with NO dataset loaded, gives the bits of game_load(X_new) + game_predict and matches the
    oracle's forward pass."""
    rng = np.random.default_rng(71)
    N = 3001
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    K = orc.num_terms(fam, d, F)
    genes = (rng.standard_normal(K) / np.sqrt(K) / (F if fam in (2, 3) else 1)).astype(np.float32)
    fresh = g.Game(fam, d, F)
    for act in (SIGMOID, IDENTITY):
        fresh.set_activation(act)
        z, y = fresh.predict_new(dev(genes), dev(X))
        ctx = make_ctx(fam, d, X, np.zeros(N, np.float32), act)
        z2, y2 = ctx.predict(dev(genes))
        assert torch.equal(z.view(torch.int32), z2.view(torch.int32)) and torch.equal(y.view(torch.int32), y2.view(torch.int32))
        zr, yr = orc.forward(fam, d, X, genes, act=act)
        assert np.allclose(z.cpu().numpy(), zr, rtol=1e-5, atol=2e-5) and np.allclose(y.cpu().numpy(), yr, rtol=1e-5, atol=2e-6)
    assert fresh.generation() == 0 and fresh.population_size() == 0


def test_genes_outside_fp16_range_are_not_clamped_silently(orc):
    """|gene| > 65504 cannot be an fp16 operand: game_set_population routes AUTO to the FP32 path (parity kept) and rejects an
    explicit tensor path; NaN genes are rejected; a caller-supplied population evaluates that chromosome to NaN on the
    tensor paths (asynchronous call) and game_fitness_host reports GAME_ERR_UNSUPPORTED."""
    rng = np.random.default_rng(72)
    fam, d, F, N, P = CHEB, 3, 8, 3000, 40
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    t = rng.integers(0, 2, N).astype(np.float32)
    pop = rng.uniform(-1, 1, (P, orc.num_terms(fam, d, F))).astype(np.float32)
    pop[7, 3] = 1.0e5
    ctx = make_ctx(fam, d, X, t)
    ctx.set_population(dev(pop))
    assert ctx.resolved_path(P) == g.GAME_PATH_FP32                      # AUTO falls back, nothing clamped
    res = ctx.evolve(0, 1, g.ga_params(P=P))
    _, fit, order = ctx.get_population_host()
    check_fitness(orc, fit, fam, d, X, t, pop, SIGMOID, MSE, 0.0, g.GAME_PATH_FP32, "big gene, FP32 fallback")
    assert res.best_index == order[0]
    for path in (g.GAME_PATH_TENSOR, g.GAME_PATH_TENSOR_SPLIT):
        c2 = make_ctx(fam, d, X, t, path=path)
        with pytest.raises(g.GameError) as e:
            c2.set_population(dev(pop))
        assert e.value.code == 5
        assert c2.population_size() == 0                                 # the rejected population was not installed
        got = c2.fitness(dev(pop)).cpu().numpy()                         # asynchronous call: NaN for THAT chromosome only
        assert np.isnan(got[7]) and np.isfinite(np.delete(got, 7)).all()
        ok = np.delete(np.arange(P), 7)
        check_fitness(orc, got[ok], fam, d, X, t, pop[ok], SIGMOID, MSE, 0.0, path, "others unaffected")
        with pytest.raises(g.GameError) as e:
            c2.fitness_host(pop)
        assert e.value.code == 5
    bad = pop.copy()
    bad[7, 3] = np.nan
    with pytest.raises(g.GameError) as e:
        ctx.set_population(dev(bad))
    assert e.value.code == 6
    pop[7, 3] = 65504.0                                                  # the largest finite fp16: still a tensor-path operand
    c3 = make_ctx(fam, d, X, t, path=g.GAME_PATH_TENSOR_SPLIT)
    c3.set_population(dev(pop))
    assert c3.resolved_path(P) == g.GAME_PATH_TENSOR_SPLIT


def test_two_contexts_with_different_shared_memory_needs(orc):
    """The dynamic-shared-memory opt-in is recorded per context (i.e. per device), not per process: two contexts whose
    launches of the SAME kernel instantiation need different amounts both run, in either order, and agree with the
    FFMA path.  (Two devices are not available here; the per-context record is what makes that case work.)"""
    rng = np.random.default_rng(73)
    N, P = 148 * 256 + 77, 200
    shapes = [(CHEB, 3, 32), (TRIG, 8, 32)]           # K = 128 (2 resident k-blocks) and K = 544 (9): same kernel template
    ctxs, pops = [], []
    for fam, d, F in shapes:
        X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
        t = rng.integers(0, 2, N).astype(np.float32)
        ctxs.append(make_ctx(fam, d, X, t, path=g.GAME_PATH_TENSOR))
        pops.append(rng.uniform(-1, 1, (P, ctxs[-1].K)).astype(np.float32))
    first = [c.fitness(dev(p)).cpu().numpy() for c, p in zip(ctxs, pops)]
    again = [c.fitness(dev(p)).cpu().numpy() for c, p in reversed(list(zip(ctxs, pops)))][::-1]
    for c, p, a, b in zip(ctxs, pops, first, again):
        assert np.array_equal(a.view(np.uint32), b.view(np.uint32))
        c.set_path(g.GAME_PATH_FP32)
        ref = c.fitness(dev(p)).cpu().numpy()
        assert np.allclose(a, ref, rtol=1e-3, atol=1e-5)


def test_tuning_knobs_are_per_context():
    ctx = g.Game(CHEB, 2, 4)
    for knob, value in ((99, 0), (-1, 0), (g.GAME_TUNE_CTA_GROUP, 3), (g.GAME_TUNE_SIGMOID, 1), (g.GAME_TUNE_RATIONAL_SHARE, 9)):
        with pytest.raises(g.GameError) as e:
            ctx.set_tuning(knob, value)
        assert e.value.code == 1
    rng = np.random.default_rng(74)
    X = rng.uniform(-1, 1, (5000, 4)).astype(np.float32)
    t = rng.integers(0, 2, 5000).astype(np.float32)
    pop = rng.uniform(-1, 1, (300, ctx.K)).astype(np.float32)
    a, b = g.Game(CHEB, 2, 4), g.Game(CHEB, 2, 4)
    b.set_tuning(g.GAME_TUNE_PDL, 0)                   # a launch attribute only: same bits
    b.set_tuning(g.GAME_TUNE_HALF_TILES, 0)
    b.set_tuning(g.GAME_TUNE_HALF_TILES, -1)           # back to automatic
    for c in (a, b):
        c.load(dev(X), dev(t))
    fa, fb = a.fitness(dev(pop)), b.fitness(dev(pop))
    assert torch.equal(fa.view(torch.int32), fb.view(torch.int32))


def test_async_advance_with_stop_equals_evolve(orc):
    """The device-resident sharded loop (asynchronous game_advance, stop flag on the device, polled) against game_evolve
    with the same stop threshold: same generations applied, same population, same fitness bits."""
    from paper_1304_0597_b200 import sharded
    w = wl.config(1)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    probe = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    hist = [probe.evolve(0, w.seed, g.ga_params(P=w.P)).best_error]
    for _ in range(60):
        hist.append(probe.evolve(1, w.seed, g.ga_params(P=w.P)).best_error)
    target = float(hist[37])
    first = next(i for i, h in enumerate(hist) if h <= target)
    gp = g.ga_params(P=w.P, stop_error=target)
    ref = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    r = ref.evolve(60, w.seed, gp)
    assert r.stopped_on_error == 1 and r.generations_run == first

    def configure(c):
        c.set_activation(w.act)
        c.set_error(w.err, w.R)
    sg = sharded.ShardedGame.load(fam, d, X, t, 1, 0, configure=configure)
    done, res = sg.evolve(60, w.seed, gp)
    assert done == first and res.stopped_on_error == 1 and sg.game.generation() == first
    pr, fr, orr = ref.get_population_host()
    ps, fs, os_ = sg.game.get_population_host()
    assert np.array_equal(pr.view(np.uint32), ps.view(np.uint32))
    assert np.array_equal(fr.view(np.uint32), fs.view(np.uint32)) and np.array_equal(orr, os_)
    assert res.best_error == r.best_error and res.best_index == r.best_index
    # a second call continues from the device-side counters and stops at once
    done2, res2 = sg.evolve(5, w.seed, gp)
    assert done2 == 0 and res2.stopped_on_error == 1 and sg.game.generation() == first


# ---- round 2: the whole loop as one persistent cooperative kernel (sub-wave problems, configs 1-2) -------------------------
@pytest.mark.parametrize("cfg,P,gens,path,act,err", [
    (1, None, 21, g.GAME_PATH_AUTO, SIGMOID, TMSE),           # config 1 as benchmarked (split path, local rank)
    (2, None, 10, g.GAME_PATH_AUTO, SIGMOID, TMSE),           # config 2 as benchmarked (P = 1024: distributed rank)
    (2, 300, 21, g.GAME_PATH_AUTO, SIGMOID, TMSE),            # ragged P over three chromosome blocks
    (2, 256, 5, g.GAME_PATH_TENSOR, SIGMOID, MSE),            # one-pass fp16 operands, tanh logistic, odd generation count
    (1, 64, 8, g.GAME_PATH_TENSOR, IDENTITY, RMSE),
    (1, None, 1, g.GAME_PATH_TENSOR_SPLIT, IDENTITY, TMSE),
    (1, None, 0, g.GAME_PATH_AUTO, SIGMOID, MSE),             # evaluation only
])
def test_persistent_loop_equals_launch_path(orc, cfg, P, gens, path, act, err):
    """game_evolve on a sub-wave problem runs ONE persistent kernel (fitness tiles -> grid barrier -> rank -> operators ->
    grid barrier, looping on the device).  It must give, bit for bit, what stepping the launch-per-kernel path one
    generation at a time gives (GAME_TUNE_PERSISTENT = 0): population, fitness, order, best -- PAPER.md L217-L220."""
    w = wl.config(cfg)
    w = w.scaled(P=P or w.P, generations=gens)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    R = 0.49 if err == TMSE else 0.0
    gp = g.ga_params(P=w.P)
    step = make_ctx(fam, d, X, t, act, err, R, path)
    step.set_tuning(g.GAME_TUNE_PERSISTENT, 0)
    n0 = step.launch_count()
    step.evolve(0, w.seed, gp)
    for _ in range(gens):
        step.evolve(1, w.seed, gp)
    ps, fs, os_ = step.get_population_host()
    launches_step = step.launch_count() - n0
    ctx = make_ctx(fam, d, X, t, act, err, R, path)
    n0 = ctx.launch_count()
    res = ctx.evolve(gens, w.seed, gp)
    launches = ctx.launch_count() - n0
    assert launches <= 4 <= launches_step, (launches, launches_step)      # init, split expansion, fp16 copy, the ONE loop kernel
    pg, fg, og = ctx.get_population_host()
    assert res.generations_run == gens and ctx.generation() == gens
    assert np.array_equal(pg.view(np.uint32), ps.view(np.uint32))
    assert np.array_equal(fg.view(np.uint32), fs.view(np.uint32)) and np.array_equal(og, os_)
    assert res.best_index == og[0] and res.best_error == fg[og[0]]
    # continuing in two more calls (resume across kernels, buffer parity) stays on the same trajectory
    for extra in (3, 2):
        for _ in range(extra):
            step.evolve(1, w.seed, gp)
        ctx.evolve(extra, w.seed, gp)
    ps, fs, os_ = step.get_population_host()
    pg, fg, og = ctx.get_population_host()
    assert np.array_equal(pg.view(np.uint32), ps.view(np.uint32)) and np.array_equal(fg.view(np.uint32), fs.view(np.uint32))
    # and a stand-alone fitness call reproduces the loop's fitness bits
    f2 = ctx.fitness(dev(pg)).cpu().numpy()
    assert np.array_equal(f2.view(np.uint32), fg.view(np.uint32))


@pytest.mark.parametrize("cfg,P,gens", [(1, None, 9), (1, 41, 6), (1, 3, 5), (2, 33, 4)])
def test_persistent_local_population_form(orc, cfg, P, gens):
    """Small populations (P K <= 4096 genes) run the persistent loop with the whole population in every CTA's shared memory
    (no population traffic, one grid barrier per generation).  Same bits as the shared-population form
    (GAME_TUNE_PERSISTENT = 2) and as the launch path (0), including odd P, P = 3 and a resumed run."""
    w = wl.config(cfg)
    w = w.scaled(P=P or w.P, generations=gens)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    gp = g.ga_params(P=w.P)
    out = {}
    for knob in (1, 2, 0):
        ctx = make_ctx(fam, d, X, t, w.act, w.err, w.R, g.GAME_PATH_AUTO)
        ctx.set_tuning(g.GAME_TUNE_PERSISTENT, knob)
        ctx.evolve(gens, w.seed, gp)
        ctx.evolve(3, w.seed, gp)                              # resume: the global copy written at the end of the first call
        out[knob] = ctx.get_population_host()
        f2 = ctx.fitness(dev(out[knob][0])).cpu().numpy()      # the fp16 copy written at the end matches the population
        assert np.array_equal(f2.view(np.uint32), out[knob][1].view(np.uint32))
        ctx.destroy()
    for knob in (2, 0):
        for a, b in zip(out[1], out[knob]):
            assert np.array_equal(np.asarray(a).view(np.uint32), np.asarray(b).view(np.uint32)), knob
    # the oracle's operators from the GPU's own order reproduce one more generation bit for bit
    pop, fit, order = out[1]
    check_fitness(orc, fit, fam, d, X, t, pop, w.act, w.err, w.R, g.GAME_PATH_TENSOR_SPLIT, "local form")
    assert np.array_equal(order, orc.rank(fit))


def test_persistent_loop_stop_criterion(orc):
    w = wl.config(1)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    ref = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    ref.set_tuning(g.GAME_TUNE_PERSISTENT, 0)
    hist = [ref.evolve(0, w.seed, g.ga_params(P=w.P)).best_error]
    for _ in range(60):
        hist.append(ref.evolve(1, w.seed, g.ga_params(P=w.P)).best_error)
    target = float(hist[33])
    first = next(i for i, h in enumerate(hist) if h <= target)
    ctx = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    r = ctx.evolve(60, w.seed, g.ga_params(P=w.P, stop_error=target))
    assert r.stopped_on_error == 1 and r.generations_run == first and ctx.generation() == first and r.best_error <= target
    ref2 = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    ref2.set_tuning(g.GAME_TUNE_PERSISTENT, 0)
    r2 = ref2.evolve(60, w.seed, g.ga_params(P=w.P, stop_error=target))
    assert (r2.generations_run, r2.best_error, r2.best_index) == (r.generations_run, r.best_error, r.best_index)
    pa, fa, oa = ctx.get_population_host()
    pb, fb, ob = ref2.get_population_host()
    assert np.array_equal(pa.view(np.uint32), pb.view(np.uint32)) and np.array_equal(fa.view(np.uint32), fb.view(np.uint32))
    assert np.array_equal(oa, ob)


# ---- round 3: boundary corners ----------------------------------------------------------------------------------
def _bits_equal_state(a, b):
    pa, fa, oa = a.get_population_host()
    pb, fb, ob = b.get_population_host()
    assert np.array_equal(pa.view(np.uint32), pb.view(np.uint32))
    assert np.array_equal(fa.view(np.uint32), fb.view(np.uint32)) and np.array_equal(oa, ob)


def test_advance_on_a_population_larger_than_any_fitness_call_saw(orc):
    """game_advance's operators also write the fp16 copy the next tensor-path fitness call reads.  That buffer used to be
    sized by fitness calls only: a context that had evaluated 64 chromosomes, then got 1024 installed and was advanced with
    totals computed ELSEWHERE (another context, another rank) wrote past its end.  Now game_advance sizes it itself: the
    step and the evaluation after it equal game_evolve's, bit for bit (L217-L220)."""
    w = wl.config(3).scaled(N=20000, P=1024)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    gp = g.ga_params(P=w.P)
    pop = dev(wl.uniform_population(w.P, w.K, 6))
    a = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    assert a.resolved_path(w.P) == g.GAME_PATH_TENSOR
    a.fitness(dev(wl.uniform_population(64, w.K, 5)))            # scratch sized for 64 chromosomes
    a.set_population(pop)
    other = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    other.set_population(pop)
    sums = other.fitness_sums(None, w.P)                         # the totals come from another context
    res = a.advance(sums, X.shape[0], w.seed, gp, True, sync=True)
    assert res.generations_run == 1
    a.evolve(0, w.seed, gp)                                      # evaluates from the fp16 copy the operators wrote
    ref = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    ref.set_population(pop)
    ref.evolve(1, w.seed, gp)
    _bits_equal_state(a, ref)


def test_async_evaluation_only_calls_inside_a_run_keep_the_trajectory(orc):
    """An asynchronous run may evaluate without stepping (apply_operators = 0, e.g. to log the fitness) between steps.  The
    operators' Philox draws are keyed on the steps APPLIED (DESIGN R3-R6), not on the evaluations made, so the trajectory is
    game_evolve's -- and so is the next run's, which must not reuse a generation key."""
    w = wl.config(1)
    fam, d = w.family, w.degree
    X, t, _ = wl.make(w, lambda X, c: orc.forward(fam, d, X, c))
    gp = g.ga_params(P=w.P)
    N = X.shape[0]
    ref = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    a = make_ctx(fam, d, X, t, w.act, w.err, w.R)
    ref.evolve(0, w.seed, gp)
    a.evolve(0, w.seed, gp)
    sums = torch.empty(w.P, dtype=torch.float64, device="cuda")
    for steps, logs in ((6, (0, 2, 3)), (5, (4,))):
        ref.evolve(steps, w.seed, gp)
        for k in range(steps):
            a.fitness_sums(None, w.P, out=sums)
            if k in logs:
                a.advance(sums, N, w.seed, gp, False, sync=False)        # evaluation only, in the middle of the run
            a.advance(sums, N, w.seed, gp, True, sync=False)
        a.fitness_sums(None, w.P, out=sums)
        a.advance(sums, N, w.seed, gp, False, sync=False)                # the returned fitness belongs to the returned population
        res = a.sync()
        assert res.generations_run == steps and a.generation() == ref.generation()
        _bits_equal_state(a, ref)


def test_set_population_rejected_while_growing_keeps_the_installed_one():
    """A population that needs larger buffers is checked BEFORE the old buffers are given up: NaN genes are refused and
    the population installed before is still there, unchanged."""
    ctx = g.Game(CHEB, 3, 2)
    old = dev(wl.uniform_population(8, ctx.K, 1))
    ctx.set_population(old)
    bad = wl.uniform_population(64, ctx.K, 2)
    bad[40, 3] = np.nan
    with pytest.raises(g.GameError) as e:
        ctx.set_population(dev(bad))
    assert e.value.code == 6
    assert ctx.population_size() == 8
    got, _, _ = ctx.get_population(want_fit=False)
    assert torch.equal(got.view(torch.int32), old.view(torch.int32))
    ctx.set_population(dev(wl.uniform_population(64, ctx.K, 3)))      # a clean one of that size is accepted
    assert ctx.population_size() == 64
