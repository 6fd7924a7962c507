"""Pins P5-P13: the oracle's fitness against the paper's worked example,
library routines, closed forms, invariants and hand-written brute force."""
import math
import os

import numpy as np

TRIG, CHEB = 0, 1
SIGMOID, IDENTITY = 0, 1
MSE, TMSE, RMSE = 0, 1, 2
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "tmse_worked_example.txt")


def _golden_rows():
    rows = []
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        rows.append((f[0], [float(v) for v in f[1:]]))
    return rows


def test_p5_paper_worked_example(orc):
    # PAPER.md L109/L118 through the public fitness call: identity activation, Chebyshev d=1,
    # F=1, X=(-1,+1): Out = c0 + c1*x, so genes ((y1+y2)/2, (y2-y1)/2) give outputs (y1, y2).
    X = np.array([[-1.0], [1.0]], dtype=np.float32)
    exact = {"first": (0.2401, 0.0), "second": (0.13005, 0.13005)}
    for name, (t1, y1, t2, y2, R, mse_print, tmse_print) in _golden_rows():
        genes = np.array([[(y1 + y2) / 2, (y2 - y1) / 2]], dtype=np.float32)
        t = np.array([t1, t2], dtype=np.float32)
        mse = orc.fitness(CHEB, 1, X, t, genes, act=IDENTITY, err=MSE)[0]
        tmse = orc.fitness(CHEB, 1, X, t, genes, act=IDENTITY, err=TMSE, R=R)[0]
        rmse = orc.fitness(CHEB, 1, X, t, genes, act=IDENTITY, err=RMSE)[0]
        assert abs(mse - mse_print) < 0.005 and abs(tmse - tmse_print) < 0.005
        assert abs(mse - exact[name][0]) < 1e-7 and abs(tmse - exact[name][1]) < 1e-7
        assert abs(rmse - math.sqrt(exact[name][0])) < 1e-7
    # the model must PREFER the first solution under TMSE and the second under MSE (L109-L118)
    assert exact["second"][0] < exact["first"][0] and exact["first"][1] < exact["second"][1]


def test_p5_tmse_boundary_is_inclusive(orc):
    # |r| == R -> 0 (eq. 10's "<=" branch, DESIGN G5); just above -> r^2, still divided by all N
    X = np.array([[-1.0], [1.0]], dtype=np.float32)
    t = np.array([0.0, 0.0], dtype=np.float32)
    g = np.array([[0.5, 0.0]], dtype=np.float32)          # outputs (0.5, 0.5) -> |r| = 0.5
    assert orc.fitness(CHEB, 1, X, t, g, act=IDENTITY, err=TMSE, R=0.5)[0] == 0.0
    g = np.array([[0.625, 0.125]], dtype=np.float32)      # outputs (0.5, 0.75)
    assert orc.fitness(CHEB, 1, X, t, g, act=IDENTITY, err=TMSE, R=0.5)[0] == 0.75 ** 2 / 2
    fit, near = orc.fitness(CHEB, 1, X, t, g, act=IDENTITY, err=TMSE, R=0.5, delta=1e-6)
    assert near[0] == 1


def test_p6_identity_mse_is_a_gemm(orc):
    rng = np.random.default_rng(2)
    for fam, d in ((TRIG, 3), (CHEB, 5)):
        X = rng.uniform(-1, 1, (300, 5)).astype(np.float32)
        K = orc.num_terms(fam, d, 5)
        pop = rng.uniform(-1, 1, (17, K)).astype(np.float32)
        t = rng.normal(size=300).astype(np.float32)
        E = orc.expand(fam, d, X)
        ref = np.mean((t.astype(np.float64)[:, None] - E @ pop.astype(np.float64).T) ** 2, axis=0)
        got = orc.fitness(fam, d, X, t, pop, act=IDENTITY, err=MSE)
        assert np.allclose(got, ref, rtol=1e-12, atol=0)
        assert np.allclose(orc.fitness(fam, d, X, t, pop, act=IDENTITY, err=RMSE), np.sqrt(ref), rtol=1e-12)


def test_p7_least_squares_optimum(orc):
    rng = np.random.default_rng(3)
    X = rng.uniform(-1, 1, (400, 3)).astype(np.float32)
    d = 3
    E = orc.expand(CHEB, d, X)
    # drop the two redundant constant columns (DESIGN G3) for a well-posed lstsq
    keep = [k for k in range(E.shape[1]) if not (k % (d + 1) == 0 and k > 0)]
    t = rng.normal(size=400)
    sol, *_ = np.linalg.lstsq(E[:, keep], t, rcond=None)
    c = np.zeros(E.shape[1])
    c[keep] = sol
    c32 = c.astype(np.float32)
    t32 = t.astype(np.float32)
    base = orc.fitness(CHEB, d, X, t32, c32[None], act=IDENTITY, err=MSE)[0]
    resid = np.mean((t32.astype(np.float64) - E @ c32.astype(np.float64)) ** 2)
    assert abs(base - resid) < 1e-12        # the mean, not the sum
    for _ in range(20):
        pert = (c + rng.normal(scale=0.05, size=c.shape)).astype(np.float32)
        assert orc.fitness(CHEB, d, X, t32, pert[None], act=IDENTITY, err=MSE)[0] >= base - 1e-9


def test_p8_planted_chromosome(orc):
    rng = np.random.default_rng(4)
    X = rng.uniform(-1, 1, (500, 6)).astype(np.float32)
    K = orc.num_terms(TRIG, 2, 6)
    c0 = rng.standard_normal(K).astype(np.float32)
    z, y = orc.forward(TRIG, 2, X, c0, act=SIGMOID)
    # regression targets = the oracle's own output: zero error in fp64 needs float64 targets, the
    # API takes float32 ones, so the residual is the float32 rounding of y: <= (2^-25)^2
    t = y.astype(np.float32)
    f = orc.fitness(TRIG, 2, X, t, c0[None], act=SIGMOID, err=MSE)[0]
    assert 0.0 <= f <= (2.0 ** -25) ** 2
    # thresholded targets, no flips: zero misclassifications; with R=0.5 the TMSE is exactly 0
    tb = (z > 0).astype(np.float32)
    assert np.all((y > 0.5) == (tb > 0.5))
    assert orc.fitness(TRIG, 2, X, tb, c0[None], act=SIGMOID, err=TMSE, R=0.5)[0] == 0.0
    other = rng.standard_normal((5, K)).astype(np.float32)
    assert np.all(orc.fitness(TRIG, 2, X, tb, other, act=SIGMOID, err=TMSE, R=0.5) > 0.0)


def test_p9_tied_gene_reduction(orc):
    # eq. 9 as printed (L100-L103): one coefficient set shared by all features, acting on the
    # per-pattern sums of cosines and sines (the paper's two precomputed vectors, L254).
    rng = np.random.default_rng(5)
    N, F, d = 200, 4, 3
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    a0 = 0.3
    a = rng.uniform(-1, 1, d).astype(np.float32)
    b = rng.uniform(-1, 1, d).astype(np.float32)
    Xd = X.astype(np.float64)
    out = np.full(N, 0.0)
    for m in range(1, d + 1):
        out += a[m - 1] * np.cos(m * Xd).sum(axis=1) + b[m - 1] * np.sin(m * Xd).sum(axis=1)
    out += a0
    # K-gene chromosome whose blocks are all equal; the single a_0 of eq. 9 goes in block 0 only
    block = np.concatenate([[0.0], a, b]).astype(np.float32)
    genes = np.tile(block, F)
    genes[0] = np.float32(a0)
    z, _ = orc.forward(TRIG, d, X, genes, act=IDENTITY)
    assert np.allclose(z, out - a0 + np.float64(np.float32(a0)), atol=1e-12)


def test_p10_row_replication(orc):
    # the paper's own scaling construction (L326): replicated rows leave mean-type errors unchanged
    rng = np.random.default_rng(6)
    X = rng.uniform(-1, 1, (64, 3)).astype(np.float32)
    t = rng.integers(0, 2, 64).astype(np.float32)
    pop = rng.uniform(-1, 1, (6, orc.num_terms(CHEB, 4, 3))).astype(np.float32)
    for err in (MSE, TMSE, RMSE):
        f1 = orc.fitness(CHEB, 4, X, t, pop, err=err, R=0.49)
        f4 = orc.fitness(CHEB, 4, np.tile(X, (4, 1)), np.tile(t, 4), pop, err=err, R=0.49)
        assert np.allclose(f1, f4, rtol=1e-13)


def test_p11_brute_force_tiny(orc):
    # every term written out by hand: N=2, F=2, d=2, trig -> K=10
    X = np.array([[0.5, -0.25], [1.0, 0.75]], dtype=np.float32)
    t = np.array([1.0, 0.0], dtype=np.float32)
    g = np.array([0.1, 0.2, -0.3, 0.4, 0.5, -0.6, 0.7, 0.8, -0.9, 0.25], dtype=np.float32)
    gd = g.astype(np.float64)
    zs = []
    for x0, x1 in X.astype(np.float64):
        z = (gd[0] + gd[1] * math.cos(x0) + gd[2] * math.cos(2 * x0) + gd[3] * math.sin(x0) + gd[4] * math.sin(2 * x0)
             + gd[5] + gd[6] * math.cos(x1) + gd[7] * math.cos(2 * x1) + gd[8] * math.sin(x1) + gd[9] * math.sin(2 * x1))
        zs.append(z)
    ys = [1 / (1 + math.exp(-z)) for z in zs]
    mse = ((1.0 - ys[0]) ** 2 + (0.0 - ys[1]) ** 2) / 2
    assert abs(orc.fitness(TRIG, 2, X, t, g[None], err=MSE)[0] - mse) < 1e-15
    assert abs(orc.fitness(TRIG, 2, X, t, g[None], err=RMSE)[0] - math.sqrt(mse)) < 1e-15
    R = 0.45
    tm = sum(r * r for r in (1.0 - ys[0], 0.0 - ys[1]) if abs(r) > R) / 2
    assert abs(orc.fitness(TRIG, 2, X, t, g[None], err=TMSE, R=R)[0] - tm) < 1e-15
    # Chebyshev, N=1, F=2, d=2 -> K=6, identity
    X = np.array([[0.5, -0.5]], dtype=np.float32)
    g = np.array([1, 2, 3, 4, 5, 6], dtype=np.float32) / 8
    z = (1 + 2 * 0.5 + 3 * (2 * 0.25 - 1) + 4 + 5 * (-0.5) + 6 * (2 * 0.25 - 1)) / 8
    zz, yy = orc.forward(CHEB, 2, X, g, act=IDENTITY)
    assert zz[0] == z and yy[0] == z


def test_p12_permutations(orc):
    rng = np.random.default_rng(7)
    X = rng.uniform(-1, 1, (128, 4)).astype(np.float32)
    t = rng.integers(0, 2, 128).astype(np.float32)
    pop = rng.uniform(-1, 1, (9, orc.num_terms(TRIG, 2, 4))).astype(np.float32)
    f = orc.fitness(TRIG, 2, X, t, pop, err=TMSE, R=0.49)
    pn = rng.permutation(128)
    assert np.allclose(orc.fitness(TRIG, 2, X[pn], t[pn], pop, err=TMSE, R=0.49), f, rtol=1e-13)
    pp = rng.permutation(9)
    assert np.array_equal(orc.fitness(TRIG, 2, X, t, pop[pp], err=TMSE, R=0.49), f[pp])


def test_p13_sigmoid(orc):
    # sigma(0) = 1/2, sigma(z) + sigma(-z) = 1, saturation without NaN at |z| = 100 (and beyond)
    X = np.zeros((1, 1), dtype=np.float32)       # T_0 = 1, T_1 = 0 -> z = gene 0
    for zval in (0.0, 0.5, 3.0, 30.0, 100.0):
        _, yp = orc.forward(CHEB, 1, X, np.array([zval, 0], dtype=np.float32))
        _, ym = orc.forward(CHEB, 1, X, np.array([-zval, 0], dtype=np.float32))
        assert abs(yp[0] + ym[0] - 1.0) < 1e-15
        assert abs(yp[0] - 1.0 / (1.0 + math.exp(-zval))) < 1e-15
        if zval == 0.0:
            assert yp[0] == 0.5
    big = np.array([[1.0, 0.0], [-1.0, 0.0]], dtype=np.float32) * 3e38
    f = orc.fitness(CHEB, 1, X, np.array([1.0], dtype=np.float32), big)
    assert f[0] == 0.0 and f[1] == 1.0 and not np.any(np.isnan(f))


def test_p24_figures_of_merit(orc):
    # L301 definitions on a hand-made case.  Identity activation, Chebyshev d=1, F=1: Out = c0 + c1*x, genes (0, 1)
    # -> Out = x.  Patterns x = (0.9, 0.8, 0.7 | 0.6, 0.2, 0.1, -0.3, -0.5), truth (1,1,1 | 0 ...) with cut 0.5:
    X = np.array([0.9, 0.8, 0.7, 0.6, 0.2, 0.1, -0.3, -0.5, 0.4, 0.3], dtype=np.float32)[:, None]
    t = np.array([1, 1, 1, 0, 0, 0, 0, 0, 1, 1], dtype=np.float32)
    g = np.array([0.0, 1.0], dtype=np.float32)
    counts, fom, near = orc.classify(CHEB, 1, X, t, g, act=IDENTITY, cut=0.5)
    # predicted GC: x > 0.5 -> first four.  TP = 3, FP = 1 (x=0.6), TN = 4, FN = 2 (x=0.4, 0.3)
    assert counts.tolist() == [3, 1, 4, 2]
    assert fom[0] == 7 / 10           # accuracy: correctly classified / total
    assert fom[1] == 3 / 5            # completeness: GCs classified as such / all GCs
    assert fom[2] == 1 / 5            # contamination: non-GCs classified as GC / all non-GCs (L301, literal)
    assert near == 0
    # the cut is exclusive (y > cut), and sigmoid(z) > 0.5 <=> z > 0
    Xz = np.array([0.0, 1e-3, -1e-3], dtype=np.float32)[:, None]
    c2, _, n2 = orc.classify(CHEB, 1, Xz, np.array([1, 1, 0], dtype=np.float32), g, act=SIGMOID, cut=0.5, delta=1e-6)
    assert c2.tolist() == [1, 0, 1, 1] and n2 == 1
    # degenerate denominators give 0, not NaN
    c3, f3, _ = orc.classify(CHEB, 1, X[:3], t[:3], g, act=IDENTITY, cut=0.5)
    assert c3.tolist() == [3, 0, 0, 0] and f3.tolist() == [1.0, 1.0, 0.0]
    # consistency with forward(): counts recomputed from the oracle's own outputs
    rng = np.random.default_rng(30)
    Xr = rng.uniform(-1, 1, (500, 4)).astype(np.float32)
    gr = rng.standard_normal(orc.num_terms(TRIG, 3, 4)).astype(np.float32)
    tr = rng.integers(0, 2, 500).astype(np.float32)
    _, y = orc.forward(TRIG, 3, Xr, gr)
    cr, fr, _ = orc.classify(TRIG, 3, Xr, tr, gr)
    pred, truth = y > 0.5, tr > 0.5
    assert cr.tolist() == [int((pred & truth).sum()), int((pred & ~truth).sum()), int((~pred & ~truth).sum()),
                           int((~pred & truth).sum())]
    assert abs(fr[0] - np.mean(pred == truth)) < 1e-15
