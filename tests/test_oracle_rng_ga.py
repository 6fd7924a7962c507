"""Pins P14-P23: Philox, the R0 integer mappings and the GA operators."""
import ctypes
import math
import os
import subprocess
import sys

import numpy as np
import pytest

TRIG, CHEB = 0, 1


# ---- P14: Philox4x32-10 against an independent implementation (torch's ATen philox_engine) ----
_SHIM = r"""
#include <ATen/core/PhiloxRNGEngine.h>
extern "C" void aten_philox(unsigned long long seed, unsigned long long subseq,
                            unsigned long long offset, unsigned int *out) {
    at::Philox4_32 eng(seed, subseq, offset);   // counter = (offset lo, offset hi, subseq lo, subseq hi)
    for (int i = 0; i < 4; ++i) out[i] = eng();
}
"""


@pytest.fixture(scope="module")
def aten_philox(tmp_path_factory):
    import torch
    inc = os.path.join(os.path.dirname(torch.__file__), "include")
    d = tmp_path_factory.mktemp("aten_philox")
    src = d / "shim.cpp"
    src.write_text(_SHIM)
    so = d / "shim.so"
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-shared", "-fPIC", "-I", inc, "-o", str(so), str(src)])
    L = ctypes.CDLL(str(so))

    def call(seed, subseq, offset):
        out = (ctypes.c_uint32 * 4)()
        L.aten_philox(ctypes.c_uint64(seed), ctypes.c_uint64(subseq), ctypes.c_uint64(offset), out)
        return np.array(list(out), dtype=np.uint32)
    return call


def test_p14_philox_matches_aten(orc, aten_philox):
    rng = np.random.default_rng(8)
    cases = [(0, (0, 0, 0, 0)), (1, (1, 2, 3, 4)), (2**64 - 1, (2**32 - 1,) * 4)]
    for _ in range(200):
        cases.append((int(rng.integers(0, 2**63)) * 2 + int(rng.integers(0, 2)),
                      tuple(int(v) for v in rng.integers(0, 2**32, 4))))
    for seed, (c0, c1, c2, c3) in cases:
        got = orc.philox4x32_10([seed & 0xFFFFFFFF, seed >> 32], [c0, c1, c2, c3])
        ref = aten_philox(seed, c2 | (c3 << 32), c0 | (c1 << 32))
        assert np.array_equal(got, ref), (seed, c0, c1, c2, c3)


def test_p14_philox_uniformity(orc):
    # weak statistical sanity on top of the exact pin: byte histogram of 4*4096 words
    words = np.concatenate([orc.philox4x32_10([7, 9], [i, 0, 0, 0]) for i in range(4096)])
    hist = np.bincount(words.view(np.uint8), minlength=256)
    exp = words.size * 4 / 256
    chi2 = ((hist - exp) ** 2 / exp).sum()
    assert chi2 < 255 + 6 * math.sqrt(2 * 255)


# ---- P15: R0 mappings ------------------------------------------------------------------------
def test_p15_integer_mappings(orc):
    assert orc.upm1(0) == -1.0 and orc.upm1(0xFFFFFFFF) == 1.0 - 2.0 ** -23
    assert orc.upm1(0x80000000) == 0.0
    assert orc.u01(0) == 0.0 and orc.u01(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    rng = np.random.default_rng(9)
    for w in rng.integers(0, 2**32, 500):
        w = int(w)
        a, b = orc.upm1(w), orc.u01(w)
        assert -1.0 <= a < 1.0 and 0.0 <= b < 1.0
        assert (a * 2.0 ** 23) == int(a * 2.0 ** 23) and (b * 2.0 ** 24) == int(b * 2.0 ** 24)
        assert a == ((w >> 8) - 2**23) / 2.0**23 and b == (w >> 8) / 2.0**24
        for n in (1, 2, 3, 20, 1024, 8192, 2**31):
            assert orc.idx(w, n) == (w * n) >> 32 < n
    assert orc.idx(0, 17) == 0 and orc.idx(0xFFFFFFFF, 17) == 16
    assert orc.thr(1.0) == (0xFFFFFFFF, True) and orc.thr(1.5)[1]
    assert orc.thr(0.0) == (0, False) and orc.thr(-0.5) == (0, False)
    assert orc.thr(0.5) == (2**31, False)
    p = float(np.float32(0.9))
    assert orc.thr(0.9) == (math.floor(p * 2.0**32), False)


# ---- P16: initial population -----------------------------------------------------------------
def test_p16_init_modes(orc):
    P, K = 400, 250
    g = orc.init_population(1, 11, P, K).astype(np.float64).ravel()     # normal in [-1,1]
    n = g.size
    assert np.all(np.abs(g) <= 1.0)
    assert abs(g.mean()) < 4 * (1 / 3) / math.sqrt(n)
    assert abs(g.std() - 1 / 3) < 0.004
    clamp = np.mean(np.abs(g) == 1.0)
    assert 0.0015 < clamp < 0.0040         # P(|Z|>3): 0.27% normal, ~0.2% for 12-term Irwin-Hall
    # quartiles of N(0,1/9)
    assert abs(np.quantile(g, 0.75) - 0.6745 / 3) < 0.006
    u = orc.init_population(0, 11, P, K).astype(np.float64).ravel()
    assert u.min() >= -1 and u.max() < 1 and abs(u.mean()) < 0.01 and abs(u.var() - 1 / 3) < 0.01
    v = orc.init_population(2, 11, P, K).astype(np.float64).ravel()
    assert v.min() >= 0 and v.max() < 1 and abs(v.mean() - 0.5) < 0.005 and abs(v.var() - 1 / 12) < 0.003
    # counter-based: a gene depends only on (seed, p, k)
    big = orc.init_population(1, 11, P + 7, K)
    assert np.array_equal(big[:P], orc.init_population(1, 11, P, K))
    assert not np.array_equal(orc.init_population(1, 12, P, K), big[:P])


def _gp(orc, P, **kw):
    d = dict(P=P, tournament_size=3, elitism=2, elite_mode=0, selection=0, init_mode=1,
             p_crossover=0.9, p_mutation=0.05, stop_error=-1.0)
    d.update(kw)
    return orc.GaParams(**d)


# ---- P21: rank -------------------------------------------------------------------------------
def test_p21_rank(orc):
    rng = np.random.default_rng(10)
    fit = rng.random(257).astype(np.float32)
    fit[[3, 77]] = np.nan
    fit[[5, 9, 200]] = 0.25          # ties
    fit[11] = np.inf
    order = orc.rank(fit)
    assert sorted(order.tolist()) == list(range(257))
    key = np.where(np.isnan(fit), np.inf, fit)
    for a, b in zip(order[:-1], order[1:]):
        assert (key[a], a) < (key[b], b)
    assert set(order[-3:].tolist()) == {3, 11, 77} and order[-3:].tolist() == [3, 11, 77]
    assert np.array_equal(order, np.lexsort((np.arange(257), key)))


# ---- P17: tournament distribution ------------------------------------------------------------
def test_p17_tournament_closed_form(orc):
    P, t, e = 16, 3, 0
    gp = _gp(orc, P, tournament_size=t, elitism=e, p_crossover=0.0, p_mutation=0.0)
    pop = np.arange(P, dtype=np.float32)[:, None] * np.ones((1, 2), dtype=np.float32)
    order = np.arange(P, dtype=np.int32)[::-1].copy()       # rank r -> chromosome P-1-r
    fit = np.zeros(P, dtype=np.float32)
    counts = np.zeros(P)
    for g in range(400):
        _, par, do, cut = orc.ga_step(gp, 123, g, order, fit, pop, debug=True)
        assert not do.any()
        ranks = (P - 1) - par.ravel()
        counts += np.bincount(ranks, minlength=P)
    n = counts.sum()
    r = np.arange(P)
    prob = ((P - r) ** t - (P - r - 1) ** t) / P ** t
    chi2 = ((counts - n * prob) ** 2 / (n * prob)).sum()
    assert chi2 < (P - 1) + 5 * math.sqrt(2 * (P - 1)), chi2
    # t = 1 is uniform; t = 5 uses a second Philox block (draws 4..)
    gp5 = _gp(orc, P, tournament_size=5, elitism=0, p_crossover=0.0, p_mutation=0.0)
    c5 = np.zeros(P)
    for g in range(400):
        _, par, _, _ = orc.ga_step(gp5, 5, g, order, fit, pop, debug=True)
        c5 += np.bincount((P - 1) - par.ravel(), minlength=P)
    prob5 = ((P - r) ** 5 - (P - r - 1) ** 5) / P ** 5
    keep = prob5 * c5.sum() > 5
    chi2 = ((c5 - c5.sum() * prob5) ** 2 / (c5.sum() * prob5))[keep].sum()
    assert chi2 < keep.sum() + 5 * math.sqrt(2 * keep.sum())


# ---- P18: crossover --------------------------------------------------------------------------
def test_p18_crossover_invariants(orc):
    P, K, e = 41, 37, 2                       # odd child count: last B dropped (G19)
    gp = _gp(orc, P, p_mutation=0.0, elitism=e)
    rng = np.random.default_rng(11)
    pop = rng.uniform(-1, 1, (P, K)).astype(np.float32)
    fit = rng.random(P).astype(np.float32)
    order = orc.rank(fit)
    applied, cuts = [], []
    for g in range(300):
        nxt, par, do, cut = orc.ga_step(gp, 77, g, order, fit, pop, debug=True)
        applied += do.tolist()
        cuts += cut.tolist()
        for q in range(len(do)):
            pa, pb = pop[par[q, 0]], pop[par[q, 1]]
            A = nxt[e + 2 * q]
            c = cut[q] if do[q] else K
            assert 1 <= cut[q] <= K - 1
            assert np.array_equal(A[:c], pa[:c]) and np.array_equal(A[c:], pb[c:])
            if e + 2 * q + 1 < P:
                B = nxt[e + 2 * q + 1]
                assert np.array_equal(B[:c], pb[:c]) and np.array_equal(B[c:], pa[c:])
        # elites: copies of the winner (paper-literal, L148)
        assert np.array_equal(nxt[0], pop[order[0]]) and np.array_equal(nxt[1], pop[order[0]])
    n = len(applied)
    frac = np.mean(applied)
    assert abs(frac - 0.9) < 4 * math.sqrt(0.9 * 0.1 / n)
    h = np.bincount(cuts, minlength=K)[1:K]
    assert h.min() > 0 and np.bincount(cuts, minlength=K)[0] == 0
    chi2 = ((h - n / (K - 1)) ** 2 / (n / (K - 1))).sum()
    assert chi2 < (K - 2) + 5 * math.sqrt(2 * (K - 2))
    # p_c = 1 -> always; p_c = 0 -> never; K = 1 -> no-op
    _, _, do, _ = orc.ga_step(_gp(orc, P, p_crossover=1.0, p_mutation=0.0), 1, 0, order, fit, pop, debug=True)
    assert do.all()
    _, _, do, _ = orc.ga_step(_gp(orc, P, p_crossover=0.0, p_mutation=0.0), 1, 0, order, fit, pop, debug=True)
    assert not do.any()
    nxt, par, do, _ = orc.ga_step(_gp(orc, P, p_crossover=1.0, p_mutation=0.0), 1, 0, order, fit,
                                  pop[:, :1].copy(), debug=True)
    assert not do.any() and np.array_equal(nxt[2::2, 0], pop[par[:, 0], 0])


def test_elite_top_e(orc):
    P, K = 12, 5
    rng = np.random.default_rng(12)
    pop = rng.uniform(-1, 1, (P, K)).astype(np.float32)
    fit = rng.random(P).astype(np.float32)
    order = orc.rank(fit)
    nxt = orc.ga_step(_gp(orc, P, elitism=3, elite_mode=1), 3, 0, order, fit, pop)
    for j in range(3):
        assert np.array_equal(nxt[j], pop[order[j]])


# ---- P19: mutation ---------------------------------------------------------------------------
def test_p19_mutation_binomial(orc):
    P, K, e, pm = 64, 101, 2, 0.05
    gp = _gp(orc, P, p_crossover=0.0, p_mutation=pm, elitism=e)
    gp0 = _gp(orc, P, p_crossover=0.0, p_mutation=0.0, elitism=e)
    rng = np.random.default_rng(13)
    pop = (rng.uniform(-1, 1, (P, K)) + 5.0).astype(np.float32)     # outside [-1,1): a hit is visible
    fit = rng.random(P).astype(np.float32)
    order = orc.rank(fit)
    changed = 0
    trials = 0
    for g in range(40):
        a = orc.ga_step(gp, 99, g, order, fit, pop)
        b = orc.ga_step(gp0, 99, g, order, fit, pop)
        diff = a != b
        assert not diff[:e].any()                                  # elites untouched
        assert np.all((a[diff] >= -1.0) & (a[diff] < 1.0))          # fresh U[-1,1)
        assert np.all(a[~diff] > 3.0)
        changed += diff.sum()
        trials += (P - e) * K
    sd = math.sqrt(trials * pm * (1 - pm))
    assert abs(changed - trials * pm) < 4 * sd
    newvals = a[diff].astype(np.float64)
    assert abs(newvals.mean()) < 0.15


# ---- P20 / P22: elitism monotonicity and resume, on the whole loop ---------------------------
def test_p20_p22_evolve_invariants(orc):
    rng = np.random.default_rng(14)
    N, F, d = 120, 3, 2
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    c0 = rng.standard_normal(orc.num_terms(TRIG, d, F)).astype(np.float32)
    z, _ = orc.forward(TRIG, d, X, c0)
    t = (z > 0).astype(np.float32)
    gp = _gp(orc, 24)
    full = orc.evolve(TRIG, d, X, t, gp, 5, 30, err=1, R=0.49, history=True)
    h = full["best_hist"]
    assert not np.isnan(h).any() and np.all(np.diff(h) <= 0.0)     # never worsens, exactly
    assert full["gen"] == 30 and full["result"].generations_run == 30
    assert full["result"].best_error == h[-1] == full["fit"][full["order"][0]]
    assert np.all(np.abs(full["pop"]) <= 1.0)
    a = orc.evolve(TRIG, d, X, t, gp, 5, 12, err=1, R=0.49)
    b = orc.evolve(TRIG, d, X, t, gp, 5, 18, err=1, R=0.49, pop=a["pop"], gen0=a["gen"])
    assert b["gen"] == 30 and np.array_equal(b["pop"], full["pop"]) and np.array_equal(b["fit"], full["fit"])
    # stop criterion (L219, L287): threshold reached -> stops before evolving
    s = orc.evolve(TRIG, d, X, t, _gp(orc, 24, stop_error=float(h[10])), 5, 30, err=1, R=0.49)
    assert s["result"].stopped_on_error == 1 and s["result"].generations_run <= 10
    assert s["result"].best_error <= h[10]


# ---- P23: roulette (weights are DESIGN G14's choice: parity unpinned; self-consistency only) --
def test_p23_roulette_frequencies(orc):
    P = 10
    fit = np.array([0.1, 0.5, 0.3, 0.9, 0.7, 0.2, np.nan, 0.4, 0.6, 0.8], dtype=np.float32)
    order = orc.rank(fit)
    w = orc.roulette_weights(fit, order).astype(np.float64)
    assert w[-1] == 0 and w[-2] == 1 and w[0] == 2**24 + 1            # NaN -> 0, worst -> 1, best -> 2^24+1
    assert np.all(np.diff(w[:-1]) <= 0)
    gp = _gp(orc, P, selection=1, elitism=0, p_crossover=0.0, p_mutation=0.0)
    pop = np.arange(P, dtype=np.float32)[:, None] * np.ones((1, 2), dtype=np.float32)
    counts = np.zeros(P)
    for g in range(1500):
        _, par, _, _ = orc.ga_step(gp, 31, g, order, fit, pop, debug=True)
        counts += np.bincount(par.ravel(), minlength=P)
    prob = np.zeros(P)
    prob[order] = w / w.sum()
    n = counts.sum()
    keep = prob * n > 5
    assert counts[~keep].sum() <= 5
    chi2 = ((counts - n * prob) ** 2 / np.maximum(n * prob, 1e-300))[keep].sum()
    assert chi2 < keep.sum() + 5 * math.sqrt(2 * keep.sum())
    # all equal -> uniform weights; all non-finite -> all 1
    eq = np.full(P, 0.5, dtype=np.float32)
    assert np.all(orc.roulette_weights(eq, orc.rank(eq)) == 1)
    nf = np.full(P, np.nan, dtype=np.float32)
    assert np.all(orc.roulette_weights(nf, orc.rank(nf)) == 1)
