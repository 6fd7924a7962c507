"""Pins for the paper-literal (tied-coefficient) families: eq. 2 and eq. 9 as printed
(PAPER.md L57, L100-L103), chromosome sizes of eq. 7 (L91, L105), precomputed sums of L254."""
import numpy as np

TRIG, CHEB, TRIG_TIED, POLY_TIED = 0, 1, 2, 3
IDENTITY, MSE = 1, 0


def test_gene_counts_follow_eq7(orc):
    # eq. 7: NUM_genes = B*d + 1; B = 2 for the trigonometric expansion (L105), 1 in the simplest case (L89)
    for d in (1, 2, 4, 8):
        assert orc.num_terms(TRIG_TIED, d, 11) == 2 * d + 1
        assert orc.num_terms(POLY_TIED, d, 11) == d + 1


def test_trig_tied_is_eq9(orc):
    rng = np.random.default_rng(40)
    N, F, d = 100, 11, 4
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    Xd = X.astype(np.float64)
    E = orc.expand(TRIG_TIED, d, X)
    assert E.shape == (N, 2 * d + 1) and np.all(E[:, 0] == 1.0)
    for m in range(1, d + 1):       # numpy's cos/sin and its own summation: the two vectors of L254
        assert np.allclose(E[:, m], np.cos(m * Xd).sum(axis=1), atol=1e-13)
        assert np.allclose(E[:, d + m], np.sin(m * Xd).sum(axis=1), atol=1e-13)
    # equals the per-feature model with all blocks equal and the constant only once (P9, the other way round)
    genes = rng.uniform(-1, 1, 2 * d + 1).astype(np.float32)
    block = genes.copy()
    block[0] = 0.0
    wide = np.tile(block, F)
    wide[0] = genes[0]
    z_tied, _ = orc.forward(TRIG_TIED, d, X, genes, act=IDENTITY)
    z_wide, _ = orc.forward(TRIG, d, X, wide, act=IDENTITY)
    assert np.allclose(z_tied, z_wide, atol=1e-12)


def test_poly_tied_is_eq2_with_powers(orc):
    rng = np.random.default_rng(41)
    N, F, d = 64, 5, 6
    X = rng.uniform(-1, 1, (N, F)).astype(np.float32)
    Xd = X.astype(np.float64)
    E = orc.expand(POLY_TIED, d, X)
    assert E.shape == (N, d + 1) and np.all(E[:, 0] == 1.0)
    for j in range(1, d + 1):
        assert np.allclose(E[:, j], (Xd ** j).sum(axis=1), atol=1e-13)
    # degree 1: Out = a_0 + a_1 * sum_i f_i -- checked by hand on one pattern
    x = np.array([[0.5, -0.25, 0.125]], dtype=np.float32)
    z, _ = orc.forward(POLY_TIED, 1, x, np.array([0.25, 2.0], dtype=np.float32), act=IDENTITY)
    assert z[0] == 0.25 + 2.0 * 0.375
    # fitness through the tied family is still the GEMM special case
    pop = rng.uniform(-1, 1, (7, d + 1)).astype(np.float32)
    t = rng.normal(size=N).astype(np.float32)
    ref = np.mean((t.astype(np.float64)[:, None] - E @ pop.astype(np.float64).T) ** 2, axis=0)
    assert np.allclose(orc.fitness(POLY_TIED, d, X, t, pop, act=IDENTITY, err=MSE), ref, rtol=1e-12)
