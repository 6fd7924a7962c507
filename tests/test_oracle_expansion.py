"""Pins P1-P4: the oracle's feature expansion against closed forms.

None of these retypes the oracle's recurrence: each uses an identity the expansion must obey.
"""
import numpy as np

TRIG, CHEB = 0, 1


def test_p1_chebyshev_cos_identity(orc):
    # T_m(cos th) = cos(m th)
    th = np.linspace(0.0, np.pi, 257)
    X = np.cos(th).astype(np.float32)[:, None]
    d = 12
    E = orc.expand(CHEB, d, X)
    thx = np.arccos(X[:, 0].astype(np.float64))      # the angle of the float32 input actually used
    for m in range(d + 1):
        assert np.allclose(E[:, m], np.cos(m * thx), atol=5e-13 * max(1, m * m)), m


def test_p1_chebyshev_special_values(orc):
    d = 9
    X = np.array([[1.0], [-1.0], [0.0]], dtype=np.float32)
    E = orc.expand(CHEB, d, X)
    for m in range(d + 1):
        assert E[0, m] == 1.0
        assert E[1, m] == (-1.0) ** m
        assert E[2, m] == (0.0 if m % 2 else (-1.0) ** (m // 2))


def test_p1_chebyshev_explicit_polynomials(orc):
    # textbook monomial forms of T_2..T_5, typed from the textbook, not from the recurrence
    x = np.linspace(-1, 1, 41).astype(np.float32)
    xd = x.astype(np.float64)
    E = orc.expand(CHEB, 5, x[:, None])
    assert np.allclose(E[:, 0], 1.0) and np.allclose(E[:, 1], xd)
    assert np.allclose(E[:, 2], 2 * xd**2 - 1, atol=1e-14)
    assert np.allclose(E[:, 3], 4 * xd**3 - 3 * xd, atol=1e-14)
    assert np.allclose(E[:, 4], 8 * xd**4 - 8 * xd**2 + 1, atol=1e-14)
    assert np.allclose(E[:, 5], 16 * xd**5 - 20 * xd**3 + 5 * xd, atol=1e-14)


def test_p2_trig_values_and_layout(orc):
    d, F = 4, 3
    B = 2 * d + 1
    X = np.zeros((1, F), dtype=np.float32)
    E = orc.expand(TRIG, d, X)
    assert E.shape == (1, F * B)
    for i in range(F):
        blk = E[0, i * B:(i + 1) * B]
        assert np.all(blk[:d + 1] == 1.0)     # a_0 column and cos(m*0)
        assert np.all(blk[d + 1:] == 0.0)     # sin(m*0)
    rng = np.random.default_rng(0)
    X = rng.uniform(-1, 1, (50, F)).astype(np.float32)
    E = orc.expand(TRIG, d, X)
    for i in range(F):
        for m in range(1, d + 1):
            c = E[:, i * B + m]
            s = E[:, i * B + d + m]
            assert np.allclose(c * c + s * s, 1.0, atol=1e-14)
            # radians, argument m*x, no pi factor (eq. 8-9 as printed); sign of sin matters
            assert np.allclose(np.arctan2(s, c), np.angle(np.exp(1j * m * X[:, i].astype(np.float64))),
                               atol=1e-12)
    # feature-major blocks: changing feature i changes only block i
    X2 = X.copy()
    X2[:, 1] += 0.125
    E2 = orc.expand(TRIG, d, X2)
    diff = np.any(E2 != E, axis=0)
    assert not diff[:B].any() and not diff[2 * B:].any() and diff[B + 1:2 * B].all()


def test_p3_cross_family(orc):
    # Chebyshev family on cos(X) == constant + cos columns of the trig family on X
    rng = np.random.default_rng(1)
    d, F = 6, 4
    X = rng.uniform(-1, 1, (64, F)).astype(np.float32)
    Xc = np.cos(X.astype(np.float64)).astype(np.float32)
    Ec = orc.expand(CHEB, d, Xc)
    # angle whose cosine is exactly the float32 value fed to the Chebyshev side
    th = np.arccos(Xc.astype(np.float64)).astype(np.float64)
    for i in range(F):
        for m in range(d + 1):
            assert np.allclose(Ec[:, i * (d + 1) + m], np.cos(m * th[:, i]), atol=1e-12 * (1 + m * m))
    Et = orc.expand(TRIG, d, X)
    B = 2 * d + 1
    for i in range(F):
        # both are cos(m x) up to the float32 rounding of cos(x): |d cos(m acos u)/du| <= m^2
        assert np.allclose(Ec[:, i * (d + 1):(i + 1) * (d + 1)], Et[:, i * B:i * B + d + 1],
                           atol=6e-8 * d * d * 2)


def test_p4_discrete_orthogonality(orc):
    # On the Chebyshev-Gauss nodes the columns are orthogonal: 0 (i!=j), N/2 (i=j>0), N (i=j=0).
    # float32 nodes perturb the sums by ~N * 6e-8 * m^2.
    N, d = 64, 10
    x = np.cos(np.pi * (np.arange(N) + 0.5) / N).astype(np.float32)
    E = orc.expand(CHEB, d, x[:, None])
    G = E.T @ E
    expect = np.diag([N] + [N / 2.0] * d)
    assert np.allclose(G, expect, atol=N * 6e-8 * d * d * 4)
