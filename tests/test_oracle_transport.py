"""Pins of the oracle's molecular-diffusion transport terms (Eq. 3-4, readings
V1-V3 of DESIGN.md): Eq. 4 by hand, its zeros, the uniform-density reduction of Eq. 3, a three-layer column expanded
by hand, zero-flux boundaries, linearity, independent atmospheres."""
import numpy as np

K_B = 1.380649e-16


def column(L, ns=2, seed=0):
    rng = np.random.default_rng(seed)
    n = 10 ** rng.uniform(5, 12, (ns, L))
    T = rng.uniform(500, 2500, L)
    N = 10 ** rng.uniform(14, 20, L)
    D = 10 ** rng.uniform(0, 6, (ns, L))
    mass = rng.uniform(1.0, 60.0, ns) * 1.66e-24
    alpha = rng.uniform(-0.4, 0.3, ns)
    return n, T, N, D, mass, alpha


def test_equation_4_by_hand_and_its_zeros(oracle):
    n, T, N, D, mass, alpha = column(5)
    mbar, g, dz = np.array([3.9e-24]), np.array([2140.0]), np.array([3.0e6])
    _, d = oracle.transport(n, T, N, D, mass, alpha, mbar, g, dz, 1, 5, want_d=True)
    for y in range(2):
        for k in range(4):
            Th, Dh = 0.5 * (T[k] + T[k + 1]), 0.5 * (D[y, k] + D[y, k + 1])
            want = Dh / (2 * dz[0] ** 2) * ((mbar[0] - mass[y]) * g[0] * dz[0] / (K_B * Th) - alpha[y] / Th * (T[k + 1] - T[k]))
            assert abs(d[y, k] - want) <= 4e-16 * (abs(Dh / (2 * dz[0] ** 2)) * (abs((mbar[0] - mass[y]) * g[0] * dz[0] / (K_B * Th)) + abs(alpha[y] / Th * (T[k + 1] - T[k]))))
        assert d[y, 4] == 0.0                                  # no half level above the top layer
    # a species as heavy as the mean gas in an isothermal column does not separate: d = 0, no transport
    Tiso = np.full(5, 1200.0)
    mass2 = np.array([mbar[0], mass[1]])
    tr, d = oracle.transport(n, Tiso, N, D, mass2, alpha, mbar, g, dz, 1, 5, want_d=True)
    assert np.all(d[0] == 0.0) and np.all(tr[0] == 0.0) and np.any(tr[1] != 0.0)
    # without gravity and thermal diffusion nothing moves either
    tr0 = oracle.transport(n, T, N, D, mass, 0 * alpha, mbar, 0 * g, dz, 1, 5)
    assert np.all(tr0 == 0.0)


def test_uniform_gas_density_reduces_equation_3_to_plain_differences(oracle):
    """N_k constant: every ratio N_{k+-1/2} / N is 1 and tr_k = -d+ n_{k+1} - (d+ - d-) n_k + d- n_{k-1}."""
    L = 7
    n, T, N, D, mass, alpha = column(L, seed=2)
    N = np.full(L, 3.0e17)
    mbar, g, dz = np.array([3.9e-24]), np.array([980.0]), np.array([1.0e6])
    tr, dp = oracle.transport(n, T, N, D, mass, alpha, mbar, g, dz, 1, L, want_d=True)
    # d_{k-1/2} seen from layer k differs from d_{(k-1)+1/2} only by the sign of the temperature difference (Eq. 4
    # writes T_{k+-1} - T_k); rebuild it here from Eq. 4
    for y in range(2):
        for k in range(L):
            dm = 0.0
            if k > 0:
                Th, Dh = 0.5 * (T[k] + T[k - 1]), 0.5 * (D[y, k] + D[y, k - 1])
                dm = Dh / (2 * dz[0] ** 2) * ((mbar[0] - mass[y]) * g[0] * dz[0] / (K_B * Th) - alpha[y] / Th * (T[k - 1] - T[k]))
            up = n[y, k + 1] if k + 1 < L else 0.0
            dn = n[y, k - 1] if k > 0 else 0.0
            want = -dp[y, k] * up - (dp[y, k] - dm) * n[y, k] + dm * dn
            scale = abs(dp[y, k]) * (up + n[y, k]) + abs(dm) * (n[y, k] + dn)
            assert abs(tr[y, k] - want) <= 1e-15 * scale


def test_three_layer_column_expanded_by_hand(oracle):
    n = np.array([[2.0e9, 5.0e8, 1.0e8]])
    T = np.array([1000.0, 900.0, 800.0])
    N = np.array([4.0e18, 1.0e18, 2.0e17])
    D = np.array([[10.0, 40.0, 160.0]])
    mass, alpha, mbar, g, dz = np.array([2.0e-24]), np.array([0.25]), np.array([4.0e-24]), np.array([1000.0]), np.array([1.0e6])

    def d(Da, Db, Ta, Tb):                                     # from layer a towards layer b
        Th = 0.5 * (Ta + Tb)
        return 0.5 * (Da + Db) / (2 * dz[0] ** 2) * ((mbar[0] - mass[0]) * g[0] * dz[0] / (K_B * Th) - alpha[0] / Th * (Tb - Ta))

    d01, d10 = d(10.0, 40.0, 1000.0, 900.0), d(40.0, 10.0, 900.0, 1000.0)
    d12, d21 = d(40.0, 160.0, 900.0, 800.0), d(160.0, 40.0, 800.0, 900.0)
    N01, N12 = 0.5 * (N[0] + N[1]), 0.5 * (N[1] + N[2])
    want = np.array([
        -d01 * (N01 / N[1]) * n[0, 1] - d01 * (N01 / N[0]) * n[0, 0],
        -d12 * (N12 / N[2]) * n[0, 2] - (d12 * (N12 / N[1]) - d10 * (N01 / N[1])) * n[0, 1] + d10 * (N01 / N[1]) * n[0, 0],
        d21 * (N12 / N[2]) * n[0, 2] + d21 * (N12 / N[2]) * n[0, 1]])
    tr = oracle.transport(n, T, N, D, mass, alpha, mbar, g, dz, 1, 3)
    assert np.allclose(tr[0], want, rtol=1e-14, atol=0)


def test_linearity_boundaries_and_independent_atmospheres(oracle):
    L, A = 6, 3
    n, T, N, D, mass, alpha = column(L * A, ns=3, seed=5)
    mbar = np.array([3.9e-24, 4.4e-24, 2.3e-24])
    g = np.array([2140.0, 980.0, 2500.0])
    dz = np.array([3.0e6, 1.0e6, 5.0e6])
    tr = oracle.transport(n, T, N, D, mass, alpha, mbar, g, dz, A, L)
    n2 = 10 ** np.random.default_rng(9).uniform(5, 12, n.shape)
    tr2 = oracle.transport(n2, T, N, D, mass, alpha, mbar, g, dz, A, L)
    both = oracle.transport(2.0 * n + n2, T, N, D, mass, alpha, mbar, g, dz, A, L)
    assert np.allclose(both, 2.0 * tr + tr2, rtol=1e-12, atol=1e-300)
    # each atmosphere alone gives the same numbers: nothing leaks across the top of one into the bottom of the next
    for a in range(A):
        sl = slice(a * L, (a + 1) * L)
        solo = oracle.transport(n[:, sl].copy(), T[sl].copy(), N[sl].copy(), D[:, sl].copy(), mass, alpha, mbar[a:a + 1], g[a:a + 1],
                                dz[a:a + 1], 1, L)
        assert np.array_equal(solo, tr[:, sl])
    # a single layer has no neighbours: zero flux on both sides, no transport
    one = oracle.transport(n[:, :1].copy(), T[:1].copy(), N[:1].copy(), D[:, :1].copy(), mass, alpha, mbar[:1], g[:1], dz[:1], 1, 1)
    assert np.all(one == 0.0)
