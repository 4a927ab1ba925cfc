"""Pins of the oracle's thermochemical-equilibrium composition (f4, reading E1) against what
the definition fixes: closed forms of one-reaction systems, the Lagrange conditions rebuilt here from the oracle's
thermo output, element conservation, the kinetic fixed point (every reversible reaction balanced, so the source
oracle returns dn/dt = 0), and the minimum property itself against feasible perturbations."""
import numpy as np
import pytest

from conftest import SimpleNet

KB = 1.380649e-16
P0 = 1.0e6


def const_g(g):
    """NASA-7 set with G/RT = g at every T (only a7 = -g is non-zero)."""
    a = np.zeros(7)
    a[6] = -g
    return a


def simple(comp, gs, reactions=()):
    ns = len(gs)
    lo = [const_g(g) for g in gs]
    rt = [1] * len(reactions)
    return SimpleNet(comp, lo, lo, [1000.0] * ns, rt, [r[0] for r in reactions], [r[1] for r in reactions],
                     [1] * len(reactions), [[1e-12, 0.0, 0.0]] * len(reactions))


def test_isomers_follow_the_boltzmann_ratio(oracle):
    """A <=> B with the same formula: x_B / x_A = exp(-(g_B - g_A)), whatever the pressure."""
    net = simple([[1], [1]], [-3.0, -1.5])
    T, P = np.array([900.0, 900.0]), np.array([1e6, 3e2])
    n, it = oracle.equilibrium(net, T, P, np.array([[1.0, 7.0]]))
    assert np.all(it > 0)
    assert np.allclose(n[1] / n[0], np.exp(-1.5), rtol=1e-14)
    assert np.allclose(n.sum(0), P / (KB * T), rtol=1e-14)


@pytest.mark.parametrize("P", [1.0e6, 1.0e3, 2.5e8])
def test_dissociation_closed_form_and_le_chatelier(oracle, P):
    """A2 <=> 2 A: x_A^2 (P/P0) / x_A2 = exp(-(2 g_A - g_A2)) and x_A + x_A2 = 1 is a quadratic in x_A."""
    gA, gA2 = -2.0, -5.5
    net = simple([[1], [2]], [gA, gA2])
    T = np.array([1500.0])
    n, it = oracle.equilibrium(net, T, np.array([P]), np.array([[3.0]]))
    K, p = np.exp(-(2 * gA - gA2)), P / P0
    xA = (-K + np.sqrt(K * K + 4 * p * K)) / (2 * p)
    x = n[:, 0] / n[:, 0].sum()
    assert it[0] > 0 and abs(x[0] - xA) <= 1e-14 and abs(x[1] - (1 - xA)) <= 1e-14
    # higher pressure favours the side with fewer molecules
    n_hi, _ = oracle.equilibrium(net, T, np.array([10 * P]), np.array([[3.0]]))
    assert n_hi[0, 0] / n_hi[:, 0].sum() < x[0]


def test_ionisation_is_neutral_and_follows_the_saha_form(oracle):
    """A <=> A+ + e-, charge as a signed element with abundance 0: x_+ = x_e and x_+ x_e (P/P0) / x_A = K."""
    gA, gp, ge = -4.0, -1.0, -0.5
    net = simple([[1, 0], [1, 1], [0, -1]], [gA, gp, ge])
    P = 2.0e4
    n, it, pi = oracle.equilibrium(net, np.array([3000.0]), np.array([P]), np.array([[1.0], [0.0]]), want_pi=True)
    x = n[:, 0] / n[:, 0].sum()
    K, p = np.exp(-(gp + ge - gA)), P / P0
    assert it[0] > 0 and abs(x[1] - x[2]) <= 1e-15 * x[1]
    assert abs(x[1] * x[2] * p / x[0] - K) <= 1e-13 * K
    # the Lagrange condition of every species with the returned element potentials
    comp = net.composition.astype(float)
    assert np.allclose(np.array([gA, gp, ge]) + np.log(x) + np.log(p), comp @ pi[:, 0], atol=1e-13)


@pytest.mark.parametrize("cfg", [1, 2])
def test_lagrange_conditions_and_conservation_on_the_config_networks(oracle, network, cfg):
    """G_i/RT + ln x_i + ln(P/P0) must lie in the column space of the composition matrix (least squares over the
    element potentials, G_i/RT taken from orc_thermo), the element ratios must be those asked for, sum x = 1."""
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    nc = atm.ncol
    comp = net.composition.astype(float)
    b = comp.T @ atm.n
    n, it = oracle.equilibrium(net, atm.T, atm.P, b, nc)
    assert np.all(it[:nc] > 0)
    g = oracle.thermo(net, atm.T, nc)[3]
    ntot = atm.P[:nc] / (KB * atm.T[:nc])
    assert np.allclose(n[:, :nc].sum(0), ntot, rtol=1e-13)
    got = comp.T @ n[:, :nc]
    assert np.allclose(got / got.sum(0), b[:, :nc] / b[:, :nc].sum(0), rtol=1e-12, atol=0)
    for c in range(nc):
        ok = n[:, c] > 1e-250          # traces below the double range are returned as (sub)normal zeros
        x = n[ok, c] / ntot[c]
        assert ok.sum() > comp.shape[1] and np.all(n[:, c] >= 0)
        mu = g[ok, c] + np.log(x) + np.log(atm.P[c] / P0)
        pi, *_ = np.linalg.lstsq(comp[ok], mu, rcond=None)
        assert np.abs(comp[ok] @ pi - mu).max() <= 1e-10 * max(1.0, np.abs(mu).max())


@pytest.mark.parametrize("cfg", [1, 2])
def test_equilibrium_is_a_fixed_point_of_the_kinetics(oracle, network, cfg):
    """At the equilibrium composition every reversible reaction has q_f = q_r (K_c comes from the same G_i/RT), so
    without photolysis the source oracle must return dn/dt = 0 to round-off; a composition with the same elements
    that is NOT the equilibrium one must not (negative control)."""
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    nc = atm.ncol
    comp = net.composition.astype(float)
    n, it = oracle.equilibrium(net, atm.T, atm.P, comp.T @ atm.n, nc)
    kf, kr = oracle.rate_coeffs(net, atm.T, atm.P, np.zeros_like(atm.J), nc)
    d, p, l = oracle.source(net, kf, kr, n, nc)
    scale = (p + l)[:, :nc]
    big = scale > 1e-200       # terms of trace species below the double range have lost their bits
    assert big.sum() > 0.5 * big.size and scale.max() > 0
    assert np.all(np.abs(d[:, :nc])[big] <= 1e-12 * scale[big])
    d0, p0, l0 = oracle.source(net, kf, kr, atm.n, nc)
    assert np.abs(d0[:, :nc]).max() > 1e-3 * (p0 + l0)[:, :nc].max()


def gibbs(g, x_unnorm, p):
    """G/RT of a composition (any scale) at reduced pressure p."""
    n = x_unnorm
    return float(np.sum(n * (g + np.log(n / n.sum()) + np.log(p))))


def test_no_feasible_perturbation_lowers_the_gibbs_energy(oracle, network):
    """The defining property, brute force: moving along any direction that keeps the element totals (null space of
    the transposed composition matrix) raises G.  In double precision the rise is visible only when the species that
    move are abundant, so the directions exchange atoms among the species with x > 1e-4, taken as a mixture of their
    own at their partial pressure (the traces enter G only through terms far below the rise, and are covered by the
    Lagrange conditions above); the rise must also be of second order in the step."""
    from paper_2512_06729_b200 import synth
    rng = np.random.default_rng(5)
    tried = 0
    for cfg in (1, 2):
        net = network(cfg)
        atm = synth.config_atmosphere(cfg, net)
        comp = net.composition.astype(float)
        n, _ = oracle.equilibrium(net, atm.T, atm.P, comp.T @ atm.n, atm.ncol)
        g = oracle.thermo(net, atm.T, atm.ncol)[3]
        for c in range(0, atm.ncol, 3):
            x = n[:, c] / n[:, c].sum()
            major = np.flatnonzero(x > 1e-4)
            _, s, vt = np.linalg.svd(comp[major].T)
            null = vt[np.sum(s > 1e-10):]
            if null.shape[0] == 0:
                continue
            p = atm.P[c] / P0
            g0 = gibbs(g[major, c], x[major], p * x[major].sum())   # G of the abundant species as a mixture of their own
            for _ in range(10):
                v = null.T @ rng.standard_normal(null.shape[0])
                eps = 0.3 * np.min(x[major] / np.maximum(np.abs(v), 1e-300))
                rise = [gibbs(g[major, c], x[major] + sgn * f * eps * v, p * x[major].sum()) - g0
                        for f in (1.0, 0.5) for sgn in (1.0, -1.0)]
                assert min(rise) > 0
                assert 2.5 < (rise[0] + rise[1]) / (rise[2] + rise[3]) < 6.5    # about 4: second order
                tried += 1
    assert tried >= 100


def test_only_the_ratios_of_the_abundances_matter(oracle, network):
    from paper_2512_06729_b200 import synth
    net = network(1)
    atm = synth.config_atmosphere(1, net)
    b = net.composition.astype(float).T @ atm.n
    n1, _ = oracle.equilibrium(net, atm.T, atm.P, b, atm.ncol)
    n2, _ = oracle.equilibrium(net, atm.T, atm.P, 3.7e-9 * b, atm.ncol)
    assert np.allclose(n1[:, :atm.ncol], n2[:, :atm.ncol], rtol=1e-12, atol=0)


def test_an_element_without_abundance_is_refused(oracle):
    net = simple([[1, 0], [0, 1]], [-1.0, -1.0])
    with pytest.raises(ArithmeticError):
        oracle.equilibrium(net, np.array([1000.0]), np.array([1e6]), np.array([[1.0], [0.0]]))


def test_a_general_purpose_minimiser_finds_the_same_composition(oracle):
    """A different algorithm on the same definition: scipy's SLSQP minimises G/RT over the mole numbers under the
    linear element constraints (no Lagrange iteration, no logarithmic variables) for a 5-species, 2-element gas;
    it converges to about 1e-7, the oracle must agree with it to that accuracy."""
    from scipy.optimize import minimize
    comp = np.array([[1, 0], [0, 1], [2, 0], [1, 1], [2, 1]], dtype=float)     # A, B, A2, AB, A2B
    gs = np.array([-1.0, -2.0, -6.5, -7.0, -11.0])
    net = simple(comp.astype(int).tolist(), gs.tolist())
    T, P = np.array([1200.0]), np.array([3.0e5])
    b = np.array([[2.0], [1.0]])
    n, it = oracle.equilibrium(net, T, P, b)
    x = n[:, 0] / n[:, 0].sum()
    p = P[0] / P0

    def G(m):
        m = np.maximum(m, 1e-300)
        return float(np.sum(m * (gs + np.log(m / m.sum()) + np.log(p))))

    cons = {"type": "eq", "fun": lambda m: comp.T @ m - b[:, 0], "jac": lambda m: comp.T}
    best = None
    for seed in range(4):
        m0 = np.random.default_rng(seed).uniform(0.05, 0.5, 5)
        r = minimize(G, m0, method="SLSQP", constraints=[cons], bounds=[(1e-12, None)] * 5,
                     options={"ftol": 1e-15, "maxiter": 500})
        if r.success and (best is None or r.fun < best.fun):
            best = r
    assert best is not None
    xs = best.x / best.x.sum()
    assert np.allclose(xs, x, rtol=0, atol=2e-6), (xs, x)
    # and the oracle's point is at least as low as the minimiser's, on the minimiser's own scale
    m_or = x * (b[0, 0] / (comp[:, 0] @ x))
    assert np.allclose(comp.T @ m_or, b[:, 0], rtol=1e-13)
    assert G(m_or) <= best.fun + 1e-9 * abs(best.fun)
