"""Pins of the oracle's NASA-7 thermochemistry (oracle O1).

Nothing here retypes the oracle's formulas: the pins are textbook thermochemistry of the
molecules whose coefficients the paper prints (Table 1), calculus identities that tie cp, H, S
and G together, and the range-selection rule.
"""
import numpy as np
import pytest

from conftest import SimpleNet, load_table1

R_GAS = 8.314462618  # J/mol/K, exact SI 2019


def thermo_net(rows_lo, rows_hi, t_mid):
    ns = len(t_mid)
    return SimpleNet(np.zeros((ns, 1)), rows_lo, rows_hi, t_mid, [], [], [], [], np.zeros((0, 3)))


def test_table1_water_and_co2_match_textbook_thermochemistry(oracle):
    """Burcat rows of Table 1 must reproduce the standard-state values every
    thermochemistry table gives at 298.15 K: H2O(g) dfH = -241.83 kJ/mol, S = 188.84 J/mol/K,
    cp = 33.59 J/mol/K; CO2 dfH = -393.51 kJ/mol, S = 213.79 J/mol/K, cp = 37.13 J/mol/K
    (NIST-JANAF / CODATA key values; the paper cites NIST-JANAF and Burcat).
    A wrong divisor, sign or index in H/RT, S/R or cp/R moves these by far more than the bound
    (e.g. a6/T dropped: 250 kJ/mol; a2 T/2 -> a2 T: 0.75 kJ/mol; a7 dropped: 7 J/mol/K)."""
    t = load_table1()
    net = thermo_net([t["H2O_burcat_lo"], t["CO2_burcat_lo"]], [t["H2O_burcat_hi"], t["CO2_burcat_hi"]],
                     [1000.0, 1000.0])
    T = np.array([298.15])
    cp, h, s, g = oracle.thermo(net, T)
    H = h[:, 0] * R_GAS * T[0] / 1e3
    S = s[:, 0] * R_GAS
    CP = cp[:, 0] * R_GAS
    assert H[0] == pytest.approx(-241.826, abs=0.05)
    assert S[0] == pytest.approx(188.835, abs=0.03)
    assert CP[0] == pytest.approx(33.59, abs=0.03)
    assert H[1] == pytest.approx(-393.51, abs=0.05)
    assert S[1] == pytest.approx(213.79, abs=0.03)
    assert CP[1] == pytest.approx(37.13, abs=0.03)
    # G = H - T S in absolute units as well (kJ/mol): -241.83 - 298.15*0.188835 = -298.13
    G = g[:, 0] * R_GAS * T[0] / 1e3
    assert G[0] == pytest.approx(-241.826 - 298.15 * 0.188835, abs=0.06)
    assert G[1] == pytest.approx(-393.51 - 298.15 * 0.21379, abs=0.06)


def test_table1_monatomic_gas_has_cp_five_halves(oracle):
    """P(2D) rows: a monatomic ideal gas has cp/R = 5/2 at every T."""
    t = load_table1()
    net = thermo_net([t["P2D_lo"]], [t["P2D_hi"]], [1000.0])
    T = np.array([10.0, 200.0, 999.0, 1001.0, 3000.0])
    cp, h, s, g = oracle.thermo(net, T)
    assert np.allclose(cp[0], 2.5, rtol=0, atol=1e-9)
    # H(T2) - H(T1) = 5/2 R (T2 - T1):  T*H/RT differences
    th = h[0] * T
    assert np.allclose(np.diff(th), 2.5 * np.diff(T), rtol=1e-7)  # printed a2..a5 are ~1e-13, not 0
    # Sackur-Tetrode: S(T2) - S(T1) = 5/2 R ln(T2/T1)
    assert np.allclose(np.diff(s[0]), 2.5 * np.diff(np.log(T)), rtol=1e-7)


def test_table1_burcat_sets_join_at_1000K(oracle):
    """The Burcat low and high sets are fitted to be continuous at their common 1000 K junction:
    pins range selection plus every term of cp/R and G/RT at once."""
    t = load_table1()
    for mol in ("H2O_burcat", "CO2_burcat"):
        net = thermo_net([t[mol + "_lo"]], [t[mol + "_hi"]], [1000.0])
        T = np.array([1000.0, np.nextafter(1000.0, 2000.0)])
        cp, h, s, g = oracle.thermo(net, T)
        assert cp[0, 0] != cp[0, 1]                       # the two sets really are different
        assert cp[0, 0] == pytest.approx(cp[0, 1], rel=5e-5)
        assert h[0, 0] == pytest.approx(h[0, 1], rel=5e-5)
        assert s[0, 0] == pytest.approx(s[0, 1], rel=5e-5)
        assert g[0, 0] == pytest.approx(g[0, 1], rel=5e-6)


def test_range_selection_rule(oracle):
    """T <= t_mid -> low set, T > t_mid -> high set, per species (reading T3)."""
    lo = np.zeros((2, 7))
    hi = np.zeros((2, 7))
    lo[:, 0], hi[:, 0] = 1.0, 2.0
    net = thermo_net(lo, hi, [300.0, 1000.0])
    T = np.array([np.nextafter(300.0, 0), 300.0, np.nextafter(300.0, 1e9), 999.0, 1000.0, 1000.5])
    cp, _, _, _ = oracle.thermo(net, T)
    assert cp[0].tolist() == [1, 1, 2, 2, 2, 2]
    assert cp[1].tolist() == [1, 1, 1, 1, 1, 2]


def _random_sets(rng, ns):
    a = np.zeros((ns, 7))
    a[:, 0] = rng.uniform(2.5, 5, ns)
    a[:, 1] = rng.uniform(-1, 1, ns) * 1e-3
    a[:, 2] = rng.uniform(-1, 1, ns) * 1e-6
    a[:, 3] = rng.uniform(-1, 1, ns) * 1e-9
    a[:, 4] = rng.uniform(-1, 1, ns) * 1e-12
    a[:, 5] = rng.uniform(-1e5, 1e5, ns)
    a[:, 6] = rng.uniform(-10, 30, ns)
    return a


def test_gibbs_is_enthalpy_minus_entropy(oracle):
    """G/RT (printed form) = H/RT - S/R (standard forms), evaluated independently."""
    rng = np.random.default_rng(7)
    ns = 40
    lo, hi = _random_sets(rng, ns), _random_sets(rng, ns)
    net = thermo_net(lo, hi, np.full(ns, 1000.0))
    T = np.array([150.0, 300.0, 800.0, 1000.0, 1500.0, 3000.0])
    cp, h, s, g = oracle.thermo(net, T)
    scale = np.abs(h) + np.abs(s)
    assert np.all(np.abs(g - (h - s)) <= 4e-16 * scale)


def test_calculus_identities(oracle):
    """d(T H/RT)/dT = cp/R,  T d(S/R)/dT = cp/R,  d(G/RT)/dT = -(H/RT)/T  (Gibbs-Helmholtz).
    Central differences; the truncation error h^2 f'''/6 is ~1e-7 of cp for these coefficients.
    Each identity fails at O(1e-2..1) if any divisor (2,3,4,5 / 2,3,4 / 2,6,12,20) is wrong."""
    rng = np.random.default_rng(11)
    ns = 30
    lo = _random_sets(rng, ns)
    t = load_table1()
    lo[0], lo[1] = t["H2O_burcat_lo"], t["P2O2_hi"]
    net = thermo_net(lo, lo, np.full(ns, 1e9))
    for T0 in (400.0, 1200.0, 2500.0):
        dT = 0.5
        T = np.array([T0 - dT, T0, T0 + dT])
        cp, h, s, g = oracle.thermo(net, T)
        d_th = (h[:, 2] * T[2] - h[:, 0] * T[0]) / (2 * dT)
        d_s = T0 * (s[:, 2] - s[:, 0]) / (2 * dT)
        d_g = (g[:, 2] - g[:, 0]) / (2 * dT)
        assert np.allclose(d_th, cp[:, 1], rtol=2e-6, atol=2e-6)
        assert np.allclose(d_s, cp[:, 1], rtol=2e-6, atol=2e-6)
        assert np.allclose(d_g, -h[:, 1] / T0, rtol=2e-6, atol=1e-9)


def test_generated_heat_capacities_respect_config_bounds(oracle, network):
    """BASELINE.json config 1: cp/R stays within 2.5..15 over 200-3000 K (checked through the
    oracle's own range selection, so a swapped lo/hi set shows up here)."""
    net = network(2)
    T = np.arange(200.0, 3001.0, 25.0)
    cp, h, s, g = oracle.thermo(net, T)
    assert cp.min() >= 2.5 - 1e-9 and cp.max() <= 15 + 1e-9
    # H and S are continuous across each species' t_mid (generator solves a6', a7' for that)
    for tm in (300.0, 500.0, 700.0, 1000.0):
        T2 = np.array([tm, np.nextafter(tm, 1e9)])
        cp2, h2, s2, g2 = oracle.thermo(net, T2)
        assert np.allclose(h2[:, 0], h2[:, 1], rtol=1e-11, atol=1e-11)
        assert np.allclose(s2[:, 0], s2[:, 1], rtol=1e-11, atol=1e-11)


def test_double_build_agrees_with_extended_build(oracle, oracle_f64, network):
    assert oracle.mant_dig == 64 and oracle_f64.mant_dig == 53
    net = network(2)
    T = np.linspace(150.0, 3100.0, 64)
    a = oracle.thermo(net, T)
    b = oracle_f64.thermo(net, T)
    for x, y in zip(a[:3], b[:3]):
        assert np.allclose(x, y, rtol=1e-13, atol=0)
    scale = np.abs(a[1]) + np.abs(a[2])
    assert np.all(np.abs(a[3] - b[3]) <= 1e-15 * scale)
