"""Pins of the oracle's forward and reverse rate coefficients (oracle O2, O3;
PAPER.md:116-159, 219-235).  Special cases, limits, symmetries and K_c recomputed by other code."""
import numpy as np
import pytest

from conftest import SimpleNet, load_table1

UNI, BI, FALLOFF, PHOTO = 0, 1, 2, 3
K_B = 1.380649e-16
P0 = 1.0e6


def zeros_thermo(ns):
    return np.zeros((ns, 7)), np.zeros((ns, 7)), np.full(ns, 1000.0)


def one_reaction(rtype, lhs, rhs, arrh, arrh_low=None, fc=None, t_ref=None, ns=4, reversible=0,
                 thermo=None):
    lo, hi, tm = thermo if thermo is not None else zeros_thermo(ns)
    return SimpleNet(np.zeros((ns, 1)), lo, hi, tm, [rtype], [lhs], [rhs], [reversible], [arrh],
                     None if arrh_low is None else [arrh_low], None if fc is None else [fc],
                     None if t_ref is None else [t_ref])


def test_arrhenius_special_cases(oracle):
    """north_star: n = 0, E = 0 gives k = A.  Also E = 0, T = T_ref gives k = A."""
    T = np.array([150.0, 800.0, 2500.0])
    P = np.full(3, 1e6)
    net = one_reaction(BI, [0, 1], [2, 3], [3.7e-11, 0.0, 0.0])
    kf, kr = oracle.rate_coeffs(net, T, P, None)
    assert kf[0].tolist() == [3.7e-11] * 3 and kr[0].tolist() == [0.0] * 3
    net = one_reaction(BI, [0, 1], [2, 3], [3.7e-11, 1.7, 0.0], t_ref=300.0)
    kf, _ = oracle.rate_coeffs(net, np.array([300.0]), P[:1], None)
    assert kf[0, 0] == 3.7e-11
    net = one_reaction(UNI, [0], [1, 2], [1e13, -2.0, 0.0], t_ref=1.0)
    kf, _ = oracle.rate_coeffs(net, np.array([1.0]), P[:1], None)
    assert kf[0, 0] == 1e13


def test_arrhenius_against_library_evaluation_and_kooij_equivalence(oracle):
    """Eq. 7 on a grid against numpy's pow/exp; Kooij alpha (T/300)^beta == (alpha 300^-beta) T^beta."""
    rng = np.random.default_rng(3)
    T = np.linspace(150.0, 3000.0, 57)
    P = np.full(T.shape, 1e5)
    for _ in range(20):
        A, n, E = 10 ** rng.uniform(-20, -9), rng.uniform(-3, 3), rng.uniform(0, 40000)
        net = one_reaction(BI, [0, 1], [2, 3], [A, n, E])
        kf, _ = oracle.rate_coeffs(net, T, P, None)
        ref = A * np.power(T, n) * np.exp(-E / T)
        assert np.allclose(kf[0], ref, rtol=2e-13, atol=0)
        kooij = one_reaction(BI, [0, 1], [2, 3], [A, n, E], t_ref=300.0)
        resc = one_reaction(BI, [0, 1], [2, 3], [A * 300.0 ** (-n), n, E], t_ref=1.0)
        k1, _ = oracle.rate_coeffs(kooij, T, P, None)
        k2, _ = oracle.rate_coeffs(resc, T, P, None)
        assert np.allclose(k1[0], k2[0], rtol=1e-14, atol=0)
        # monotone in T for n >= 0, E >= 0
        if n >= 0:
            assert np.all(np.diff(kf[0]) > 0)


def _falloff_net(A0, Ainf, fc, n0=0.0, E0=0.0, ninf=0.0, Einf=0.0):
    return one_reaction(FALLOFF, [0, 1], [2], [Ainf, ninf, Einf], [A0, n0, E0], fc)


def test_lindemann_form_and_limits(oracle):
    """Fc = 1 is Eq. 12 exactly; k -> k0[M] at low pressure and k -> k_inf at high pressure
    (north_star).  With Fc = 1 the approach is algebraic, 1/(1 + Pr), so the limits are tight."""
    A0, Ainf = 2e-30, 5e-11
    T = np.full(7, 1000.0)
    M = np.array([1e-2, 1e3, 1e10, Ainf / A0, 1e25, 1e31, 1e36])
    P = M * K_B * T
    net = _falloff_net(A0, Ainf, 1.0)
    kf, _ = oracle.rate_coeffs(net, T, P, None)
    Pr = A0 * M / Ainf
    assert np.allclose(kf[0], A0 * M / (1 + Pr), rtol=1e-14)
    assert kf[0, 0] / (A0 * M[0]) == pytest.approx(1.0, abs=1e-14)      # Pr ~ 4e-22
    assert kf[0, 3] == pytest.approx(0.5 * Ainf, rel=1e-14)             # Pr = 1
    assert kf[0, 6] / Ainf == pytest.approx(1.0, abs=1e-14)             # Pr ~ 4e16
    assert np.all(kf[0] <= np.minimum(A0 * M, Ainf) * (1 + 1e-15))


def test_troe_broadening_properties(oracle):
    """Reading F1: F(Pr = 1) = Fc, F(Pr) = F(1/Pr), Fc <= F <= 1, F -> 1 in both limits, and
    k (1 + Pr) / (k0 [M]) = F."""
    A0, Ainf = 2e-30, 5e-11
    for fc in (0.3, 0.55, 0.9):
        lp = np.array([-30.0, -8.0, -2.0, -0.5, 0.0, 0.5, 2.0, 8.0, 30.0])
        Pr = 10.0 ** lp
        M = Pr * Ainf / A0
        T = np.full(lp.shape, 700.0)
        P = M * K_B * T
        kf, _ = oracle.rate_coeffs(_falloff_net(A0, Ainf, fc), T, P, None)
        F = kf[0] * (1 + Pr) / (A0 * M)
        assert F[4] == pytest.approx(fc, rel=1e-13)
        assert np.allclose(F, F[::-1], rtol=1e-12)
        assert np.all(F >= fc * (1 - 1e-13)) and np.all(F <= 1 + 1e-13)
        assert np.all(np.diff(F[:5]) < 0) and np.all(np.diff(F[4:]) > 0)
        assert F[0] > 0.995 and F[-1] > 0.995
        assert np.all(kf[0] <= np.minimum(A0 * M, Ainf) * (1 + 1e-13))
    # the limit F -> 1 is only algebraic in log Pr (SURVEY: F(1e-30; 0.3) = 0.99734)
    kf, _ = oracle.rate_coeffs(_falloff_net(A0, Ainf, 0.3), np.array([700.0]),
                               np.array([1e-30 * Ainf / A0 * K_B * 700.0]), None)
    assert kf[0, 0] / (A0 * 1e-30 * Ainf / A0) == pytest.approx(0.99734, abs=2e-5)


def test_falloff_uses_both_temperature_dependences(oracle):
    """k0 and k_inf each carry their own (alpha, beta, gamma), Eq. 10-11; swapping them changes k."""
    T = np.array([900.0])
    M = 1e19
    P = M * K_B * T
    a = one_reaction(FALLOFF, [0, 1], [2], [5e-11, 0.5, 300.0], [2e-30, -2.5, 1200.0], 1.0)
    kf, _ = oracle.rate_coeffs(a, T, P, None)
    k0 = 2e-30 * 900.0 ** -2.5 * np.exp(-1200.0 / 900.0)
    kinf = 5e-11 * 900.0 ** 0.5 * np.exp(-300.0 / 900.0)
    assert kf[0, 0] == pytest.approx(k0 * M / (1 + k0 * M / kinf), rel=1e-13)


def test_photolysis_rows_follow_user_order_and_are_irreversible(oracle):
    """k_f of the p-th PHOTO reaction (user order) is row p of J; k_r = 0 (reading R2)."""
    lo, hi, tm = zeros_thermo(4)
    net = SimpleNet(np.zeros((4, 1)), lo, hi, tm, [PHOTO, BI, PHOTO, UNI, PHOTO],
                    [[0], [0, 1], [1], [2], [3]], [[1, 2], [2, 3], [0, 3], [0, 1], [0, 0]],
                    [0, 1, 0, 1, 0], [[0, 0, 0], [1e-10, 0, 0], [0, 0, 0], [1e3, 0, 0], [0, 0, 0]])
    T = np.array([1000.0, 1500.0])
    P = np.array([1e6, 1e3])
    J = np.array([[1e-3, 2e-3], [3e-5, 4e-5], [5e-7, 6e-7]])
    kf, kr = oracle.rate_coeffs(net, T, P, J)
    assert np.array_equal(kf[0], J[0]) and np.array_equal(kf[2], J[1]) and np.array_equal(kf[4], J[2])
    assert not kr[[0, 2, 4]].any()
    assert kr[1].all() and kr[3].all()


def test_equilibrium_constant_unit_check(oracle):
    """All G = 0, A + B <=> C at 1000 K: K_c = (P0/k_B T)^-1 = k_B T / P0 = 1.380649e-19 cm^3
    (P0/k_B T = 7.242971e18 cm^-3).  A <=> B + C gives the inverse; A + B <=> C + D gives 1."""
    T = np.array([1000.0])
    P = np.array([1e6])
    kf, kr = oracle.rate_coeffs(one_reaction(BI, [0, 1], [2], [1e-10, 0, 0], reversible=1), T, P, None)
    assert kf[0, 0] / kr[0, 0] == pytest.approx(1.380649e-19, rel=1e-14)
    kf, kr = oracle.rate_coeffs(one_reaction(UNI, [0], [1, 2], [1e5, 0, 0], reversible=1), T, P, None)
    assert kf[0, 0] / kr[0, 0] == pytest.approx(7.242970516e18, rel=1e-9)
    kf, kr = oracle.rate_coeffs(one_reaction(BI, [0, 1], [2, 3], [1e-10, 0, 0], reversible=1), T, P, None)
    assert kf[0, 0] == kr[0, 0]
    # three products (Eq. 13): A + B <=> X + Y + Z has dnu = +1
    kf, kr = oracle.rate_coeffs(one_reaction(BI, [0, 1], [2, 3, 3], [1e-10, 0, 0], reversible=1), T, P, None)
    assert kf[0, 0] / kr[0, 0] == pytest.approx(7.242970516e18, rel=1e-9)
    # irreversible thermal reaction
    kf, kr = oracle.rate_coeffs(one_reaction(BI, [0, 1], [2, 3], [1e-10, 0, 0], reversible=0), T, P, None)
    assert kr[0, 0] == 0.0


def test_detailed_balance_against_thermo_outputs(oracle, network):
    """north_star: k_f / k_r equals K_c computed independently from the thermo.  K_c is rebuilt
    here with numpy from orc_thermo's G/RT output: K_c = exp(-dG/RT) (P0/k_B T)^dnu."""
    from paper_2512_06729_b200 import synth
    net = network(2)
    atm = synth.config_atmosphere(2, net)
    kf, kr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    _, _, _, g = oracle.thermo(net, atm.T, atm.ncol)
    T = atm.T[:atm.ncol]
    checked = 0
    for r in range(net.n_reactions):
        if net.type[r] == PHOTO:
            assert not kr[r].any()
            continue
        lhs = [s for s in net.reactants[r] if s >= 0]
        rhs = [s for s in net.products[r] if s >= 0]
        dG = g[rhs, :atm.ncol].sum(axis=0) - g[lhs, :atm.ncol].sum(axis=0)
        dnu = len(rhs) - len(lhs)
        with np.errstate(over="ignore"):
            Kc = np.exp(-dG) * (P0 / (K_B * T)) ** dnu
        ratio = kf[r, :atm.ncol] / kr[r, :atm.ncol]
        ok = np.isfinite(Kc) & (Kc > 1e-290) & np.isfinite(ratio)
        # exp() of a double-rounded dG: relative error ~ |dG| * 2^-53 per rounded term
        tol = 1e-15 * (np.abs(g[rhs, :atm.ncol]).sum(axis=0) + np.abs(g[lhs, :atm.ncol]).sum(axis=0)) + 1e-14
        assert np.all(np.abs(ratio[ok] / Kc[ok] - 1) <= tol[ok])
        checked += int(ok.sum())
    assert checked > 0.9 * (net.n_reactions - net.n_photo) * atm.ncol


def test_equilibrium_constant_symmetries(oracle):
    """Isomers with identical coefficients -> K_c = 1; a thermodynamic cycle A->B->C->A has
    prod K_c = 1; swapping the listed direction inverts K_c."""
    t = load_table1()
    lo = np.array([t["H2O_burcat_lo"], t["H2O_burcat_lo"], t["CO2_burcat_lo"], t["P2O_lo"]])
    hi = np.array([t["H2O_burcat_hi"], t["H2O_burcat_hi"], t["CO2_burcat_hi"], t["P2O_hi"]])
    tm = np.array([1000.0, 1000.0, 1000.0, 350.0])
    net = SimpleNet(np.zeros((4, 1)), lo, hi, tm, [UNI] * 5,
                    [[0], [1], [2], [3], [2]], [[1], [2], [3], [1], [1]], [1] * 5,
                    [[1e3, 0.5, 100.0]] * 5)
    T = np.array([200.0, 400.0, 900.0, 1000.0, 1700.0, 2900.0])
    kf, kr = oracle.rate_coeffs(net, T, np.full(T.shape, 1e4), None)
    K = kf / kr
    assert np.array_equal(kf[0], kr[0])                                  # isomerisation, same G
    assert np.allclose(K[1] * K[2] * K[3], 1.0, rtol=1e-12)              # cycle 1 -> 2 -> 3 -> 1
    assert np.allclose(K[1] * K[4], 1.0, rtol=1e-12)                     # 1 -> 2 and 2 -> 1


def test_reverse_coefficient_saturates_like_ieee(oracle, oracle_f64):
    """Reading R5: K_c outside the double range must not overflow before k_r is rounded."""
    lo = np.zeros((2, 7))
    lo[1, 5] = 1.2e5                      # G_B/RT - G_A/RT = 1.2e5/T  -> K_c = exp(-800) at 150 K
    net = SimpleNet(np.zeros((2, 1)), lo, lo, [1000.0, 1000.0], [UNI], [[0]], [[1]], [1], [[1e-40, 0, 0]])
    T = np.array([150.0, 100.0])
    kf, kr = oracle.rate_coeffs(net, T, np.full(2, 1e6), None)
    # k_r = 1e-40 * exp(800) = 2.7e307 (finite) and 1e-40 * exp(1200) = inf
    assert kr[0, 0] == pytest.approx(float(np.longdouble(1e-40) * np.exp(np.longdouble(800.0))), rel=1e-13)
    assert 2.72e307 < kr[0, 0] < 2.73e307       # e^800 = 2.7264e347
    assert np.isinf(kr[0, 1])


def test_table1_phosphorus_network_equilibrium_constant(oracle):
    """The only element-balanced reaction among the paper's Table 1 species, 2 P2O <=> P2O2 + 2 P(2D)
    (SURVEY section 4), with the PRINTED coefficients: K_c from the oracle's
    k_f/k_r against G/RT evaluated here from the printed line-671 formula with exact fractions.
    dnu = 3 - 2 = +1, so K_c = exp(-dG/RT) * P0/(k_B T) [cm^-3]."""
    from fractions import Fraction
    rows = load_table1()
    names = ["P2O", "P2O2", "P2D"]
    lo = np.array([rows[n + "_lo"] for n in names])
    hi = np.array([rows[n + "_hi"] for n in names])
    t_mid = np.array([350.0, 300.0, 1000.0])       # junctions found in Table 1 (reading T3)
    net = SimpleNet([[2, 1], [2, 2], [1, 0]], lo, hi, t_mid, [BI], [[0, 0]], [[1, 2, 2]], [1],
                    [[1e-11, 0.5, 1000.0]], element_names=["P", "O"])
    T = np.array([280.0, 400.0, 900.0, 1500.0, 2500.0])
    kf, kr = oracle.rate_coeffs(net, T, np.full(T.size, 1e6), None)

    def g_rt(a, t):                                  # PAPER.md:671, exact rational arithmetic except ln T
        a = [Fraction(float(x)) for x in a]
        t = Fraction(float(t))
        poly = -a[1] * t / 2 - a[2] * t ** 2 / 6 - a[3] * t ** 3 / 12 - a[4] * t ** 4 / 20 + a[5] / t - a[6]
        return float(poly) + float(a[0]) * (1.0 - np.log(float(t)))

    for c, t in enumerate(T):
        sets = [lo[i] if t <= t_mid[i] else hi[i] for i in range(3)]
        dg = g_rt(sets[1], t) + 2 * g_rt(sets[2], t) - 2 * g_rt(sets[0], t)
        kc = np.exp(-dg) * P0 / (K_B * t)
        assert kf[0, c] / kr[0, c] == pytest.approx(kc, rel=5e-12)
        assert kf[0, c] == pytest.approx(1e-11 * t ** 0.5 * np.exp(-1000.0 / t), rel=1e-14)
