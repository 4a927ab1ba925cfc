"""Pins of the oracle's rates of progress, production/loss, Jacobian and CSR layouts
(oracle O4-O6; BASELINE.json north_star): hand-expanded rate laws, element
conservation, the equilibrium fixed point, homogeneity, Euler's identity, finite differences
and brute-force CSR construction."""
import numpy as np
import pytest

from conftest import SimpleNet

UNI, BI, FALLOFF, PHOTO = 0, 1, 2, 3
K_B = 1.380649e-16
P0 = 1.0e6


def hand_network():
    """3 species X0, X1, X2.
       R0: 2 X0 <=> X1 + 2 X2   (repeated reactant, three products with a repeat; cf. the Table-1-only
                                 network 2 P2O <=> P2O2 + 2 P(2D))
       R1: X1 -> X0 + X2        (photolysis)
       R2: X0 + X2 <=> X1       (falloff-type recombination)
       R3: X2 + X0 <=> X1 + X0  (X0 on both sides, nu = 0; needs no balance for the oracle)"""
    z = np.zeros((3, 7))
    return SimpleNet(np.zeros((3, 1)), z, z, [1000.0] * 3, [BI, PHOTO, FALLOFF, BI],
                     [[0, 0], [1], [0, 2], [2, 0]], [[1, 2, 2], [0, 2], [1], [1, 0]], [1, 0, 1, 1],
                     np.zeros((4, 3)))


def test_hand_expanded_rate_laws_on_three_species(oracle):
    """north_star: brute-force hand-expanded rate laws on a 3-species network."""
    net = hand_network()
    rng = np.random.default_rng(5)
    ncol = 9
    n = 10 ** rng.uniform(-3, 12, size=(3, ncol))
    n[1, 4] = 0.0                                     # a zero density must give exact zeros
    kf = 10 ** rng.uniform(-14, -2, size=(4, ncol))
    kr = 10 ** rng.uniform(-14, -2, size=(4, ncol))
    kr[1] = 0.0
    n0, n1, n2 = n
    a = kf[0] * n0 * n0 - kr[0] * n1 * n2 * n2        # R0 net
    b = kf[1] * n1                                    # R1
    c = kf[2] * n0 * n2 - kr[2] * n1                  # R2 net
    d = kf[3] * n2 * n0 - kr[3] * n1 * n0             # R3 net
    want = np.array([-2 * a + b - c, a - b + c + d, 2 * a + b - c - d])
    gross = np.array([
        2 * kf[0] * n0 * n0 + 2 * kr[0] * n1 * n2 * n2 + b + kf[2] * n0 * n2 + kr[2] * n1,
        kf[0] * n0 * n0 + kr[0] * n1 * n2 * n2 + b + kf[2] * n0 * n2 + kr[2] * n1
        + kf[3] * n2 * n0 + kr[3] * n1 * n0,
        2 * kf[0] * n0 * n0 + 2 * kr[0] * n1 * n2 * n2 + b + kf[2] * n0 * n2 + kr[2] * n1
        + kf[3] * n2 * n0 + kr[3] * n1 * n0])
    dndt, prod, loss = oracle.source(net, kf, kr, n)
    assert np.all(np.abs(dndt - want) <= 4e-16 * gross)
    assert np.all(np.abs(prod + loss - gross) <= 4e-16 * gross)
    assert np.all(np.abs((prod - loss) - dndt) <= 4e-16 * gross)
    assert np.all(prod >= 0) and np.all(loss >= 0)
    # production of X0: reverse of R0 (x2), R1; of X1: R0 fwd, R2 fwd, R3 fwd; ...
    p0 = 2 * kr[0] * n1 * n2 * n2 + b + kr[2] * n1
    assert np.all(np.abs(prod[0] - p0) <= 4e-16 * gross[0])
    # rates of progress
    qf, qr = oracle.rates(net, kf, kr, n)
    assert np.allclose(qf[0], kf[0] * n0 * n0, rtol=4e-16) and np.allclose(qr[0], kr[0] * n1 * n2 * n2, rtol=4e-16)
    assert np.array_equal(qr[1], np.zeros(ncol))
    # Jacobian, hand-differentiated
    J = np.zeros((3, 3, ncol))
    da = [2 * kf[0] * n0, -kr[0] * n2 * n2, -2 * kr[0] * n1 * n2]
    db = [0 * n0, kf[1], 0 * n0]
    dc = [kf[2] * n2, -kr[2], kf[2] * n0]
    dd = [kf[3] * n2 - kr[3] * n1, -kr[3] * n0, kf[3] * n0]
    for j in range(3):
        J[0, j] = -2 * da[j] + db[j] - dc[j]
        J[1, j] = da[j] - db[j] + dc[j] + dd[j]
        J[2, j] = 2 * da[j] + db[j] - dc[j] - dd[j]
    for c_ in range(ncol):
        dense, scale = oracle.jacobian_dense(net, kf, kr, n, c_)
        assert np.all(np.abs(dense - J[:, :, c_]) <= 1e-15 * scale + 1e-300)
    # the zero density column: d/dn1 terms stay finite and exact (never q / n_j)
    dense, _ = oracle.jacobian_dense(net, kf, kr, n, 4)
    assert np.isfinite(dense).all() and dense[0, 1] == pytest.approx(
        2 * kr[0, 4] * n2[4] ** 2 + kf[1, 4] + kr[2, 4], rel=1e-15)


def _element_residual(net, x, scale):
    a = net.composition.astype(np.float64)            # [ns][ne]
    res = a.T @ x                                     # [ne][...]
    ref = np.abs(a).T @ scale
    return res, ref


@pytest.mark.parametrize("cfg", [1, 2])
def test_element_conservation(oracle, network, cfg):
    """north_star: for every element, sum_species atoms x dn/dt = 0 to round-off (relative to
    sum |atoms| (P + L)); paper: "ensuring mass conservation"."""
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    dndt, prod, loss = oracle.source_from_state(net, atm.T, atm.P, atm.J, atm.n, atm.ncol)
    assert np.isfinite(dndt).all()
    res, ref = _element_residual(net, dndt, prod + loss)
    assert np.all(np.abs(res) <= 1e-15 * ref)
    assert np.any(np.abs(dndt) > 1e-3 * (prod + loss))  # not trivially zero


@pytest.mark.parametrize("cfg", [1, 2])
def test_equilibrium_composition_is_a_fixed_point(oracle, network, cfg):
    """n_i = (P0/k_B T) exp(-G_i/RT) prod_e lambda_e^(a_ie) makes q_f = q_r for every reversible
    reaction, so dn/dt = 0 when J = 0 (paper: "nearly equal forward and reverse reaction rates"
    at thermochemical equilibrium).  Pins the sign of dnu, P0 and the K_c
    convention in one shot: any of them wrong leaves O(1) relative residuals."""
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    ncol = atm.ncol
    T, P = atm.T[:ncol], atm.P[:ncol]
    _, _, _, g = oracle.thermo(net, T)
    rng = np.random.default_rng(17)
    loglam = rng.uniform(-3, 3, size=net.n_elements)
    ln_n = np.log(P0 / (K_B * T))[None, :] - g + (net.composition @ loglam)[:, None]
    n = np.exp(ln_n)
    assert np.isfinite(n).all() and (n > 0).all()
    J = np.zeros_like(atm.J[:, :ncol])
    dndt, prod, loss = oracle.source_from_state(net, T, P, J, n)
    scale = prod + loss
    live = scale > 0
    assert live.sum() >= net.n_species * ncol * 0.9
    # exp() of doubles |G| ~ 1e2 carries ~1e-14 relative error into each n_i
    assert np.all(np.abs(dndt[live]) <= 2e-12 * scale[live])
    # negative control: doubling one species' density breaks the balance at O(1)
    n2 = n.copy()
    n2[net.n_species // 2] *= 2.0
    d2, p2, l2 = oracle.source_from_state(net, T, P, J, n2)
    assert np.any(np.abs(d2) > 1e-3 * (p2 + l2))


def test_rates_are_homogeneous_in_density(oracle, network):
    """Scaling every n by s scales q_f by s^(#reactants) and q_r by s^(#products)."""
    from paper_2512_06729_b200 import synth
    net = network(1)
    atm = synth.config_atmosphere(1, net)
    kf, kr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    qf, qr = oracle.rates(net, kf, kr, atm.n)
    s = 4.0                                            # power of two: exact scaling
    qf2, qr2 = oracle.rates(net, kf, kr, s * atm.n)
    of = (net.reactants >= 0).sum(axis=1)
    orv = (net.products >= 0).sum(axis=1)
    assert np.array_equal(qf2, qf * (s ** of)[:, None])
    assert np.array_equal(qr2, qr * (s ** orv)[:, None])


@pytest.mark.parametrize("cfg", [1, 2])
def test_jacobian_invariants(oracle, network, cfg):
    """Element conservation of every Jacobian column, and Euler's identity for homogeneous
    polynomials: sum_j Jac_ij n_j = sum_r nu_ir (order_f q_f - order_r q_r)."""
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    ncol = min(atm.ncol, 8)
    kf, kr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    row_ptr, col = oracle.jac_pattern(net)
    jac, sc = oracle.jacobian(net, kf, kr, atm.n, row_ptr, col, ncol)
    qf, qr = oracle.rates(net, kf, kr, atm.n)
    ns = net.n_species
    a = net.composition.astype(np.float64)
    of = (net.reactants >= 0).sum(axis=1)
    orv = (net.products >= 0).sum(axis=1)
    nu = np.zeros((ns, net.n_reactions))
    for r in range(net.n_reactions):
        for s_ in net.products[r]:
            if s_ >= 0:
                nu[s_, r] += 1
        for s_ in net.reactants[r]:
            if s_ >= 0:
                nu[s_, r] -= 1
    for c in range(ncol):
        dense = np.zeros((ns, ns))
        scale = np.zeros((ns, ns))
        for i in range(ns):
            sl = slice(row_ptr[i], row_ptr[i + 1])
            dense[i, col[sl]] = jac[sl, c]
            scale[i, col[sl]] = sc[sl, c]
        d2, s2 = oracle.jacobian_dense(net, kf, kr, atm.n, c)
        assert np.array_equal(dense, d2) and np.array_equal(scale, s2)
        res = a.T @ dense                              # [ne][ns]
        ref = np.abs(a).T @ scale
        assert np.all(np.abs(res) <= 1e-15 * ref)
        euler_l = dense @ atm.n[:, c]
        euler_r = nu @ (of * qf[:, c] - orv * qr[:, c])
        ref = scale @ np.abs(atm.n[:, c])
        assert np.all(np.abs(euler_l - euler_r) <= 1e-14 * ref + 1e-300)


def test_jacobian_against_finite_differences(oracle, network):
    """dn/dt is a polynomial of degree <= 3 in each n_j.  In a direction with multiplicity <= 2
    everywhere the central difference is exact up to round-off; otherwise its error is
    h^2 f'''/6 = h^2 * (third-order coefficient).  Checked on every (i, j) of config 1."""
    from paper_2512_06729_b200 import synth
    net = network(1)
    atm = synth.config_atmosphere(1, net)
    kf, kr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    ns = net.n_species
    eps = 2.0 ** -52
    checked = 0
    for c in (0, 3, 7, 11, 15, 19):
        dense, scale = oracle.jacobian_dense(net, kf, kr, atm.n, c)
        base = atm.n[:, c:c + 1].copy()
        _, p0, l0 = oracle.source(net, kf[:, c:c + 1], kr[:, c:c + 1], base)
        s0 = (p0 + l0)[:, 0]
        for j in range(ns):
            h = base[j, 0] * 2.0 ** -8
            up, dn = base.copy(), base.copy()
            up[j, 0] += h
            dn[j, 0] -= h
            fu, pu, lu = oracle.source(net, kf[:, c:c + 1], kr[:, c:c + 1], up)
            fd, _, _ = oracle.source(net, kf[:, c:c + 1], kr[:, c:c + 1], dn)
            fdiff = (fu[:, 0] - fd[:, 0]) / (2 * h)
            # round-off of the difference + cubic truncation (only where some multiplicity is 3:
            # none in config 1, whose reactions have at most a doubled species)
            noise = 8 * eps * np.maximum(s0, (pu + lu)[:, 0]) / (2 * h)
            trunc = 2.0 ** -16 * scale[:, j]           # (h/n_j)^2 x (terms that are cubic in n_j)
            assert np.all(np.abs(fdiff - dense[:, j]) <= noise + trunc + 1e-300), (c, j)
            checked += int(np.count_nonzero(scale[:, j] > 64 * noise))
    assert checked > 100                               # the check is sharp for many entries


def _brute_source_csr(net):
    rows = [[] for _ in range(net.n_species)]
    for r in range(net.n_reactions):
        nu = {}
        for s_ in net.reactants[r]:
            if s_ >= 0:
                nu[int(s_)] = nu.get(int(s_), 0) - 1
        for s_ in net.products[r]:
            if s_ >= 0:
                nu[int(s_)] = nu.get(int(s_), 0) + 1
        for i, v in nu.items():
            if v:
                rows[i].append((r, v))
    return rows


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_csr_layouts_against_brute_force(oracle, network, cfg):
    """Readings S2, J1, J2: a second, set-based construction in Python must match bit for bit."""
    net = network(cfg)
    row_ptr, rxn, nu = oracle.source_csr(net)
    rows = _brute_source_csr(net)
    assert row_ptr[0] == 0 and row_ptr[-1] == sum(len(x) for x in rows) == rxn.shape[0]
    for i, lst in enumerate(rows):
        sl = slice(row_ptr[i], row_ptr[i + 1])
        assert rxn[sl].tolist() == [r for r, _ in lst]
        assert nu[sl].tolist() == [v for _, v in lst]
    assert np.all(np.abs(nu) <= 3) and np.all(nu != 0)
    jp, jc = oracle.jac_pattern(net)
    pat = [set([i]) for i in range(net.n_species)]
    for r in range(net.n_reactions):
        sp = {int(s_) for s_ in list(net.reactants[r]) + list(net.products[r]) if s_ >= 0}
        for i in sp:
            pat[i] |= sp
    assert jp[0] == 0 and jp[-1] == sum(len(x) for x in pat) == jc.shape[0]
    for i, st in enumerate(pat):
        assert jc[jp[i]:jp[i + 1]].tolist() == sorted(st)
    # structure: symmetric, diagonal present
    dense = np.zeros((net.n_species, net.n_species), dtype=bool)
    for i in range(net.n_species):
        dense[i, jc[jp[i]:jp[i + 1]]] = True
    assert np.array_equal(dense, dense.T) and dense.diagonal().all()
    if cfg == 3:
        he = net.element_names.index("He")
        inert = int(np.flatnonzero(net.composition[:, he])[0])
        assert row_ptr[inert] == row_ptr[inert + 1]            # empty source row
        assert jc[jp[inert]:jp[inert + 1]].tolist() == [inert]  # diagonal only


def test_double_build_of_source_agrees(oracle, oracle_f64, network):
    from paper_2512_06729_b200 import synth
    net = network(2)
    atm = synth.config_atmosphere(2, net)
    a = oracle.source_from_state(net, atm.T, atm.P, atm.J, atm.n, atm.ncol)
    b = oracle_f64.source_from_state(net, atm.T, atm.P, atm.J, atm.n, atm.ncol)
    scale = a[1] + a[2]
    # k_r in pure double carries |dG/RT| * 2^-53 relative error (~1e-13 at these temperatures)
    assert np.all(np.abs(a[0] - b[0]) <= 5e-12 * scale)


@pytest.mark.parametrize("seed", [11, 13, 16])
def test_invariants_on_random_networks_with_one_way_reactions(oracle, seed):
    """The conservation laws do not care which reactions are reversible or which rate form they use: on seeded random
    networks with 30 % one-way thermal reactions and Kooij forms mixed in (the networks of the kernel tests), dn/dt
    conserves every element, so does every Jacobian column, one-way reactions have k_r = 0 exactly, and reversible
    ones obey k_f / k_r = K_c rebuilt here from the thermo output."""
    from paper_2512_06729_b200 import synth
    rng = np.random.default_rng(seed)
    elements = ["H", "C", "O", "N", "S"][:int(rng.integers(2, 6))]
    ns = int(rng.integers(6, 40))
    nr = int(rng.integers(5, 330))
    net = synth.make_network(900 + seed, elements, ns, nr, inert=())
    flip = rng.random(net.n_reactions) < 0.3
    net.reversible = np.where(flip & (net.type != 3), 0, net.reversible).astype(np.uint8)
    net.t_ref = np.where(rng.random(net.n_reactions) < 0.3, 300.0, 1.0)
    atm = synth.make_atmosphere(1900 + seed, net, 1, 12)
    ncol = atm.ncol
    kf, kr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    assert np.all(kr[net.reversible == 0, :ncol] == 0.0) and np.all(kr[net.reversible == 1, :ncol] > 0.0)
    g = oracle.thermo(net, atm.T, ncol)[3]
    kB, P0 = 1.380649e-16, 1.0e6
    for r in np.flatnonzero(net.reversible == 1)[:40]:
        dg = sum(g[s] for s in net.products[r] if s >= 0) - sum(g[s] for s in net.reactants[r] if s >= 0)
        dnu = int((net.products[r] >= 0).sum()) - int((net.reactants[r] >= 0).sum())
        kc = np.exp(-dg[:ncol]) * (P0 / (kB * atm.T[:ncol])) ** dnu
        assert np.allclose(kf[r, :ncol] / kr[r, :ncol], kc, rtol=1e-11, atol=0)
    dndt, prod, loss = oracle.source(net, kf, kr, atm.n, ncol)
    res, ref = _element_residual(net, dndt[:, :ncol], (prod + loss)[:, :ncol])
    assert np.all(np.abs(res) <= 1e-15 * ref)
    row_ptr, col = oracle.jac_pattern(net)
    jac, sc = oracle.jacobian(net, kf, kr, atm.n, row_ptr, col, 3)
    a = net.composition.astype(np.float64)
    rows = np.repeat(np.arange(net.n_species), np.diff(row_ptr))
    for c in range(3):
        dense, scale = np.zeros((net.n_species,) * 2), np.zeros((net.n_species,) * 2)
        dense[rows, col], scale[rows, col] = jac[:, c], sc[:, c]
        assert np.all(np.abs(a.T @ dense) <= 1e-15 * (np.abs(a).T @ scale))
