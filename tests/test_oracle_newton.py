"""Pins of the oracle's implicit step (the chemistry is a stiff ODE
integrated with implicit solvers, backward Euler being the lowest order).  One Newton iteration of the
backward-Euler step solves (I - dt Jac(y)) delta = -(y - n_old - dt f(y)).  The pins are what the
mathematics fixes without this code: closed forms of linear networks, conservation, the equilibrium fixed
point, the explicit limit, quadratic convergence, and an independent library solve of the same system."""
import numpy as np
import pytest

from conftest import SimpleNet

UNI, BI, FALLOFF, PHOTO = 0, 1, 2, 3
K_B = 1.380649e-16
P0 = 1.0e6


def linear_pair(reversible):
    """X0 -> X1 (unimolecular), optionally reversible; thermo all zero so K_c = 1 and k_r = k_f when reversible."""
    z = np.zeros((2, 7))
    return SimpleNet(np.ones((2, 1)), z, z, [1000.0] * 2, [UNI], [[0]], [[1]], [reversible], [[1.0, 0.0, 0.0]])


def test_first_order_decay_is_the_backward_euler_closed_form(oracle):
    """dn/dt = -k n: backward Euler gives n0 / (1 + dt k) exactly, and for a LINEAR network one Newton
    iteration from any iterate lands on it."""
    net = linear_pair(0)
    k = np.array([[2.5e-3, 40.0, 1e6]])
    dt = np.array([100.0, 0.5, 3.0])
    n0 = np.array([[1e10, 3e4, 7.0], [0.0, 5.0, 1e3]])
    exact_a = n0[0] / (1 + dt * k[0])
    for y in (n0, n0 * np.array([[0.3], [2.0]])):              # start at n_old, and off it
        delta, y_new = oracle.newton_step(net, k, np.zeros_like(k), n0, dt, y)
        assert np.all(np.abs(y_new[0] - exact_a) <= 4e-16 * n0[0])
        assert np.all(np.abs(y_new[1] - (n0[1] + n0[0] - exact_a)) <= 4e-16 * (n0[0] + n0[1]))
        assert np.all(np.abs(delta - (y_new - y)) <= 4e-16 * (np.abs(y_new) + np.abs(y)))


def test_reversible_pair_two_by_two_by_hand(oracle):
    """X0 <=> X1 with k_f = a, k_r = b: (I - dt J) = [[1 + dt a, -dt b], [-dt a, 1 + dt b]], solved by hand."""
    net = linear_pair(1)
    a, b, dt = 3.0, 0.25, 2.0
    n0 = np.array([[10.0], [4.0]])
    y = np.array([[7.0], [9.0]])
    f = np.array([-a * y[0, 0] + b * y[1, 0], a * y[0, 0] - b * y[1, 0]])
    rhs = -(y[:, 0] - n0[:, 0] - dt * f)
    det = (1 + dt * a) * (1 + dt * b) - dt * dt * a * b
    want = np.array([(1 + dt * b) * rhs[0] + dt * b * rhs[1], dt * a * rhs[0] + (1 + dt * a) * rhs[1]]) / det
    delta, y_new = oracle.newton_step(net, np.array([[a]]), np.array([[b]]), n0, np.array([dt]), y)
    assert np.allclose(delta[:, 0], want, rtol=1e-15, atol=0)
    A, rb = oracle.newton_system(net, np.array([[a]]), np.array([[b]]), n0, np.array([dt]), y, 0)
    assert np.array_equal(A, [[1 + dt * a, -dt * b], [-dt * a, 1 + dt * b]]) and np.allclose(rb, rhs, rtol=1e-15)


def _state(network, oracle, cfg, stiffness, seed=3):
    """Config network + atmosphere, coefficients, and a per-column dt = stiffness / max_i |Jac_ii|."""
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    ncol = min(atm.ncol, 12)
    kf, kr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    kf, kr, n = kf[:, :ncol].copy(), kr[:, :ncol].copy(), atm.n[:, :ncol].copy()
    dt = np.zeros(ncol)
    for c in range(ncol):
        d, _ = oracle.jacobian_dense(net, kf, kr, n, c)
        dt[c] = stiffness / np.abs(np.diag(d)).max()
    return net, kf, kr, n, dt, ncol


@pytest.mark.parametrize("cfg,stiffness", [(1, 1.0), (1, 1e3), (2, 10.0)])
def test_step_conserves_every_element(oracle, network, cfg, stiffness):
    """a^T f = 0 and a^T Jac = 0 (element conservation of O5, O6) give a^T (I - dt Jac) = a^T, hence
    a^T delta = -a^T (y - n_old): from y = n_old the Newton update moves no atoms."""
    net, kf, kr, n, dt, ncol = _state(network, oracle, cfg, stiffness)
    a = net.composition.astype(np.float64)
    delta, y_new = oracle.newton_step(net, kf, kr, n, dt, n)
    scale = np.abs(a).T @ np.abs(delta)
    assert np.all(np.abs(a.T @ delta) <= 1e-13 * scale + 1e-300)
    rng = np.random.default_rng(1)
    y = n * 10 ** rng.uniform(-0.3, 0.3, size=n.shape)
    delta2, _ = oracle.newton_step(net, kf, kr, n, dt, y)
    want = -(a.T @ (y - n))
    scale2 = np.abs(a).T @ (np.abs(delta2) + np.abs(y) + np.abs(n))
    assert np.all(np.abs(a.T @ delta2 - want) <= 1e-13 * scale2)


def test_equilibrium_composition_is_a_fixed_point_of_the_step(oracle, network):
    """At n_i = (P0/k_B T) exp(-G_i/RT) prod_e lambda_e^(a_ie) with J = 0, f = 0 (test_oracle_source), so
    from y = n_old = n the Newton update vanishes for any dt."""
    from paper_2512_06729_b200 import synth
    net = network(2)
    atm = synth.config_atmosphere(2, net)
    ncol = 6
    T, P = atm.T[:ncol], atm.P[:ncol]
    g = oracle.thermo(net, T)[3]
    loglam = np.random.default_rng(17).uniform(-3, 3, size=net.n_elements)
    n = np.exp(np.log(P0 / (K_B * T))[None, :] - g + (net.composition @ loglam)[:, None])
    J = np.zeros((net.n_photo, ncol))
    kf, kr = oracle.rate_coeffs(net, T, P, J)
    rate = np.array([np.abs(np.diag(oracle.jacobian_dense(net, kf, kr, n, c)[0])).max() for c in range(ncol)])
    y_off = n * 10 ** np.random.default_rng(5).uniform(-0.3, 0.3, size=n.shape)   # negative control: off equilibrium
    for stiffness in (1e-3, 1.0, 1e3, 1e9):
        dt = stiffness / rate
        delta, _ = oracle.newton_step(net, kf, kr, n, dt, n)
        # f = 0 up to the ~1e-14 relative round-off that exp(|G| ~ 1e2) leaves in n
        assert np.all(np.abs(delta) <= 1e-12 * n), stiffness
        d_off, _ = oracle.newton_step(net, kf, kr, y_off, dt, y_off)
        assert np.abs(d_off / y_off).max() >= 1e-4 * min(stiffness, 1.0), stiffness


def test_small_step_limit_is_explicit_euler(oracle, network):
    """dt -> 0: (I - dt Jac)^-1 = I + dt Jac + O(dt^2), so delta / dt = f + dt Jac f + O(dt^2): the gap to
    explicit Euler is bounded by dt |Jac| |f| and shrinks in proportion to dt."""
    gaps = []
    for stiffness in (1e-6, 1e-9):
        net, kf, kr, n, dt, ncol = _state(network, oracle, 1, stiffness)
        f, prod, loss = oracle.source(net, kf, kr, n)
        delta, _ = oracle.newton_step(net, kf, kr, n, dt, n)
        gap = np.abs(delta / dt[None, :] - f)
        bound = np.stack([dt[c] * (np.abs(oracle.jacobian_dense(net, kf, kr, n, c)[0]) @ np.abs(f[:, c])) for c in range(ncol)], axis=1)
        assert np.all(gap <= 1.01 * bound + 1e-13 * (prod + loss))
        gaps.append(float((gap / (prod + loss).max(axis=0, keepdims=True)).max()))
    assert gaps[1] <= 2e-3 * gaps[0]


@pytest.mark.parametrize("cfg,stiffness", [(1, 30.0), (2, 30.0)])
def test_newton_iteration_converges_quadratically_to_the_backward_euler_root(oracle, network, cfg, stiffness):
    net, kf, kr, n, dt, ncol = _state(network, oracle, cfg, stiffness)
    y = n.copy()
    norms = []
    for it in range(8):
        f, prod, loss = oracle.source(net, kf, kr, y)
        F = y - n - dt[None, :] * f
        scale = np.abs(y) + np.abs(n) + dt[None, :] * (prod + loss)
        norms.append(float((np.abs(F) / scale).max()))
        if norms[-1] < 1e-15:
            break
        _, y = oracle.newton_step(net, kf, kr, n, dt, y)
    assert norms[-1] <= 1e-13, norms
    big = [x for x in norms if 1e-12 < x < 1e-2]
    for a, b in zip(big, big[1:]):
        assert b <= 10 * a * a + 1e-13, norms            # quadratic once inside the basin
    assert np.all(np.isfinite(y))


@pytest.mark.parametrize("cfg", [1, 2])
def test_solution_agrees_with_a_library_solver_on_the_same_system(oracle, network, cfg):
    """The exported dense system solved by LAPACK (numpy) in double: an independent elimination."""
    net, kf, kr, n, dt, ncol = _state(network, oracle, cfg, 100.0)
    y = n * 10 ** np.random.default_rng(2).uniform(-0.2, 0.2, size=n.shape)
    delta, _ = oracle.newton_step(net, kf, kr, n, dt, y)
    for c in range(ncol):
        A, b = oracle.newton_system(net, kf, kr, n, dt, y, c)
        x = np.linalg.solve(A, b)
        cond = np.linalg.cond(A)
        assert np.all(np.abs(x - delta[:, c]) <= 1e-15 * cond * np.abs(delta[:, c]).max() + 1e-300)
        # Gaussian elimination with partial pivoting is backward stable NORMWISE (densities span 40 decades, so
        # a componentwise bound does not hold for the small rows); the residual is evaluated in double here
        r = A @ delta[:, c] - b
        bound = np.abs(A).sum(axis=1).max() * np.abs(delta[:, c]).max() + np.abs(b).max()
        assert np.abs(r).max() <= (net.n_species + 2) * 2.3e-16 * bound
