"""`-m gpu` parity tests: the CUDA path, called through the C ABI (paper_2512_06729_b200.binding),
against the CPU oracle on the same seeded inputs, element by element.

Tolerances (BASELINE.json north_star): k_f, k_r relative 1e-12; dn/dt and Jacobian entries 1e-11
of sum |contributing terms| per entry; CSR layouts bit-exact (tests/test_boundary.py).  Thermo:
1e-13 of sum |polynomial terms|.  Overflow rule: DESIGN.md reading R5."""
import numpy as np
import pytest

import gpu_common as G

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def xod():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests need the B200 box (there is no CPU fallback)")
    from paper_2512_06729_b200 import binding, build
    build.build()
    binding.lib()
    return binding


_handles = {}


@pytest.fixture(autouse=True)
def _device_clean_after_each_test(xod):
    """After every test: synchronise and, in the bounds-checked build (XOD_CHECK=1), fail if a kernel
    saw an out-of-range table index (the check build clamps and records instead of faulting)."""
    yield
    for h in _handles.values():
        h.check_status()


def handle(xod, network, cfg):
    key = 3 if cfg in (3, 4, 5) else cfg
    if key not in _handles:
        _handles[key] = xod.Network(network(key), device=0)
    return _handles[key]


def atmosphere(cfg, net, n_atm=None):
    from paper_2512_06729_b200 import synth
    return synth.config_atmosphere(cfg, net, n_atm)


def thermo_scale(net, T):
    """sum |terms| of each NASA-7 form (tolerance scale only)."""
    T = np.asarray(T)[None, :]
    a = np.where((T <= net.t_mid[:, None])[:, :, None], net.nasa_lo[:, None, :], net.nasa_hi[:, None, :])
    a = np.abs(a)
    lnT = np.abs(np.log(T))
    p = [a[:, :, k] * T ** k for k in range(5)]
    cp = sum(p)
    h = p[0] + p[1] / 2 + p[2] / 3 + p[3] / 4 + p[4] / 5 + a[:, :, 5] / T
    s = a[:, :, 0] * lnT + p[1] + p[2] / 2 + p[3] / 3 + p[4] / 4 + a[:, :, 6]
    g = a[:, :, 0] * (1 + lnT) + p[1] / 2 + p[2] / 6 + p[3] / 12 + p[4] / 20 + a[:, :, 5] / T + a[:, :, 6]
    return cp, h, s, g


# ------------------------------------------------------------------------------- a2 thermo
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_thermo_matches_oracle(xod, oracle, network, cfg):
    net = network(cfg)
    h = handle(xod, network, cfg)
    atm = atmosphere(cfg, net)
    want = oracle.thermo(net, atm.T, atm.ncol)
    outs = [G.empty(net.n_species, atm.ld) for _ in range(4)]
    h.thermo(atm.ncol, atm.ld, G.dev(atm.T), *outs)
    scales = thermo_scale(net, atm.T)
    c = slice(0, atm.ncol)
    for name, got, w, s in zip(("cp/R", "H/RT", "S/R", "G/RT"), outs, want, scales):
        got = G.host(got)
        assert np.all(np.abs(got[:, c] - w[:, c]) <= G.TOL_THERMO * s[:, c]), name
        assert np.all(np.isnan(got[:, atm.ncol:])), "%s: padding columns were written" % name
    # optional outputs: only G/RT requested
    g_only = G.empty(net.n_species, atm.ld)
    h.thermo(atm.ncol, atm.ld, G.dev(atm.T), None, None, None, g_only)
    assert np.array_equal(G.host(g_only)[:, c], G.host(outs[3])[:, c])


def test_thermo_range_selection_at_t_mid(xod, oracle, network):
    """Reading T3: T <= t_mid -> low set; exactly t_mid -> low."""
    net = network(2)
    h = handle(xod, network, 2)
    tm = float(net.t_mid[0])
    T = np.array([np.nextafter(tm, 0), tm, np.nextafter(tm, 1e9), 300.0, 500.0, 700.0, 1000.0, 150.0, 6000.0])
    want = oracle.thermo(net, T)
    outs = [G.empty(net.n_species, T.size) for _ in range(4)]
    h.thermo(T.size, T.size, G.dev(T), *outs)
    for got, w, s in zip(outs, want, thermo_scale(net, T)):
        assert np.all(np.abs(G.host(got) - w) <= G.TOL_THERMO * s)


# ------------------------------------------------------------------------------- a1, a3-a6 coefficients
def run_rate_coeffs(h, atm, ncol=None, ld=None):
    ncol = atm.ncol if ncol is None else ncol
    ld = atm.ld if ld is None else ld
    kf, kr = G.empty(h.n_reactions, ld), G.empty(h.n_reactions, ld)
    ws = G.workspace(h.rate_coeffs_workspace_bytes(ncol))
    h.rate_coeffs(ncol, ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), kf, kr, ws)
    return G.host(kf), G.host(kr)


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_rate_coeffs_match_oracle(xod, oracle, network, cfg):
    net = network(cfg)
    h = handle(xod, network, cfg)
    atm = atmosphere(cfg, net)
    kf, kr = run_rate_coeffs(h, atm)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    c = slice(0, atm.ncol)
    G.check_k(kf[:, c], okf[:, c], "k_f config %d" % cfg)
    G.check_k(kr[:, c], okr[:, c], "k_r config %d" % cfg)
    assert np.all(np.isnan(kf[:, atm.ncol:])) and np.all(np.isnan(kr[:, atm.ncol:]))
    photo = net.type == 3
    assert np.array_equal(kf[photo][:, c], atm.J[:, c])           # a5: k_f = J bit for bit
    assert np.all(kr[photo][:, c] == 0.0)


def test_rate_coeffs_cold_columns_overflow_rule(xod, oracle, network):
    """Config 4's cold T shifts drive |dG/RT| past the double range (reading R5): inf where the
    oracle (long double, rounded at the end) is inf, tiny where it underflows, 1e-12 elsewhere."""
    net = network(4)
    h = handle(xod, network, 4)
    atm = atmosphere(4, net, n_atm=6)
    assert atm.T[:atm.ncol].min() < 450.0
    kf, kr = run_rate_coeffs(h, atm)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    c = slice(0, atm.ncol)
    G.check_k(kf[:, c], okf[:, c], "k_f config 4")
    G.check_k(kr[:, c], okr[:, c], "k_r config 4")
    assert np.isinf(okr[:, c]).any(), "the sample was meant to contain overflowing k_r"


def test_kooij_reference_temperature(xod, oracle, network):
    """Reading K1: t_ref = 300 (Kooij) on some reactions."""
    import copy
    net = copy.copy(network(1))
    net.t_ref = np.where(np.arange(net.n_reactions) % 2 == 0, 300.0, 1.0)
    h = xod.Network(net, device=0)
    atm = atmosphere(1, net)
    kf, kr = run_rate_coeffs(h, atm)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    G.check_k(kf[:, :atm.ncol], okf[:, :atm.ncol], "k_f Kooij")
    G.check_k(kr[:, :atm.ncol], okr[:, :atm.ncol], "k_r Kooij")
    h.close()


# ------------------------------------------------------------------------------- a7-a8 source
def element_residual(net, dndt, scale, cols):
    """max over (element, column) of |sum_i a_ie dn_i/dt| / sum_i |a_ie| S_i."""
    a = net.composition.astype(np.float64)
    num = np.abs(a.T @ dndt[:, cols])
    den = np.abs(a).T @ scale[:, cols]
    m = den > 0
    return float((num[m] / den[m]).max())


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_source_from_stored_coefficients(xod, oracle, network, cfg):
    net = network(cfg)
    h = handle(xod, network, cfg)
    atm = atmosphere(cfg, net)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, atm.ncol)
    ns, ld = net.n_species, atm.ld
    ws = G.workspace(h.source_workspace_bytes(atm.ncol))
    d0 = G.empty(ns, ld)
    h.source(atm.ncol, ld, G.dev(okf), G.dev(okr), G.dev(atm.n), d0, workspace=ws)
    d1, p1, l1 = G.empty(ns, ld), G.empty(ns, ld), G.empty(ns, ld)
    h.source(atm.ncol, ld, G.dev(okf), G.dev(okr), G.dev(atm.n), d1, p1, l1, workspace=ws)
    cols = np.arange(atm.ncol)
    scale = wp + wl
    for got in (G.host(d0), G.host(d1)):
        G.check_sum(got, want, scale, cols, "dn/dt config %d" % cfg)
        assert np.all(np.isnan(got[:, atm.ncol:]))
        assert element_residual(net, got, scale, cols) <= 1e-13
    G.check_sum(G.host(p1), wp, scale, cols, "P")
    G.check_sum(G.host(l1), wl, scale, cols, "L")


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_source_fused_matches_oracle(xod, oracle, network, cfg):
    """The headline path a1-a8: (T, P, J, n) -> dn/dt with k_f, k_r never stored."""
    net = network(cfg)
    h = handle(xod, network, cfg)
    atm = atmosphere(cfg, net)
    want, wp, wl = oracle.source_from_state(net, atm.T, atm.P, atm.J, atm.n, atm.ncol)
    ns, ld = net.n_species, atm.ld
    ws = G.workspace(h.source_fused_workspace_bytes(atm.ncol))
    d0 = G.empty(ns, ld)
    h.source_fused(atm.ncol, ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n), d0, workspace=ws)
    d1, p1, l1 = G.empty(ns, ld), G.empty(ns, ld), G.empty(ns, ld)
    h.source_fused(atm.ncol, ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n), d1, p1, l1,
                   workspace=ws)
    cols = np.arange(atm.ncol)
    scale = wp + wl
    for got in (G.host(d0), G.host(d1)):
        G.check_sum(got, want, scale, cols, "fused dn/dt config %d" % cfg)
        assert np.all(np.isnan(got[:, atm.ncol:]))
        assert element_residual(net, got, scale, cols) <= 1e-13
    G.check_sum(G.host(p1), wp, scale, cols, "fused P")
    G.check_sum(G.host(l1), wl, scale, cols, "fused L")
    # the host-buffer entry point runs the same kernels
    out = np.full((ns, ld), np.nan)
    h.source_fused_host(atm.ncol, ld, atm.T, atm.P, atm.J, atm.n, out)
    assert np.array_equal(out[:, :atm.ncol], G.host(d0)[:, :atm.ncol])


def test_source_fused_config4_batch(xod, oracle, network):
    """Config 4 family (T shifts, metallicity): several chunks, a ragged tail, and columns with
    non-finite k_r excluded by reading R5 (their count is reported, and must be > 0 here)."""
    net = network(4)
    h = handle(xod, network, 4)
    atm = atmosphere(4, net, n_atm=9)                 # 1350 columns: 84 full tiles and a ragged one (6 columns)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, atm.ncol)
    ns, ld = net.n_species, atm.ld
    ws = G.workspace(h.source_fused_workspace_bytes(atm.ncol))
    d0 = G.empty(ns, ld)
    h.source_fused(atm.ncol, ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n), d0, workspace=ws)
    ok = G.finite_columns(okf[:, :atm.ncol], okr[:, :atm.ncol], want[:, :atm.ncol], wp[:, :atm.ncol], wl[:, :atm.ncol])
    cols = np.flatnonzero(ok)
    excluded = atm.ncol - cols.size
    print("config 4 sample: %d of %d columns excluded by R5" % (excluded, atm.ncol))
    assert 0 < excluded < atm.ncol
    got = G.host(d0)
    scale = wp + wl
    G.check_sum(got, want, scale, cols, "fused dn/dt config 4")
    assert element_residual(net, got, scale, cols) <= 1e-13


# ------------------------------------------------------------------------------- a9 Jacobian
@pytest.mark.parametrize("cfg,n_atm", [(1, None), (2, None), (5, 1)])
def test_jacobian_matches_oracle(xod, oracle, network, cfg, n_atm):
    net = network(cfg)
    h = handle(xod, network, cfg)
    atm = atmosphere(cfg, net, n_atm)
    ncol = atm.ncol if cfg != 5 else 40               # the dense oracle is O(ns^2) per column
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    rp, col = h.jac_pattern()
    want, scale = oracle.jacobian(net, okf, okr, atm.n, rp, col, ncol)
    assert h.jac_info()["enabled"] == 1
    for tiled in (0, 1):      # the one-warp-per-entry gather kernel, then the tiled kernel (the default)
        h.tune(xod.XOD_TUNE_JAC_TILED, tiled)
        jac = G.empty(h.nnz_jac, atm.ld)
        h.jacobian(ncol, atm.ld, G.dev(okf), G.dev(okr), G.dev(atm.n), jac)
        got = G.host(jac)
        worst = G.check_sum(got, want, scale, np.arange(ncol), "Jacobian config %d (tiled %d)" % (cfg, tiled))
        assert np.all(np.isnan(got[:, ncol:]))
        print("Jacobian config %d, %d columns, tiled kernel %d: worst |err|/scale %.2e" % (cfg, ncol, tiled, worst))
    # element conservation of the Jacobian: sum_i a_ie Jac_ij = 0 for every (e, j)
    rows = np.repeat(np.arange(net.n_species), np.diff(rp))
    a = net.composition.astype(np.float64)
    for e in range(net.n_elements):
        num = np.zeros((net.n_species, ncol))
        den = np.zeros((net.n_species, ncol))
        np.add.at(num, col, a[rows, e][:, None] * got[:, :ncol])
        np.add.at(den, col, np.abs(a[rows, e])[:, None] * scale[:, :ncol])
        m = den > 0
        assert np.all(np.abs(num[m]) <= 1e-13 * den[m])


# ------------------------------------------------------------------------------- edge cases
def test_zero_densities_give_exact_zeros(xod, oracle, network):
    """Reading Q2: n = 0 is legal; the Jacobian never divides by n_j."""
    net = network(2)
    h = handle(xod, network, 2)
    atm = atmosphere(2, net)
    n = atm.n.copy()
    n[::3, :] = 0.0
    n[:, 5] = 0.0
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    want, wp, wl = oracle.source(net, okf, okr, n, atm.ncol)
    ws = G.workspace(h.source_fused_workspace_bytes(atm.ncol))
    d0 = G.empty(net.n_species, atm.ld)
    h.source_fused(atm.ncol, atm.ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(n), d0, workspace=ws)
    got = G.host(d0)
    G.check_sum(got, want, wp + wl, np.arange(atm.ncol), "dn/dt with zeros")
    assert np.all(got[:, 5] == 0.0)
    rp, col = h.jac_pattern()
    wj, sj = oracle.jacobian(net, okf, okr, n, rp, col, atm.ncol)
    jac = G.empty(h.nnz_jac, atm.ld)
    h.jacobian(atm.ncol, atm.ld, G.dev(okf), G.dev(okr), G.dev(n), jac)
    G.check_sum(G.host(jac), wj, sj, np.arange(atm.ncol), "Jacobian with zeros")


@pytest.mark.parametrize("ncol,ld", [(0, 32), (1, 1), (31, 40), (33, 64), (150, 150), (97, 256)])
def test_ragged_sizes_and_pitches(xod, oracle, network, ncol, ld):
    """Empty, single-column, sub-warp, just-over-a-warp sizes and pitches that are not multiples
    of 32; columns beyond ncol are never touched."""
    from paper_2512_06729_b200 import synth
    net = network(2)
    h = handle(xod, network, 2)
    atm = synth.make_atmosphere(77, net, 1, max(ncol, 1), ld=ld)
    want, wp, wl = oracle.source_from_state(net, atm.T, atm.P, atm.J, atm.n, ncol)
    ws = G.workspace(h.source_fused_workspace_bytes(ncol))
    d0 = G.empty(net.n_species, ld)
    h.source_fused(ncol, ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n), d0, workspace=ws)
    got = G.host(d0)
    G.check_sum(got, want, wp + wl, np.arange(ncol), "ragged dn/dt")
    assert np.all(np.isnan(got[:, ncol:]))
    kf, kr = run_rate_coeffs(h, atm, ncol, ld)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    G.check_k(kf[:, :ncol], okf[:, :ncol], "ragged k_f")
    G.check_k(kr[:, :ncol], okr[:, :ncol], "ragged k_r")
    assert np.all(np.isnan(kf[:, ncol:]))


def test_chunk_boundaries_do_not_change_results(xod, network):
    """The column-chunk pipeline (multi-kernel path: col0 > 0 in k_prologue / k_rates / k_source) must be
    invisible: 64-column chunks == one chunk, bit for bit."""
    net = network(3)
    atm = atmosphere(3, net)
    outs = []
    for chunk in (0, 64):
        h = xod.Network(net, device=0)
        h.tune(xod.XOD_TUNE_FUSED_KERNEL, 0)
        h.tune(xod.XOD_TUNE_CHUNK_COLS, chunk)
        ws = G.workspace(h.source_fused_workspace_bytes(atm.ncol))
        d0 = G.empty(net.n_species, atm.ld)
        h.source_fused(atm.ncol, atm.ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n), d0, workspace=ws)
        outs.append(G.host(d0)[:, :atm.ncol])
        h.close()
    assert np.array_equal(outs[0], outs[1])


def test_workspace_too_small_is_an_error(xod, network):
    net = network(1)
    h = handle(xod, network, 1)
    atm = atmosphere(1, net)
    d0 = G.empty(net.n_species, atm.ld)
    with pytest.raises(xod.XodError) as e:
        h.source_fused(atm.ncol, atm.ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n), d0,
                       workspace=G.dev(np.zeros(4)))
    assert e.value.status == 5
    with pytest.raises(xod.XodError) as e:
        h.source_fused(atm.ncol, atm.ncol - 1, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n), d0,
                       workspace=G.workspace(h.source_fused_workspace_bytes(atm.ncol)))
    assert e.value.status == 1


# ------------------------------------------------------------------------------- full sizes, sampled
def _gather_columns(atm, cols):
    """A compact atmosphere holding only the sampled columns (oracle input)."""
    return atm.T[cols].copy(), atm.P[cols].copy(), atm.J[:, cols].copy(), atm.n[:, cols].copy()


def test_full_size_config4_whole_batch(xod, oracle, network):
    """BASELINE config 4 at full size (256 x 150 = 38 400 columns) in the launch configuration
    bench.py times (one xod_source_fused call), every column against the oracle (about a minute of
    oracle time); columns with k_r beyond the double range are excluded by reading R5 and counted."""
    net = network(4)
    h = handle(xod, network, 4)
    atm = atmosphere(4, net)
    assert atm.ncol == 38400
    ws = G.workspace(h.source_fused_workspace_bytes(atm.ncol))
    d0, p0, l0 = G.empty(net.n_species, atm.ld), G.empty(net.n_species, atm.ld), G.empty(net.n_species, atm.ld)
    dT, dP, dJ, dn = G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n)
    h.source_fused(atm.ncol, atm.ld, dT, dP, dJ, dn, d0, workspace=ws)
    got = G.host(d0)
    h.source_fused(atm.ncol, atm.ld, dT, dP, dJ, dn, d0, p0, l0, workspace=ws)
    got_pl, gp, gl = G.host(d0), G.host(p0), G.host(l0)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, atm.ncol)
    c = slice(0, atm.ncol)
    ok = G.finite_columns(okf[:, c], okr[:, c], want[:, c], wp[:, c], wl[:, c])
    cols = np.flatnonzero(ok)
    scale = wp + wl
    worst = G.check_sum(got, want, scale, cols, "full-size fused dn/dt")
    res = element_residual(net, got, scale, cols)
    print("config 4, all %d columns: %d excluded by R5; worst |err|/scale = %.2e; element residual %.2e"
          % (atm.ncol, atm.ncol - cols.size, worst, res))
    assert 0 < atm.ncol - cols.size < atm.ncol // 2
    assert res <= 1e-13
    G.check_sum(got_pl, want, scale, cols, "full-size fused dn/dt (P/L variant)")
    G.check_sum(gp, wp, scale, cols, "full-size fused P")
    G.check_sum(gl, wl, scale, cols, "full-size fused L")
    # excluded columns: wherever the oracle's value left the double range (an overflowed k_r), the GPU's did too; the
    # GPU may have more such entries, because a partial product of k n n n can overflow first (reading R5, second part)
    assert not np.isfinite(got[:, c][~np.isfinite(want[:, c])]).any()


def test_full_size_config5_jacobian_whole_atmospheres(xod, oracle, network):
    """BASELINE config 5 at full size (64 x 150 = 9 600 columns): rate coefficients, dn/dt and
    Jacobian values, checked on sampled columns."""
    net = network(5)
    h = handle(xod, network, 5)
    atm = atmosphere(5, net)
    assert atm.ncol == 9600
    nr, ns, ld = net.n_reactions, net.n_species, atm.ld
    T, P, J, n = G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n)
    kf, kr = G.empty(nr, ld), G.empty(nr, ld)
    h.rate_coeffs(atm.ncol, ld, T, P, J, kf, kr, G.workspace(h.rate_coeffs_workspace_bytes(atm.ncol)))
    jac = G.empty(h.nnz_jac, ld)
    h.jacobian(atm.ncol, ld, kf, kr, n, jac)
    d0 = G.empty(ns, ld)
    h.source(atm.ncol, ld, kf, kr, n, d0, workspace=G.workspace(h.source_workspace_bytes(atm.ncol)))
    # two whole atmospheres (the first and one from the middle) plus the edges of the last tiles
    cols = np.unique(np.concatenate([np.arange(150), np.arange(31 * 150, 32 * 150), [9567, 9568, 9583, 9584, 9599]]))
    Tc, Pc, Jc, nc = _gather_columns(atm, cols)
    okf, okr = oracle.rate_coeffs(net, Tc, Pc, Jc)
    G.check_k(G.host(kf)[:, cols], okf, "full-size k_f")
    G.check_k(G.host(kr)[:, cols], okr, "full-size k_r")
    rp, col = h.jac_pattern()
    wj, sj = oracle.jacobian(net, okf, okr, nc, rp, col)
    wj_worst = G.check_sum(G.host(jac)[:, cols], wj, sj, np.arange(cols.size), "full-size Jacobian (%d columns)" % cols.size)
    want, wp, wl = oracle.source(net, okf, okr, nc)
    wd = G.check_sum(G.host(d0)[:, cols], want, wp + wl, np.arange(cols.size), "full-size dn/dt (sampled)")
    print("config 5, %d of %d columns: worst |err|/scale Jacobian %.2e, dn/dt %.2e" % (cols.size, atm.ncol, wj_worst, wd))


def test_reaction_split_path_matches_single_pass(xod, oracle, network):
    """Few columns: the chunks of a tile are split over several CTAs and combined in split order.
    Forced splits must agree with the oracle like the automatic choice does."""
    net = network(3)
    atm = atmosphere(3, net)
    want, wp, wl = oracle.source_from_state(net, atm.T, atm.P, atm.J, atm.n, atm.ncol)
    for split in (1, 3, 31):
        h = xod.Network(net, device=0)
        h.tune(xod.XOD_TUNE_SPLIT, split)
        ws = G.workspace(h.source_fused_workspace_bytes(atm.ncol))
        d0 = G.empty(net.n_species, atm.ld)
        h.source_fused(atm.ncol, atm.ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n), d0, workspace=ws)
        G.check_sum(G.host(d0), want, wp + wl, np.arange(atm.ncol), "split %d" % split)
        assert np.all(np.isnan(G.host(d0)[:, atm.ncol:]))
        h.close()


def test_many_thermo_breakpoints_fall_back_to_the_multi_kernel_path(xod, oracle, network):
    """More than 31 distinct t_mid values: the fused single-kernel tables are disabled and
    xod_source_fused runs the multi-kernel pipeline; results still match the oracle."""
    import copy
    net = copy.copy(network(2))
    net.t_mid = 300.0 + 10.0 * np.arange(net.n_species)
    h = xod.Network(net, device=0)
    assert h.fused_info()["enabled"] == 0
    atm = atmosphere(2, net)
    want, wp, wl = oracle.source_from_state(net, atm.T, atm.P, atm.J, atm.n, atm.ncol)
    ws = G.workspace(h.source_fused_workspace_bytes(atm.ncol))
    d0 = G.empty(net.n_species, atm.ld)
    h.source_fused(atm.ncol, atm.ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n), d0, workspace=ws)
    G.check_sum(G.host(d0), want, wp + wl, np.arange(atm.ncol), "fallback dn/dt")
    kf, kr = run_rate_coeffs(h, atm)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    G.check_k(kf[:, :atm.ncol], okf[:, :atm.ncol], "fallback k_f")
    G.check_k(kr[:, :atm.ncol], okr[:, :atm.ncol], "fallback k_r")
    h.close()


def test_multi_kernel_pipeline_can_be_forced(xod, oracle, network):
    """XOD_TUNE_FUSED_KERNEL = 0: xod_rate_coeffs and xod_source_fused run the multi-kernel pipeline
    (prologue + rates + source kernels); both pipelines must match the oracle."""
    net = network(3)
    atm = atmosphere(3, net)
    h = xod.Network(net, device=0)
    h.tune(xod.XOD_TUNE_FUSED_KERNEL, 0)
    kf, kr = run_rate_coeffs(h, atm)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    G.check_k(kf[:, :atm.ncol], okf[:, :atm.ncol], "multi-kernel k_f")
    G.check_k(kr[:, :atm.ncol], okr[:, :atm.ncol], "multi-kernel k_r")
    want, wp, wl = oracle.source(net, okf, okr, atm.n, atm.ncol)
    ws = G.workspace(h.source_fused_workspace_bytes(atm.ncol))
    d0 = G.empty(net.n_species, atm.ld)
    h.source_fused(atm.ncol, atm.ld, G.dev(atm.T), G.dev(atm.P), G.dev(atm.J), G.dev(atm.n), d0, workspace=ws)
    G.check_sum(G.host(d0), want, wp + wl, np.arange(atm.ncol), "multi-kernel dn/dt")
    h.close()


def test_host_entry_point_pipelines_column_chunks(xod, oracle, network):
    """xod_source_fused_host on 5 000 columns: three chunks (2 x 2 368 + 264, the last one on the
    reaction-split path) through the staging slots; checked on sampled columns of every chunk."""
    from paper_2512_06729_b200 import synth
    net = network(3)
    h = handle(xod, network, 3)
    atm = synth.make_atmosphere(91, net, 1, 5000)
    out = np.full((net.n_species, atm.ld), np.nan)
    h.source_fused_host(atm.ncol, atm.ld, atm.T, atm.P, atm.J, atm.n, out)
    assert np.all(np.isfinite(out[:, :atm.ncol])) and np.all(np.isnan(out[:, atm.ncol:]))
    cols = np.array([0, 15, 16, 2367, 2368, 2369, 4735, 4736, 4737, 4999])
    T, P, J, n = _gather_columns(atm, cols)
    want, wp, wl = oracle.source_from_state(net, T, P, J, n)
    G.check_sum(out[:, cols], want, wp + wl, np.arange(cols.size), "host pipeline dn/dt (sampled)")


# ------------------------------------------------------------------------------- the edge-case network
@pytest.fixture(scope="module")
def edge(xod, oracle):
    from paper_2512_06729_b200 import synth
    net = synth.edge_network()
    atm = synth.edge_atmosphere(net)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, atm.ncol)
    c = slice(0, atm.ncol)
    cols = np.flatnonzero(G.finite_columns(okf[:, c], okr[:, c], want[:, c], wp[:, c], wl[:, c]))
    h = xod.Network(net, device=0)
    _handles["edge"] = h
    return net, atm, h, okf, okr, want, wp, wl, cols


def test_edge_network_rate_coefficients(xod, edge):
    """Irreversible thermal reactions (k_r = 0 exactly), Fc = 1 (Eq. 12), Kooij forms, ions, and T on /
    one ulp beside every thermo breakpoint (reading T3) -- through k_rate_coeffs and the multi-kernel pipeline."""
    net, atm, h, okf, okr, *_ = edge
    c = slice(0, atm.ncol)
    for fused in (1, 0):
        h.tune(xod.XOD_TUNE_FUSED_KERNEL, fused)
        kf, kr = run_rate_coeffs(h, atm)
        wf = G.check_k(kf[:, c], okf[:, c], "edge k_f (fused tables %d)" % fused)
        wr = G.check_k(kr[:, c], okr[:, c], "edge k_r (fused tables %d)" % fused)
        assert np.all(kr[net.reversible == 0][:, c] == 0.0)
        print("edge network k (single-kernel %d): worst relative error k_f %.2e, k_r %.2e" % (fused, wf, wr))
    h.tune(xod.XOD_TUNE_FUSED_KERNEL, 1)
    assert np.isinf(okr[:, c]).any()


def test_edge_network_source_all_paths(xod, edge):
    """nu = +-3, an empty CSR row, a zero species, a zero column, a negative density: xod_source and
    xod_source_fused, with and without P/L, single-kernel and multi-kernel, reaction-split or not."""
    net, atm, h, okf, okr, want, wp, wl, cols = edge
    ns, ld, ncol = net.n_species, atm.ld, atm.ncol
    scale = wp + wl
    dT, dP, dJ, dn, dkf, dkr = (G.dev(a) for a in (atm.T, atm.P, atm.J, atm.n, okf, okr))
    ws = G.workspace(max(h.source_fused_workspace_bytes(ncol), h.source_workspace_bytes(ncol)) + (64 << 20))
    for fused, split in ((1, 0), (1, 2), (0, 0)):
        h.tune(xod.XOD_TUNE_FUSED_KERNEL, fused)
        h.tune(xod.XOD_TUNE_SPLIT, split)
        for pl in (False, True):
            for stored in (False, True):
                d0 = G.empty(ns, ld)
                p0, l0 = (G.empty(ns, ld), G.empty(ns, ld)) if pl else (None, None)
                if stored:
                    h.source(ncol, ld, dkf, dkr, dn, d0, p0, l0, workspace=ws)
                else:
                    h.source_fused(ncol, ld, dT, dP, dJ, dn, d0, p0, l0, workspace=ws)
                what = "edge dn/dt (single-kernel %d, split %d, P/L %d, stored k %d)" % (fused, split, pl, stored)
                got = G.host(d0)
                worst = G.check_sum(got, want, scale, cols, what)
                G.check_sum_entries(got, want, scale, ncol, what + " entry-wise")
                assert np.all(np.isnan(got[:, ncol:])), what
                assert np.all(got[net.meta["lone"], cols] == 0.0) and np.all(got[:, atm.meta["zero_column"]] == 0.0)
                assert element_residual(net, got, scale, cols) <= 1e-13, what
                if pl:
                    G.check_sum(G.host(p0), wp, scale, cols, what + " P")
                    G.check_sum(G.host(l0), wl, scale, cols, what + " L")
                print("%s: worst |err|/scale %.2e" % (what, worst))
    h.tune(xod.XOD_TUNE_FUSED_KERNEL, 1)
    h.tune(xod.XOD_TUNE_SPLIT, 0)


def test_edge_network_jacobian_and_thermo(xod, oracle, edge):
    net, atm, h, okf, okr, want, wp, wl, cols = edge
    ncol, ld = atm.ncol, atm.ld
    okr_f = np.where(np.isfinite(okr), okr, 0.0)      # finite inputs for the dense oracle; those columns are not compared
    rp, col = h.jac_pattern()
    wj, sj = oracle.jacobian(net, okf, okr_f, atm.n, rp, col, ncol)
    for tiled in (0, 1):
        h.tune(xod.XOD_TUNE_JAC_TILED, tiled)
        for split in (0, 3):
            h.tune(xod.XOD_TUNE_SPLIT, split)
            jac = G.empty(h.nnz_jac, ld)
            h.jacobian(ncol, ld, G.dev(okf), G.dev(okr_f), G.dev(atm.n), jac)
            worst = G.check_sum(G.host(jac), wj, sj, cols, "edge Jacobian (tiled %d, split %d)" % (tiled, split))
            assert np.all(np.isnan(G.host(jac)[:, ncol:]))
            print("edge network Jacobian (tiled %d, split %d): worst |err|/scale %.2e" % (tiled, split, worst))
    h.tune(xod.XOD_TUNE_SPLIT, 0)
    outs = [G.empty(net.n_species, ld) for _ in range(4)]
    h.thermo(ncol, ld, G.dev(atm.T), *outs)
    for got, w, s in zip(outs, oracle.thermo(net, atm.T, ncol), thermo_scale(net, atm.T)):
        assert np.all(np.abs(G.host(got)[:, :ncol] - w[:, :ncol]) <= G.TOL_THERMO * s[:, :ncol])


def test_production_and_loss_over_several_column_chunks(xod, oracle, network):
    """P and L on 2 500 columns of the config-4 family: several chunks / rounds of tiles with a ragged tail,
    for xod_source and xod_source_fused, single-kernel and multi-kernel (64-column chunks, col0 > 0)."""
    net = network(4)
    atm = atmosphere(4, net, n_atm=17)
    atm.ncol = 2500
    ncol, ld, ns = atm.ncol, atm.ld, net.n_species
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, ncol)
    c = slice(0, ncol)
    cols = np.flatnonzero(G.finite_columns(okf[:, c], okr[:, c], want[:, c], wp[:, c], wl[:, c]))
    scale = wp + wl
    okr_f = np.where(np.isfinite(okr), okr, 0.0)
    dT, dP, dJ, dn, dkf, dkr = (G.dev(a) for a in (atm.T, atm.P, atm.J, atm.n, okf, okr_f))
    for fused, chunk in ((1, 0), (0, 64)):
        h = xod.Network(net, device=0)
        h.tune(xod.XOD_TUNE_FUSED_KERNEL, fused)
        h.tune(xod.XOD_TUNE_CHUNK_COLS, chunk)
        ws = G.workspace(max(h.source_fused_workspace_bytes(ncol), h.source_workspace_bytes(ncol)))
        for stored in (False, True):
            d0, p0, l0 = G.empty(ns, ld), G.empty(ns, ld), G.empty(ns, ld)
            if stored:
                h.source(ncol, ld, dkf, dkr, dn, d0, p0, l0, workspace=ws)
            else:
                h.source_fused(ncol, ld, dT, dP, dJ, dn, d0, p0, l0, workspace=ws)
            what = "P/L over chunks (single-kernel %d, stored k %d)" % (fused, stored)
            G.check_sum(G.host(d0), want, scale, cols, what + " dn/dt")
            G.check_sum(G.host(p0), wp, scale, cols, what + " P")
            G.check_sum(G.host(l0), wl, scale, cols, what + " L")
            assert np.all(np.isnan(G.host(d0)[:, ncol:])) and np.all(np.isnan(G.host(p0)[:, ncol:]))
        h.check_status()
        h.close()


@pytest.mark.parametrize("seed", [11, 12, 13, 14, 15, 16])
def test_random_networks(xod, oracle, seed):
    """The seeded random networks of tests/test_kernel_emulation.py (odd segment lengths, reaction counts around
    the chunk size, irreversible reactions and Kooij forms mixed in, ragged column counts, cold and hot columns)
    through xod_rate_coeffs, xod_source_fused, xod_source and xod_jacobian, reaction-split or not."""
    from paper_2512_06729_b200 import synth
    rng = np.random.default_rng(seed)
    elements = ["H", "C", "O", "N", "S"][:int(rng.integers(2, 6))]
    ns = int(rng.integers(6, 40))
    nr = int(rng.integers(5, 330))
    net = synth.make_network(900 + seed, elements, ns, nr, inert=())
    flip = rng.random(net.n_reactions) < 0.3
    net.reversible = np.where(flip & (net.type != 3), 0, net.reversible).astype(np.uint8)
    net.t_ref = np.where(rng.random(net.n_reactions) < 0.3, 300.0, 1.0)
    n_layers = int(rng.integers(3, 45))
    atm = synth.make_atmosphere(1900 + seed, net, 1, n_layers, t_shift=(-300.0, 300.0))
    ncol, ld, ns = atm.ncol, atm.ld, net.n_species
    h = xod.Network(net, device=0)
    h.selfcheck()
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    dT, dP, dJ, dn = (G.dev(a) for a in (atm.T, atm.P, atm.J, atm.n))
    ws = G.workspace(max(h.source_fused_workspace_bytes(ncol), h.source_workspace_bytes(ncol), h.rate_coeffs_workspace_bytes(ncol)) + (8 << 20))
    kf, kr = G.empty(net.n_reactions, ld), G.empty(net.n_reactions, ld)
    h.rate_coeffs(ncol, ld, dT, dP, dJ, kf, kr, ws)
    G.check_k(G.host(kf)[:, :ncol], okf[:, :ncol], "random net %d k_f" % seed)
    G.check_k(G.host(kr)[:, :ncol], okr[:, :ncol], "random net %d k_r" % seed)
    assert np.all(G.host(kr)[net.reversible == 0, :ncol] == 0.0)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, ncol)
    okr_f = np.where(np.isfinite(okr), okr, 0.0)
    want_f, wpf, wlf = oracle.source(net, okf, okr_f, atm.n, ncol)
    dkf, dkr = G.dev(okf), G.dev(okr_f)
    for split in (0, 2):
        h.tune(xod.XOD_TUNE_SPLIT, split)
        d0 = G.empty(ns, ld)
        h.source_fused(ncol, ld, dT, dP, dJ, dn, d0, workspace=ws)
        G.check_sum_entries(G.host(d0), want, wp + wl, ncol, "random net %d xod_source_fused split %d" % (seed, split))
        d1 = G.empty(ns, ld)
        h.source(ncol, ld, dkf, dkr, dn, d1, workspace=ws)
        G.check_sum_entries(G.host(d1), want_f, wpf + wlf, ncol, "random net %d xod_source split %d" % (seed, split))
        assert np.all(np.isnan(G.host(d0)[:, ncol:])) and np.all(np.isnan(G.host(d1)[:, ncol:]))
    h.tune(xod.XOD_TUNE_SPLIT, 0)
    rp, col = h.jac_pattern()
    wj, sj = oracle.jacobian(net, okf, okr_f, atm.n, rp, col, ncol)
    for tiled in (1, 0):
        h.tune(xod.XOD_TUNE_JAC_TILED, tiled)
        jac = G.empty(h.nnz_jac, ld)
        h.jacobian(ncol, ld, dkf, dkr, dn, jac)
        G.check_sum_entries(G.host(jac), wj, sj, ncol, "random net %d xod_jacobian (tiled %d)" % (seed, tiled))
    h.check_status()
    h.close()


def test_network_too_large_for_the_fused_tables_and_its_jacobian(xod, oracle):
    """950 species: k_fused's tiles do not fit shared memory, so every call must take the multi-kernel pipeline
    (xod_network_fused_info says so); the tiled Jacobian still fits.  Ragged column count."""
    from paper_2512_06729_b200 import synth
    net = synth.make_network(777, ["H", "C", "O", "N", "S"], 950, 300, inert=())
    atm = synth.make_atmosphere(2777, net, 1, 19)
    h = xod.Network(net, device=0)
    assert h.fused_info()["enabled"] == 0 and h.jac_info()["enabled"] == 1
    ns, ld, ncol = net.n_species, atm.ld, atm.ncol
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, ncol)
    dT, dP, dJ, dn = (G.dev(a) for a in (atm.T, atm.P, atm.J, atm.n))
    ws = G.workspace(max(h.source_fused_workspace_bytes(ncol), h.source_workspace_bytes(ncol), h.rate_coeffs_workspace_bytes(ncol)))
    kf, kr = G.empty(net.n_reactions, ld), G.empty(net.n_reactions, ld)
    h.rate_coeffs(ncol, ld, dT, dP, dJ, kf, kr, ws)
    G.check_k(G.host(kf)[:, :ncol], okf[:, :ncol], "950 species k_f")
    G.check_k(G.host(kr)[:, :ncol], okr[:, :ncol], "950 species k_r")
    cols = np.arange(ncol)
    d0, p0, l0 = G.empty(ns, ld), G.empty(ns, ld), G.empty(ns, ld)
    h.source_fused(ncol, ld, dT, dP, dJ, dn, d0, p0, l0, workspace=ws)
    G.check_sum(G.host(d0), want, wp + wl, cols, "950 species dn/dt")
    G.check_sum(G.host(p0), wp, wp + wl, cols, "950 species P")
    G.check_sum(G.host(l0), wl, wp + wl, cols, "950 species L")
    d1 = G.empty(ns, ld)
    h.source(ncol, ld, G.dev(okf), G.dev(okr), dn, d1, workspace=ws)
    G.check_sum(G.host(d1), want, wp + wl, cols, "950 species dn/dt from stored k")
    rp, col = h.jac_pattern()
    wj, sj = oracle.jacobian(net, okf, okr, atm.n, rp, col, ncol)
    jac = G.empty(h.nnz_jac, ld)
    h.jacobian(ncol, ld, G.dev(okf), G.dev(okr), dn, jac)
    G.check_sum(G.host(jac), wj, sj, cols, "950 species Jacobian")
    h.check_status()
    h.close()


def test_network_without_reactions_and_its_jacobian(xod):
    """The empty reaction list: dn/dt, P, L and the Jacobian (pattern = the diagonal) are exact zeros; xod_rate_coeffs
    has nothing to write; padding columns stay untouched."""
    import torch
    from conftest import SimpleNet
    net = SimpleNet([[1], [2], [1]], np.zeros((3, 7)), np.zeros((3, 7)), [1000.0] * 3, [], [], [], [], np.zeros((0, 3)))
    h = xod.Network(net, device=0)
    ncol, ld = 37, 64
    T, P = G.dev(np.full(ld, 1200.0)), G.dev(np.full(ld, 1e5))
    n = G.dev(np.abs(np.random.default_rng(3).normal(size=(3, ld))) * 1e10)
    ws = G.workspace(max(h.source_fused_workspace_bytes(ncol), h.source_workspace_bytes(ncol)) + 4096)
    for pl in (False, True):
        d0, p0, l0 = G.empty(3, ld), G.empty(3, ld), G.empty(3, ld)
        h.source_fused(ncol, ld, T, P, None, n, d0, p0 if pl else None, l0 if pl else None, workspace=ws)
        outs = (d0, p0, l0) if pl else (d0,)
        for a in outs:
            got = G.host(a)
            assert np.all(got[:, :ncol] == 0.0) and np.all(np.isnan(got[:, ncol:]))
        d1 = G.empty(3, ld)
        h.source(ncol, ld, None, None, n, d1, workspace=ws)
        assert np.all(G.host(d1)[:, :ncol] == 0.0)
    jac = G.empty(h.nnz_jac, ld)
    h.jacobian(ncol, ld, None, None, n, jac)
    got = G.host(jac)
    assert h.nnz_jac == 3 and np.all(got[:, :ncol] == 0.0) and np.all(np.isnan(got[:, ncol:]))
    h.check_status()
    h.close()
