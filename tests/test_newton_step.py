"""f1, the batched implicit step: host-side symbolic factorisation, the kernel
SOURCE executed on CPU threads (tests/kernel_emu) against the oracle, and the `-m gpu` parity tests through
the C ABI.

Tolerance (derived from the arithmetic): both sides solve (I - dt Jac) delta = b in fp64-or-better; the library
eliminates WITHOUT pivoting in a fixed minimum-degree order (as DLSODES' sparse solver does), the oracle with
partial pivoting in long double.  For a matrix of condition number kappa the two solutions differ by about
kappa eps ||delta||; the tests pick dt = stiffness / max_i |Jac_ii| so that kappa stays below ~1e6 and compare
|delta_lib - delta_oracle| <= 1e-9 max_i |delta_oracle| per column, plus the normwise residual of the library's
delta in the oracle's system, ||A delta - b|| <= 1e-11 (||A|| ||delta|| + ||b||), which holds at any kappa."""
import ctypes as C

import numpy as np
import pytest

import gpu_common as G
from paper_2512_06729_b200 import binding

TOL_DELTA = 1e-9
TOL_RESID = 1e-11


def lu_handle(net, device=-1):
    return binding.Network(net, device=device, flags=binding.XOD_FLAG_BUILD_LU)


def case(network, oracle, cfg, stiffness, ncol_max, seed=4):
    """network, k_f, k_r, n_old, dt (per column, = stiffness / fastest loss frequency), a perturbed iterate y."""
    from paper_2512_06729_b200 import synth
    net = synth.edge_network() if cfg == "edge" else network(cfg)
    atm = synth.edge_atmosphere(net) if cfg == "edge" else synth.config_atmosphere(cfg, net)
    ncol = min(atm.ncol, ncol_max)
    ld = (ncol + 31) // 32 * 32
    T = atm.T[:ld].copy()
    if cfg == "edge":
        T[T < 400.0] = 900.0           # keep k_r inside the double range: the solve needs finite inputs
    kf, kr = oracle.rate_coeffs(net, T, atm.P[:ld], atm.J[:, :ld], ncol)
    n = np.ascontiguousarray(atm.n[:, :ld])
    n = np.abs(n)                       # the edge atmosphere carries a negative density; keep the test matrix benign
    dt = np.ones(ld)
    for c in range(ncol):
        d, _ = oracle.jacobian_dense(net, kf, kr, n, c)
        dt[c] = stiffness / np.abs(np.diag(d)).max()
    y = n * 10 ** np.random.default_rng(seed).uniform(-0.1, 0.1, size=n.shape)
    return net, kf, kr, n, dt, y, ncol, ld


def compare(oracle, net, kf, kr, n, dt, y, ncol, got_delta, got_y, what):
    want_delta, want_y = oracle.newton_step(net, kf, kr, n, dt, y, ncol)
    worst_d = worst_r = 0.0
    for c in range(ncol):
        scale = np.abs(want_delta[:, c]).max()
        if scale == 0.0:                                  # e.g. a column of zero densities: nothing may move
            assert np.all(got_delta[:, c] == 0.0), what
            continue
        worst_d = max(worst_d, float(np.abs(got_delta[:, c] - want_delta[:, c]).max() / scale))
        A, b = oracle.newton_system(net, kf, kr, n, dt, y, c)
        r = A @ got_delta[:, c] - b
        worst_r = max(worst_r, float(np.abs(r).max() / (np.abs(A).sum(axis=1).max() * np.abs(got_delta[:, c]).max() + np.abs(b).max())))
    assert worst_d <= TOL_DELTA, "%s: delta differs by %.2e of its largest component" % (what, worst_d)
    assert worst_r <= TOL_RESID, "%s: normwise residual %.2e" % (what, worst_r)
    assert np.all(np.abs(got_y[:, :ncol] - (y[:, :ncol] + got_delta[:, :ncol])) <= 4e-16 * (np.abs(y[:, :ncol]) + np.abs(got_delta[:, :ncol])))
    print("%s: %d columns, worst |delta - oracle| / max|delta| = %.2e, worst normwise residual = %.2e" % (what, ncol, worst_d, worst_r))
    return worst_d, worst_r


# ------------------------------------------------------------------------------- host: symbolic factorisation
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_symbolic_lu_is_the_elimination_closure_of_the_jacobian_pattern(network, cfg):
    """Brute force on a dense boolean matrix: permute the Jacobian pattern by `perm`, eliminate in order with no
    pivoting, and compare the filled pattern row by row; rows sorted, diagonal present, pattern symmetric."""
    net = network(cfg)
    h = lu_handle(net)
    info = h.lu_info()
    assert info["enabled"] == 1
    perm, rp, col = h.lu_pattern()
    ns = net.n_species
    assert sorted(perm.tolist()) == list(range(ns))
    jrp, jcol = h.jac_pattern()
    pos = np.empty(ns, dtype=np.int64)
    pos[perm] = np.arange(ns)
    m = np.zeros((ns, ns), dtype=bool)
    rows = np.repeat(np.arange(ns), np.diff(jrp))
    m[pos[rows], pos[jcol]] = True
    for k in range(ns):                                   # symbolic Gaussian elimination
        below = np.flatnonzero(m[k + 1:, k]) + k + 1
        right = np.flatnonzero(m[k, k + 1:]) + k + 1
        if below.size and right.size:
            m[np.ix_(below, right)] = True
    got = np.zeros_like(m)
    for p in range(ns):
        c = col[rp[p]:rp[p + 1]]
        assert np.all(np.diff(c) > 0) and p in c
        got[p, c] = True
    assert np.array_equal(got, m)
    assert np.array_equal(got, got.T)
    assert info["nnz_lu"] == int(m.sum()) and info["max_row"] == int(m.sum(axis=1).max())
    assert info["updates"] == sum(int(m[k + 1:, k].sum()) * int(m[k, k + 1:].sum()) for k in range(ns))
    print("config %d: nnz(Jac) %d -> nnz(L+U) %d, %d multiply-add updates per factorisation" % (cfg, jcol.size, info["nnz_lu"], info["updates"]))
    # the update and block schedules, decoded on the host as k_lu_factor decodes them: every (row, pivot) pair once,
    # pivots ascending inside a block, target slots holding the right columns
    h.selfcheck()
    assert 1 <= info["block_rows"] <= 6 and info["steps"] <= info["pairs"]
    # a pivot's U row is read once per block instead of once per row: between updates / block_rows and updates
    assert info["updates"] / info["block_rows"] <= info["u_loads"] <= info["updates"]


def test_networks_without_the_flag_have_no_lu_tables(network):
    h = binding.Network(network(1), device=-1)
    assert h.lu_info()["enabled"] == 0 and h.newton_workspace_bytes(10) == 0
    with pytest.raises(binding.XodError):
        h.lu_pattern()


# ------------------------------------------------------------------------------- kernel source on CPU threads
def run_emulated(net, kf, kr, n, dt, y, ncol, ld):
    import test_kernel_emulation as tk
    import os
    import subprocess
    if not os.path.exists(tk.LIB) or any(os.path.getmtime(d) > os.path.getmtime(tk.LIB) for d in tk.DEPS):
        subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-shared", "-fPIC", "-I" + os.path.join(tk.EMU_DIR, "shim"),
                        "-o", tk.LIB] + tk.SOURCES, check=True)
    lib = C.CDLL(tk.LIB)
    d, keep = tk.descriptor(net)
    y2 = np.ascontiguousarray(y).copy()
    delta = np.full_like(y2, np.nan)
    rc = lib.emu_newton_step(C.byref(d), C.c_int64(ncol), C.c_int64(ld), tk.ptr(kf), tk.ptr(kr), tk.ptr(n), tk.ptr(dt),
                             tk.ptr(y2), tk.ptr(delta))
    assert rc == 0
    return delta, y2


@pytest.mark.parametrize("cfg,stiffness,ncol_max", [(1, 1.0, 20), (1, 1e3, 20), (2, 30.0, 40), ("edge", 10.0, 37)])
def test_emulated_newton_step_matches_oracle(oracle, network, cfg, stiffness, ncol_max):
    net, kf, kr, n, dt, y, ncol, ld = case(network, oracle, cfg, stiffness, ncol_max)
    delta, y_new = run_emulated(net, kf, kr, n, dt, y, ncol, ld)
    compare(oracle, net, kf, kr, n, dt, y, ncol, delta, y_new, "emulated xod_newton_step, config %s, stiffness %g" % (cfg, stiffness))
    assert np.all(np.isnan(delta[:, ncol:])) and np.array_equal(y_new[:, ncol:], y[:, ncol:]), "padding columns touched"


def test_emulated_newton_iteration_reaches_the_backward_euler_root(oracle, network):
    """Iterating the emulated step drives F(y) = y - n_old - dt f(y) to round-off (the oracle's own iteration is
    pinned to converge quadratically in test_oracle_newton.py)."""
    net, kf, kr, n, dt, y, ncol, ld = case(network, oracle, 2, 30.0, 20)
    y = n.copy()
    for it in range(7):
        _, y = run_emulated(net, kf, kr, n, dt, y, ncol, ld)
    f, prod, loss = oracle.source(net, kf, kr, y, ncol)
    F = (y - n - dt[None, :] * f)[:, :ncol]
    scale = (np.abs(y) + np.abs(n) + dt[None, :] * (prod + loss))[:, :ncol]
    assert np.all(np.abs(F) <= 1e-13 * scale)


# ------------------------------------------------------------------------------- GPU parity through the C ABI
@pytest.mark.gpu
@pytest.mark.parametrize("cfg,stiffness,ncol_max", [(1, 1.0, 20), (2, 30.0, 120), ("edge", 10.0, 75), (5, 10.0, 40)])
def test_newton_step_matches_oracle_on_gpu(oracle, network, cfg, stiffness, ncol_max):
    import torch
    assert torch.cuda.is_available(), "no CUDA device: the gpu tests need the B200 box (there is no CPU fallback)"
    from paper_2512_06729_b200 import build
    build.build()
    net, kf, kr, n, dt, y, ncol, ld = case(network, oracle, cfg, stiffness, ncol_max)
    h = lu_handle(net, device=0)
    ws = G.workspace(h.newton_workspace_bytes(ncol))
    dy, dd = G.dev(y), G.empty(net.n_species, ld)
    h.newton_step(ncol, ld, G.dev(kf), G.dev(kr), G.dev(n), G.dev(dt), dy, dd, workspace=ws)
    h.check_status()
    delta, y_new = G.host(dd), G.host(dy)
    compare(oracle, net, kf, kr, n, dt, y, ncol, delta, y_new, "xod_newton_step, config %s, stiffness %g" % (cfg, stiffness))
    assert np.all(np.isnan(delta[:, ncol:])) and np.array_equal(y_new[:, ncol:], y[:, ncol:])
    h.close()


@pytest.mark.gpu
def test_newton_step_several_column_chunks_on_gpu(oracle, network):
    """2 500 columns = two passes of 2 368 + 132 (the call works through the batch in passes of 148 x 16 columns to
    bound its workspace): columns from both passes and the ragged tail against the oracle."""
    import torch
    assert torch.cuda.is_available()
    from paper_2512_06729_b200 import synth
    net = network(2)
    atm = synth.make_atmosphere(71, net, 1, 2500)
    ncol, ld = atm.ncol, atm.ld
    kf, kr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    n = atm.n
    rng = np.random.default_rng(8)
    dt = np.ones(ld)                     # reading N2: parity of the unpivoted solve holds for dt = stiffness / max |Jac_ii|
    for c in range(ncol):
        d, _ = oracle.jacobian_dense(net, kf, kr, n, c)
        dt[c] = 30.0 / np.abs(np.diag(d)).max()
    y = n * 10 ** rng.uniform(-0.1, 0.1, size=n.shape)
    h = lu_handle(net, device=0)
    ws = G.workspace(h.newton_workspace_bytes(ncol))
    dy, dd = G.dev(y), G.empty(net.n_species, ld)
    h.newton_step(ncol, ld, G.dev(kf), G.dev(kr), G.dev(n), G.dev(dt), dy, dd, workspace=ws)
    h.check_status()
    delta, y_new = G.host(dd), G.host(dy)
    cols = np.array([0, 31, 32, 2367, 2368, 2369, 2399, 2400, 2499])
    sub = lambda a: np.ascontiguousarray(a[..., cols])
    compare(oracle, net, sub(kf), sub(kr), sub(n), sub(dt), sub(y), cols.size, sub(delta), sub(y_new), "xod_newton_step over column chunks")
    assert np.all(np.isfinite(delta[:, :ncol])) and np.all(np.isnan(delta[:, ncol:]))
    h.close()
