"""f4, the thermochemical-equilibrium composition (reading E1): the kernel
SOURCE executed on the CPU against the oracle, and the `-m gpu` parity tests through the C ABI.

The equilibrium composition is unique (a strictly convex minimisation), so the two sides are compared species by
species.  Tolerance: both iterate to a relative correction <= 1e-13, the kernel in fp64, the
oracle in long double; what remains is the rounding of the (n_e + 1) system, amplified by its condition number
(<= ~1e4 for these inputs after row scaling), which enters every species through sum_e a_ie pi_e with up to ~12 atoms:
relative 1e-9 on every n_i that lies inside the double range is asked, and the worst ratio is printed.  Independent of
the oracle, the result must conserve the element ratios and sum to P / (k_B T) to 1e-12."""
import ctypes as C

import numpy as np
import pytest

import gpu_common as G

KB = 1.380649e-16
TOL = 1e-9


def case(network, cfg, ncol_max, shift=0.0):
    from paper_2512_06729_b200 import synth
    net = synth.edge_network() if cfg == "edge" else network(cfg)
    atm = synth.edge_atmosphere(net) if cfg == "edge" else synth.config_atmosphere(cfg, net)
    ncol = min(atm.ncol, ncol_max)
    ld = (ncol + 31) // 32 * 32
    T = np.ascontiguousarray(atm.T[:ld]) + shift
    P = np.ascontiguousarray(atm.P[:ld])
    comp = np.asarray(net.composition, dtype=np.float64)
    n0 = np.abs(np.ascontiguousarray(atm.n[:, :ld])) + 1e-30      # the edge atmosphere has zero and negative densities
    b = comp.T @ n0
    b[np.asarray(net.composition).min(axis=0) < 0] = 0.0          # a signed column is the charge: neutral gas
    return net, T, P, np.ascontiguousarray(b), ncol, ld


def check(net, T, P, b, ncol, got, want, what):
    n, pi, iters = got
    wn, wit = want
    assert np.all(wit[:ncol] > 0), what + ": the oracle did not converge"
    assert np.all(iters[:ncol] > 0), what + ": not converged in columns %s" % np.flatnonzero(iters[:ncol] <= 0)[:8]
    g, w = n[:, :ncol], wn[:, :ncol]
    inside = w > 1e-250
    assert np.all(g[~inside] <= 1e-240) and np.all(g >= 0), what
    rel = np.abs(g[inside] - w[inside]) / w[inside]
    worst = float(rel.max())
    assert worst <= TOL, "%s: worst relative error %.2e" % (what, worst)
    ntot = P[:ncol] / (KB * T[:ncol])
    assert np.allclose(g.sum(0), ntot, rtol=1e-12, atol=0), what + ": sum n != P / (k_B T)"
    comp = np.asarray(net.composition, dtype=np.float64)
    have = comp.T @ g
    pos = b[:, :ncol].sum(0)
    ratio_err = np.abs(have / have[b[:, 0] > 0].sum(0) - b[:, :ncol] / pos).max()
    assert ratio_err <= 1e-12, "%s: element ratios off by %.2e" % (what, ratio_err)
    assert np.all(np.isnan(n[:, ncol:])) and np.all(iters[ncol:] == -7), what + ": padding columns written"
    # the element potentials reproduce every species (Lagrange conditions), G_i/RT from the oracle's thermo
    print("%s: %d columns, %d..%d iterations (oracle %d..%d), worst relative error %.2e, element ratios %.1e" % (
        what, ncol, iters[:ncol].min(), iters[:ncol].max(), wit[:ncol].min(), wit[:ncol].max(), worst, ratio_err))


def touched_by_underflow(net, n, ncol):
    """[species][column] mask: the species takes part in a reaction one of whose participants has an equilibrium
    density below the double range in that column.  There the balance q_f = q_r holds mathematically (k_r ~ 1e260
    times n ~ 1e-380) but cannot be formed in fp64 (n is returned as 0), so the kinetic cross-check skips it."""
    tiny = n[:, :ncol] < 1e-280
    out = np.zeros_like(tiny)
    for r in range(net.n_reactions):
        sp = [s for s in list(net.reactants[r]) + list(net.products[r]) if s >= 0]
        bad = tiny[sp].any(axis=0)
        for s in sp:
            out[s] |= bad
    return out


def run_emulated(net, T, P, b, ncol, ld, max_iter=0, tol=0.0):
    import os
    import subprocess
    import test_kernel_emulation as tk
    if not os.path.exists(tk.LIB) or any(os.path.getmtime(d) > os.path.getmtime(tk.LIB) for d in tk.DEPS):
        subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-shared", "-fPIC", "-I" + os.path.join(tk.EMU_DIR, "shim"),
                        "-o", tk.LIB] + tk.SOURCES, check=True)
    lib = C.CDLL(tk.LIB)
    d, keep = tk.descriptor(net)
    ne = np.asarray(net.composition).shape[1]
    n = np.full((net.n_species, ld), np.nan)
    pi = np.full((ne, ld), np.nan)
    iters = np.full(ld, -7, dtype=np.int32)
    rc = lib.emu_equilibrium(C.byref(d), C.c_int64(ncol), C.c_int64(ld), tk.ptr(T), tk.ptr(P), tk.ptr(b), C.c_int(max_iter),
                             C.c_double(tol), tk.ptr(n), tk.ptr(pi), tk.ptr(iters))
    assert rc == 0
    return n, pi, iters


@pytest.mark.parametrize("cfg,ncol_max,shift", [(1, 20, 0.0), (2, 70, 0.0), (2, 120, -550.0), ("edge", 40, 0.0), (3, 6, 0.0)])
def test_emulated_equilibrium_matches_oracle(oracle, network, cfg, ncol_max, shift):
    net, T, P, b, ncol, ld = case(network, cfg, ncol_max, shift)
    want = oracle.equilibrium(net, T, P, b, ncol)
    got = run_emulated(net, T, P, b, ncol, ld)
    check(net, T, P, b, ncol, got, want, "emulated xod_equilibrium config %s (T shift %+.0f K)" % (cfg, shift))


def coldest_config4_atmosphere(network):
    """The coldest of the 256 atmospheres of config 4 (T down to ~175 K at the top, |G/RT| of several hundred)."""
    from paper_2512_06729_b200 import synth
    net = network(3)
    atm = synth.config_atmosphere(4, net)
    a = int(np.argmin(atm.T[:atm.ncol])) // 150
    sl = slice(a * 150, (a + 1) * 150)
    ncol, ld = 150, 160
    T, P = np.full(ld, 1000.0), np.full(ld, 1.0e6)
    T[:150], P[:150] = atm.T[sl], atm.P[sl]
    n0 = np.ones((net.n_species, ld))
    n0[:, :150] = atm.n[:, sl]
    b = np.ascontiguousarray(np.asarray(net.composition, dtype=np.float64).T @ n0)
    return net, T, P, b, ncol, ld


def test_emulated_equilibrium_on_the_coldest_atmosphere_of_config_4(oracle, network):
    net, T, P, b, ncol, ld = coldest_config4_atmosphere(network)
    assert T[:ncol].min() < 200.0
    want = oracle.equilibrium(net, T, P, b, ncol)
    got = run_emulated(net, T, P, b, ncol, ld)
    check(net, T, P, b, ncol, got, want, "emulated xod_equilibrium, coldest atmosphere of config 4")


def test_emulated_equilibrium_reports_rejected_and_unconverged_columns(network):
    """Column 1 has a missing element, column 2 a negative temperature: iters = 0 and NaN; with max_iter = 3 nothing
    converges: iters = -3 and NaN; the other columns are unaffected by their neighbours."""
    net, T, P, b, ncol, ld = case(network, 1, 8)
    b2, T2 = b.copy(), T.copy()
    b2[1, 1] = 0.0
    T2[2] = -5.0
    n, pi, iters = run_emulated(net, T2, P, b2, ncol, ld)
    assert iters[1] == 0 and iters[2] == 0 and np.all(np.isnan(n[:, 1:3])) and np.all(np.isnan(pi[:, 1:3]))
    ref = run_emulated(net, T, P, b, ncol, ld)
    keep = [0, 3, 4, 5, 6, 7]
    assert np.array_equal(n[:, keep], ref[0][:, keep]) and np.all(iters[keep] > 0)
    n3, _, it3 = run_emulated(net, T, P, b, ncol, ld, max_iter=3)
    assert np.all(it3[:ncol] == -3) and np.all(np.isnan(n3[:, :ncol]))


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,ncol_max,shift", [(1, 20, 0.0), (2, 120, 0.0), (2, 120, -550.0), ("edge", 75, 0.0), (3, 150, 0.0),
                                                (4, 450, 0.0), ("cold4", 150, 0.0)])
def test_equilibrium_matches_oracle_on_gpu(oracle, network, cfg, ncol_max, shift):
    import torch
    assert torch.cuda.is_available(), "no CUDA device: the gpu tests need the B200 box (there is no CPU fallback)"
    from paper_2512_06729_b200 import binding, build
    build.build()
    net, T, P, b, ncol, ld = coldest_config4_atmosphere(network) if cfg == "cold4" else case(network, cfg, ncol_max, shift)
    want = oracle.equilibrium(net, T, P, b, ncol)
    h = binding.Network(net, device=0)
    ne = np.asarray(net.composition).shape[1]
    n, pi = G.empty(net.n_species, ld), G.empty(ne, ld)
    iters = torch.full((ld,), -7, dtype=torch.int32, device="cuda")
    h.equilibrium(ncol, ld, G.dev(T), G.dev(P), G.dev(b), n, pi, iters)
    h.check_status()
    got = (G.host(n), G.host(pi), iters.cpu().numpy())
    check(net, T, P, b, ncol, got, want, "xod_equilibrium config %s (T shift %+.0f K)" % (cfg, shift))
    if np.any((np.asarray(net.reversible) == 0) & (np.asarray(net.type) != 3)):
        h.close()
        return        # one-way thermal reactions (the edge network) are not balanced at equilibrium: no kinetic cross-check
    # the kinetics agree: without photolysis dn/dt vanishes at the returned composition (xod_source_fused vs its own P + L scale)
    J = torch.zeros((max(net.n_photo, 1), ld), dtype=torch.float64, device="cuda")
    d = G.empty(net.n_species, ld)
    ws = G.workspace(h.source_fused_workspace_bytes(ncol, prod_loss=False))
    h.source_fused(ncol, ld, G.dev(T), G.dev(P), J, n, d, workspace=ws)
    kf, kr = oracle.rate_coeffs(net, T, P, np.zeros((net.n_photo, ld)), ncol)
    _, wp, wl = oracle.source(net, kf, kr, got[0], ncol)
    scale = (wp + wl)[:, :ncol]
    big = np.isfinite(scale) & (scale > 1e-200) & ~touched_by_underflow(net, got[0], ncol)
    assert big.any()
    assert np.all(np.abs(G.host(d)[:, :ncol])[big] <= 1e-7 * scale[big])
    h.close()
