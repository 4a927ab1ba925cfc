"""f3, the molecular-diffusion transport terms: the kernel SOURCE executed on the CPU
against the oracle, and the `-m gpu` parity tests through the C ABI.

Tolerance: tr is a sum of up to four products, each holding d = D/(2 dz^2) (gravity term - thermal term); the bar is
|tr - oracle| <= 1e-12 x S with S the same sum taken over absolute values (both parts of d and all four products), which
the test forms independently with numpy."""
import ctypes as C

import numpy as np
import pytest

import gpu_common as G

K_B = 1.380649e-16


def inputs(network, cfg, n_atm, seed=61):
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net, n_atm)
    tr = synth.make_transport(seed, net, atm)
    return net, atm, tr


def scale(net, atm, t):
    """sum of |terms| of Eq. 3-4 per (species, column)."""
    L, A = atm.meta["n_layers"], atm.meta["n_atm"]
    ns, ncol = net.n_species, atm.ncol
    S = np.zeros((ns, atm.ld))
    n, T, N, D = atm.n, atm.T, t["n_gas"], t["D"]
    for a in range(A):
        h = t["dz"][a]
        for k in range(L):
            c = a * L + k
            for sgn in (+1, -1):
                if not (0 <= k + sgn < L):
                    continue
                cn = c + sgn
                Th, Nh, Dh = 0.5 * (T[c] + T[cn]), 0.5 * (N[c] + N[cn]), 0.5 * (D[:, c] + D[:, cn])
                dabs = Dh / (2 * h * h) * (np.abs(t["mbar"][a] - t["mass"]) * t["grav"][a] * h / (K_B * Th) + np.abs(t["alpha_T"]) / Th * abs(T[cn] - T[c]))
                if sgn > 0:      # - d+ (N+/N_{k+1}) n_{k+1} - d+ (N+/N_k) n_k
                    S[:, c] += dabs * (Nh / N[cn] * np.abs(n[:, cn]) + Nh / N[c] * np.abs(n[:, c]))
                else:            # + d- (N-/N_k) n_k + d- (N-/N_k) n_{k-1}
                    S[:, c] += dabs * (Nh / N[c] * np.abs(n[:, c]) + Nh / N[c] * np.abs(n[:, cn]))
    return S


def check(got, want, S, ncol, what):
    err = np.abs(got[:, :ncol] - want[:, :ncol])
    assert np.all(err <= 1e-12 * S[:, :ncol]), "%s: worst ratio %.2e" % (what, float((err / np.maximum(S[:, :ncol], 1e-300)).max()))
    assert np.all(np.isnan(got[:, ncol:])), what + ": padding columns written"
    nz = S[:, :ncol] > 0
    print("%s: %d x %d values, worst |err| / sum|terms| = %.2e" % (what, got.shape[0], ncol, float((err[nz] / S[:, :ncol][nz]).max()) if nz.any() else 0.0))


def oracle_tr(oracle, atm, t):
    return oracle.transport(atm.n, atm.T, t["n_gas"], t["D"], t["mass"], t["alpha_T"], t["mbar"], t["grav"], t["dz"],
                            atm.meta["n_atm"], atm.meta["n_layers"])


@pytest.mark.parametrize("cfg,n_atm,spb", [(1, 1, 12), (1, 7, 5), (2, 3, 16)])
def test_emulated_transport_matches_oracle(oracle, network, cfg, n_atm, spb):
    import test_kernel_emulation as tk
    net, atm, t = inputs(network, cfg, n_atm)
    want = oracle_tr(oracle, atm, t)
    import os
    import subprocess
    if not os.path.exists(tk.LIB) or any(os.path.getmtime(d) > os.path.getmtime(tk.LIB) for d in tk.DEPS):
        subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-shared", "-fPIC", "-I" + os.path.join(tk.EMU_DIR, "shim"),
                        "-o", tk.LIB] + tk.SOURCES, check=True)
    lib = C.CDLL(tk.LIB)
    got = np.full((net.n_species, atm.ld), np.nan)
    c = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    arrs = [c(atm.n), c(atm.T), c(t["n_gas"]), c(t["D"]), c(t["mass"]), c(t["alpha_T"]), c(t["mbar"]), c(t["grav"]), c(t["dz"])]
    rc = lib.emu_transport(C.c_int(net.n_species), C.c_int64(atm.meta["n_atm"]), C.c_int64(atm.meta["n_layers"]), C.c_int64(atm.ld),
                           *[tk.ptr(x) for x in arrs], tk.ptr(got), C.c_int(spb))
    assert rc == 0
    check(got, want, scale(net, atm, t), atm.ncol, "emulated xod_transport config %d, %d atmospheres" % (cfg, n_atm))


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,n_atm", [(1, 7), (2, 3), (5, 4)])
def test_transport_matches_oracle_on_gpu(oracle, network, cfg, n_atm):
    import torch
    assert torch.cuda.is_available(), "no CUDA device: the gpu tests need the B200 box (there is no CPU fallback)"
    from paper_2512_06729_b200 import binding, build
    build.build()
    net, atm, t = inputs(network, cfg, n_atm)
    want = oracle_tr(oracle, atm, t)
    h = binding.Network(net, device=0)
    tr = G.empty(net.n_species, atm.ld)
    h.transport(atm.meta["n_atm"], atm.meta["n_layers"], atm.ld, G.dev(atm.n), G.dev(atm.T), G.dev(t["n_gas"]), G.dev(t["D"]),
                G.dev(t["mass"]), G.dev(t["alpha_T"]), G.dev(t["mbar"]), G.dev(t["grav"]), G.dev(t["dz"]), tr)
    h.check_status()
    check(G.host(tr), want, scale(net, atm, t), atm.ncol, "xod_transport config %d, %d atmospheres" % (cfg, n_atm))
    h.close()


@pytest.mark.parametrize("n_layers", [1, 2, 3])
def test_emulated_transport_on_the_thinnest_atmospheres(oracle, network, n_layers):
    """One layer (both boundaries at once: no term survives), two layers (every layer touches a
    boundary) and three; five atmospheres side by side, so neighbours in memory belong to other atmospheres."""
    import test_kernel_emulation as tk
    from paper_2512_06729_b200 import synth
    net = network(1)
    atm = synth.make_atmosphere(2401, net, 5, n_layers)
    t = synth.make_transport(62, net, atm)
    want = oracle_tr(oracle, atm, t)
    lib = C.CDLL(tk.LIB)
    got = np.full((net.n_species, atm.ld), np.nan)
    c = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    arrs = [c(atm.n), c(atm.T), c(t["n_gas"]), c(t["D"]), c(t["mass"]), c(t["alpha_T"]), c(t["mbar"]), c(t["grav"]), c(t["dz"])]
    rc = lib.emu_transport(C.c_int(net.n_species), C.c_int64(5), C.c_int64(n_layers), C.c_int64(atm.ld),
                           *[tk.ptr(x) for x in arrs], tk.ptr(got), C.c_int(4))
    assert rc == 0
    check(got, want, scale(net, atm, t), atm.ncol, "emulated xod_transport, %d layer(s)" % n_layers)
    if n_layers == 1:
        assert np.all(got[:, :atm.ncol] == 0.0)
