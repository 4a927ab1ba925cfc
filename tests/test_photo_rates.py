"""f2, the photolysis rate constants: the kernel SOURCE executed on CPU threads
against the oracle, and the `-m gpu` parity tests through the C ABI.

Tolerance: every term of k_ph is >= 0, so the sums are well conditioned; the only amplified rounding is the
exponent of exp(-tau/mu), |tau/mu| eps <= 745 x 1.1e-16 for any result that is not yet subnormal.  Bar: relative
1e-12 where the oracle is a normal number; |value| <= 1e-300 where the oracle underflows (the rule of reading R5)."""
import ctypes as C

import numpy as np
import pytest

import gpu_common as G


def inputs(network, cfg, n_atm, n_bins, seed=51, diffuse=True):
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net, n_atm)
    ph = synth.make_photo(seed, net, n_bins=n_bins)
    dz, j0, jd, mu, tf = synth.make_irradiation(seed + 1, net, atm, ph, with_diffuse=diffuse)
    return net, atm, ph, dz, j0, jd, mu, tf


def check(got, want, ncol, what):
    g, w = got[:, :ncol], want[:, :ncol]
    tiny = np.abs(w) < 2.2250738585072014e-308
    assert np.all(np.abs(g[tiny]) <= 1e-300), what
    rel = np.abs(g[~tiny] - w[~tiny]) / np.abs(w[~tiny])
    worst = float(rel.max()) if rel.size else 0.0
    assert worst <= 1e-12, "%s: max relative error %.3e" % (what, worst)
    assert np.all(np.isnan(got[:, ncol:])), what + ": padding columns written"
    print("%s: %d x %d values, %d underflowed, worst relative error %.2e" % (what, g.shape[0], ncol, int(tiny.sum()), worst))


def run_emulated(net, atm, ph, dz, j0, jd, mu, tf):
    import test_kernel_emulation as tk
    import os
    import subprocess
    if not os.path.exists(tk.LIB) or any(os.path.getmtime(d) > os.path.getmtime(tk.LIB) for d in tk.DEPS):
        subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-shared", "-fPIC", "-I" + os.path.join(tk.EMU_DIR, "shim"),
                        "-o", tk.LIB] + tk.SOURCES, check=True)
    lib = C.CDLL(tk.LIB)
    J = np.full((net.n_photo, atm.ld), np.nan)
    c = lambda a, dt=np.float64: np.ascontiguousarray(a, dtype=dt)
    ab, se, sp, dl = c(ph.abs_species, np.int32), c(ph.sigma_ext), c(ph.sigma_ph), c(ph.dlambda)
    n, dz, j0, mu, tf = c(atm.n), c(dz), c(j0), c(mu), c(tf)
    jd = None if jd is None else c(jd)
    rc = lib.emu_photo_rates(C.c_int(net.n_species), C.c_int(net.n_photo), C.c_int(ph.n_bins), C.c_int(ab.shape[0]), tk.ptr(ab),
                             tk.ptr(se), tk.ptr(sp), tk.ptr(dl), C.c_int64(atm.meta["n_atm"]), C.c_int64(atm.meta["n_layers"]),
                             C.c_int64(atm.ld), tk.ptr(n), tk.ptr(dz), tk.ptr(j0), tk.ptr(jd), tk.ptr(mu), tk.ptr(tf), tk.ptr(J))
    assert rc == 0
    return J


@pytest.mark.parametrize("cfg,n_atm,n_bins,diffuse", [(1, 3, 70, True), (2, 1, 45, False), (2, 2, 130, True)])
def test_emulated_photo_rates_match_oracle(oracle, network, cfg, n_atm, n_bins, diffuse):
    """Ragged in every dimension: bins, photolysis rows and columns that are not multiples of the 64 x 64 x 16 tiles
    or of the 32-bin groups; several atmospheres (each scanned from its own top); with and without J_diff."""
    net, atm, ph, dz, j0, jd, mu, tf = inputs(network, cfg, n_atm, n_bins, diffuse=diffuse)
    want = oracle.photo_rates(ph, atm.n, dz, j0, jd, mu, tf, atm.meta["n_atm"], atm.meta["n_layers"])
    got = run_emulated(net, atm, ph, dz, j0, jd, mu, tf)
    check(got, want, atm.ncol, "emulated xod_photo_rates config %d" % cfg)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,n_atm,n_bins,diffuse", [(1, 3, 70, True), (2, 2, 1000, True), (5, 4, 2000, False)])
def test_photo_rates_match_oracle_on_gpu(oracle, network, cfg, n_atm, n_bins, diffuse):
    import torch
    assert torch.cuda.is_available(), "no CUDA device: the gpu tests need the B200 box (there is no CPU fallback)"
    from paper_2512_06729_b200 import binding, build
    build.build()
    net, atm, ph, dz, j0, jd, mu, tf = inputs(network, cfg, n_atm, n_bins, diffuse=diffuse)
    want = oracle.photo_rates(ph, atm.n, dz, j0, jd, mu, tf, atm.meta["n_atm"], atm.meta["n_layers"])
    h = binding.Network(net, device=0)
    p = binding.Photo(h, ph)
    J = G.empty(net.n_photo, atm.ld)
    ws = G.workspace(p.workspace_bytes(atm.ncol))
    p.rates(atm.meta["n_atm"], atm.meta["n_layers"], atm.ld, G.dev(atm.n), G.dev(dz), G.dev(j0), None if jd is None else G.dev(jd),
            G.dev(mu), G.dev(tf), J, ws)
    h.check_status()
    check(G.host(J), want, atm.ncol, "xod_photo_rates config %d, %d bins" % (cfg, n_bins))
    # the result is the J input of the source term: feed it through xod_source_fused and compare with the oracle's chain
    dndt = G.empty(net.n_species, atm.ld)
    ws2 = G.workspace(h.source_fused_workspace_bytes(atm.ncol))
    h.source_fused(atm.ncol, atm.ld, G.dev(atm.T), G.dev(atm.P), J, G.dev(atm.n), dndt, workspace=ws2)
    d_want, wp, wl = oracle.source_from_state(net, atm.T, atm.P, want, atm.n, atm.ncol)
    G.check_sum(G.host(dndt), d_want, wp + wl, np.arange(atm.ncol), "dn/dt with computed J")
    p.close()
    h.close()


def test_photo_create_validates_its_tables(network):
    from paper_2512_06729_b200 import binding, synth
    net = network(1)
    h = binding.Network(net, device=-1)
    ph = synth.make_photo(5, net, n_bins=20)
    binding.Photo(h, ph).close()
    bad = synth.make_photo(5, net, n_bins=20)
    bad.abs_species = bad.abs_species.copy()
    bad.abs_species[0] = net.n_species
    with pytest.raises(binding.XodError):
        binding.Photo(h, bad)
    bad2 = synth.make_photo(5, net, n_bins=20)
    bad2.sigma_ph = -bad2.sigma_ph
    bad2.sigma_ph[0, 0] = -1.0
    with pytest.raises(binding.XodError):
        binding.Photo(h, bad2)


@pytest.mark.parametrize("n_abs,n_layers,n_bins", [(0, 7, 5), (3, 1, 33), (2, 40, 1)])
def test_emulated_photo_rates_degenerate_shapes(oracle, network, n_abs, n_layers, n_bins):
    """No absorber at all (a transparent atmosphere: the contraction over absorbers has K = 0), atmospheres of a
    single layer (tau = half the layer's own slab), a single wavelength bin."""
    from paper_2512_06729_b200 import synth
    net = network(1)
    atm = synth.make_atmosphere(2301, net, 3, n_layers)
    ph = synth.make_photo(77, net, n_bins=n_bins, n_abs=max(n_abs, 1))
    if n_abs == 0:
        ph.abs_species = np.zeros(0, dtype=np.int32)
        ph.sigma_ext = np.zeros((0, n_bins))
    dz, j0, jd, mu, tf = synth.make_irradiation(78, net, atm, ph, with_diffuse=False)
    want = oracle.photo_rates(ph, atm.n, dz, j0, jd, mu, tf, 3, n_layers)
    got = run_emulated(net, atm, ph, dz, j0, jd, mu, tf)
    check(got, want, atm.ncol, "emulated xod_photo_rates, %d absorbers, %d layers, %d bins" % (n_abs, n_layers, n_bins))
    if n_abs == 0:      # transparent: k_ph = t_f sum_b J0 sigma dlambda in every layer (PAPER.md:207 with tau = 0)
        flat = (np.asarray(tf)[:, None] * (np.asarray(j0) * ph.dlambda[None, :]) @ ph.sigma_ph.T)     # [atm][photo]
        for a in range(3):
            assert np.allclose(got[:, a * n_layers:(a + 1) * n_layers], flat[a][:, None], rtol=1e-12, atol=0)
