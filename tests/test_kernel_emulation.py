"""The CUDA kernel SOURCE executed on CPU threads (tests/kernel_emu: one std::thread per CUDA thread,
std::barrier as __syncthreads, blocks one after another) against the oracle.  No GPU needed: this
checks the kernels' indexing, table decoding, chunk schedule and arithmetic as written, for the fused
source kernel (both modes), its reaction-split/combine path, the persistent tile loop and the
rate-coefficient kernel.  It cannot see races or memory-model effects; the `-m gpu` tests do that."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from conftest import ROOT
import gpu_common as G

from paper_2512_06729_b200 import binding

EMU_DIR = os.path.join(ROOT, "tests", "kernel_emu")
CSRC = os.path.join(ROOT, "paper_2512_06729_b200", "csrc")
LIB = os.path.join(EMU_DIR, "libxod_emu.so")
SOURCES = [os.path.join(EMU_DIR, "emu.cpp")] + [os.path.join(CSRC, f) for f in ("pack.cpp", "pack_fused.cpp", "pack_jac.cpp", "pack_lu.cpp", "pack_path.cpp")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("fused.cuh", "rates2.cuh", "kernels.cuh", "jac_tiled.cuh", "newton.cuh", "photo.cuh", "transport.cuh", "pathway.cuh", "equil.cuh", "sched.cuh", "xod_math.cuh", "xod_internal.h")] + [
    os.path.join(EMU_DIR, "shim", "cuda_runtime.h"), os.path.join(EMU_DIR, "shim", "xod_cta.cuh")]


@pytest.fixture(scope="module")
def emu():
    if not os.path.exists(LIB) or any(os.path.getmtime(d) > os.path.getmtime(LIB) for d in DEPS):
        subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-shared", "-fPIC",
                        "-I" + os.path.join(EMU_DIR, "shim"), "-o", LIB] + SOURCES, check=True)
    return C.CDLL(LIB)


def descriptor(net):
    keep = dict(
        composition=np.ascontiguousarray(net.composition, dtype=np.int32), nasa_lo=np.ascontiguousarray(net.nasa_lo),
        nasa_hi=np.ascontiguousarray(net.nasa_hi), t_mid=np.ascontiguousarray(net.t_mid),
        type=np.ascontiguousarray(net.type, dtype=np.int32), reactants=np.ascontiguousarray(net.reactants, dtype=np.int32),
        products=np.ascontiguousarray(net.products, dtype=np.int32), reversible=np.ascontiguousarray(net.reversible, dtype=np.uint8),
        arrh=np.ascontiguousarray(net.arrh), arrh_low=np.ascontiguousarray(net.arrh_low),
        troe_fc=np.ascontiguousarray(net.troe_fc), t_ref=np.ascontiguousarray(net.t_ref))
    ns, ne = keep["composition"].shape
    d = binding._Desc(ns, ne, keep["type"].shape[0], *[C.c_void_p(keep[k].ctypes.data) for k in (
        "composition", "nasa_lo", "nasa_hi", "t_mid", "type", "reactants", "products", "reversible", "arrh",
        "arrh_low", "troe_fc", "t_ref")], 0)
    return d, keep


def ptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


def run_fused(emu, net, atm, ncol, kf=None, kr=None, grid=2, nsplit=1):
    d, keep = descriptor(net)
    out = np.full((net.n_species, atm.ld), np.nan)
    rc = emu.emu_source_fused(C.byref(d), C.c_int64(ncol), C.c_int64(atm.ld), ptr(atm.T), ptr(atm.P), ptr(atm.J),
                              ptr(kf), ptr(kr), ptr(atm.n), ptr(out), C.c_int(grid), C.c_int(nsplit))
    assert rc == 0
    return out


def check(got, want, scale, ncol, what):
    err = np.abs(got[:, :ncol] - want[:, :ncol])
    assert np.all(err <= 1e-11 * scale[:, :ncol]), what
    assert np.all(np.isnan(got[:, ncol:])), what + ": padding columns written"


@pytest.mark.parametrize("cfg,grid,nsplit", [(1, 1, 1), (1, 2, 1), (2, 3, 1), (2, 5, 3)])
def test_fused_kernel_source_matches_oracle(emu, oracle, network, cfg, grid, nsplit):
    """k_fused<false> (a1-a8): config 1 (one chunk, 2 tiles) and config 2 (3 chunks, 8 tiles) with fewer
    blocks than work items (persistent loop) and with the chunks of a tile split over blocks."""
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    want, wp, wl = oracle.source_from_state(net, atm.T, atm.P, atm.J, atm.n, atm.ncol)
    got = run_fused(emu, net, atm, atm.ncol, grid=grid, nsplit=nsplit)
    check(got, want, wp + wl, atm.ncol, "emulated k_fused config %d" % cfg)


def test_fused_kernel_source_on_the_594_species_network(emu, oracle, network):
    """The production network (config 3: 33 chunks of 240 reactions, 609 accumulator rows with hub-species extras,
    227 KB of shared memory) on 20 columns = one full and one ragged tile, chunks split 3 ways, fewer blocks than
    work items -- the launch shape of the few-column path."""
    from paper_2512_06729_b200 import synth
    net = network(3)
    atm = synth.make_atmosphere(2033, net, 1, 20)
    want, wp, wl = oracle.source_from_state(net, atm.T, atm.P, atm.J, atm.n, atm.ncol)
    got = run_fused(emu, net, atm, atm.ncol, grid=4, nsplit=3)
    check(got, want, wp + wl, atm.ncol, "emulated k_fused config 3")
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    got_k = run_fused(emu, net, atm, atm.ncol, kf=np.ascontiguousarray(okf), kr=np.ascontiguousarray(okr), grid=2, nsplit=1)
    check(got_k, want, wp + wl, atm.ncol, "emulated k_fused<FROMK> config 3")


def test_fused_kernel_source_from_stored_coefficients_and_mixed_intervals(emu, oracle, network):
    """k_fused<true> (xod_source), and a tile whose columns straddle thermo breakpoints (the rare
    per-thread second parameter block) with cold columns whose k_r overflow."""
    from paper_2512_06729_b200 import synth
    net = network(2)
    atm = synth.make_atmosphere(5, net, 1, 37, t_shift=(-600.0, -600.0))
    atm.T[:37] = np.linspace(180.0, 1100.0, 37)          # crosses 300, 500, 700, 1000 K inside tiles
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, atm.ncol)
    fin = np.all(np.isfinite(okr[:, :atm.ncol]), axis=0) & np.all(np.isfinite(want[:, :atm.ncol]), axis=0)
    assert 5 < fin.sum() < atm.ncol
    got = run_fused(emu, net, atm, atm.ncol, grid=2)
    err = np.abs(got[:, :atm.ncol] - want[:, :atm.ncol])[:, fin]
    assert np.all(err <= 1e-11 * (wp + wl)[:, :atm.ncol][:, fin])
    got_k = run_fused(emu, net, atm, atm.ncol, kf=np.ascontiguousarray(okf), kr=np.ascontiguousarray(okr), grid=3)
    err = np.abs(got_k[:, :atm.ncol] - want[:, :atm.ncol])[:, fin]
    assert np.all(err <= 1e-11 * (wp + wl)[:, :atm.ncol][:, fin])


@pytest.mark.parametrize("cfg,slice_", [(1, 64), (2, 8)])
def test_rate_coefficient_kernel_source_matches_oracle(emu, oracle, network, cfg, slice_):
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    d, keep = descriptor(net)
    kf = np.full((net.n_reactions, atm.ld), np.nan)
    kr = np.full((net.n_reactions, atm.ld), np.nan)
    rc = emu.emu_rate_coeffs(C.byref(d), C.c_int64(atm.ncol), C.c_int64(atm.ld), ptr(atm.T), ptr(atm.P), ptr(atm.J),
                             ptr(kf), ptr(kr), C.c_int(slice_))
    assert rc == 0
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    c = slice(0, atm.ncol)
    assert np.all(np.abs(kf[:, c] - okf[:, c]) <= 1e-12 * np.abs(okf[:, c]))
    assert np.all(np.abs(kr[:, c] - okr[:, c]) <= 1e-12 * np.abs(okr[:, c]))
    assert np.all(np.isnan(kf[:, atm.ncol:])) and np.all(np.isnan(kr[:, atm.ncol:]))


@pytest.mark.parametrize("cfg", [1, 2])
def test_thermo_and_jacobian_kernel_sources_match_oracle(emu, oracle, network, cfg):
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    d, keep = descriptor(net)
    ns, ld, ncol = net.n_species, atm.ld, atm.ncol
    outs = [np.full((ns, ld), np.nan) for _ in range(4)]
    assert emu.emu_thermo(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(atm.T), *[ptr(o) for o in outs], C.c_int(5)) == 0
    want = oracle.thermo(net, atm.T, ncol)
    for got, w in zip(outs, want):
        assert np.all(np.abs(got[:, :ncol] - w[:, :ncol]) <= 1e-12 * (1 + np.abs(w[:, :ncol])))
        assert np.all(np.isnan(got[:, ncol:]))
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    h = binding.Network(net, device=-1)
    rp, col = h.jac_pattern()
    wj, sj = oracle.jacobian(net, okf, okr, atm.n, rp, col, ncol)
    jac = np.full((col.shape[0], ld), np.nan)
    assert emu.emu_jacobian(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(okf), ptr(okr), ptr(atm.n), ptr(jac), C.c_int(3)) == 0
    assert np.all(np.abs(jac[:, :ncol] - wj[:, :ncol]) <= 1e-11 * sj[:, :ncol])
    assert np.all(np.isnan(jac[:, ncol:]))


@pytest.mark.parametrize("cfg,grid,nsplit", [(1, 1, 1), (2, 2, 1), (2, 3, 3), (2, 30, 5)])
def test_tiled_jacobian_kernel_source_matches_oracle(emu, oracle, network, cfg, grid, nsplit):
    """k_jac_tiled: slots evaluated once per column tile, scheduled row reduction, per-unit flush; fewer blocks
    than work items (persistent loop) and the units of a tile split over several blocks."""
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    d, keep = descriptor(net)
    ncol, ld = atm.ncol, atm.ld
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    h = binding.Network(net, device=-1)
    rp, col = h.jac_pattern()
    wj, sj = oracle.jacobian(net, okf, okr, atm.n, rp, col, ncol)
    jac = np.full((col.shape[0], ld), np.nan)
    assert emu.emu_jacobian_tiled(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(okf), ptr(okr), ptr(atm.n), ptr(jac),
                                  C.c_int(grid), C.c_int(nsplit)) == 0
    worst = G.check_sum(jac, wj, sj, np.arange(ncol), "emulated k_jac_tiled config %d" % cfg)
    assert np.all(np.isnan(jac[:, ncol:])), "padding columns written"
    print("k_jac_tiled config %d (grid %d, split %d): worst |err|/scale %.2e" % (cfg, grid, nsplit, worst))


def test_tiled_jacobian_kernel_source_hub_columns_over_several_chunks(emu, oracle, network):
    """Config-3 network: hub species own units of several chunks (accumulators carried across chunks, extra rows
    for entries with more than 16 terms in a chunk); 20 columns = one full and one ragged tile, units split 3 ways."""
    from paper_2512_06729_b200 import synth
    net = network(3)
    atm = synth.make_atmosphere(2033, net, 1, 20)
    d, keep = descriptor(net)
    ncol, ld = atm.ncol, atm.ld
    h = binding.Network(net, device=-1)
    info = h.jac_info()
    assert info["enabled"] and info["nchunk"] > info["units"], "some unit must span several chunks"
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    rp, col = h.jac_pattern()
    wj, sj = oracle.jacobian(net, okf, okr, atm.n, rp, col, ncol)
    jac = np.full((col.shape[0], ld), np.nan)
    assert emu.emu_jacobian_tiled(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(okf), ptr(okr), ptr(atm.n), ptr(jac),
                                  C.c_int(2), C.c_int(3)) == 0
    worst = G.check_sum(jac, wj, sj, np.arange(ncol), "emulated k_jac_tiled config 3")
    assert np.all(np.isnan(jac[:, ncol:]))
    print("k_jac_tiled config 3 (%d slots for %d terms, %d chunks, %d units): worst |err|/scale %.2e"
          % (info["slots"], h.n_jac_terms, info["nchunk"], info["units"], worst))


@pytest.mark.parametrize("cfg", [1, 2])
def test_multi_kernel_pipeline_sources_match_oracle(emu, oracle, network, cfg):
    """k_prologue + k_rates + k_source (the prod/loss variants and the fallback of the fused path), and
    k_rates_from_k + k_source for xod_source with prod/loss."""
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    d, keep = descriptor(net)
    ns, ld, ncol = net.n_species, atm.ld, atm.ncol
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, ncol)
    scale = wp + wl
    for kf_in, kr_in in ((None, None), (okf, okr)):
        for pl in (False, True):
            dn, pr, lo = (np.full((ns, ld), np.nan) for _ in range(3))
            rc = emu.emu_source_pipeline(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(atm.T), ptr(atm.P), ptr(atm.J),
                                         ptr(kf_in), ptr(kr_in), ptr(atm.n), ptr(dn), ptr(pr) if pl else None,
                                         ptr(lo) if pl else None, C.c_int(16))
            assert rc == 0
            check(dn, want, scale, ncol, "pipeline dn/dt")
            if pl:
                check(pr, wp, scale, ncol, "pipeline P")
                check(lo, wl, scale, ncol, "pipeline L")
    kf = np.full((net.n_reactions, ld), np.nan)
    kr = np.full((net.n_reactions, ld), np.nan)
    assert emu.emu_rate_coeffs_pipeline(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(atm.T), ptr(atm.P), ptr(atm.J),
                                        ptr(kf), ptr(kr), C.c_int(16)) == 0
    assert np.all(np.abs(kf[:, :ncol] - okf[:, :ncol]) <= 1e-12 * np.abs(okf[:, :ncol]))
    assert np.all(np.abs(kr[:, :ncol] - okr[:, :ncol]) <= 1e-12 * np.abs(okr[:, :ncol]))


# ------------------------------------------------------------------------------- the edge-case network
@pytest.fixture(scope="module")
def edge(oracle):
    """synth.edge_network / edge_atmosphere with the oracle's results (shared by the tests below)."""
    from paper_2512_06729_b200 import synth
    net = synth.edge_network()
    atm = synth.edge_atmosphere(net)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, atm.ncol)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, atm.ncol)
    c = slice(0, atm.ncol)
    fin = G.finite_columns(okf[:, c], okr[:, c], want[:, c], wp[:, c], wl[:, c])
    assert 0 < (~fin).sum() <= 8, "only the cold columns (170 K, 300 K) hold k_r beyond the double range (reading R5)"
    return net, atm, okf, okr, want, wp, wl, np.flatnonzero(fin)


def test_edge_network_has_every_shape():
    from paper_2512_06729_b200 import synth
    net = synth.edge_network()
    h = binding.Network(net, device=-1)
    h.selfcheck()
    rp, rxn, nu = h.source_csr()
    assert nu.min() == -3 and nu.max() == 3
    assert rp[net.meta["lone"] + 1] == rp[net.meta["lone"]], "a species in no reaction has an empty CSR row"
    irr = net.reversible == 0
    assert {0, 1, 2} <= set(net.type[irr].tolist())
    assert np.any((net.type == 2) & (net.troe_fc == 1.0)) and np.any((net.type == 2) & (net.troe_fc < 1.0))
    assert np.any(net.t_ref == 300.0) and np.any(net.t_ref == 1.0)
    assert net.composition[net.meta["ion"], -1] == 1 and net.composition[net.meta["electron"], -1] == -1
    atm = synth.edge_atmosphere(net)
    for tm in np.unique(net.t_mid):
        assert np.any(atm.T[:atm.ncol] == tm) and np.any(atm.T[:atm.ncol] == np.nextafter(tm, 0)) \
            and np.any(atm.T[:atm.ncol] == np.nextafter(tm, 1e9))


@pytest.mark.parametrize("grid,nsplit,fromk", [(2, 1, False), (3, 2, False), (2, 1, True)])
def test_edge_network_fused_kernel_source(emu, edge, grid, nsplit, fromk):
    """k_fused on irreversible reactions (C0 = -inf), Fc = 1, nu = +-3, ions, an empty CSR row, Kooij
    forms, and columns sitting exactly on / one ulp beside every thermo breakpoint inside a tile."""
    net, atm, okf, okr, want, wp, wl, cols = edge
    kw = dict(kf=np.ascontiguousarray(okf), kr=np.ascontiguousarray(okr)) if fromk else {}
    got = run_fused(emu, net, atm, atm.ncol, grid=grid, nsplit=nsplit, **kw)
    worst = G.check_sum(got, want, wp + wl, cols, "emulated k_fused, edge network")
    # columns with some overflowing k_r (T = 300 K -+ 1 ulp among them): every entry they do not reach still matches
    w2, skipped = G.check_sum_entries(got, want, wp + wl, atm.ncol, "emulated k_fused, edge network, entry-wise")
    assert skipped > 0
    assert np.all(np.isnan(got[:, atm.ncol:]))
    assert np.all(got[net.meta["lone"], cols] == 0.0)
    zc = atm.meta["zero_column"]
    assert np.all(got[:, zc] == 0.0), "a column of zero densities gives exact zeros"
    print("edge network, k_fused(fromk=%s, split %d): worst |err|/scale = %.2e on %d columns" % (fromk, nsplit, worst, cols.size))


def test_edge_network_rate_coefficient_kernel_source(emu, edge):
    net, atm, okf, okr, *_ = edge
    d, keep = descriptor(net)
    kf = np.full((net.n_reactions, atm.ld), np.nan)
    kr = np.full((net.n_reactions, atm.ld), np.nan)
    assert emu.emu_rate_coeffs(C.byref(d), C.c_int64(atm.ncol), C.c_int64(atm.ld), ptr(atm.T), ptr(atm.P), ptr(atm.J),
                               ptr(kf), ptr(kr), C.c_int(12)) == 0
    c = slice(0, atm.ncol)
    wf = G.check_k(kf[:, c], okf[:, c], "emulated k_rate_coeffs k_f, edge network")
    wr = G.check_k(kr[:, c], okr[:, c], "emulated k_rate_coeffs k_r, edge network")
    irr = net.reversible == 0
    assert np.all(kr[irr][:, c] == 0.0), "irreversible reactions have k_r = 0 exactly"
    assert np.isinf(okr[:, c]).any(), "the cold column overflows (reading R5)"
    print("edge network, k_rate_coeffs: worst relative error k_f %.2e, k_r %.2e" % (wf, wr))


def test_edge_network_other_kernel_sources(emu, oracle, edge):
    """k_thermo, k_jacobian and the multi-kernel pipeline (with P and L) on the edge network."""
    net, atm, okf, okr, want, wp, wl, cols = edge
    d, keep = descriptor(net)
    ns, ld, ncol = net.n_species, atm.ld, atm.ncol
    outs = [np.full((ns, ld), np.nan) for _ in range(4)]
    assert emu.emu_thermo(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(atm.T), *[ptr(o) for o in outs], C.c_int(7)) == 0
    for got, w in zip(outs, oracle.thermo(net, atm.T, ncol)):
        assert np.all(np.abs(got[:, :ncol] - w[:, :ncol]) <= 1e-12 * (1 + np.abs(w[:, :ncol])))
    scale = wp + wl
    for kf_in, kr_in in ((None, None), (okf, okr)):
        dn, pr, lo = (np.full((ns, ld), np.nan) for _ in range(3))
        assert emu.emu_source_pipeline(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(atm.T), ptr(atm.P), ptr(atm.J),
                                       ptr(kf_in), ptr(kr_in), ptr(atm.n), ptr(dn), ptr(pr), ptr(lo), C.c_int(16)) == 0
        G.check_sum(dn, want, scale, cols, "pipeline dn/dt, edge network")
        G.check_sum(pr, wp, scale, cols, "pipeline P, edge network")
        G.check_sum(lo, wl, scale, cols, "pipeline L, edge network")
    h = binding.Network(net, device=-1)
    rp, col = h.jac_pattern()
    okf_f, okr_f = okf.copy(), okr.copy()
    okr_f[~np.isfinite(okr_f)] = 0.0            # the dense oracle wants finite inputs; those columns are not compared
    wj, sj = oracle.jacobian(net, okf_f, okr_f, atm.n, rp, col, ncol)
    jac = np.full((col.shape[0], ld), np.nan)
    assert emu.emu_jacobian(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(okf_f), ptr(okr_f), ptr(atm.n), ptr(jac), C.c_int(3)) == 0
    G.check_sum(jac, wj, sj, cols, "emulated k_jacobian, edge network")
    jac2 = np.full((col.shape[0], ld), np.nan)
    assert emu.emu_jacobian_tiled(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(okf_f), ptr(okr_f), ptr(atm.n), ptr(jac2),
                                  C.c_int(2), C.c_int(2)) == 0
    G.check_sum(jac2, wj, sj, cols, "emulated k_jac_tiled, edge network")
    assert np.all(np.isnan(jac2[:, ncol:]))


TSAN_CHILD = r"""
import sys, ctypes as C
sys.path.insert(0, sys.argv[1]); sys.path.insert(0, sys.argv[1] + "/tests")
import numpy as np
import test_kernel_emulation as tk
from paper_2512_06729_b200 import synth
from paper_2512_06729_b200 import binding
def binding_nnz(net):
    return binding.Network(net, device=-1).nnz_jac
emu = C.CDLL(sys.argv[2])
net = synth.config_network(2)
atm = synth.config_atmosphere(2, net)
for grid, nsplit in ((3, 1), (5, 3)):
    got = tk.run_fused(emu, net, atm, atm.ncol, grid=grid, nsplit=nsplit)
    assert np.all(np.isfinite(got[:, :atm.ncol]))
# the tiled Jacobian kernel: slot buffers, accumulator rows flushed and zeroed per unit
d, keep = tk.descriptor(net)
ncol = 40
kf = np.abs(np.random.default_rng(1).normal(size=(net.n_reactions, atm.ld)))
jac = np.zeros((binding_nnz(net), atm.ld))
assert emu.emu_jacobian_tiled(C.byref(d), C.c_int64(ncol), C.c_int64(atm.ld), tk.ptr(kf), tk.ptr(kf), tk.ptr(atm.n),
                              tk.ptr(jac), C.c_int(2), C.c_int(2)) == 0
# the implicit step: k_lu_factor's shared row, one barrier per pivot
net1 = synth.config_network(1)
atm1 = synth.config_atmosphere(1, net1)
d1, keep1 = tk.descriptor(net1)
k1 = np.abs(np.random.default_rng(2).normal(size=(net1.n_reactions, atm1.ld))) * 1e-12
y1 = atm1.n.copy()
delta1 = np.zeros_like(y1)
dt1 = np.full(atm1.ld, 1e-3)
assert emu.emu_newton_step(C.byref(d1), C.c_int64(atm1.ncol), C.c_int64(atm1.ld), tk.ptr(k1), tk.ptr(k1), tk.ptr(atm1.n),
                           tk.ptr(dt1), tk.ptr(y1), tk.ptr(delta1)) == 0
# the pathway analyser: double-buffered distance tiles, partial minima combined after a barrier, __syncthreads_or
dist1 = np.zeros_like(y1)
pred1, via1 = np.zeros(y1.shape, dtype=np.int32), np.zeros(y1.shape, dtype=np.int32)
assert emu.emu_pathway(C.byref(d1), C.c_int64(atm1.ncol), C.c_int64(atm1.ld), tk.ptr(k1), tk.ptr(k1), tk.ptr(atm1.n), C.c_int(2),
                       tk.ptr(dist1), tk.ptr(pred1), tk.ptr(via1), C.c_int(2)) == 0
# the photolysis contraction: shared operand tiles of the GEMM, the scan tile of k_photo_flux
import test_photo_rates as tp
tk.LIB = sys.argv[2]
atm3 = synth.config_atmosphere(1, net1, 2)
ph = synth.make_photo(51, net1, n_bins=70)
tp.run_emulated(net1, atm3, ph, *synth.make_irradiation(52, net1, atm3, ph))
print("emulated-ok")
"""


ASAN_CHILD = r"""
import sys, ctypes as C
sys.path.insert(0, sys.argv[1]); sys.path.insert(0, sys.argv[1] + "/tests")
import numpy as np
import test_kernel_emulation as tk
import test_photo_rates as tp
from paper_2512_06729_b200 import synth, binding
emu = C.CDLL(sys.argv[2])
tk.LIB = tp_lib = sys.argv[2]
# exact-size heap buffers (numpy) around every kernel: any access outside [0, rows x ld) is reported
for net, atm in ((synth.config_network(2), None), (synth.edge_network(), None)):
    atm = synth.edge_atmosphere(net) if net.meta.get("name") == "edge" else synth.config_atmosphere(2, net)
    ncol = atm.ncol - 3                                   # ragged: the last tile and the last warp are partial
    tk.run_fused(emu, net, atm, ncol, grid=3, nsplit=2)
    d, keep = tk.descriptor(net)
    nr, ns, ld = net.n_reactions, net.n_species, atm.ld
    kf, kr = np.full((nr, ld), 1e-12), np.full((nr, ld), 1e-13)
    assert emu.emu_rate_coeffs(C.byref(d), C.c_int64(ncol), C.c_int64(ld), tk.ptr(atm.T), tk.ptr(atm.P), tk.ptr(atm.J),
                               tk.ptr(kf), tk.ptr(kr), C.c_int(12)) == 0
    kr[~np.isfinite(kr)] = 0.0
    tk.run_fused(emu, net, atm, ncol, kf=kf, kr=kr, grid=2, nsplit=1)
    nnz = binding.Network(net, device=-1).nnz_jac
    jac = np.zeros((nnz, ld))
    assert emu.emu_jacobian_tiled(C.byref(d), C.c_int64(ncol), C.c_int64(ld), tk.ptr(kf), tk.ptr(kr), tk.ptr(atm.n), tk.ptr(jac),
                                  C.c_int(2), C.c_int(3)) == 0
    assert emu.emu_jacobian(C.byref(d), C.c_int64(ncol), C.c_int64(ld), tk.ptr(kf), tk.ptr(kr), tk.ptr(atm.n), tk.ptr(jac), C.c_int(3)) == 0
    dn, pr, lo = (np.zeros((ns, ld)) for _ in range(3))
    assert emu.emu_source_pipeline(C.byref(d), C.c_int64(ncol), C.c_int64(ld), tk.ptr(atm.T), tk.ptr(atm.P), tk.ptr(atm.J),
                                   None, None, tk.ptr(atm.n), tk.ptr(dn), tk.ptr(pr), tk.ptr(lo), C.c_int(16)) == 0
    y, delta, n_old, dt = np.abs(atm.n).copy(), np.zeros((ns, ld)), np.abs(atm.n).copy(), np.full(ld, 1e-9)
    assert emu.emu_newton_step(C.byref(d), C.c_int64(min(ncol, 37)), C.c_int64(ld), tk.ptr(kf), tk.ptr(kr), tk.ptr(n_old),
                               tk.ptr(dt), tk.ptr(y), tk.ptr(delta)) == 0
net = synth.config_network(1)
atm = synth.config_atmosphere(1, net, 3)
ph = synth.make_photo(51, net, n_bins=70)
tp.run_emulated(net, atm, ph, *synth.make_irradiation(52, net, atm, ph))
t = synth.make_transport(61, net, atm)
arrs = [np.ascontiguousarray(x, dtype=np.float64) for x in (atm.n, atm.T, t["n_gas"], t["D"], t["mass"], t["alpha_T"], t["mbar"], t["grav"], t["dz"])]
tr = np.zeros((net.n_species, atm.ld))
assert emu.emu_transport(C.c_int(net.n_species), C.c_int64(3), C.c_int64(20), C.c_int64(atm.ld), *[tk.ptr(x) for x in arrs], tk.ptr(tr), C.c_int(5)) == 0
import test_pathway as tpw
net2 = synth.config_network(2)
atm2 = synth.config_atmosphere(2, net2)
k2 = np.full((net2.n_reactions, atm2.ld), 1e-12)
tpw.run_emulated(net2, k2, k2, atm2.n, 37, atm2.ld, 5, 2)
import test_equilibrium as teq
comp2 = np.asarray(net2.composition, dtype=np.float64)
b2 = np.ascontiguousarray(comp2.T @ atm2.n)
n_eq, pi_eq, it_eq = teq.run_emulated(net2, np.ascontiguousarray(atm2.T), np.ascontiguousarray(atm2.P), b2, 37, atm2.ld)
assert np.all(it_eq[:37] > 0)
print("emulated-ok")
"""


def test_kernel_sources_touch_no_memory_outside_their_buffers_under_address_sanitizer():
    """memcheck substitute (compute-sanitizer is closed on the GPU pool): the emulation built with AddressSanitizer
    and UndefinedBehaviorSanitizer (alignment, bounds, shifts), every kernel run on exact-size heap buffers with ragged
    column counts: an access one element past a [rows][ld] array, a misaligned 16-byte vector access or an index
    beyond a static shared array aborts the child."""
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("libasan not available")
    lib = os.path.join(EMU_DIR, "libxod_emu_asan.so")
    if not os.path.exists(lib) or any(os.path.getmtime(d) > os.path.getmtime(lib) for d in DEPS):
        subprocess.run(["g++", "-std=c++20", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                        "-pthread", "-shared", "-fPIC", "-I" + os.path.join(EMU_DIR, "shim"), "-o", lib] + SOURCES, check=True)
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:halt_on_error=1", UBSAN_OPTIONS="print_stacktrace=1")
    out = subprocess.run([os.sys.executable, "-c", ASAN_CHILD, ROOT, lib], capture_output=True, text=True, env=env, timeout=1800)
    assert "emulated-ok" in out.stdout, (out.stdout[-1000:], out.stderr[-3000:])
    assert "AddressSanitizer" not in out.stderr and "runtime error" not in out.stderr, out.stderr[-3000:]


def test_barrier_synchronised_kernel_sources_are_race_free_under_thread_sanitizer():
    """racecheck substitute (compute-sanitizer is closed on the GPU pool): the emulated CUDA threads are
    real threads and __syncthreads a real barrier, so ThreadSanitizer sees every shared-memory access
    of k_fused, k_jac_tiled, k_lu_factor, k_pathway, k_photo_gemm and k_photo_flux between barriers: the double-buffered values and schedule, the accumulator
    read-modify-writes of the row tasks, the per-unit flush, the tile prologue/epilogue.  (Removing the per-chunk barrier makes it report.)"""
    tsan = subprocess.run(["gcc", "-print-file-name=libtsan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(tsan) or not os.path.exists(tsan):
        pytest.skip("libtsan not available")
    lib = os.path.join(EMU_DIR, "libxod_emu_tsan.so")
    if not os.path.exists(lib) or any(os.path.getmtime(d) > os.path.getmtime(lib) for d in DEPS):
        subprocess.run(["g++", "-std=c++20", "-O1", "-g", "-fsanitize=thread", "-pthread", "-shared", "-fPIC",
                        "-I" + os.path.join(EMU_DIR, "shim"), "-o", lib] + SOURCES, check=True)
    env = dict(os.environ, LD_PRELOAD=tsan, TSAN_OPTIONS="halt_on_error=0 report_signal_unsafe=0 exitcode=0")
    out = subprocess.run([os.sys.executable, "-c", TSAN_CHILD, ROOT, lib], capture_output=True, text=True, env=env,
                         timeout=900)
    assert "emulated-ok" in out.stdout, out.stderr[-2000:]
    assert "ThreadSanitizer" not in out.stderr, out.stderr[-3000:]


@pytest.mark.parametrize("seed", [11, 12, 13, 14, 15, 16])
def test_random_networks_through_the_kernel_sources(emu, oracle, seed):
    """Seeded random networks of odd sizes (segment lengths that are not multiples of 4, reaction counts around
    the chunk size, one to five elements, some reactions made irreversible, Kooij forms mixed in) and ragged column
    counts through k_fused (both modes, split or not), k_rate_coeffs and k_jac_tiled against the oracle: the
    packer's padding, chunking and schedules must hold for shapes nobody picked by hand; xod_network_selfcheck
    must accept the tables."""
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
    ncol, ld = atm.ncol, atm.ld
    h = binding.Network(net, device=-1)
    h.selfcheck()
    d, keep = descriptor(net)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    # rate coefficients (reading R5 rules)
    kf, kr = np.full((net.n_reactions, ld), np.nan), np.full((net.n_reactions, ld), np.nan)
    assert emu.emu_rate_coeffs(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(atm.T), ptr(atm.P), ptr(atm.J), ptr(kf), ptr(kr),
                               C.c_int(8)) == 0
    G.check_k(kf[:, :ncol], okf[:, :ncol], "random net %d k_f" % seed)
    G.check_k(kr[:, :ncol], okr[:, :ncol], "random net %d k_r" % seed)
    assert np.all(kr[net.reversible == 0, :ncol] == 0.0)
    # source term, evaluated and from stored coefficients, split or not
    want, wp, wl = oracle.source(net, okf, okr, atm.n, ncol)
    scale = wp + wl
    okr_f = np.where(np.isfinite(okr), okr, 0.0)
    want_f, wpf, wlf = oracle.source(net, okf, okr_f, atm.n, ncol)
    for nsplit in (1, 2):
        got = run_fused(emu, net, atm, ncol, grid=2, nsplit=nsplit)
        G.check_sum_entries(got, want, scale, ncol, "random net %d k_fused split %d" % (seed, nsplit))
        got = run_fused(emu, net, atm, ncol, kf=okf, kr=okr_f, grid=3, nsplit=nsplit)
        G.check_sum_entries(got, want_f, wpf + wlf, ncol, "random net %d k_fused<FROMK> split %d" % (seed, nsplit))
    # Jacobian values
    rp, col = h.jac_pattern()
    wj, sj = oracle.jacobian(net, okf, okr_f, atm.n, rp, col, ncol)
    jac = np.full((col.shape[0], ld), np.nan)
    assert emu.emu_jacobian_tiled(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(okf), ptr(okr_f), ptr(atm.n), ptr(jac),
                                  C.c_int(2), C.c_int(2)) == 0
    G.check_sum_entries(jac, wj, sj, ncol, "random net %d k_jac_tiled" % seed)
    print("random network %d: %d species, %d reactions (%d irreversible), %d columns: ok" % (
        seed, net.n_species, net.n_reactions, int((net.reversible == 0).sum()), ncol))


def test_kernel_sources_at_the_ends_of_the_temperature_range(emu, oracle, network):
    """the network is "valid" from 100 K to 30 000 K, far outside the 200-3000 K of the thermo fits
    (reading T4: extrapolate, no clamp).  Columns at 100, 120, 3 000, 10 000 and 30 000 K: most reverse coefficients
    over- or underflow at the cold end and the extrapolated quartic does at the hot end (reading R5 decides what the
    kernels must return there); everything in between must match to 1e-12."""
    from paper_2512_06729_b200 import synth
    net = network(2)
    atm = synth.make_atmosphere(2077, net, 1, 20)
    atm.T[:20] = np.array([100.0, 120.0, 150.0, 200.0, 3000.0, 5000.0, 10000.0, 20000.0, 30000.0, 30000.0] * 2)
    ncol, ld = atm.ncol, atm.ld
    d, keep = descriptor(net)
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    kf, kr = np.full((net.n_reactions, ld), np.nan), np.full((net.n_reactions, ld), np.nan)
    assert emu.emu_rate_coeffs(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(atm.T), ptr(atm.P), ptr(atm.J), ptr(kf), ptr(kr),
                               C.c_int(16)) == 0
    worst_f = G.check_k(kf[:, :ncol], okf[:, :ncol], "k_f at the ends of the range")
    worst_r = G.check_k(kr[:, :ncol], okr[:, :ncol], "k_r at the ends of the range")
    cold, hot = atm.T[:ncol] <= 200.0, atm.T[:ncol] >= 10000.0      # both ends leave the double range for some reactions:
    assert np.isinf(okr[:, :ncol][:, cold]).any() and np.isinf(okr[:, :ncol][:, hot]).any()   # a6 / T when cold, a5 T^4 when hot
    want, wp, wl = oracle.source(net, okf, okr, atm.n, ncol)
    got = run_fused(emu, net, atm, ncol, grid=2, nsplit=1)
    worst, skipped = G.check_sum_entries(got, want, wp + wl, ncol, "k_fused at the ends of the range")
    print("100 K .. 30 000 K: worst relative error k_f %.2e, k_r %.2e; dn/dt %.2e of scale, %d non-finite entries skipped"
          % (worst_f, worst_r, worst, skipped))


def test_a_network_too_large_for_the_single_kernel_tables(emu, oracle):
    """950 species: the n tile and the accumulator tile of k_fused no longer fit one CTA's shared memory together, so
    the library must disable the fused tables (xod_network_fused_info) and serve xod_rate_coeffs / xod_source /
    xod_source_fused by the multi-kernel pipeline; the tiled Jacobian (one accumulator set per unit only) still fits.
    Both are run here against the oracle, with a ragged column count."""
    from paper_2512_06729_b200 import synth
    net = synth.make_network(777, ["H", "C", "O", "N", "S"], 950, 300, inert=())
    atm = synth.make_atmosphere(2777, net, 1, 19)
    h = binding.Network(net, device=-1)
    assert h.fused_info()["enabled"] == 0 and h.jac_info()["enabled"] == 1
    h.selfcheck()
    d, keep = descriptor(net)
    ns, ld, ncol = net.n_species, atm.ld, atm.ncol
    okf, okr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    want, wp, wl = oracle.source(net, okf, okr, atm.n, ncol)
    kf, kr = np.full((net.n_reactions, ld), np.nan), np.full((net.n_reactions, ld), np.nan)
    assert emu.emu_rate_coeffs_pipeline(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(atm.T), ptr(atm.P), ptr(atm.J),
                                        ptr(kf), ptr(kr), C.c_int(16)) == 0
    G.check_k(kf[:, :ncol], okf[:, :ncol], "950 species k_f")
    G.check_k(kr[:, :ncol], okr[:, :ncol], "950 species k_r")
    dn, pr, lo = (np.full((ns, ld), np.nan) for _ in range(3))
    assert emu.emu_source_pipeline(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(atm.T), ptr(atm.P), ptr(atm.J), None, None,
                                   ptr(atm.n), ptr(dn), ptr(pr), ptr(lo), C.c_int(16)) == 0
    check(dn, want, wp + wl, ncol, "950 species dn/dt")
    check(pr, wp, wp + wl, ncol, "950 species P")
    check(lo, wl, wp + wl, ncol, "950 species L")
    rp, col = h.jac_pattern()
    wj, sj = oracle.jacobian(net, okf, okr, atm.n, rp, col, ncol)
    jac = np.full((col.shape[0], ld), np.nan)
    assert emu.emu_jacobian_tiled(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(okf), ptr(okr), ptr(atm.n), ptr(jac),
                                  C.c_int(2), C.c_int(2)) == 0
    G.check_sum(jac, wj, sj, np.arange(ncol), "950 species k_jac_tiled")


def test_a_network_without_reactions(emu):
    """The empty reaction list: dn/dt, P and L are exact zeros for every species and the Jacobian (its pattern is the
    diagonal alone) is zero too; nothing outside the asked columns is written."""
    from conftest import SimpleNet
    net = SimpleNet([[1], [2], [1]], np.zeros((3, 7)), np.zeros((3, 7)), [1000.0] * 3, [], [], [], [], np.zeros((0, 3)))
    h = binding.Network(net, device=-1)
    assert h.fused_info()["enabled"] == 0 and h.jac_info()["enabled"] == 0 and h.nnz_jac == 3
    d, keep = descriptor(net)
    ncol, ld = 37, 64
    T, P = np.full(ld, 1200.0), np.full(ld, 1e5)
    J = np.zeros((0, ld))
    n = np.abs(np.random.default_rng(3).normal(size=(3, ld))) * 1e10
    dn, pr, lo = (np.full((3, ld), np.nan) for _ in range(3))
    assert emu.emu_source_pipeline(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(T), ptr(P), ptr(J), None, None, ptr(n), ptr(dn),
                                   ptr(pr), ptr(lo), C.c_int(16)) == 0
    for a in (dn, pr, lo):
        assert np.all(a[:, :ncol] == 0.0) and np.all(np.isnan(a[:, ncol:]))
    jac = np.full((3, ld), np.nan)
    empty = np.zeros((0, ld))
    assert emu.emu_jacobian(C.byref(d), C.c_int64(ncol), C.c_int64(ld), ptr(empty), ptr(empty), ptr(n), ptr(jac), C.c_int(3)) == 0
    assert np.all(jac[:, :ncol] == 0.0) and np.all(np.isnan(jac[:, ncol:]))
