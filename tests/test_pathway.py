"""f4, the reaction pathway analyser: the kernel SOURCE executed on CPU threads
against the oracle, and the `-m gpu` parity tests through the C ABI.

What is unique is compared exactly: the set of reachable species must be identical, and dist must agree to relative
1e-13 (both sides add the same edge weights 1/q from the source outwards; the oracle accumulates in long double and
rounds, the kernel in fp64, and 1/q itself carries the few-ulp difference of q = k prod n).  pred / via are not
unique when routes tie, so they are checked for validity instead: the named reaction direction consumes pred and
forms the species, and dist[pred] + 1/q equals dist to 1e-12 (a tight tree edge)."""
import ctypes as C

import numpy as np
import pytest

import gpu_common as G

REV = 1 << 30


def case(network, oracle, cfg, ncol_max):
    from paper_2512_06729_b200 import synth
    net = synth.edge_network() if cfg == "edge" else network(cfg)
    atm = synth.edge_atmosphere(net) if cfg == "edge" else synth.config_atmosphere(cfg, net)
    ncol = min(atm.ncol, ncol_max)
    ld = (ncol + 31) // 32 * 32
    kf, kr = oracle.rate_coeffs(net, atm.T[:ld], atm.P[:ld], atm.J[:, :ld], ncol)
    return net, kf, kr, np.ascontiguousarray(atm.n[:, :ld]), ncol, ld


def check(net, kf, kr, n, ncol, source, got, want, what):
    dist, pred, via = got
    wd = want[0]
    g, w = dist[:, :ncol], wd[:, :ncol]
    assert np.array_equal(np.isfinite(g), np.isfinite(w)), what + ": reachable sets differ"
    fin = np.isfinite(w)
    rel = np.abs(g[fin] - w[fin]) / np.maximum(w[fin], 1e-300)
    worst = float(rel.max()) if rel.size else 0.0
    assert worst <= 1e-13, "%s: dist differs by %.2e" % (what, worst)
    assert np.all(g[source] == 0.0)
    assert np.all(np.isnan(dist[:, ncol:])) and np.all(pred[:, ncol:] == -7) and np.all(via[:, ncol:] == -7), what + ": padding columns written"
    # validity of the tree
    for c in range(ncol):
        for v in range(net.n_species):
            if v == source or not np.isfinite(g[v, c]):
                assert pred[v, c] == -1 and via[v, c] == -1, what
                continue
            u, r, rev = int(pred[v, c]), int(via[v, c] & ~REV), bool(via[v, c] & REV)
            assert 0 <= r < net.n_reactions and 0 <= u < net.n_species
            frm, to = (net.products[r], net.reactants[r]) if rev else (net.reactants[r], net.products[r])
            assert u in frm and v in to and (not rev or net.reversible[r]), what
            q = (kr if rev else kf)[r, c] * np.prod([n[s, c] for s in frm if s >= 0])
            assert abs(g[u, c] + 1.0 / q - g[v, c]) <= 1e-12 * g[v, c], what + ": predecessor edge is not tight"
    print("%s: %d columns, %d reachable of %d, worst relative error of dist %.2e" % (what, ncol, int(fin.sum()), fin.size, worst))


def run_emulated(net, kf, kr, n, ncol, ld, source, grid):
    import os
    import subprocess
    import test_kernel_emulation as tk
    if not os.path.exists(tk.LIB) or any(os.path.getmtime(d) > os.path.getmtime(tk.LIB) for d in tk.DEPS):
        subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-shared", "-fPIC", "-I" + os.path.join(tk.EMU_DIR, "shim"),
                        "-o", tk.LIB] + tk.SOURCES, check=True)
    lib = C.CDLL(tk.LIB)
    d, keep = tk.descriptor(net)
    dist = np.full((net.n_species, ld), np.nan)
    pred = np.full((net.n_species, ld), -7, dtype=np.int32)
    via = np.full((net.n_species, ld), -7, dtype=np.int32)
    rc = lib.emu_pathway(C.byref(d), C.c_int64(ncol), C.c_int64(ld), tk.ptr(kf), tk.ptr(kr), tk.ptr(n), C.c_int(source),
                         tk.ptr(dist), tk.ptr(pred), tk.ptr(via), C.c_int(grid))
    assert rc == 0
    return dist, pred, via


@pytest.mark.parametrize("cfg,ncol_max,source,grid", [(1, 20, 0, 1), (1, 20, 7, 2), (2, 37, 11, 2), ("edge", 20, 3, 1)])
def test_emulated_pathway_matches_oracle(oracle, network, cfg, ncol_max, source, grid):
    net, kf, kr, n, ncol, ld = case(network, oracle, cfg, ncol_max)
    if cfg == "edge":
        kr = np.where(np.isfinite(kr), kr, 0.0)
    want = oracle.pathway(net, kf, kr, n, source, ncol)
    got = run_emulated(net, kf, kr, n, ncol, ld, source, grid)
    check(net, kf, kr, n, ncol, source, got, want, "emulated xod_pathway config %s from species %d" % (cfg, source))


def test_emulated_pathway_with_hub_species_split_over_warps(oracle, network):
    """The 594-species network: hub species own thousands of incoming edges and are cut into parts on several warps."""
    from paper_2512_06729_b200 import binding
    net, kf, kr, n, ncol, ld = case(network, oracle, 3, 5)
    want = oracle.pathway(net, kf, kr, n, 17, ncol)
    got = run_emulated(net, kf, kr, n, ncol, ld, 17, 1)
    check(net, kf, kr, n, ncol, 17, got, want, "emulated xod_pathway config 3")


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,ncol_max,source", [(1, 20, 0), (2, 120, 11), ("edge", 75, 3), (3, 150, 17), (5, 300, 100)])
def test_pathway_matches_oracle_on_gpu(oracle, network, cfg, ncol_max, source):
    import torch
    assert torch.cuda.is_available(), "no CUDA device: the gpu tests need the B200 box (there is no CPU fallback)"
    from paper_2512_06729_b200 import binding, build
    build.build()
    net, kf, kr, n, ncol, ld = case(network, oracle, cfg, ncol_max)
    if cfg == "edge":
        kr = np.where(np.isfinite(kr), kr, 0.0)
    want = oracle.pathway(net, kf, kr, n, source, ncol)
    h = binding.Network(net, device=0)
    dist = G.empty(net.n_species, ld)
    pred = torch.full((net.n_species, ld), -7, dtype=torch.int32, device="cuda")
    via = torch.full((net.n_species, ld), -7, dtype=torch.int32, device="cuda")
    ws = G.workspace(h.pathway_workspace_bytes(ncol))
    h.pathway(ncol, ld, G.dev(kf), G.dev(kr), G.dev(n), source, dist, pred, via, ws)
    h.check_status()
    got = (G.host(dist), pred.cpu().numpy(), via.cpu().numpy())
    check(net, kf, kr, n, ncol, source, got, want, "xod_pathway config %s from species %d" % (cfg, source))
    h.close()
