"""CPU-side checks of the C-ABI boundary: the library loads and exports every symbol that
include/xodiac.h declares, the host packer's CSR layouts are bit-identical to the oracle's
independently built ones, the type sort is stable, and argument errors are reported.
No compute call runs here (no GPU): networks are created with cuda_device = -1."""
import os
import re

import numpy as np
import pytest

from conftest import ROOT, SimpleNet

from paper_2512_06729_b200 import binding, build


@pytest.fixture(scope="module")
def built():
    build.build()
    return binding.lib()


def test_library_exports_every_declared_symbol(built):
    header = open(os.path.join(ROOT, "include", "xodiac.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(xod_[a-z0-9_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(built, name), name


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_csr_layouts_bit_exact_against_oracle(built, oracle, network, cfg):
    """north_star: "the CSR layout bit-exact".  Two code bases, two constructions (oracle: dense
    boolean matrix and nested loops; library: sort-based), compared bitwise."""
    net = network(cfg)
    h = binding.Network(net, device=-1)
    rp, rxn, nu = h.source_csr()
    orp, orxn, onu = oracle.source_csr(net)
    assert rp.dtype == orp.dtype == np.int64 and rxn.dtype == orxn.dtype == np.int32
    assert np.array_equal(rp, orp) and np.array_equal(rxn, orxn) and np.array_equal(nu, onu)
    jp, jc = h.jac_pattern()
    ojp, ojc = oracle.jac_pattern(net)
    assert np.array_equal(jp, ojp) and np.array_equal(jc, ojc)
    assert h.nnz_source == rxn.shape[0] and h.nnz_jac == jc.shape[0]
    assert (h.n_species, h.n_reactions, h.n_photo) == (net.n_species, net.n_reactions, net.n_photo)


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_type_sort_is_stable_and_photo_rows_follow_user_order(built, network, cfg):
    net = network(cfg)
    h = binding.Network(net, device=-1)
    perm = h.perm()
    assert sorted(perm.tolist()) == list(range(net.n_reactions))
    want = np.argsort(net.type, kind="stable").astype(np.int32)
    assert np.array_equal(perm, want)
    assert np.array_equal(h.photo_index(), np.flatnonzero(net.type == binding.XOD_PHOTO).astype(np.int32))


def _tiny(**over):
    z = np.zeros((3, 7))
    kw = dict(composition=[[1], [1], [2]], nasa_lo=z, nasa_hi=z, t_mid=[1000.0] * 3, rtype=[1, 3],
              reactants=[[0, 1], [2]], products=[[2], [0, 1]], reversible=[1, 0],
              arrh=[[1e-10, 0, 0], [0, 0, 0]])
    kw.update(over)
    return SimpleNet(**kw)


def test_argument_errors_are_reported(built):
    ok = binding.Network(_tiny(), device=-1)
    assert ok.n_photo == 1
    with pytest.raises(binding.XodError) as e:
        binding.Network(_tiny(composition=[[1], [1], [3]]), device=-1)
    assert e.value.status == 2 and "reaction 0" in str(e.value)              # XOD_ERR_UNBALANCED
    binding.Network(_tiny(composition=[[1], [1], [3]]), device=-1,
                    flags=binding.XOD_FLAG_SKIP_BALANCE_CHECK)
    for bad in (dict(reversible=[1, 1]),                                        # reversible photolysis
                dict(rtype=[1, 7]),                                             # bad type
                dict(reactants=[[0, 5], [2]]),                                  # index out of range
                dict(arrh=[[-1.0, 0, 0], [0, 0, 0]]),                           # alpha <= 0
                dict(rtype=[2, 3], troe_fc=[1.5, 1.0], arrh_low=[[1e-30, 0, 0], [0, 0, 0]])):  # Fc > 1
        with pytest.raises(binding.XodError) as e:
            binding.Network(_tiny(**bad), device=-1)
        assert e.value.status == 1, bad


def test_compute_without_device_fails_loudly(built):
    h = binding.Network(_tiny(), device=-1)
    st = built.xod_thermo(h._h, binding.C.c_int64(1), binding.C.c_int64(1), None, None, None, None, None, None)
    assert st == 4                                                              # XOD_ERR_CUDA, never a CPU fallback
    assert h.source_fused_workspace_bytes(150) > 0
    C = binding.C
    st = built.xod_equilibrium(h._h, C.c_int64(1), C.c_int64(1), None, None, None, C.c_int32(0), C.c_double(0.0), None, None, None, None)
    assert st == 4


def test_charge_as_an_element_and_padding_anywhere(built, oracle):
    """C -> C+ + e- (PAPER.md:363): charge carried as an extra 'element' that may be negative;
    the -1 padding may sit before a species index."""
    z = np.zeros((3, 7))
    net = SimpleNet([[1, 0], [1, 1], [0, -1]], z, z, [1000.0] * 3, [3, 1], [[-1, 0], [1, 2]],
                    [[1, -1, 2], [0]], [0, 1], [[0, 0, 0], [1e-9, 0, 0]], element_names=["C", "q"])
    h = binding.Network(net, device=-1)
    assert np.array_equal(h.source_csr()[1], oracle.source_csr(net)[1])
    assert np.array_equal(h.jac_pattern()[1], oracle.jac_pattern(net)[1])


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_fused_path_tables_are_consistent(built, network, cfg):
    """Host-side check of the single-kernel path's tables, decoded as the kernel decodes them: every
    source-CSR entry is scheduled exactly once, no accumulator row is shared by two row tasks of a
    chunk (the atomic-free guarantee), species slots and J rows survive the packing."""
    net = network(cfg)
    h = binding.Network(net, device=-1)
    info = h.fused_info()
    assert info["enabled"] == 1 and info["smem_bytes"] <= 227 * 1024
    assert info["chunk"] % 80 == 0 and info["npad"] == info["chunk"] * info["nchunk"] >= net.n_reactions
    h.selfcheck()


def test_fused_path_disabled_for_many_thermo_intervals(built, network):
    import copy
    net = copy.copy(network(2))
    net.t_mid = 300.0 + 10.0 * np.arange(net.n_species)
    h = binding.Network(net, device=-1)
    assert h.fused_info()["enabled"] == 0
    h.selfcheck()
