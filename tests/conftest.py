import functools
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (runs on the B200 box)")


# `pytest -x -m gpu` stops at the first failure: the hot path (test_gpu_parity.py) must have run
# before any of the section 8(f) rows gets its chance to stop the session.  Everything else keeps its order.
_GPU_ORDER = ["test_gpu_parity", "test_newton_step", "test_photo_rates", "test_transport", "test_pathway", "test_equilibrium"]


def pytest_collection_modifyitems(session, config, items):
    def rank(item):
        if item.get_closest_marker("gpu") is None:
            return -1
        name = item.module.__name__.rsplit(".", 1)[-1]
        r = _GPU_ORDER.index(name) if name in _GPU_ORDER else len(_GPU_ORDER)
        # inside the hot-path file: a1-a8 (kernels that ran on a GPU in round 1) before a9's tiled Jacobian kernel
        # (new in round 2) and before the tests that mix both
        if "jacobian" in item.name or "zero_densities" in item.name:
            r += 0.5
        elif "random_networks" in item.name:
            r += 0.6
        return r
    items.sort(key=rank)       # stable: the order inside a module and among the CPU tests is unchanged


@functools.lru_cache(maxsize=None)
def _network(cfg):
    from paper_2512_06729_b200 import synth
    return synth.config_network(cfg)


@pytest.fixture(scope="session")
def network():
    return _network


@pytest.fixture(scope="session")
def oracle():
    from oracle import Oracle
    return Oracle()


@pytest.fixture(scope="session")
def oracle_f64():
    from oracle import Oracle
    return Oracle(extended=False)


def load_table1():
    rows = {}
    with open(os.path.join(ROOT, "tests", "golden", "table1_nasa7.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            p = line.split()
            rows[p[0]] = np.array([float(x) for x in p[1:8]])
    return rows


class SimpleNet:
    """Hand-written network description with the same attribute names as synth.Network."""

    def __init__(self, composition, nasa_lo, nasa_hi, t_mid, rtype, reactants, products, reversible,
                 arrh, arrh_low=None, troe_fc=None, t_ref=None, element_names=None):
        self.composition = np.asarray(composition, dtype=np.int32).reshape(len(t_mid), -1)
        self.nasa_lo = np.asarray(nasa_lo, dtype=np.float64).reshape(-1, 7)
        self.nasa_hi = np.asarray(nasa_hi, dtype=np.float64).reshape(-1, 7)
        self.t_mid = np.asarray(t_mid, dtype=np.float64)
        self.type = np.asarray(rtype, dtype=np.int32)
        nr = self.type.shape[0]

        def pad(side):
            out = -np.ones((nr, 3), dtype=np.int32)
            for r, s in enumerate(side):
                out[r, :len(s)] = s
            return out

        self.reactants = pad(reactants)
        self.products = pad(products)
        self.reversible = np.asarray(reversible, dtype=np.uint8)
        self.arrh = np.asarray(arrh, dtype=np.float64).reshape(nr, 3)
        self.arrh_low = (np.zeros((nr, 3)) if arrh_low is None
                         else np.asarray(arrh_low, dtype=np.float64).reshape(nr, 3))
        self.troe_fc = np.ones(nr) if troe_fc is None else np.asarray(troe_fc, dtype=np.float64)
        self.t_ref = np.ones(nr) if t_ref is None else np.asarray(t_ref, dtype=np.float64)
        self.element_names = element_names or ["E%d" % e for e in range(self.composition.shape[1])]

    n_species = property(lambda self: self.composition.shape[0])
    n_elements = property(lambda self: self.composition.shape[1])
    n_reactions = property(lambda self: self.type.shape[0])
    n_photo = property(lambda self: int(np.count_nonzero(self.type == 3)))
