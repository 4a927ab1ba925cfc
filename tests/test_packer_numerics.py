"""CPU test of the packer's arithmetic (no GPU): the log2-domain coefficient tables of the fused path,
evaluated here with numpy exactly as the kernels' formulas read (include/xodiac.h,
xod_network_fused_params), must reproduce the oracle's k_f and k_r to the GPU tolerance.  This pins
the folding of Eq. 7 / 10-12 / 15 and of the per-interval sums of NASA-7
Gibbs polynomials without a device."""
import os

import numpy as np
import pytest

from conftest import ROOT
from paper_2512_06729_b200 import binding, build

LOG2_KB = np.log2(1.380649e-16)


@pytest.fixture(scope="module")
def built():
    build.build()
    return binding.lib()


def evaluate_tables(h, T, P, J):
    """k_f, k_r [n_reactions][ncol] from the parameter blocks (numpy longdouble, formulas of the header)."""
    info = h.fused_info()
    T = np.asarray(T, dtype=np.longdouble)
    l2T, iT = np.log2(T), 1 / T
    lM = np.log2(np.asarray(P, dtype=np.longdouble)) - np.longdouble(LOG2_KB) - l2T
    kf = np.zeros((h.n_reactions, T.size))
    kr = np.zeros((h.n_reactions, T.size))
    bp = h.fused_params(0)[3]
    interval = (T[:, None] > bp[None, :]).sum(axis=1)
    photo_rows = {int(u): p for p, u in enumerate(h.photo_index())}
    for g in np.unique(interval):
        user, kind, coef, _ = h.fused_params(int(g))
        cols = np.flatnonzero(interval == g)
        c = coef.astype(np.longdouble)
        for pp in np.flatnonzero(user >= 0):
            r = user[pp]
            if kind[pp] == 2:
                kf[r, cols] = J[photo_rows[r], cols]
                continue
            y = c[pp, 0] + c[pp, 1] * l2T[cols] + c[pp, 2] * iT[cols]
            Tc = T[cols]
            z = c[pp, 3] + c[pp, 4] * l2T[cols] + c[pp, 5] * iT[cols] - Tc * (
                c[pp, 6] + Tc * (c[pp, 7] + Tc * (c[pp, 8] + Tc * c[pp, 9])))
            if kind[pp] == 0:
                kf[r, cols] = np.exp2(y)
                kr[r, cols] = np.exp2(z)
            else:
                w = c[pp, 10] + c[pp, 11] * l2T[cols] + c[pp, 12] * iT[cols] + lM[cols]
                lp = w - y
                lF = c[pp, 13] / (1 + (lp * c[pp, 14]) ** 2)
                ym = np.minimum(w, y) + lF
                den = 1 / (1 + np.exp2(-np.abs(lp)))
                kf[r, cols] = np.exp2(ym) * den
                kr[r, cols] = np.exp2(ym + z) * den
    return kf, kr


@pytest.mark.parametrize("cfg", [1, 2])
def test_tables_reproduce_oracle_coefficients(built, oracle, network, cfg):
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    h = binding.Network(net, device=-1)
    atm = synth.config_atmosphere(cfg, net)
    # add columns on both sides of every breakpoint so each interval table is exercised
    T = np.concatenate([atm.T[:atm.ncol], [250.0, 300.0, 300.5, 499.0, 500.0, 650.0, 700.0, 701.0, 999.0, 1000.0, 1001.0]])
    P = np.concatenate([atm.P[:atm.ncol], np.full(11, 1.0e5)])
    J = np.concatenate([atm.J[:, :atm.ncol], np.full((net.n_photo, 11), 1e-5)], axis=1)
    kf, kr = evaluate_tables(h, T, P, J)
    okf, okr = oracle.rate_coeffs(net, T, P, J)
    fin = np.isfinite(okr) & (np.abs(okr) > 1e-300)
    assert np.all(np.abs(kf - okf) <= 1e-12 * np.abs(okf))
    assert np.all(np.abs(kr[fin] - okr[fin]) <= 1e-12 * np.abs(okr[fin]))
    assert np.array_equal(np.isinf(kr), np.isinf(okr))
    assert np.all(kr[net.type == 3] == 0.0)


def test_large_network_tables_on_sampled_reactions(built, oracle, network):
    """Config 3 (594 species / 7 720 reactions): the same check on a few columns (python loop over reactions)."""
    from paper_2512_06729_b200 import synth
    net = network(3)
    h = binding.Network(net, device=-1)
    atm = synth.config_atmosphere(3, net)
    cols = np.array([0, 40, 75, 110, 149])
    T = np.concatenate([atm.T[cols], [480.0, 980.0]])
    P = np.concatenate([atm.P[cols], [1e4, 1e2]])
    J = np.concatenate([atm.J[:, cols], np.full((net.n_photo, 2), 1e-6)], axis=1)
    kf, kr = evaluate_tables(h, T, P, J)
    okf, okr = oracle.rate_coeffs(net, T, P, J)
    fin = np.isfinite(okr) & (np.abs(okr) > 1e-300)
    assert np.all(np.abs(kf - okf) <= 1e-12 * np.abs(okf))
    assert np.all(np.abs(kr[fin] - okr[fin]) <= 1e-12 * np.abs(okr[fin]))


def test_exp2_polynomial_constants_match_their_generator():
    """kExp2C in csrc/xod_math.cuh must be what csrc/gen_exp2_coeffs.py prints (degree 9), and the polynomial
    must hold the 3.7e-14 relative error the kernel documentation claims (exact rational evaluation)."""
    import re
    import subprocess
    import sys
    from fractions import Fraction
    mp = pytest.importorskip("mpmath")
    csrc = os.path.join(ROOT, "paper_2512_06729_b200", "csrc")
    text = open(os.path.join(csrc, "xod_math.cuh")).read()
    body = re.search(r"kExp2C\[10\]\s*=\s*\{([^}]*)\}", text).group(1)
    in_header = [float(x) for x in body.replace("\n", " ").split(",")]
    out = subprocess.run([sys.executable, os.path.join(csrc, "gen_exp2_coeffs.py"), "9"], capture_output=True, text=True, check=True).stdout
    generated = {int(m.group(1)): float(m.group(2)) for m in re.finditer(r"c(\d+)\s*=\s*(\S+)", out)}
    assert in_header == [generated[k] for k in range(10)]
    mp.mp.dps = 50
    worst = 0.0
    for k in range(-400, 401):
        f = Fraction(k, 800)
        p = Fraction(0)
        for c in reversed(in_header):
            p = p * f + Fraction(c)
        exact = mp.power(2, mp.mpf(f.numerator) / f.denominator)
        worst = max(worst, abs(float((mp.mpf(p.numerator) / p.denominator - exact) / exact)))
    assert worst <= 4e-14
