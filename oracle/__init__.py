"""ctypes front end of the CPU oracle (oracle/xodiac_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this.  It imports nothing from the CUDA package; it takes any object with the
network attributes (composition, nasa_lo, ..., t_ref) as plain numpy arrays.

`Oracle()` loads the long-double build (parity checks); `Oracle(extended=False)` loads the
pure-fp64 build (the one timed as the CPU baseline).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "xodiac_oracle.c")
_LIBS = {True: os.path.join(_HERE, "liboracle.so"), False: os.path.join(_HERE, "liboracle_f64.so")}


def build(force=False):
    """Compile both oracle builds with gcc -O2 (no fast-math)."""
    for extended, out in _LIBS.items():
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-o", out, _SRC, "-lm"]
        if not extended:
            cmd.insert(1, "-DXOD_ORACLE_DOUBLE")
        subprocess.run(cmd, check=True)


class _Net(C.Structure):
    _fields_ = [("n_species", C.c_int), ("n_elements", C.c_int), ("n_reactions", C.c_int),
                ("composition", C.c_void_p), ("nasa_lo", C.c_void_p), ("nasa_hi", C.c_void_p),
                ("t_mid", C.c_void_p), ("type", C.c_void_p), ("reactants", C.c_void_p),
                ("products", C.c_void_p), ("reversible", C.c_void_p), ("arrh", C.c_void_p),
                ("arrh_low", C.c_void_p), ("troe_fc", C.c_void_p), ("t_ref", C.c_void_p)]


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


class Oracle:
    def __init__(self, extended=True):
        build()
        self.lib = C.CDLL(_LIBS[bool(extended)])
        self.extended = bool(extended)
        L = self.lib
        L.orc_real_mant_dig.restype = C.c_int
        for name in ("orc_source_csr", "orc_jac_pattern", "orc_jacobian"):
            getattr(L, name).restype = C.c_long
        self.mant_dig = L.orc_real_mant_dig()

    # -- network marshalling (keeps the numpy arrays alive next to the struct)
    def _net(self, net):
        keep = {
            "composition": np.ascontiguousarray(net.composition, dtype=np.int32),
            "nasa_lo": _f64(net.nasa_lo), "nasa_hi": _f64(net.nasa_hi), "t_mid": _f64(net.t_mid),
            "type": np.ascontiguousarray(net.type, dtype=np.int32),
            "reactants": np.ascontiguousarray(net.reactants, dtype=np.int32),
            "products": np.ascontiguousarray(net.products, dtype=np.int32),
            "reversible": np.ascontiguousarray(net.reversible, dtype=np.uint8),
            "arrh": _f64(net.arrh), "arrh_low": _f64(net.arrh_low), "troe_fc": _f64(net.troe_fc),
            "t_ref": None if getattr(net, "t_ref", None) is None else _f64(net.t_ref),
        }
        ns, ne = keep["composition"].shape
        s = _Net(ns, ne, keep["type"].shape[0], *[_ptr(keep[k]) for k in (
            "composition", "nasa_lo", "nasa_hi", "t_mid", "type", "reactants", "products",
            "reversible", "arrh", "arrh_low", "troe_fc", "t_ref")])
        return s, keep

    @staticmethod
    def _dims(net):
        return int(np.shape(net.composition)[0]), int(np.shape(net.type)[0])

    def thermo(self, net, T, ncol=None):
        """cp/R, H/RT, S/R, G/RT, each [n_species][ld]."""
        T = _f64(T)
        ld = T.shape[0]
        ncol = ld if ncol is None else ncol
        ns, _ = self._dims(net)
        s, keep = self._net(net)
        out = [np.zeros((ns, ld)) for _ in range(4)]
        self.lib.orc_thermo(C.byref(s), C.c_long(ncol), C.c_long(ld), _ptr(T), *[_ptr(o) for o in out])
        return tuple(out)

    def rate_coeffs(self, net, T, P, J, ncol=None):
        """k_f, k_r [n_reactions][ld] in user reaction order."""
        T, P = _f64(T), _f64(P)
        ld = T.shape[0]
        ncol = ld if ncol is None else ncol
        _, nr = self._dims(net)
        J = _f64(J).reshape(-1, ld) if J is not None and np.size(J) else np.zeros((0, ld))
        s, keep = self._net(net)
        kf, kr = np.zeros((nr, ld)), np.zeros((nr, ld))
        self.lib.orc_rate_coeffs(C.byref(s), C.c_long(ncol), C.c_long(ld), _ptr(T), _ptr(P), _ptr(J),
                                 _ptr(kf), _ptr(kr))
        return kf, kr

    def rates(self, net, kf, kr, n, ncol=None):
        kf, kr, n = _f64(kf), _f64(kr), _f64(n)
        ld = n.shape[1]
        ncol = ld if ncol is None else ncol
        s, keep = self._net(net)
        qf, qr = np.zeros_like(kf), np.zeros_like(kr)
        self.lib.orc_rates(C.byref(s), C.c_long(ncol), C.c_long(ld), _ptr(kf), _ptr(kr), _ptr(n),
                           _ptr(qf), _ptr(qr))
        return qf, qr

    def source(self, net, kf, kr, n, ncol=None):
        """dn/dt, P, L [n_species][ld]."""
        kf, kr, n = _f64(kf), _f64(kr), _f64(n)
        ld = n.shape[1]
        ncol = ld if ncol is None else ncol
        s, keep = self._net(net)
        out = [np.zeros_like(n) for _ in range(3)]
        rc = self.lib.orc_source(C.byref(s), C.c_long(ncol), C.c_long(ld), _ptr(kf), _ptr(kr), _ptr(n),
                                 *[_ptr(o) for o in out])
        assert rc == 0
        return tuple(out)

    def source_from_state(self, net, T, P, J, n, ncol=None):
        """The whole path a1..a8: (T, P, J, n) -> dn/dt, P, L (k_f, k_r rounded to double between)."""
        kf, kr = self.rate_coeffs(net, T, P, J, ncol)
        return self.source(net, kf, kr, n, ncol)

    def source_csr(self, net):
        ns, _ = self._dims(net)
        s, keep = self._net(net)
        row_ptr = np.zeros(ns + 1, dtype=np.int64)
        nnz = self.lib.orc_source_csr(C.byref(s), _ptr(row_ptr), None, None)
        rxn, nu = np.zeros(nnz, dtype=np.int32), np.zeros(nnz, dtype=np.int32)
        self.lib.orc_source_csr(C.byref(s), _ptr(row_ptr), _ptr(rxn), _ptr(nu))
        return row_ptr, rxn, nu

    def jac_pattern(self, net):
        ns, _ = self._dims(net)
        s, keep = self._net(net)
        row_ptr = np.zeros(ns + 1, dtype=np.int64)
        nnz = self.lib.orc_jac_pattern(C.byref(s), _ptr(row_ptr), None)
        col = np.zeros(nnz, dtype=np.int32)
        self.lib.orc_jac_pattern(C.byref(s), _ptr(row_ptr), _ptr(col))
        return row_ptr, col

    def jacobian_dense(self, net, kf, kr, n, c):
        """Dense [n_species][n_species] Jacobian and tolerance scale of column c."""
        kf, kr, n = _f64(kf), _f64(kr), _f64(n)
        ns, _ = self._dims(net)
        s, keep = self._net(net)
        d, sc = np.zeros((ns, ns)), np.zeros((ns, ns))
        rc = self.lib.orc_jacobian_dense(C.byref(s), C.c_long(n.shape[1]), _ptr(kf), _ptr(kr), _ptr(n),
                                         C.c_long(c), _ptr(d), _ptr(sc))
        assert rc == 0
        return d, sc

    def jacobian(self, net, kf, kr, n, row_ptr, col, ncol=None):
        """Pattern values and scales [nnz][ld]; asserts the dense matrix is zero off-pattern."""
        kf, kr, n = _f64(kf), _f64(kr), _f64(n)
        ld = n.shape[1]
        ncol = ld if ncol is None else ncol
        s, keep = self._net(net)
        row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
        col = np.ascontiguousarray(col, dtype=np.int32)
        jac, sc = np.zeros((col.shape[0], ld)), np.zeros((col.shape[0], ld))
        bad = self.lib.orc_jacobian(C.byref(s), C.c_long(ncol), C.c_long(ld), _ptr(kf), _ptr(kr),
                                    _ptr(n), _ptr(row_ptr), _ptr(col), _ptr(jac), _ptr(sc))
        if bad != 0:
            raise AssertionError("oracle: %d dense Jacobian entries outside the pattern are non-zero" % bad)
        return jac, sc

    # ---- f1: backward-Euler Newton step
    def newton_system(self, net, kf, kr, n_old, dt, y, c):
        """A = I - dt Jac(y) [ns][ns] and b = -(y - n_old - dt f(y)) [ns] of column c, rounded to double."""
        kf, kr, n_old, y, dt = _f64(kf), _f64(kr), _f64(n_old), _f64(y), _f64(dt)
        ns, _ = self._dims(net)
        s, keep = self._net(net)
        A, b = np.zeros((ns, ns)), np.zeros(ns)
        rc = self.lib.orc_newton_system(C.byref(s), C.c_long(y.shape[1]), _ptr(kf), _ptr(kr), _ptr(n_old), _ptr(dt),
                                        _ptr(y), C.c_long(c), _ptr(A), _ptr(b))
        assert rc == 0
        return A, b

    def newton_step(self, net, kf, kr, n_old, dt, y, ncol=None):
        """delta, y + delta [n_species][ld] of one Newton iteration of the backward-Euler step."""
        kf, kr, n_old, y, dt = _f64(kf), _f64(kr), _f64(n_old), _f64(y), _f64(dt)
        ld = y.shape[1]
        ncol = ld if ncol is None else ncol
        s, keep = self._net(net)
        delta, y_new = np.zeros_like(y), np.zeros_like(y)
        rc = self.lib.orc_newton_step(C.byref(s), C.c_long(ncol), C.c_long(ld), _ptr(kf), _ptr(kr), _ptr(n_old),
                                      _ptr(dt), _ptr(y), _ptr(delta), _ptr(y_new))
        if rc != 0:
            raise ArithmeticError("oracle Newton step failed (%d: -2 = singular matrix)" % rc)
        return delta, y_new

    # ---- f2: photolysis rate constants
    def photo_rates(self, ph, n, dz, j0, j_diff, mu, t_f, n_atm, n_layers, want_tau=False):
        """k_ph [n_photo][ld] (and the layer-centre optical depths [n_bins][ld]).  `ph` is any object with
        abs_species [n_abs], sigma_ext [n_abs][n_bins], sigma_ph [n_photo][n_bins], dlambda [n_bins]."""
        n, dz, j0, mu, t_f = _f64(n), _f64(dz), _f64(j0), _f64(mu), _f64(t_f)
        ld = n.shape[1]
        sig_e, sig_p, dl = _f64(ph.sigma_ext), _f64(ph.sigma_ph), _f64(ph.dlambda)
        ab = np.ascontiguousarray(ph.abs_species, dtype=np.int32)
        nph, nb = sig_p.shape
        jd = None if j_diff is None else _f64(j_diff)
        kph = np.zeros((nph, ld))
        tau = np.zeros((nb, ld)) if want_tau else None
        rc = self.lib.orc_photo_rates(C.c_int(nph), C.c_int(nb), C.c_int(ab.shape[0]), _ptr(ab), _ptr(sig_e), _ptr(sig_p),
                                      _ptr(dl), C.c_long(n_atm), C.c_long(n_layers), C.c_long(ld), _ptr(n), _ptr(dz), _ptr(j0),
                                      _ptr(jd), _ptr(mu), _ptr(t_f), _ptr(kph), _ptr(tau))
        assert rc == 0
        return (kph, tau) if want_tau else kph

    # ---- f3: molecular-diffusion transport terms (Eq. 3-4)
    def transport(self, n, T, n_gas, D, mass, alpha_T, mbar, grav, dz, n_atm, n_layers, want_d=False):
        """tr [n_species][ld] (and d_{k+1/2} [n_species][ld])."""
        n, T, n_gas, D = _f64(n), _f64(T), _f64(n_gas), _f64(D)
        mass, alpha_T, mbar, grav, dz = _f64(mass), _f64(alpha_T), _f64(mbar), _f64(grav), _f64(dz)
        ns, ld = n.shape
        tr = np.zeros((ns, ld))
        d = np.zeros((ns, ld)) if want_d else None
        rc = self.lib.orc_transport(C.c_int(ns), C.c_long(n_atm), C.c_long(n_layers), C.c_long(ld), _ptr(n), _ptr(T), _ptr(n_gas),
                                    _ptr(D), _ptr(mass), _ptr(alpha_T), _ptr(mbar), _ptr(grav), _ptr(dz), _ptr(tr), _ptr(d))
        assert rc == 0
        return (tr, d) if want_d else tr

    # ---- f4: reaction pathway analyser
    def pathway(self, net, kf, kr, n, source, ncol=None):
        """dist [n_species][ld] (sum of 1/rate along the fastest route from `source`), pred, via (int32)."""
        kf, kr, n = _f64(kf), _f64(kr), _f64(n)
        ld = n.shape[1]
        ncol = ld if ncol is None else ncol
        ns, _ = self._dims(net)
        s, keep = self._net(net)
        dist = np.full((ns, ld), np.nan)
        pred, via = np.full((ns, ld), -2, dtype=np.int32), np.full((ns, ld), -2, dtype=np.int32)
        rc = self.lib.orc_pathway(C.byref(s), C.c_long(ncol), C.c_long(ld), _ptr(kf), _ptr(kr), _ptr(n), C.c_int(source),
                                  _ptr(dist), _ptr(pred), _ptr(via))
        assert rc == 0
        return dist, pred, via

    # ---- f4: thermochemical-equilibrium composition
    def equilibrium(self, net, T, P, b, ncol=None, max_iter=2000, tol=1e-15, want_pi=False):
        """n [n_species][ld] minimising the Gibbs energy at (T, P) for element abundances b [n_elements][ld];
        also the iterations used per column (negative: not converged) and, on request, the element potentials."""
        T, P, b = _f64(T), _f64(P), _f64(b)
        ld = b.shape[1]
        ncol = ld if ncol is None else ncol
        ns, _ = self._dims(net)
        ne = np.asarray(net.composition).shape[1]
        s, keep = self._net(net)
        n = np.full((ns, ld), np.nan)
        pi = np.full((ne, ld), np.nan)
        iters = np.zeros(ld, dtype=np.int32)
        rc = self.lib.orc_equilibrium(C.byref(s), C.c_long(ncol), C.c_long(ld), _ptr(T), _ptr(P), _ptr(b), C.c_int(max_iter),
                                      C.c_double(tol), _ptr(n), _ptr(pi), _ptr(iters))
        if rc != 0:
            raise ArithmeticError("oracle equilibrium failed (%d: -2 singular system, -3 element without abundance)" % rc)
        return (n, iters, pi) if want_pi else (n, iters)
