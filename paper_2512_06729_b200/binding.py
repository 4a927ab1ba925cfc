"""Thin ctypes binding of libxodiac.so: the same names as include/xodiac.h, argument marshalling
only.  Device buffers are torch tensors (fp64, CUDA); every step of the path runs in the CUDA
kernels of the library.  There is no CPU fallback: a missing library raises at first use."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# XOD_CHECK=1 selects the bounds-checked debugging build (same sources, -DXOD_CHECK; see build.py)
_LIB_PATH = os.path.join(_HERE, "libxodiac_check.so" if os.environ.get("XOD_CHECK") else "libxodiac.so")
_lib = None

XOD_OK = 0
XOD_UNI, XOD_BI, XOD_FALLOFF, XOD_PHOTO = 0, 1, 2, 3
XOD_FLAG_SKIP_BALANCE_CHECK, XOD_FLAG_BUILD_LU = 1, 2
XOD_TUNE_CHUNK_COLS, XOD_TUNE_TIMING, XOD_TUNE_SPLIT, XOD_TUNE_FUSED_KERNEL, XOD_TUNE_JAC_TILED = 0, 1, 2, 3, 4
KERNEL_NAMES = ["thermo", "prologue", "rates", "rates_from_k", "source", "jacobian", "fused", "fused_combine", "rate_coeffs", "jac_tiled", "newton_assemble", "lu_factor", "lu_solve", "photo_gemm", "photo_flux", "transport", "path_weights", "pathway", "equilibrium"]
STATUS_NAMES = {0: "XOD_OK", 1: "XOD_ERR_INVALID_ARG", 2: "XOD_ERR_UNBALANCED", 3: "XOD_ERR_ALLOC",
                4: "XOD_ERR_CUDA", 5: "XOD_ERR_WORKSPACE"}

EXPORTS = ["xod_network_create", "xod_network_destroy", "xod_last_error", "xod_network_sizes",
           "xod_network_perm", "xod_network_photo_index", "xod_network_source_csr",
           "xod_network_jac_pattern", "xod_network_tune", "xod_thermo",
           "xod_rate_coeffs_workspace_bytes", "xod_rate_coeffs", "xod_source_workspace_bytes",
           "xod_source", "xod_source_fused_workspace_bytes", "xod_source_fused", "xod_jacobian",
           "xod_source_fused_host", "xod_probe_fp64_peak", "xod_network_timing_read", "xod_launch_count", "xod_network_fused_info", "xod_network_selfcheck", "xod_network_fused_params",
           "xod_check_status", "xod_build_has_checks", "xod_network_jac_info", "xod_network_lu_info", "xod_network_lu_pattern",
           "xod_newton_workspace_bytes", "xod_newton_step", "xod_photo_create", "xod_photo_destroy",
           "xod_photo_workspace_bytes", "xod_photo_rates", "xod_transport",
           "xod_pathway_workspace_bytes", "xod_pathway", "xod_equilibrium",
           "xod_source_workspace_bytes_dndt", "xod_source_fused_workspace_bytes_dndt"]


class XodError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("%s: %s" % (STATUS_NAMES.get(status, status), message))
        self.status = status


class _Desc(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_elements", C.c_int32), ("n_reactions", C.c_int32),
                ("composition", C.c_void_p), ("nasa_lo", C.c_void_p), ("nasa_hi", C.c_void_p),
                ("t_mid", C.c_void_p), ("type", C.c_void_p), ("reactants", C.c_void_p),
                ("products", C.c_void_p), ("reversible", C.c_void_p), ("arrh", C.c_void_p),
                ("arrh_low", C.c_void_p), ("troe_fc", C.c_void_p), ("t_ref", C.c_void_p),
                ("flags", C.c_uint32)]


def lib():
    """Load libxodiac.so (fails loudly if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(os.path.basename(_LIB_PATH) + " is missing: run `python -m paper_2512_06729_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        L.xod_last_error.restype = C.c_char_p
        for name in ("xod_rate_coeffs_workspace_bytes", "xod_source_workspace_bytes",
                     "xod_source_fused_workspace_bytes", "xod_newton_workspace_bytes", "xod_pathway_workspace_bytes",
                     "xod_source_workspace_bytes_dndt", "xod_source_fused_workspace_bytes_dndt"):
            getattr(L, name).restype = C.c_size_t
            getattr(L, name).argtypes = [C.c_void_p, C.c_int64]
        L.xod_photo_workspace_bytes.restype = C.c_size_t
        L.xod_photo_workspace_bytes.argtypes = [C.c_void_p, C.c_int64]
        L.xod_photo_destroy.restype = None
        L.xod_photo_destroy.argtypes = [C.c_void_p]
        L.xod_launch_count.restype = C.c_int64
        L.xod_network_destroy.restype = None
        L.xod_network_destroy.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _check(st):
    if st != XOD_OK:
        raise XodError(st, lib().xod_last_error().decode())


def _np(a, dtype):
    return None if a is None else np.ascontiguousarray(a, dtype=dtype)


def _hp(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


def _dp(t):
    """Device pointer of a torch tensor (fp64, CUDA, contiguous rows) or None."""
    if t is None:
        return None
    assert t.is_cuda and t.dtype.is_floating_point and t.element_size() == 8 and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(int(stream))


class Network:
    """xod_network handle.  `net` is any object with the attributes of synth.Network."""

    def __init__(self, net, device=0, flags=0):
        L = lib()
        keep = dict(
            composition=_np(net.composition, np.int32), nasa_lo=_np(net.nasa_lo, np.float64),
            nasa_hi=_np(net.nasa_hi, np.float64), t_mid=_np(net.t_mid, np.float64),
            type=_np(net.type, np.int32), reactants=_np(net.reactants, np.int32),
            products=_np(net.products, np.int32), reversible=_np(net.reversible, np.uint8),
            arrh=_np(net.arrh, np.float64), arrh_low=_np(getattr(net, "arrh_low", None), np.float64),
            troe_fc=_np(getattr(net, "troe_fc", None), np.float64),
            t_ref=_np(getattr(net, "t_ref", None), np.float64))
        ns, ne = keep["composition"].shape
        d = _Desc(ns, ne, keep["type"].shape[0], *[_hp(keep[k]) for k in (
            "composition", "nasa_lo", "nasa_hi", "t_mid", "type", "reactants", "products", "reversible",
            "arrh", "arrh_low", "troe_fc", "t_ref")], flags)
        h = C.c_void_p()
        _check(L.xod_network_create(C.byref(d), C.c_int(device), C.byref(h)))
        self._h = h
        self.device = device
        v = [C.c_int32(), C.c_int32(), C.c_int32(), C.c_int64(), C.c_int64(), C.c_int64()]
        _check(L.xod_network_sizes(h, *[C.byref(x) for x in v]))
        (self.n_species, self.n_reactions, self.n_photo, self.nnz_source, self.nnz_jac,
         self.n_jac_terms) = [x.value for x in v]

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:     # at interpreter exit the module globals may be gone already
            _lib.xod_network_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- introspection
    def perm(self):
        out = np.zeros(self.n_reactions, dtype=np.int32)
        _check(lib().xod_network_perm(self._h, _hp(out)))
        return out

    def photo_index(self):
        out = np.zeros(self.n_photo, dtype=np.int32)
        _check(lib().xod_network_photo_index(self._h, _hp(out)))
        return out

    def source_csr(self):
        rp = np.zeros(self.n_species + 1, dtype=np.int64)
        rxn, nu = np.zeros(self.nnz_source, dtype=np.int32), np.zeros(self.nnz_source, dtype=np.int32)
        _check(lib().xod_network_source_csr(self._h, _hp(rp), _hp(rxn), _hp(nu)))
        return rp, rxn, nu

    def jac_pattern(self):
        rp = np.zeros(self.n_species + 1, dtype=np.int64)
        col = np.zeros(self.nnz_jac, dtype=np.int32)
        _check(lib().xod_network_jac_pattern(self._h, _hp(rp), _hp(col)))
        return rp, col

    def fused_info(self):
        v = (C.c_int64 * 10)()
        _check(lib().xod_network_fused_info(self._h, v))
        keys = ("enabled", "chunk", "nchunk", "n_acc", "n_bp", "smem_bytes", "npad", "tasks", "entries", "rev_bytes")
        return dict(zip(keys, [int(x) for x in v]))

    def jac_info(self):
        v = (C.c_int64 * 8)()
        _check(lib().xod_network_jac_info(self._h, v))
        keys = ("enabled", "chunk", "nchunk", "units", "acc_rows", "smem_bytes", "slots", "entries")
        return dict(zip(keys, [int(x) for x in v]))

    def lu_info(self):
        v = (C.c_int64 * 8)()
        _check(lib().xod_network_lu_info(self._h, v))
        return dict(zip(("enabled", "nnz_lu", "pairs", "updates", "max_row", "block_rows", "u_loads", "steps"), [int(x) for x in v]))

    def lu_pattern(self):
        info = self.lu_info()
        perm = np.zeros(self.n_species, dtype=np.int32)
        rp = np.zeros(self.n_species + 1, dtype=np.int64)
        col = np.zeros(info["nnz_lu"], dtype=np.int32)
        _check(lib().xod_network_lu_pattern(self._h, _hp(perm), _hp(rp), _hp(col)))
        return perm, rp, col

    def fused_params(self, interval):
        """(user_rxn [npad], kind [npad], coef [npad][16], breakpoints) of one thermo interval."""
        info = self.fused_info()
        user = np.zeros(info["npad"], dtype=np.int32)
        kind = np.zeros(info["npad"], dtype=np.int32)
        coef = np.zeros((info["npad"], 16))
        bp = np.zeros(info["n_bp"])
        _check(lib().xod_network_fused_params(self._h, C.c_int32(interval), _hp(user), _hp(kind), _hp(coef), _hp(bp)))
        return user, kind, coef, bp

    def selfcheck(self):
        _check(lib().xod_network_selfcheck(self._h))

    def check_status(self):
        """Synchronise the device; in the XOD_CHECK build raise if a kernel saw an out-of-range table index."""
        _check(lib().xod_check_status(self._h))

    def tune(self, knob, value):
        _check(lib().xod_network_tune(self._h, C.c_int32(knob), C.c_int64(value)))

    def timing_read(self):
        """{kernel name: (total ms, launches)} since the last read (XOD_TUNE_TIMING on)."""
        ms = (C.c_double * len(KERNEL_NAMES))()
        cnt = (C.c_int64 * len(KERNEL_NAMES))()
        _check(lib().xod_network_timing_read(self._h, ms, cnt))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(KERNEL_NAMES)}

    # ---- workspace sizes
    def rate_coeffs_workspace_bytes(self, ncol):
        return lib().xod_rate_coeffs_workspace_bytes(self._h, ncol)

    def source_workspace_bytes(self, ncol, prod_loss=True):
        f = lib().xod_source_workspace_bytes if prod_loss else lib().xod_source_workspace_bytes_dndt
        return f(self._h, ncol)

    def source_fused_workspace_bytes(self, ncol, prod_loss=True):
        """Upper bound for any arguments; prod_loss=False: the requirement when prod and loss are not asked for."""
        f = lib().xod_source_fused_workspace_bytes if prod_loss else lib().xod_source_fused_workspace_bytes_dndt
        return f(self._h, ncol)

    # ---- compute calls (device tensors)
    def thermo(self, ncol, ld, T, cp_R=None, h_RT=None, s_R=None, g_RT=None, stream=None):
        _check(lib().xod_thermo(self._h, C.c_int64(ncol), C.c_int64(ld), _dp(T), _dp(cp_R), _dp(h_RT),
                                _dp(s_R), _dp(g_RT), _stream(stream)))

    def rate_coeffs(self, ncol, ld, T, P, J, kf, kr, workspace, stream=None):
        _check(lib().xod_rate_coeffs(self._h, C.c_int64(ncol), C.c_int64(ld), _dp(T), _dp(P), _dp(J),
                                     _dp(kf), _dp(kr), _dp(workspace),
                                     C.c_size_t(0 if workspace is None else workspace.numel() * 8),
                                     _stream(stream)))

    def source(self, ncol, ld, kf, kr, n, dndt, prod=None, loss=None, workspace=None, stream=None):
        _check(lib().xod_source(self._h, C.c_int64(ncol), C.c_int64(ld), _dp(kf), _dp(kr), _dp(n),
                                _dp(dndt), _dp(prod), _dp(loss), _dp(workspace),
                                C.c_size_t(0 if workspace is None else workspace.numel() * 8),
                                _stream(stream)))

    def source_fused(self, ncol, ld, T, P, J, n, dndt, prod=None, loss=None, workspace=None, stream=None):
        _check(lib().xod_source_fused(self._h, C.c_int64(ncol), C.c_int64(ld), _dp(T), _dp(P), _dp(J),
                                      _dp(n), _dp(dndt), _dp(prod), _dp(loss), _dp(workspace),
                                      C.c_size_t(0 if workspace is None else workspace.numel() * 8),
                                      _stream(stream)))

    def jacobian(self, ncol, ld, kf, kr, n, jac, stream=None):
        _check(lib().xod_jacobian(self._h, C.c_int64(ncol), C.c_int64(ld), _dp(kf), _dp(kr), _dp(n),
                                  _dp(jac), _stream(stream)))

    # ---- f1: one Newton iteration of a backward-Euler step (y updated in place)
    def newton_workspace_bytes(self, ncol):
        return lib().xod_newton_workspace_bytes(self._h, ncol)

    def newton_step(self, ncol, ld, kf, kr, n_old, dt, y, delta=None, workspace=None, stream=None):
        _check(lib().xod_newton_step(self._h, C.c_int64(ncol), C.c_int64(ld), _dp(kf), _dp(kr), _dp(n_old), _dp(dt),
                                     _dp(y), _dp(delta), _dp(workspace),
                                     C.c_size_t(0 if workspace is None else workspace.numel() * 8), _stream(stream)))

    # ---- f3: molecular-diffusion transport terms (Eq. 3-4)
    def transport(self, n_atm, n_layers, ld, n, T, n_gas, D, mass, alpha_T, mbar, grav, dz, tr, stream=None):
        _check(lib().xod_transport(self._h, C.c_int64(n_atm), C.c_int64(n_layers), C.c_int64(ld), _dp(n), _dp(T), _dp(n_gas),
                                   _dp(D), _dp(mass), _dp(alpha_T), _dp(mbar), _dp(grav), _dp(dz), _dp(tr), _stream(stream)))

    # ---- f4: pathway analyser (dist fp64, pred / via int32 tensors)
    def pathway_workspace_bytes(self, ncol):
        return lib().xod_pathway_workspace_bytes(self._h, ncol)

    def pathway(self, ncol, ld, kf, kr, n, source, dist, pred, via, workspace, stream=None):
        assert pred.is_cuda and via.is_cuda and pred.element_size() == 4 and via.element_size() == 4
        _check(lib().xod_pathway(self._h, C.c_int64(ncol), C.c_int64(ld), _dp(kf), _dp(kr), _dp(n), C.c_int32(source), _dp(dist),
                                 C.c_void_p(pred.data_ptr()), C.c_void_p(via.data_ptr()), _dp(workspace),
                                 C.c_size_t(0 if workspace is None else workspace.numel() * 8), _stream(stream)))

    # ---- f4: thermochemical-equilibrium composition (n, pi fp64, iters int32 tensors)
    def equilibrium(self, ncol, ld, T, P, b, n, pi=None, iters=None, max_iter=0, tol=0.0, stream=None):
        assert iters is None or (iters.is_cuda and iters.element_size() == 4)
        _check(lib().xod_equilibrium(self._h, C.c_int64(ncol), C.c_int64(ld), _dp(T), _dp(P), _dp(b), C.c_int32(max_iter),
                                     C.c_double(tol), _dp(n), _dp(pi), None if iters is None else C.c_void_p(iters.data_ptr()),
                                     _stream(stream)))

    # ---- end to end on HOST buffers (numpy arrays or pinned torch CPU tensors)
    def source_fused_host(self, ncol, ld, T, P, J, n, dndt):
        def hp(a):
            if a is None:
                return None
            if isinstance(a, np.ndarray):
                assert a.dtype == np.float64 and a.flags.c_contiguous
                return C.c_void_p(a.ctypes.data)
            assert (not a.is_cuda) and a.element_size() == 8 and a.is_contiguous()
            return C.c_void_p(a.data_ptr())
        _check(lib().xod_source_fused_host(self._h, C.c_int64(ncol), C.c_int64(ld), hp(T), hp(P), hp(J),
                                           hp(n), hp(dndt)))


class _PhotoDesc(C.Structure):
    _fields_ = [("n_bins", C.c_int32), ("n_abs", C.c_int32), ("dlambda", C.c_void_p), ("abs_species", C.c_void_p),
                ("sigma_ext", C.c_void_p), ("sigma_ph", C.c_void_p)]


class Photo:
    """xod_photo handle (f2).  `ph` is any object with dlambda, abs_species, sigma_ext, sigma_ph (synth.Photo)."""

    def __init__(self, network, ph):
        keep = dict(dlambda=_np(ph.dlambda, np.float64), abs_species=_np(ph.abs_species, np.int32),
                    sigma_ext=_np(ph.sigma_ext, np.float64), sigma_ph=_np(ph.sigma_ph, np.float64))
        d = _PhotoDesc(keep["dlambda"].shape[0], keep["abs_species"].shape[0],
                       *[_hp(keep[k]) for k in ("dlambda", "abs_species", "sigma_ext", "sigma_ph")])
        h = C.c_void_p()
        _check(lib().xod_photo_create(network._h, C.byref(d), C.byref(h)))
        self._h, self._net = h, network          # the photo object points into the network: keep it alive
        self.n_bins = d.n_bins

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.xod_photo_destroy(self._h)
            self._h = None

    __del__ = close

    def workspace_bytes(self, ncol):
        return lib().xod_photo_workspace_bytes(self._h, ncol)

    def rates(self, n_atm, n_layers, ld, n, dz, j0, j_diff, mu, t_f, J, workspace, stream=None):
        _check(lib().xod_photo_rates(self._h, C.c_int64(n_atm), C.c_int64(n_layers), C.c_int64(ld), _dp(n), _dp(dz), _dp(j0),
                                     _dp(j_diff), _dp(mu), _dp(t_f), _dp(J), _dp(workspace),
                                     C.c_size_t(0 if workspace is None else workspace.numel() * 8), _stream(stream)))


def build_has_checks():
    return bool(lib().xod_build_has_checks())


def launch_count():
    return lib().xod_launch_count()


def probe_fp64_peak(device=0, iters=20):
    out = C.c_double()
    _check(lib().xod_probe_fp64_peak(C.c_int(device), C.c_int32(iters), C.byref(out)))
    return out.value
