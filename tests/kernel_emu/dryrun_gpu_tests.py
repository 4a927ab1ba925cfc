"""Run the `-m gpu` tests WITHOUT a GPU, against the CPU execution of the kernel text (tests/kernel_emu).

TEST INFRASTRUCTURE ONLY, and not GPU evidence: torch stays on the CPU (`.cuda()` is a copy, `device="cuda"` is
dropped) and every compute method of the binding is routed to the matching `emu_*` entry point of libxod_emu.so,
i.e. to the kernel source run on CPU threads on the tables of the real host packer, following the same path choice
as the library (single kernel / multi-kernel pipeline / tiled or gather Jacobian, reaction splits).  What it finds:
mistakes in GPU tests that have never run (names, argument order, shapes, aliasing, tolerance rules that no input
had exercised).  What it cannot find: anything about the GPU (launch configuration, cp.async, memory model, speed).
Argument validation of the C ABI is not reproduced (test_workspace_too_small_is_an_error needs the real library).

    python tests/kernel_emu/dryrun_gpu_tests.py [pytest arguments, e.g. tests/test_gpu_parity.py -k "not full_size"]
"""

import ctypes as C
import os, sys
import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT); sys.path.insert(0, os.path.join(ROOT, "tests"))

# ---- torch: everything stays on the CPU
torch.cuda.is_available = lambda: True
torch.cuda.synchronize = lambda *a, **k: None
torch.cuda.current_device = lambda: 0
torch.Tensor.cuda = lambda self, *a, **k: self.clone()
torch.Tensor.is_cuda = property(lambda self: True)
for name in ("full", "zeros", "empty", "ones"):
    orig = getattr(torch, name)
    def mk(orig):
        def f(*a, **k):
            k.pop("device", None)
            return orig(*a, **k)
        return f
    setattr(torch, name, mk(orig))

from paper_2512_06729_b200 import binding, build
import test_kernel_emulation as tk
build.build = lambda *a, **k: None
import subprocess
if not os.path.exists(tk.LIB) or any(os.path.getmtime(d) > os.path.getmtime(tk.LIB) for d in tk.DEPS):
    subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-shared", "-fPIC", "-I" + os.path.join(tk.EMU_DIR, "shim"), "-o", tk.LIB] + tk.SOURCES, check=True)
EMU = C.CDLL(tk.LIB)

def P(t):
    if t is None: return None
    assert isinstance(t, torch.Tensor) and t.is_contiguous(), type(t)
    return C.c_void_p(t.data_ptr())

RealNetwork = binding.Network
class FakeNetwork(RealNetwork):
    def __init__(self, net, device=0, flags=0):
        super().__init__(net, device=-1, flags=flags)
        self._net = net
        self._d, self._keep = tk.descriptor(net)
        self._tune = {}
        self.calls = []
    def tune(self, knob, value):
        self._tune[knob] = value
        super().tune(knob, value)
    def check_status(self): pass
    def timing_read(self): return {k: (0.0, 0) for k in binding.KERNEL_NAMES}
    def _fused_on(self): return self.fused_info()["enabled"] and self._tune.get(binding.XOD_TUNE_FUSED_KERNEL, 1)
    def _ws(self, workspace, need):
        if workspace is None or workspace.numel() * 8 < need:
            raise binding.XodError(5, "workspace too small: %d < %d" % (0 if workspace is None else workspace.numel() * 8, need))
    def thermo(self, ncol, ld, T, cp_R=None, h_RT=None, s_R=None, g_RT=None, stream=None):
        if ncol == 0: return
        assert EMU.emu_thermo(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(T), P(cp_R), P(h_RT), P(s_R), P(g_RT), C.c_int(5)) == 0
    def rate_coeffs(self, ncol, ld, T, Pp, J, kf, kr, workspace=None, stream=None):
        if ncol == 0: return
        self._ws(workspace, self.rate_coeffs_workspace_bytes(ncol))
        if self._fused_on():
            rc = EMU.emu_rate_coeffs(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(T), P(Pp), P(J), P(kf), P(kr), C.c_int(16))
        else:
            rc = EMU.emu_rate_coeffs_pipeline(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(T), P(Pp), P(J), P(kf), P(kr), C.c_int(16))
        assert rc == 0
    def source(self, ncol, ld, kf, kr, n, dndt, prod=None, loss=None, workspace=None, stream=None):
        if ncol == 0: return
        self._ws(workspace, self.source_workspace_bytes(ncol) if prod is not None else lib_dndt(self, ncol, False))
        if prod is None and self._fused_on() and self.n_reactions > 0:
            rc = EMU.emu_source_fused(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), None, None, None, P(kf), P(kr), P(n), P(dndt), C.c_int(2), C.c_int(max(1, self._tune.get(binding.XOD_TUNE_SPLIT, 0))))
        else:
            z = torch.zeros(max(ld, 1), dtype=torch.float64) + 1000.0
            rc = EMU.emu_source_pipeline(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(z), P(z), None, P(kf) if kf is not None else P(torch.zeros(1)), P(kr) if kr is not None else P(torch.zeros(1)), P(n), P(dndt), P(prod), P(loss), C.c_int(16))
        assert rc == 0
    def source_fused(self, ncol, ld, T, Pp, J, n, dndt, prod=None, loss=None, workspace=None, stream=None):
        if ncol == 0: return
        self._ws(workspace, self.source_fused_workspace_bytes(ncol) if prod is not None else lib_dndt(self, ncol, True))
        if prod is None and self._fused_on():
            rc = EMU.emu_source_fused(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(T), P(Pp), P(J), None, None, P(n), P(dndt), C.c_int(2), C.c_int(max(1, self._tune.get(binding.XOD_TUNE_SPLIT, 0))))
        else:
            rc = EMU.emu_source_pipeline(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(T), P(Pp), P(J), None, None, P(n), P(dndt), P(prod), P(loss), C.c_int(16))
        assert rc == 0
    def jacobian(self, ncol, ld, kf, kr, n, jac, stream=None):
        if ncol == 0: return
        if self.jac_info()["enabled"] and self._tune.get(binding.XOD_TUNE_JAC_TILED, 1) and self.n_reactions > 0:
            rc = EMU.emu_jacobian_tiled(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(kf), P(kr), P(n), P(jac), C.c_int(2), C.c_int(max(1, self._tune.get(binding.XOD_TUNE_SPLIT, 0))))
        else:
            e = torch.zeros(1)
            rc = EMU.emu_jacobian(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(kf if kf is not None else e), P(kr if kr is not None else e), P(n), P(jac), C.c_int(3))
        assert rc == 0
    def newton_step(self, ncol, ld, kf, kr, n_old, dt, y, delta=None, workspace=None, stream=None):
        self._ws(workspace, self.newton_workspace_bytes(ncol))
        assert EMU.emu_newton_step(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(kf), P(kr), P(n_old), P(dt), P(y), P(delta)) == 0
    def transport(self, n_atm, n_layers, ld, n, T, n_gas, D, mass, alpha_T, mbar, grav, dz, tr, stream=None):
        assert EMU.emu_transport(C.c_int(self.n_species), C.c_int64(n_atm), C.c_int64(n_layers), C.c_int64(ld), P(n), P(T), P(n_gas), P(D), P(mass), P(alpha_T), P(mbar), P(grav), P(dz), P(tr), C.c_int(7)) == 0
    def pathway(self, ncol, ld, kf, kr, n, source, dist, pred, via, workspace, stream=None):
        self._ws(workspace, self.pathway_workspace_bytes(ncol))
        assert pred.dtype == torch.int32 and via.dtype == torch.int32
        assert EMU.emu_pathway(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(kf), P(kr), P(n), C.c_int(source), P(dist), P(pred), P(via), C.c_int(2)) == 0
    def equilibrium(self, ncol, ld, T, Pp, b, n, pi=None, iters=None, max_iter=0, tol=0.0, stream=None):
        assert iters is None or iters.dtype == torch.int32
        assert EMU.emu_equilibrium(C.byref(self._d), C.c_int64(ncol), C.c_int64(ld), P(T), P(Pp), P(b), C.c_int(max_iter), C.c_double(tol), P(n), P(pi), P(iters)) == 0
    def source_fused_host(self, ncol, ld, T, Pp, J, n, dndt):
        t = lambda a: torch.from_numpy(a) if isinstance(a, np.ndarray) else a
        ws = torch.empty(lib_dndt(self, ncol, True) // 8 + 64, dtype=torch.float64)
        self.source_fused(ncol, ld, t(T), t(Pp), t(J), t(n), t(dndt), workspace=ws)

def lib_dndt(h, ncol, fused):
    L = binding.lib()
    return (L.xod_source_fused_workspace_bytes_dndt if fused else L.xod_source_workspace_bytes_dndt)(h._h, ncol)

binding.Network = FakeNetwork

RealPhoto = binding.Photo
class FakePhoto:
    def __init__(self, h, ph):
        self.h, self.ph = h, ph
        self._real = RealPhoto(h, ph)      # validates the tables (host-only)
    def workspace_bytes(self, ncol): return self._real.workspace_bytes(ncol)
    def rates(self, n_atm, n_layers, ld, n, dz, j0, j_diff, mu, t_f, J, workspace, stream=None):
        assert workspace.numel() * 8 >= self.workspace_bytes(n_atm * n_layers)
        ph = self.ph
        c = lambda a, dt=np.float64: np.ascontiguousarray(a, dtype=dt)
        ab, se, sp, dl = c(ph.abs_species, np.int32), c(ph.sigma_ext), c(ph.sigma_ph), c(ph.dlambda)
        assert EMU.emu_photo_rates(C.c_int(self.h.n_species), C.c_int(self.h.n_photo), C.c_int(ph.n_bins), C.c_int(ab.shape[0]), tk.ptr(ab), tk.ptr(se), tk.ptr(sp), tk.ptr(dl),
                                   C.c_int64(n_atm), C.c_int64(n_layers), C.c_int64(ld), P(n), P(dz), P(j0), P(j_diff), P(mu), P(t_f), P(J)) == 0
    def close(self): self._real.close()
binding.Photo = FakePhoto


if __name__ == "__main__":
    import pytest
    sys.exit(pytest.main(["-p", "no:cacheprovider", "-m", "gpu", "-q"] + sys.argv[1:]))
