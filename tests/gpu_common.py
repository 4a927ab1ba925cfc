"""Helpers of the `-m gpu` parity tests: device buffers, the tolerance rules of BASELINE.json
north_star and DESIGN.md reading R5.  Marshalling and comparison only; no method arithmetic."""
import numpy as np

TOL_K = 1e-12        # k_f, k_r: relative (north_star)
TOL_SUM = 1e-11      # dn/dt and Jacobian: of sum |contributing terms| per entry (north_star)
TOL_THERMO = 1e-13   # thermo: of sum |polynomial terms| (derived from the arithmetic)


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def empty(rows, ld, fill=np.nan):
    import torch
    return torch.full((rows, ld), fill, dtype=torch.float64, device="cuda")


def workspace(nbytes):
    import torch
    return torch.empty((nbytes + 7) // 8 + 32, dtype=torch.float64, device="cuda")


def host(t):
    import torch
    torch.cuda.synchronize()
    return t.cpu().numpy()


def check_k(got, want, what):
    """Reading R5: oracle inf -> GPU inf; oracle 0 or subnormal -> |GPU| <= 1e-300; else rel 1e-12."""
    want_inf = np.isinf(want)
    assert np.array_equal(np.isinf(got), want_inf), "%s: inf pattern differs" % what
    tiny = np.abs(want) < 2.2250738585072014e-308
    assert np.all(np.abs(got[tiny]) <= 1e-300), "%s: oracle underflow but GPU not tiny" % what
    m = ~want_inf & ~tiny
    rel = np.abs(got[m] - want[m]) / np.abs(want[m])
    worst = float(rel.max()) if rel.size else 0.0
    assert worst <= TOL_K, "%s: max relative error %.3e > %.0e" % (what, worst, TOL_K)
    return worst


# Reading R5, second part: a rate of progress is formed in fp64 as k n n n, left to right, so a PARTIAL
# product can leave the double range although the term itself (which the oracle forms in long double) is still below
# it: k ~ 1e300 times n ~ 1e10 times n ~ 1e-3.  Partial products exceed the term by at most max(n)^2 < (3e21)^2, hence
# values at or beyond 1e260 count as "beyond the double range" in the comparisons of dn/dt, P, L and the Jacobian.
R5_LIMIT = 1e260


def finite_columns(*arrays):
    """Columns on which every entry of every array is finite and below R5_LIMIT (reading R5: dn/dt, Jacobian and
    conservation are compared only there)."""
    ok = None
    for a in arrays:
        with np.errstate(invalid="ignore"):
            f = np.all(np.isfinite(a) & (np.abs(a) < R5_LIMIT), axis=0)
        ok = f if ok is None else ok & f
    return ok


def check_sum(got, want, scale, cols, what, tol=TOL_SUM):
    """|got - want| <= tol * scale on the given columns; scale == 0 demands exact equality."""
    g, w, s = got[:, cols], want[:, cols], scale[:, cols]
    err = np.abs(g - w)
    bad = err > tol * s
    assert not bad.any(), "%s: %d entries beyond %.0e x scale (worst ratio %.3e)" % (
        what, int(bad.sum()), tol, float((err[bad] / np.maximum(s[bad], 1e-300)).max()))
    nz = s > 0
    return float((err[nz] / s[nz]).max()) if nz.any() else 0.0


def check_sum_entries(got, want, scale, ncol, what, tol=TOL_SUM):
    """Entry-wise form of check_sum for inputs with overflowing k_r (reading R5): every entry whose
    contributing terms are all finite (finite tolerance scale) must match; the others must not be
    finite on the GPU side either.  Returns (worst ratio, number of non-finite entries skipped)."""
    g, w, s = got[:, :ncol], want[:, :ncol], scale[:, :ncol]
    with np.errstate(invalid="ignore"):
        fin = np.isfinite(s) & np.isfinite(w) & (s < R5_LIMIT)
    err = np.abs(g[fin] - w[fin])
    bad = err > tol * s[fin]
    assert not bad.any(), "%s: %d entries beyond %.0e x scale" % (what, int(bad.sum()), tol)
    nz = s[fin] > 0
    return (float((err[nz] / s[fin][nz]).max()) if nz.any() else 0.0), int((~fin).sum())
