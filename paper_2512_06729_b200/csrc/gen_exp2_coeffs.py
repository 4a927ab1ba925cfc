"""Generate the polynomial coefficients of xexp2 (xod_math.cuh): 2^f on |f| <= 1/2.

p(f) = 1 + f g(f), g = Chebyshev-node interpolant of (2^f - 1)/f of degree DEG-1 (near-minimax),
computed with mpmath at 60 digits and rounded to double.  Prints the coefficients (highest
degree first, as the Horner chain in xexp2 uses them) and the maximum relative error of the
double-rounded polynomial evaluated exactly, over a dense grid.

    python gen_exp2_coeffs.py [DEG]      (default 9: max relative error ~2e-14, far below the
                                          1e-12 tolerance of the rate coefficients)
"""
import sys

import mpmath as mp

mp.mp.dps = 60


def fit(deg):
    m = deg                                # g has degree deg-1 -> deg nodes
    half = mp.mpf(1) / 2
    nodes = [half * mp.cos(mp.pi * (2 * k + 1) / (2 * m)) for k in range(m)]

    def g(x):
        return mp.expm1(x * mp.log(2)) / x if abs(x) > mp.mpf(10) ** -30 else mp.log(2)

    A = mp.matrix(m, m)
    b = mp.matrix(m, 1)
    for r, x in enumerate(nodes):
        for c in range(m):
            A[r, c] = x ** c
        b[r] = g(x)
    sol = mp.lu_solve(A, b)
    coeffs = [mp.mpf(1)] + [sol[c] for c in range(m)]      # c0 = 1 exactly
    return [float(c) for c in coeffs]


def max_rel_error(coeffs, npts=20001):
    worst = mp.mpf(0)
    for k in range(npts):
        x = mp.mpf(-1) / 2 + mp.mpf(k) / (npts - 1)
        p = mp.mpf(0)
        for c in reversed(coeffs):
            p = p * x + mp.mpf(c)
        worst = max(worst, abs(p / mp.power(2, x) - 1))
    return worst


if __name__ == "__main__":
    deg = int(sys.argv[1]) if len(sys.argv) > 1 else 9
    c = fit(deg)
    print("// degree %d, max relative error %s (double-rounded coefficients, exact evaluation)"
          % (deg, mp.nstr(max_rel_error(c), 3)))
    for k in range(deg, -1, -1):
        print("  c%-2d = %s" % (k, repr(c[k])))
