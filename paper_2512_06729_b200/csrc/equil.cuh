// equil.cuh -- k_equilibrium: the thermochemical-equilibrium composition, sm_100a.
//
// "the initial atmospheric composition can be specified using ... equilibrium abundances from the built-in
// equilibrium chemistry solver".  The paper gives no method; the composition is DEFINED as the
// minimiser of the Gibbs energy of an ideal gas mixture at (T, P) for given element abundances b_e (DESIGN.md
// reading E1), which the Lagrange conditions characterise:
//     G_i/RT + ln x_i + ln(P/P0) = sum_e a_ie pi_e,     sum_i x_i = 1,     sum_i a_ie x_i ~ b_e.
// They are solved per column by the damped Newton iteration in (ln n_i, ln N) of Gordon & McBride (NASA RP-1311,
// 1994, gas phase): an (n_e + 1) x (n_e + 1) linear system per iteration whose coefficients are sums over the
// species, then d ln n_i = -mu_i + sum_e a_ie pi_e + d ln N with a step-size control.
//
// thread = column (every global access is a coalesced row segment); ln n_i lives in the caller's output array
// while the iteration runs; the small dense system of a thread sits in shared memory as [entry][64 threads]
// (conflict-free, no barrier: threads never share an entry); G_i/RT is re-evaluated from the NASA-7
// coefficients where it is needed (8 FMA) rather than stored.  One iteration is two sweeps over the species:
//   sweep 1  d ln n_i and the two step-size maxima;
//   sweep 2  ln n_i += lambda d ln n_i, the convergence sums, and the NEXT iteration's system from the new n_i.
// The composition matrix is stored as a short (element, count) list per species, uniform over the warp.
// Converged columns leave the loop; the final composition is taken from the element potentials for EVERY species
// (trace species sit exactly on their Lagrange condition) and scaled to sum n_i = P / (k_B T).
#pragma once
#include <cuda_runtime.h>

#include "xod_internal.h"
#include <xod_cta.cuh>

namespace xod {

struct EquilArgs {
  int64_t ncol, ld;
  const double *T, *P, *b;   // [ld], [ld], [ne][ld]
  double *n;                 // [ns][ld] out (ln n_i during the iteration)
  double *pi;                // [ne][ld] out or NULL
  int32_t *iters;            // [ld] out or NULL
  int32_t max_iter;
  double tol;
};

// doubles of shared memory per thread: augmented system m x (m + 1) | solution m | abundances ne | sum |a| n ne   (m = ne + 1)
inline int equil_smem_doubles(int ne) { return (ne + 1) * (ne + 2) + (ne + 1) + 2 * ne; }

__global__ void __launch_bounds__(kEqThreads) k_equilibrium(EquilDev d, EquilArgs a) {
  const int64_t col = (int64_t)blockIdx.x * kEqThreads + threadIdx.x;
  if (col >= a.ncol) return;
  const int ns = d.ns, ne = d.ne, m = ne + 1, mw = m + 1;
  double *S = reinterpret_cast<double *>(cta_dyn_smem()) + threadIdx.x;
  auto M = [&](int r, int c) -> double & { return S[(size_t)(r * mw + c) * kEqThreads]; };    // column m = right-hand side
  auto sol = [&](int e) -> double & { return S[(size_t)(m * mw + e) * kEqThreads]; };
  auto bb = [&](int e) -> double & { return S[(size_t)(m * mw + m + e) * kEqThreads]; };
  auto ab = [&](int e) -> double & { return S[(size_t)(m * mw + m + ne + e) * kEqThreads]; };   // sum_i |a_ie| n_i
  double *lnn = a.n + col;
  const double nan = __longlong_as_double(0x7ff8000000000000LL);

  const double Tc = a.T[col], Pc = a.P[col];
  const double lnT = log(Tc), invT = 1.0 / Tc, lnP = log(Pc / 1.0e6);   // P0 = 1 bar (reading T2)
  // c_i = G_i/RT + ln(P/P0), NASA-7 form of PAPER.md:671 with the range rule of reading T3
  auto c_of = [&](int i) {
    const double *q = d.nasa + (size_t)i * 14 + (Tc <= __ldg(d.tmid + i) ? 0 : 7);
    const double poly = fma(Tc, fma(Tc, fma(Tc, __ldg(q + 4) * 0.05, __ldg(q + 3) * (1.0 / 12.0)), __ldg(q + 2) * (1.0 / 6.0)), __ldg(q + 1) * 0.5);
    return fma(__ldg(q + 5), invT, fma(__ldg(q), 1.0 - lnT, -fma(Tc, poly, __ldg(q + 6)))) + lnP;
  };
  // sum_e a_ie v_e over the species' element list
  auto dot_pi = [&](int i) {
    double s = 0.0;
    for (int k = __ldg(d.sp_ptr + i); k < __ldg(d.sp_ptr + i + 1); ++k) {
      const int ea = __ldg(d.sp_ea + k);
      s = fma((double)(ea >> 8), sol(XOD_IDX(ea & 0xff, ne)), s);
    }
    return s;
  };

  // ---- abundances: scaled to sum 1 over the positive ones; an element without abundance must have a signed column
  bool ok = Tc > 0.0 && Pc > 0.0 && Tc < 1.0e300 && Pc < 1.0e300;
  double bsum = 0.0;
  for (int e = 0; e < ne; ++e) {
    const double be = a.b[(size_t)e * a.ld + col];
    bb(e) = be;
    if (be > 0.0) bsum += be;
    if (!(be > 0.0) && !(be == 0.0 && __ldg(d.el_neg + e))) ok = false;
  }
  if (!ok || !(bsum > 0.0) || !(bsum < 1.0e300)) {
    for (int i = 0; i < ns; ++i) lnn[(size_t)i * a.ld] = nan;
    if (a.pi) for (int e = 0; e < ne; ++e) a.pi[(size_t)e * a.ld + col] = nan;
    if (a.iters) a.iters[col] = 0;
    return;
  }
  for (int e = 0; e < ne; ++e) bb(e) /= bsum;

  double lnN = log(0.1), lam = 0.0, dlnN = 0.0;
  {
    const double l0 = log(0.1 / (double)ns);
    for (int i = 0; i < ns; ++i) lnn[(size_t)i * a.ld] = l0;
  }
  for (int e = 0; e < m; ++e) sol(e) = 0.0;
  int it = 0;
  bool done = false;
  while (true) {
    // ---- sweep 2 of iteration `it` (it = 0: the start composition, lambda = 0): update ln n_i, the convergence
    // sums of the step just taken, and the system of the next iteration from the new composition
    const double lnN_old = lnN;
    lnN += lam * dlnN;
    const double N = exp(lnN);
    for (int r = 0; r < m; ++r)
      for (int c = 0; c < mw; ++c) M(r, c) = 0.0;
    for (int e = 0; e < ne; ++e) ab(e) = 0.0;
    double sumn = 0.0, sumnmu = 0.0, wmax = 0.0;
    for (int i = 0; i < ns; ++i) {
      const double ci = c_of(i);
      double li = lnn[(size_t)i * a.ld], dl = 0.0;
      if (it > 0) {
        dl = -(ci + li - lnN_old) + dot_pi(i) + dlnN;
        li = fma(lam, dl, li);
        lnn[(size_t)i * a.ld] = li;
      }
      const double ni = exp(li), mu = ci + li - lnN;
      sumn += ni, sumnmu = fma(ni, mu, sumnmu);
      wmax = fmax(wmax, ni * fabs(dl));
      const int k0 = __ldg(d.sp_ptr + i), k1 = __ldg(d.sp_ptr + i + 1);
      for (int k = k0; k < k1; ++k) {
        const int ea = __ldg(d.sp_ea + k), e = XOD_IDX(ea & 0xff, ne);
        const double an = (double)(ea >> 8) * ni;
        for (int l = k0; l < k1; ++l) {
          const int fa = __ldg(d.sp_ea + l);
          M(e, XOD_IDX(fa & 0xff, ne)) = fma(an, (double)(fa >> 8), M(e, fa & 0xff));
        }
        M(e, ne) += an;            // also sum_i a_ie n_i, the element total of the new composition
        ab(e) += fabs(an);
        M(e, m) = fma(an, mu, M(e, m));
      }
    }
    if (it > 0) {
      double err = fmax(wmax, N * fabs(dlnN)) / sumn, res = 0.0;
      // element residuals relative to the element's own abundance (to the charge carried, for a signed column): a
      // trace element carried by one inert species is decoupled from the others and only this residual sees it
      for (int e = 0; e < ne; ++e) res = fmax(res, fabs(M(e, ne) - bb(e)) / fmax(bb(e), ab(e)));
      done = lam == 1.0 && err <= a.tol && res <= a.tol;
      if (done || it >= a.max_iter) break;
    }
    ++it;
    for (int e = 0; e < ne; ++e) {
      M(ne, e) = M(e, ne);
      M(e, m) += bb(e) - M(e, ne);
    }
    M(ne, ne) = sumn - N;
    M(ne, m) = N - sumn + sumnmu;
    // ---- the (ne + 1) system: rows scaled by their largest entry (a charge row is many orders below the
    // element rows), Gaussian elimination with partial pivoting.  A zero pivot leaves IEEE inf/NaN: the column
    // then never converges and is reported as such.
    for (int r = 0; r < m; ++r) {
      double big = 0.0;
      for (int c = 0; c < m; ++c) big = fmax(big, fabs(M(r, c)));
      const double inv = 1.0 / big;
      for (int c = 0; c < mw; ++c) M(r, c) *= inv;
    }
    for (int k = 0; k < m; ++k) {
      int p = k;
      for (int r = k + 1; r < m; ++r)
        if (fabs(M(r, k)) > fabs(M(p, k))) p = r;
      if (p != k)
        for (int c = k; c < mw; ++c) {
          const double t = M(k, c);
          M(k, c) = M(p, c), M(p, c) = t;
        }
      const double ipiv = 1.0 / M(k, k);
      for (int r = k + 1; r < m; ++r) {
        const double l = M(r, k) * ipiv;
        if (l == 0.0) continue;
        for (int c = k + 1; c < mw; ++c) M(r, c) = fma(-l, M(k, c), M(r, c));
      }
    }
    for (int r = m - 1; r >= 0; --r) {
      double s = M(r, m);
      for (int c = r + 1; c < m; ++c) s = fma(-M(r, c), sol(c), s);
      sol(r) = s / M(r, r);
    }
    dlnN = sol(ne);
    // ---- sweep 1: the step-size control (Gordon & McBride, section 3.3)
    double big = 5.0 * fabs(dlnN), lam2 = 1.0;
    for (int i = 0; i < ns; ++i) {
      const double li = lnn[(size_t)i * a.ld];
      const double dl = -(c_of(i) + li - lnN) + dot_pi(i) + dlnN, lx = li - lnN;
      if (lx > -18.420681) {
        big = fmax(big, fabs(dl));
      } else if (dl > 0.0) {
        lam2 = fmin(lam2, fabs((-lx - 9.2103404) / (dl - dlnN)));
      }
    }
    lam = fmin(big > 2.0 ? 2.0 / big : 1.0, lam2);
    if (!(lam == lam)) lam = 1.0;   // NaN (singular system): keep going, the column will report non-convergence
  }
  // ---- every species from the element potentials, scaled to the gas density P / (k_B T)
  const double ntot = Pc / (1.380649e-16 * Tc);
  for (int i = 0; i < ns; ++i) lnn[(size_t)i * a.ld] = done ? ntot * exp(dot_pi(i) - c_of(i)) : nan;
  if (a.pi)
    for (int e = 0; e < ne; ++e) a.pi[(size_t)e * a.ld + col] = done ? sol(e) : nan;
  if (a.iters) a.iters[col] = done ? it : -it;
}

}  // namespace xod
