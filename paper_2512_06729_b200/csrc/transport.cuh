// transport.cuh -- k_transport: the molecular-diffusion transport terms of the continuity equation
// (PAPER.md:73-83), sm_100a.
//
//   d_{k+-1/2} = D_{k+-1/2} / (2 dz^2) [ (mbar - m_y) g dz / (k_B T_{k+-1/2}) - alpha_T / T_{k+-1/2} (T_{k+-1} - T_k) ]      (Eq. 4)
//   tr_{y,k}   = - d_{k+1/2} (N_{k+1/2} / N_{k+1}) n_{y,k+1} - [ d_{k+1/2} (N_{k+1/2} / N_k) - d_{k-1/2} (N_{k-1/2} / N_k) ] n_{y,k}
//                + d_{k-1/2} (N_{k-1/2} / N_k) n_{y,k-1}                                                          (Eq. 3 minus P - L)
// half levels are arithmetic means; the two extraction garbles of Eq. 3 are dropped (reading V1);
// zero-flux boundaries: no term reaches across the bottom or the top of an atmosphere (reading V2).
// thread = column (layers of an atmosphere are consecutive columns, so the k +- 1 neighbours are the adjacent lanes'
// values and every access is a coalesced row segment); a CTA loops over a block of species.  Everything that depends
// only on the column (the half-level temperatures, gas-density ratios, 1 / (2 dz^2), g dz / k_B) is computed once per
// thread.  HBM-bound: n and D read (neighbours come from L1), tr written: 24 B per (species, column).
#pragma once
#include <cuda_runtime.h>

#include "xod_internal.h"

namespace xod {

struct TransportArgs {
  int64_t ncol, n_layers, ld;
  int32_t ns;
  const double *n, *T, *n_gas, *D;      // [ns][ld], [ld], [ld], [ns][ld]
  const double *mass, *alpha_T;         // [ns]
  const double *mbar, *grav, *dz;       // [n_atm]
  double *tr;                           // [ns][ld]
  int32_t spb;                          // species per blockIdx.y
};

// grid (ceil(ncol / 128), species blocks)
__global__ void __launch_bounds__(128) k_transport(TransportArgs a) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= a.ncol) return;
  const int64_t atm = c / a.n_layers, k = c - atm * a.n_layers;
  const bool up = k + 1 < a.n_layers, dn = k > 0;
  const double h = a.dz[atm], g = a.grav[atm], mb = a.mbar[atm];
  const double Tc = a.T[c], Nc = a.n_gas[c];
  const double Tu = up ? a.T[c + 1] : Tc, Td = dn ? a.T[c - 1] : Tc;
  const double Nu = up ? a.n_gas[c + 1] : Nc, Nd = dn ? a.n_gas[c - 1] : Nc;
  const double kB = 1.380649e-16;
  const double inv2h2 = 1.0 / (2.0 * h * h);
  const double Thu = (Tc + Tu) / 2, Thd = (Tc + Td) / 2;
  const double gu = g * h / (kB * Thu), gd = g * h / (kB * Thd);     // g dz / (k_B T_{k+-1/2})
  const double tu = (Tu - Tc) / Thu, td = (Td - Tc) / Thd;           // (T_{k+-1} - T_k) / T_{k+-1/2}
  const double Nhu = (Nc + Nu) / 2, Nhd = (Nc + Nd) / 2;
  const double ru_up = Nhu / Nu, ru_c = Nhu / Nc, rd_c = Nhd / Nc;    // N_{k+1/2}/N_{k+1}, N_{k+1/2}/N_k, N_{k-1/2}/N_k
  const int y0 = blockIdx.y * a.spb, y1 = min(a.ns, y0 + a.spb);
  for (int y = y0; y < y1; ++y) {
    const double *ny = a.n + (size_t)y * a.ld, *Dy = a.D + (size_t)y * a.ld;
    const double dm = mb - __ldg(a.mass + y), al = __ldg(a.alpha_T + y);
    const double nc = ny[c], Dc = Dy[c];
    double t = 0.0, dp = 0.0, dmn = 0.0;
    if (up) dp = (Dc + Dy[c + 1]) / 2 * inv2h2 * (dm * gu - al * tu);
    if (dn) dmn = (Dc + Dy[c - 1]) / 2 * inv2h2 * (dm * gd - al * td);
    if (up) t -= dp * ru_up * ny[c + 1];
    t -= (dp * ru_c - dmn * rd_c) * nc;
    if (dn) t += dmn * rd_c * ny[c - 1];
    a.tr[(size_t)y * a.ld + c] = t;
  }
}

}  // namespace xod
