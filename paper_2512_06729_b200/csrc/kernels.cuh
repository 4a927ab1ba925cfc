// kernels.cuh -- the CUDA kernels of libxodiac (sm_100a).  Lanes are columns everywhere: a warp
// holds 32 consecutive (atmosphere, layer) columns of ONE row (species / reaction / CSR entry),
// so every global access is a coalesced 256-byte line and everything indexed by the row
// (reaction parameters, species indices, CSR entries) is warp-uniform.
#pragma once
#include <cuda_runtime.h>

#include "xod_internal.h"
#include "xod_math.cuh"
#include <xod_cta.cuh>

namespace xod {

enum { MODE_K = 0, MODE_QNET = 1, MODE_QSEP = 2 };

// per-chunk scratch in the caller's workspace (column pitch ldw, chunk-local column index)
struct ChunkScratch {
  double *l2T;   // [ldw] log2 T
  double *invT;  // [ldw] 1/T
  double *lM;    // [ldw] log2 [M],  [M] = P/(k_B T)   (north_star)
  double *u;     // [ns][ldw] u_i = log2(e) G_i/RT - log2(P0/(k_B T))
  double *q;     // [nr][ldw] net rate of progress, or q_f when prod/loss are wanted
  double *qr;    // [nr][ldw] q_r (only when prod/loss are wanted)
  int64_t ldw;
};

// ------------------------------------------------------------------------------------------
// a2  xod_thermo: NASA-7 polynomials, PAPER.md:671-673 (+ standard H/RT, S/R, reading T1).
// grid (ceil(ncol/128), species blocks); thread = column, loops over the block's species.
// HBM-write bound: 8 B per requested output per (species, column).
__global__ void __launch_bounds__(128) k_thermo(DevTables d, int64_t ncol, int64_t ld,
                                                const double *__restrict__ T, double *__restrict__ cp,
                                                double *__restrict__ h, double *__restrict__ s,
                                                double *__restrict__ g, int spb) {
  int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncol) return;
  const double Tc = T[c];
  const double lnT = log(Tc), invT = 1.0 / Tc;
  const int i0 = blockIdx.y * spb, i1 = min(d.ns, i0 + spb);
  for (int i = i0; i < i1; ++i) {
    const double *a = d.nasa + (size_t)i * 14 + (Tc <= __ldg(d.tmid + i) ? 0 : 7);
    const double a1 = __ldg(a), a2 = __ldg(a + 1), a3 = __ldg(a + 2), a4 = __ldg(a + 3),
                 a5 = __ldg(a + 4), a6 = __ldg(a + 5), a7 = __ldg(a + 6);
    const size_t o = (size_t)i * ld + c;
    if (cp) cp[o] = fma(Tc, fma(Tc, fma(Tc, fma(Tc, a5, a4), a3), a2), a1);
    if (h)
      h[o] = fma(a6, invT,
                 fma(Tc, fma(Tc, fma(Tc, fma(Tc, a5 * 0.2, a4 * 0.25), a3 * (1.0 / 3.0)), a2 * 0.5), a1));
    if (s)
      s[o] = fma(a1, lnT,
                 fma(Tc, fma(Tc, fma(Tc, fma(Tc, a5 * 0.25, a4 * (1.0 / 3.0)), a3 * 0.5), a2), a7));
    if (g) {
      double poly = fma(Tc, fma(Tc, fma(Tc, a5 * 0.05, a4 * (1.0 / 12.0)), a3 * (1.0 / 6.0)), a2 * 0.5);
      g[o] = fma(a6, invT, fma(a1, 1.0 - lnT, -fma(Tc, poly, a7)));
    }
  }
}

// ------------------------------------------------------------------------------------------
// a1 + the thermo half of a6: per-column scalars and u_i for one chunk of columns.
//   u_i = log2(e) G_i/RT - log2(P0/(k_B T)),  so that for a reversible reaction
//   log2 k_r = log2 k_f + sum_products u - sum_reactants u        (Eq. 15, K_c of Tsai+ 2017 App. E)
//   (the (P0/k_B T)^dnu factor is carried per species: dnu = #products - #reactants).
// grid (chunk column groups, species split); block 256 = 8 warps; lane = column.
__global__ void __launch_bounds__(256) k_prologue(DevTables d, int64_t ncol, int64_t col0,
                                                  const double *__restrict__ T,
                                                  const double *__restrict__ P, ChunkScratch w,
                                                  double log2_kb) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t c = (int64_t)blockIdx.x * 32 + lane;
  const int64_t gc = col0 + c;
  const bool valid = gc < ncol;
  const double Tc = valid ? T[gc] : 1000.0;
  const double l2T = log2(Tc), invT = 1.0 / Tc;
  if (blockIdx.y == 0 && warp == 0) {
    const double Pc = valid ? P[gc] : 1.0e6;
    w.l2T[c] = l2T;
    w.invT[c] = invT;
    w.lM[c] = log2(Pc) - log2_kb - l2T;
  }
  for (int i = blockIdx.y * 8 + warp; i < d.ns; i += 8 * gridDim.y) {
    const double *b = d.nasa_l2 + (size_t)i * 14 + (Tc <= __ldg(d.tmid + i) ? 0 : 7);
    const double b0 = __ldg(b), b1 = __ldg(b + 1), b2 = __ldg(b + 2), b3 = __ldg(b + 3),
                 b4 = __ldg(b + 4), b5 = __ldg(b + 5), b6 = __ldg(b + 6);
    double poly = fma(Tc, fma(Tc, fma(Tc, b5, b4), b3), b2);
    double u = fma(b6, invT, fma(-b1, l2T, fma(-Tc, poly, b0)));
    w.u[(size_t)i * w.ldw + c] = u;
  }
}

// ------------------------------------------------------------------------------------------
// a3-a7: forward and reverse coefficients (and rates of progress) of one chunk.
//   UNI/BI   log2 k_f = c0 + c1 log2 T + c2 / T                                 (Eq. 7)
//   FALLOFF  k0[M], k_inf as above;  k = k0[M]/(1 + Pr) F,  Pr = k0[M]/k_inf    (Eq. 10-12)
//            evaluated as 2^(min(log2 k0[M], log2 k_inf) + log2 F) / (1 + 2^-|log2 Pr|)
//            log2 F = log2 Fc / (1 + (cN log2 Pr)^2)                            (reading F1)
//   PHOTO    k_f = J
//   reverse  k_r = 2^(log2 k_f + z), z = sum_products u - sum_reactants u        (Eq. 15)
//            -- in the exponent, so K_c never overflows on its own (reading R5)
// A warp owns (32 columns) x (a slice of `rw` packed reactions); tasks are strided over warps
// with the column group fastest, so neighbouring warps share a slice's parameters in L1.
template <int MODE>
__global__ void __launch_bounds__(128) k_rates(DevTables d, int64_t ncol, int64_t col0, int64_t ld,
                                               ChunkScratch w, const double *__restrict__ J,
                                               const double *__restrict__ n, double *__restrict__ kf_out,
                                               double *__restrict__ kr_out, int rw, int ncg, int64_t ntasks) {
  const int lane = threadIdx.x & 31;
  const int64_t gw = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  for (int64_t t = gw; t < ntasks; t += nw) {
    const int cg = (int)(t % ncg);
    const int p0 = (int)(t / ncg) * rw, p1 = min(d.nr, p0 + rw);
    const int64_t c = (int64_t)cg * 32 + lane;
    const bool valid = col0 + c < ncol;
    const int64_t cc = valid ? c : 0;             // chunk-local column (clamped for idle lanes)
    const int64_t gc = col0 + cc;                 // caller's column
    const double l2T = w.l2T[cc], invT = w.invT[cc];
    for (int p = p0; p < p1; ++p) {
      const int2 s01 = __ldg(reinterpret_cast<const int2 *>(d.sp + (size_t)p * 6));
      const int2 s23 = __ldg(reinterpret_cast<const int2 *>(d.sp + (size_t)p * 6 + 2));
      const int2 s45 = __ldg(reinterpret_cast<const int2 *>(d.sp + (size_t)p * 6 + 4));
      const int r0 = s01.x, r1 = s01.y, r2 = s23.x, q0 = s23.y, q1 = s45.x, q2 = s45.y;
      double kf, kr = 0.0;
      if (p >= d.ph_begin) {
        kf = J[(size_t)__ldg(d.photo_row + (p - d.ph_begin)) * ld + gc];
      } else {
        const bool rev = __ldg(d.flags + p) & 1;
        double z = 0.0;
        if (rev) {
          z = w.u[(size_t)q0 * w.ldw + cc];
          if (q1 >= 0) z += w.u[(size_t)q1 * w.ldw + cc];
          if (q2 >= 0) z += w.u[(size_t)q2 * w.ldw + cc];
          double zr = w.u[(size_t)r0 * w.ldw + cc];
          if (r1 >= 0) zr += w.u[(size_t)r1 * w.ldw + cc];
          if (r2 >= 0) zr += w.u[(size_t)r2 * w.ldw + cc];
          z -= zr;
        }
        const double yi = fma(__ldg(d.c2 + p), invT, fma(__ldg(d.c1 + p), l2T, __ldg(d.c0 + p)));
        if (p < d.fo_begin) {
          kf = xexp2(yi);
          if (rev) kr = xexp2(yi + z);
        } else {
          const int f = p - d.fo_begin;
          const double y0 =
              fma(__ldg(d.l2 + f), invT, fma(__ldg(d.l1 + f), l2T, __ldg(d.l0 + f))) + w.lM[cc];
          const double lpr = y0 - yi;
          const double x = lpr * __ldg(d.cN + f);
          const double lF = __ldg(d.fcl + f) / fma(x, x, 1.0);
          const double den = 1.0 / (1.0 + xexp2(-fabs(lpr)));
          const double ym = fmin(y0, yi) + lF;
          kf = xexp2(ym) * den;
          if (rev) kr = xexp2(ym + z) * den;
        }
      }
      if (MODE == MODE_K) {
        if (valid) {
          const size_t o = (size_t)__ldg(d.user + p) * ld + gc;
          if (kf_out) kf_out[o] = kf;
          if (kr_out) kr_out[o] = kr;
        }
      } else {
        double qf = kf * n[(size_t)r0 * ld + gc];
        if (r1 >= 0) qf *= n[(size_t)r1 * ld + gc];
        if (r2 >= 0) qf *= n[(size_t)r2 * ld + gc];
        double qr = 0.0;
        if (kr != 0.0 || kr != kr) {  // warp-divergent only where some k_r are exactly 0
          qr = kr * n[(size_t)q0 * ld + gc];
          if (q1 >= 0) qr *= n[(size_t)q1 * ld + gc];
          if (q2 >= 0) qr *= n[(size_t)q2 * ld + gc];
        }
        if (MODE == MODE_QNET) {
          w.q[(size_t)p * w.ldw + cc] = qf - qr;
        } else {
          w.q[(size_t)p * w.ldw + cc] = qf;
          w.qr[(size_t)p * w.ldw + cc] = qr;
        }
      }
    }
  }
}

// a7 from stored coefficients (xod_source): q = k_f prod n_reactant - k_r prod n_product.
// kf, kr rows are in USER order; q rows in packed order.  HBM-read bound (16 B per evaluation).
template <int MODE>
__global__ void __launch_bounds__(128) k_rates_from_k(DevTables d, int64_t ncol, int64_t col0, int64_t ld,
                                                      ChunkScratch w, const double *__restrict__ kfa,
                                                      const double *__restrict__ kra,
                                                      const double *__restrict__ n, int rw, int ncg,
                                                      int64_t ntasks) {
  const int lane = threadIdx.x & 31;
  const int64_t gw = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  for (int64_t t = gw; t < ntasks; t += nw) {
    const int cg = (int)(t % ncg);
    const int p0 = (int)(t / ncg) * rw, p1 = min(d.nr, p0 + rw);
    const int64_t c = (int64_t)cg * 32 + lane;
    const bool valid = col0 + c < ncol;
    const int64_t cc = valid ? c : 0;
    const int64_t gc = col0 + cc;
    for (int p = p0; p < p1; ++p) {
      const int2 s01 = __ldg(reinterpret_cast<const int2 *>(d.sp + (size_t)p * 6));
      const int2 s23 = __ldg(reinterpret_cast<const int2 *>(d.sp + (size_t)p * 6 + 2));
      const int2 s45 = __ldg(reinterpret_cast<const int2 *>(d.sp + (size_t)p * 6 + 4));
      const int r0 = s01.x, r1 = s01.y, r2 = s23.x, q0 = s23.y, q1 = s45.x, q2 = s45.y;
      const size_t o = (size_t)__ldg(d.user + p) * ld + gc;
      double qf = kfa[o] * n[(size_t)r0 * ld + gc];
      if (r1 >= 0) qf *= n[(size_t)r1 * ld + gc];
      if (r2 >= 0) qf *= n[(size_t)r2 * ld + gc];
      double qr = 0.0;
      if (p < d.ph_begin && (__ldg(d.flags + p) & 1)) {
        qr = kra[o] * n[(size_t)q0 * ld + gc];
        if (q1 >= 0) qr *= n[(size_t)q1 * ld + gc];
        if (q2 >= 0) qr *= n[(size_t)q2 * ld + gc];
      }
      if (MODE == MODE_QNET) {
        w.q[(size_t)p * w.ldw + cc] = qf - qr;
      } else {
        w.q[(size_t)p * w.ldw + cc] = qf;
        w.qr[(size_t)p * w.ldw + cc] = qr;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// a8: atomic-free production/loss.  dn_i/dt = sum_r nu_ir (q_f,r - q_r,r)   (Eq. 1)
// as a segmented sum over the source CSR.  grid (CTA tasks, chunk column groups); block = 8
// warps; each warp sums one segment of one species row for 32 columns (a per-lane sequential
// loop, no cross-lane reduction); rows cut into several segments are combined through shared
// memory in segment order, so the result is deterministic.
template <bool PL>
__global__ void __launch_bounds__(256) k_source(DevTables d, int64_t ncol, int64_t col0, int64_t ld,
                                                ChunkScratch w, double *__restrict__ dndt,
                                                double *__restrict__ prod, double *__restrict__ loss) {
  __shared__ double part[PL ? 3 : 1][kSrcWarpsPerCta][32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const SrcSeg seg = d.src_seg[(size_t)blockIdx.x * kSrcWarpsPerCta + warp];
  const int64_t c = (int64_t)blockIdx.y * 32 + lane;
  const bool valid = col0 + c < ncol;
  const int64_t cc = valid ? c : 0;
  double a0 = 0.0, a1 = 0.0, sp = 0.0, sl = 0.0;
  if (seg.row >= 0) {
    int k = seg.begin;
    if (!PL) {
      for (; k + 1 < seg.end; k += 2) {
        const double qa = w.q[(size_t)__ldg(d.src_rxn + k) * w.ldw + cc];
        const double qb = w.q[(size_t)__ldg(d.src_rxn + k + 1) * w.ldw + cc];
        a0 = fma((double)__ldg(d.src_nu + k), qa, a0);
        a1 = fma((double)__ldg(d.src_nu + k + 1), qb, a1);
      }
      if (k < seg.end) a0 = fma((double)__ldg(d.src_nu + k), w.q[(size_t)__ldg(d.src_rxn + k) * w.ldw + cc], a0);
      a0 += a1;
    } else {
      for (; k < seg.end; ++k) {
        const size_t o = (size_t)__ldg(d.src_rxn + k) * w.ldw + cc;
        const double nu = (double)__ldg(d.src_nu + k);
        const double tf = nu * w.q[o], tr = -nu * w.qr[o];
        a0 += tf;
        a0 += tr;
        if (tf > 0) sp += tf; else sl -= tf;
        if (tr > 0) sp += tr; else sl -= tr;
      }
    }
  }
  part[0][warp][lane] = a0;
  if (PL) {
    part[1][warp][lane] = sp;
    part[PL ? 2 : 0][warp][lane] = sl;
  }
  __syncthreads();
  if (seg.row >= 0 && seg.nseg > 0 && valid) {
    double t0 = part[0][warp][lane];
    for (int s = 1; s < seg.nseg; ++s) t0 += part[0][warp + s][lane];
    const size_t o = (size_t)seg.row * ld + col0 + c;
    dndt[o] = t0;
    if (PL) {
      double t1 = part[1][warp][lane], t2 = part[PL ? 2 : 0][warp][lane];
      for (int s = 1; s < seg.nseg; ++s) {
        t1 += part[1][warp + s][lane];
        t2 += part[PL ? 2 : 0][warp + s][lane];
      }
      prod[o] = t1;
      loss[o] = t2;
    }
  }
}

// ------------------------------------------------------------------------------------------
// a9: Jacobian values as a gather (BASELINE.json config 5).  One warp per (pattern entry, 32
// columns): loops over the entry's term list  coef * k[dir][rxn] * n[o1] * n[o2]  and writes
// jac[e][col].  No division by n_j; entries without terms are written as 0.
__global__ void __launch_bounds__(256) k_jacobian(DevTables d, int64_t ncol, int64_t ld,
                                                  const double *__restrict__ kf,
                                                  const double *__restrict__ kr,
                                                  const double *__restrict__ n, double *__restrict__ jac) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t c = (int64_t)blockIdx.y * 32 + lane;
  const bool valid = c < ncol;
  const int64_t cc = valid ? c : 0;
  for (int64_t e = (int64_t)blockIdx.x * 8 + warp; e < d.nnz_jac; e += (int64_t)gridDim.x * 8) {
    const int64_t t0 = __ldg(d.jac_term_ptr + e), t1 = __ldg(d.jac_term_ptr + e + 1);
    double acc = 0.0;
    for (int64_t t = t0; t < t1; ++t) {
      const int4 tm = __ldg(reinterpret_cast<const int4 *>(d.jac_terms + t));
      const double *k = tm.x < 0 ? kr : kf;
      double v = (double)__int_as_float(tm.w) * k[(size_t)XOD_IDX(tm.x & 0x7fffffff, d.nr) * ld + cc];
      if (tm.y >= 0) v *= n[(size_t)XOD_IDX(tm.y, d.ns) * ld + cc];
      if (tm.z >= 0) v *= n[(size_t)XOD_IDX(tm.z, d.ns) * ld + cc];
      acc += v;
    }
    if (valid) jac[(size_t)e * ld + c] = acc;
  }
}

// ------------------------------------------------------------------------------------------
// measurement helper: 16 independent DFMA chains per thread, no memory traffic.
__global__ void __launch_bounds__(256) k_probe_dfma(double *out, int iters, double a, double b) {
  double x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = a + i + threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = fma(x[i], b, a);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace xod
