// fused.cuh -- k_fused: the whole source term a1-a8 of one column tile in ONE kernel (sm_100a).
//
// A CTA (16 warps) owns a tile of kFW = 16 consecutive columns and a range of reaction chunks.
// Shared memory holds, as [row][16] fp64 rows of 128 bytes (= all 32 banks, so gathers of whole
// rows by different lane groups never conflict):
//   n_s   [ns + 1]      number densities of the tile (+ a row of ones for absent species slots)
//   acc_s [n_acc]       dn/dt accumulators (+ extra rows of hub species, see pack_fused.cpp)
//   q_s   [2][chunk+1]  net rates of progress of the current / next chunk (+ a zero row)
// Per chunk: phase A (FP64-pipe bound) evaluates k_f, k_r and q = k_f prod n - k_r prod n for
// chunk x 16 (reaction, column) pairs, 8 lanes x 2 columns per reaction, 4 reactions per warp
// pass, reaction parameters read once per 64 pairs; one __syncthreads; phase B (shared-memory
// bound) runs the packer's row tasks: lane groups sum nu q over <= kFSegMax entries and add the
// result to "their" accumulator row.  q is double-buffered, so warps that finish phase B early
// start phase A of the next chunk at once.  No atomics; the summation order is fixed.
//
//   UNI/BI   log2 k_f = c0 + c1 log2 T + c2 / T                                  (Eq. 7)
//            log2 k_r = C0 + C1 log2 T + C2 / T - T (D2 + T (D3 + T (D4 + T D5)))  (Eq. 15 with the
//                        NASA-7 Gibbs polynomials of PAPER.md:671 summed per reaction)
//   FALLOFF  k0[M], k_inf as Eq. 7;  k = k0[M]/(1 + Pr) F   (Eq. 10-12; Troe F:
//            DESIGN.md reading F1);  k_r = k_f 2^z, z from the same seven coefficients
//   PHOTO    k_f = J
#pragma once
#include <cuda_runtime.h>

#include "xod_internal.h"
#include "xod_math.cuh"

namespace xod {

struct FusedArgs {
  int64_t ncol, ld;           // caller's columns and row pitch
  const double *T, *P, *J, *n;
  double *out;                // nsplit == 1: dndt [ns][ld]; else partial sums [nsplit][ns][ldp]
  int64_t ldp;                // pitch of the partial sums
  int32_t ntiles, nsplit;
  double log2_kb;
};

__device__ __forceinline__ double2 lds2(const double *p) { return *reinterpret_cast<const double2 *>(p); }

// seven reverse coefficients of reaction pp in interval g
struct Rev7 { double c[7]; };
__device__ __forceinline__ Rev7 load_rev(const FusedDev &f, int g, int pp) {
  Rev7 r;
  const double *base = f.rev + ((size_t)g * 7) * f.npad + pp;
#pragma unroll
  for (int k = 0; k < 7; ++k) r.c[k] = __ldg(base + (size_t)k * f.npad);
  return r;
}
// z-polynomial: C0 + C1 log2 T + C2 / T - T (D2 + T (D3 + T (D4 + T D5)))
__device__ __forceinline__ double rev_eval(const Rev7 &r, double T, double l2T, double invT) {
  const double poly = fma(T, fma(T, fma(T, r.c[6], r.c[5]), r.c[4]), r.c[3]);
  return fma(r.c[2], invT, fma(r.c[1], l2T, fma(-T, poly, r.c[0])));
}

__global__ void __launch_bounds__(kFWarps * 32, 1) k_fused(FusedDev f, int ns, FusedArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *n_s = reinterpret_cast<double *>(smem_raw);
  double *acc_s = n_s + (size_t)(ns + 1) * kFW;
  double *q_s = acc_s + (size_t)f.n_acc * kFW;
  double *cT = q_s + (size_t)2 * (f.chunk + 1) * kFW;
  double *cL2T = cT + kFW, *cInvT = cL2T + kFW, *cLM = cInvT + kFW;
  int *cG = reinterpret_cast<int *>(cLM + kFW);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int grp = lane >> 3, l2 = (lane & 7) * 2;  // lane group (reaction slot) and first column
  const int qrows = f.chunk + 1;

  for (int item = blockIdx.x; item < a.ntiles * a.nsplit; item += gridDim.x) {
    const int tile = item / a.nsplit, split = item - tile * a.nsplit;
    const int k_begin = (int)((int64_t)f.nchunk * split / a.nsplit);
    const int k_end = (int)((int64_t)f.nchunk * (split + 1) / a.nsplit);
    const int64_t col0 = (int64_t)tile * kFW;

    __syncthreads();  // the previous item's readers are done with shared memory
    // ---- a1: column scalars (idle columns of a ragged tile reuse the last valid column)
    if (tid < kFW) {
      const int64_t gc = min(col0 + tid, a.ncol - 1);
      const double Tc = a.T[gc], Pc = a.P[gc];
      const double l2T = log2(Tc);
      cT[tid] = Tc, cL2T[tid] = l2T, cInvT[tid] = 1.0 / Tc;
      cLM[tid] = log2(Pc) - a.log2_kb - l2T;  // log2 [M], [M] = P/(k_B T)
      int g = 0;
      for (int k = 0; k < f.n_bp; ++k) g += __ldg(f.bp + k) < Tc;
      cG[tid] = g;
    }
    // ---- n tile, ones row, zeroed accumulators and zero rows of q
    {
      const int c = tid & (kFW - 1);
      const int64_t gc = min(col0 + c, a.ncol - 1);
      for (int i = tid >> 4; i < ns; i += (kFWarps * 32) >> 4) n_s[i * kFW + c] = a.n[(size_t)i * a.ld + gc];
      for (int i = tid; i < f.n_acc * kFW; i += kFWarps * 32) acc_s[i] = 0.0;
      if (tid < kFW) {
        n_s[ns * kFW + tid] = 1.0;
        q_s[(size_t)f.chunk * kFW + tid] = 0.0;
        q_s[(size_t)(qrows + f.chunk) * kFW + tid] = 0.0;
      }
    }
    __syncthreads();
    const double T0 = cT[l2], T1 = cT[l2 + 1], lT0 = cL2T[l2], lT1 = cL2T[l2 + 1];
    const double iT0 = cInvT[l2], iT1 = cInvT[l2 + 1];
    const int g0 = cG[l2], g1 = cG[l2 + 1];
    const int64_t gc0 = min(col0 + l2, a.ncol - 1), gc1 = min(col0 + l2 + 1, a.ncol - 1);

    for (int k = k_begin; k < k_end; ++k) {
      double *qb = q_s + (size_t)((k - k_begin) & 1) * qrows * kFW;
      // ------------------------------------------------------------ phase A
      const int pp_chunk = k * f.chunk;
      for (int pass = 0; pass < f.chunk / kFPass; ++pass) {
        const int rloc = pass * kFPass + warp * kFRxnPerWarp + grp;
        const int pp = pp_chunk + rloc;
        const int ppw = pp_chunk + pass * kFPass + warp * kFRxnPerWarp;  // warp-uniform
        if (ppw >= f.ph_end) break;                                    // only padding left
        const int4 sa = __ldg(reinterpret_cast<const int4 *>(f.sp + (size_t)pp * 8));
        const int4 sb = __ldg(reinterpret_cast<const int4 *>(f.sp + (size_t)pp * 8 + 4));
        double kf0, kf1, kr0, kr1;
        if (ppw < f.fo_end) {
          const double c0 = __ldg(f.c + pp), c1 = __ldg(f.c + f.npad + pp), c2 = __ldg(f.c + 2 * (size_t)f.npad + pp);
          const double y0 = fma(c2, iT0, fma(c1, lT0, c0)), y1 = fma(c2, iT1, fma(c1, lT1, c0));
          const Rev7 ra = load_rev(f, g0, pp);
          double z0 = rev_eval(ra, T0, lT0, iT0), z1;
          if (g1 == g0) {
            z1 = rev_eval(ra, T1, lT1, iT1);
          } else {
            const Rev7 rb = load_rev(f, g1, pp);
            z1 = rev_eval(rb, T1, lT1, iT1);
          }
          if (ppw < f.arr_end) {  // UNI, BI
            kf0 = xexp2(y0), kf1 = xexp2(y1);
            kr0 = xexp2(z0), kr1 = xexp2(z1);
          } else {                // FALLOFF
            const int q = pp - f.arr_end, nfo = f.fo_end - f.arr_end;
            const double m0 = __ldg(f.l + q), m1 = __ldg(f.l + nfo + q), m2 = __ldg(f.l + 2 * nfo + q);
            const double fcl = __ldg(f.l + 3 * nfo + q), cN = __ldg(f.l + 4 * nfo + q);
            const double w0 = fma(m2, iT0, fma(m1, lT0, m0)) + cLM[l2];
            const double w1 = fma(m2, iT1, fma(m1, lT1, m0)) + cLM[l2 + 1];
            const double lp0 = w0 - y0, lp1 = w1 - y1;             // log2 Pr
            const double x0 = lp0 * cN, x1 = lp1 * cN;
            const double lF0 = fcl / fma(x0, x0, 1.0), lF1 = fcl / fma(x1, x1, 1.0);
            const double d0 = 1.0 / (1.0 + xexp2(-fabs(lp0))), d1 = 1.0 / (1.0 + xexp2(-fabs(lp1)));
            const double ym0 = fmin(w0, y0) + lF0, ym1 = fmin(w1, y1) + lF1;
            kf0 = xexp2(ym0) * d0, kf1 = xexp2(ym1) * d1;
            kr0 = xexp2(ym0 + z0) * d0, kr1 = xexp2(ym1 + z1) * d1;
          }
        } else {                  // PHOTO
          kf0 = a.J[(size_t)sb.z * a.ld + gc0], kf1 = a.J[(size_t)sb.z * a.ld + gc1];
          kr0 = kr1 = 0.0;
        }
        double2 v = lds2(n_s + sa.x * kFW + l2);
        double qf0 = kf0 * v.x, qf1 = kf1 * v.y;
        if (sa.y != ns) { v = lds2(n_s + sa.y * kFW + l2); qf0 *= v.x, qf1 *= v.y; }
        if (sa.z != ns) { v = lds2(n_s + sa.z * kFW + l2); qf0 *= v.x, qf1 *= v.y; }
        v = lds2(n_s + sa.w * kFW + l2);
        double qr0 = kr0 * v.x, qr1 = kr1 * v.y;
        if (sb.x != ns) { v = lds2(n_s + sb.x * kFW + l2); qr0 *= v.x, qr1 *= v.y; }
        if (sb.y != ns) { v = lds2(n_s + sb.y * kFW + l2); qr0 *= v.x, qr1 *= v.y; }
        *reinterpret_cast<double2 *>(qb + (size_t)rloc * kFW + l2) = make_double2(qf0 - qr0, qf1 - qr1);
      }
      __syncthreads();
      // ------------------------------------------------------------ phase B
      const int t_begin = __ldg(f.task_ptr + (size_t)k * kFWarps + warp);
      const int t_end = __ldg(f.task_ptr + (size_t)k * kFWarps + warp + 1);
      for (int t = t_begin; t < t_end; ++t) {
        const int4 tk = __ldg(reinterpret_cast<const int4 *>(f.task + t));
        const unsigned rows = (grp & 2) ? (unsigned)tk.w : (unsigned)tk.z;
        const int row = (int)((grp & 1) ? rows >> 16 : rows & 0xffffu);
        const uint32_t *e = f.entry + tk.x + grp;
        double s0 = 0.0, s1 = 0.0;
        for (int st = 0; st < tk.y; ++st) {
          const uint32_t en = __ldg(e + st * 4);
          const double nu = __hiloint2double((int)(en & 0xffff0000u), 0);
          const double2 qv = lds2(qb + (size_t)(en & 0xffffu) * kFW + l2);
          s0 = fma(nu, qv.x, s0), s1 = fma(nu, qv.y, s1);
        }
        if (row != 0xffff) {
          double2 *dst = reinterpret_cast<double2 *>(acc_s + (size_t)row * kFW + l2);
          double2 cur = *dst;
          cur.x += s0, cur.y += s1;
          *dst = cur;
        }
      }
    }
    __syncthreads();
    // ---- extra rows of hub species -> their species row, in row order (fixed order)
    if (tid < kFW) {
      for (int x = 0; x < f.n_extra; ++x) {
        const int er = __ldg(f.extra + 2 * x), sp = __ldg(f.extra + 2 * x + 1);
        acc_s[sp * kFW + tid] += acc_s[er * kFW + tid];
      }
    }
    __syncthreads();
    // ---- write the tile
    {
      const int c = tid & (kFW - 1);
      if (col0 + c < a.ncol) {
        double *o = a.nsplit == 1 ? a.out + col0 + c : a.out + (size_t)split * ns * a.ldp + col0 + c;
        const int64_t pitch = a.nsplit == 1 ? a.ld : a.ldp;
        for (int i = tid >> 4; i < ns; i += (kFWarps * 32) >> 4) o[(size_t)i * pitch] = acc_s[i * kFW + c];
      }
    }
  }
}

// dn/dt = sum over the reaction splits, in split order.  thread = column.
__global__ void __launch_bounds__(128) k_fused_combine(int ns, int64_t ncol, int64_t ld, int64_t ldp, int nsplit,
                                                       const double *__restrict__ part, double *__restrict__ dndt) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int i = blockIdx.y;
  if (c >= ncol) return;
  double s = part[(size_t)i * ldp + c];
  for (int k = 1; k < nsplit; ++k) s += part[((size_t)k * ns + i) * ldp + c];
  dndt[(size_t)i * ld + c] = s;
}

}  // namespace xod
