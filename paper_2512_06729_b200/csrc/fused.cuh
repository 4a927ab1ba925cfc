// fused.cuh -- k_fused: the whole source term a1-a8 of one column tile in ONE kernel (sm_100a).
//
// A CTA (kFWarps = 20 warps, one per SM, persistent over tiles) owns a tile of kFW = 16
// consecutive columns and a range of reaction chunks.
// Shared memory holds, as [row][16] fp64 rows of 128 bytes (= all 32 banks, so gathers of whole
// rows by different lane groups never conflict):
//   n_s   [ns + 1]      number densities of the tile (+ a row of ones for absent species slots)
//   acc_s [n_acc]       dn/dt accumulators (+ extra rows of hub species, see pack_fused.cpp)
//   q_s   [2][chunk+1]  net rates of progress of the current / next chunk (+ a zero row)
//   meta_s[2][meta_cap] the production/loss schedule of the current / next chunk (cp.async)
// Per chunk: phase A (FP64-pipe bound) evaluates k_f, k_r and q = k_f prod n - k_r prod n for
// chunk x 16 (reaction, column) pairs, 8 lanes x 2 columns per reaction, 4 reactions per warp
// pass; the parameters of those 4 reactions are one contiguous block read with 16-byte loads at
// immediate offsets.  One __syncthreads; phase B (shared-memory bound) runs the packer's row
// tasks: lane groups sum nu q over <= kFSegMax entries and add the result to "their"
// accumulator row.  q and the schedule are double-buffered, so warps that finish phase B early
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
#include <xod_cta.cuh>  // CTA primitives (dynamic shared memory, cp.async); resolved through -I csrc
#include "sched.cuh"

namespace xod {

struct FusedArgs {
  int64_t ncol, ld;           // caller's columns and the row pitch of the inputs
  int64_t ldo;                // row pitch of dndt (= ld in the public calls; the implicit step writes into its workspace)
  const double *T, *P, *J, *n;
  const double *kf, *kr;      // FROMK only: stored coefficients [n_reactions][ld]
  double *out;                // nsplit == 1: dndt [ns][ld]; else partial sums [nsplit][ns][ldp]
  int64_t ldp;                // pitch of the partial sums
  int32_t ntiles, nsplit;
  int32_t nr, n_photo;        // rows of kf/kr and of J (bounds of the -DXOD_CHECK build)
  double log2_kb;
};

__device__ __forceinline__ double2 ldg2(const unsigned char *p) { return __ldg(reinterpret_cast<const double2 *>(p)); }

// log2 k_r (UNI/BI) or z (FALLOFF) from the block of interval g
__device__ __forceinline__ double rev_eval(const unsigned char *blk, int slot16, double c0r /*C0*/, double T,
                                           double l2T, double invT) {
  const double2 c12 = ldg2(blk + 4 * 64 + slot16), d23 = ldg2(blk + 5 * 64 + slot16), d45 = ldg2(blk + 6 * 64 + slot16);
  const double poly = fma(T, fma(T, fma(T, d45.y, d45.x), d23.y), d23.x);
  return fma(c12.y, invT, fma(c12.x, l2T, fma(-T, poly, c0r)));
}

// FROMK = false: xod_source_fused (coefficients evaluated here, a1-a8).
// FROMK = true : xod_source (a7-a8): k_f, k_r are read from the caller's arrays (USER reaction order).
// byte offset of the parameter block (4 reactions) that holds padded reaction pp, inside an interval
__device__ __forceinline__ size_t block_offset(const FusedDev &f, int pp) {
  if (pp < f.arr_end) return (size_t)(pp >> 2) * kFBlkArr;
  if (pp < f.fo_end) return (size_t)f.blk_fo_off + (size_t)((pp - f.arr_end) >> 2) * kFBlkFo;
  return (size_t)f.blk_ph_off + (size_t)((pp - f.fo_end) >> 2) * kFBlkPh;
}

template <bool FROMK>
__global__ void __launch_bounds__(kFWarps * 32, 1) k_fused(FusedDev f, int ns, FusedArgs a) {
  unsigned char *smem_raw = cta_dyn_smem();
  double *n_s = reinterpret_cast<double *>(smem_raw);
  double *acc_s = n_s + (size_t)(ns + 1) * kFW;
  double *q_s = acc_s + (size_t)f.n_acc * kFW;
  int4 *meta_s = reinterpret_cast<int4 *>(q_s + (size_t)2 * (f.chunk + 1) * kFW);
  double *cT = reinterpret_cast<double *>(meta_s + 2 * f.meta_cap);
  double *cL2T = cT + kFW, *cInvT = cL2T + kFW, *cLM = cInvT + kFW;
  int *cG = reinterpret_cast<int *>(cLM + kFW);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int grp = lane >> 3, l2 = (lane & 7) * 2;  // lane group (reaction slot) and first column
  const int slot16 = grp * 16;
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
      const double Tc = FROMK ? 1000.0 : a.T[gc], Pc = FROMK ? 1.0e6 : a.P[gc];
      const double l2T = log2(Tc);
      cT[tid] = Tc, cL2T[tid] = l2T, cInvT[tid] = 1.0 / Tc;
      cLM[tid] = log2(Pc) - a.log2_kb - l2T;  // log2 [M], [M] = P/(k_B T)
      int g = 0;
      for (int k = 0; k < f.n_bp; ++k) g += __ldg(f.bp + k) < Tc;
      cG[tid] = XOD_IDX(g, f.n_bp + 1);
    }
    // ---- n tile, ones row, zeroed accumulators and zero rows of q
    {
      const int c = tid & (kFW - 1);
      const int64_t gc = min(col0 + c, a.ncol - 1);
      // all loads of the tile in flight at once (cp.async), not one round trip per row
      for (int i = tid >> 4; i < ns; i += (kFWarps * 32) >> 4) cp_async8(n_s + i * kFW + c, a.n + (size_t)i * a.ld + gc);
      for (int i = tid; i < f.n_acc * kFW; i += kFWarps * 32) acc_s[i] = 0.0;
      if (tid < kFW) {
        n_s[ns * kFW + tid] = 1.0;
        q_s[(size_t)f.chunk * kFW + tid] = 0.0;
        q_s[(size_t)(qrows + f.chunk) * kFW + tid] = 0.0;
      }
    }
    cp_async_wait_all();
    __syncthreads();
    const double T0 = cT[l2], T1 = cT[l2 + 1], lT0 = cL2T[l2], lT1 = cL2T[l2 + 1];
    const double iT0 = cInvT[l2], iT1 = cInvT[l2 + 1];
    const int64_t gc0 = min(col0 + l2, a.ncol - 1), gc1 = min(col0 + l2 + 1, a.ncol - 1);
    const unsigned char *blk0 = f.blk + (size_t)cG[l2] * f.blk_stride;
    const unsigned char *blk1 = f.blk + (size_t)cG[l2 + 1] * f.blk_stride;
    const bool same_g = blk0 == blk1;
    const double *n_l = n_s + l2;

    for (int k = k_begin; k < k_end; ++k) {
      const int buf = (k - k_begin) & 1;
      double *qb = q_s + (size_t)buf * qrows * kFW;
      int4 *mb = meta_s + (size_t)buf * f.meta_cap;
      // schedule of this chunk -> shared memory, overlapped with phase A
      {
        const int m0 = __ldg(f.meta_ptr + k), m1 = __ldg(f.meta_ptr + k + 1);
        for (int u = m0 + tid; u < m1; u += kFWarps * 32) cp_async16(mb + XOD_IDX(u - m0, f.meta_cap), f.meta + u);
      }
      // ------------------------------------------------------------ phase A
      const int pp_chunk = k * f.chunk;
#pragma unroll 1
      for (int pass = 0; pass < f.chunk / kFPass; ++pass) {
        const int rbase = pass * kFPass + warp * kFRxnPerWarp;
        const int ppw = pp_chunk + rbase;  // first of the warp's 4 reactions (one segment)
        if (ppw >= f.ph_end) break;        // only padding left
        double kf0, kf1, kr0, kr1;
        int4 sa;  // species slots as 16-bit indices: r0 r1 | r2 p0 | p1 p2 | J row
        if (FROMK) {
          const int pp = ppw + grp;
          const unsigned char *b0 = blk0 + XOD_IDX(block_offset(f, pp), (size_t)f.blk_stride) + slot16;
          sa = __ldg(reinterpret_cast<const int4 *>(b0));
          const int user = XOD_IDX(max(__ldg(f.pp_user + pp), 0), a.nr);  // padding slots read row 0 (their q is never used)
          const int64_t gc0 = min(col0 + l2, a.ncol - 1), gc1 = min(col0 + l2 + 1, a.ncol - 1);
          const double *kfr = a.kf + (size_t)user * a.ld, *krr = a.kr + (size_t)user * a.ld;
          kf0 = __ldg(kfr + gc0), kf1 = __ldg(kfr + gc1), kr0 = __ldg(krr + gc0), kr1 = __ldg(krr + gc1);
        } else if (ppw < f.fo_end) {
          const bool arr = ppw < f.arr_end;
          const size_t off = arr ? (size_t)(ppw >> 2) * kFBlkArr
                                 : (size_t)f.blk_fo_off + (size_t)((ppw - f.arr_end) >> 2) * kFBlkFo;
          const unsigned char *b0 = blk0 + XOD_IDX(off, (size_t)f.blk_stride);
          sa = __ldg(reinterpret_cast<const int4 *>(b0 + slot16));
          const double2 c01 = ldg2(b0 + 2 * 64 + slot16), c2C = ldg2(b0 + 3 * 64 + slot16);
          const double y0 = fma(c2C.x, iT0, fma(c01.y, lT0, c01.x)), y1 = fma(c2C.x, iT1, fma(c01.y, lT1, c01.x));
          const double z0 = rev_eval(b0, slot16, c2C.y, T0, lT0, iT0);
          double z1 = rev_eval(b0, slot16, c2C.y, T1, lT1, iT1);
          if (!same_g) {  // the thread's two columns sit in different thermo intervals (rare): redo column 1
            const unsigned char *b1 = blk1 + off;
            z1 = rev_eval(b1, slot16, ldg2(b1 + 3 * 64 + slot16).y, T1, lT1, iT1);
          }
          if (arr) {  // UNI, BI
            const unsigned m = max(max(xexp2_mag(y0), xexp2_mag(y1)), max(xexp2_mag(z0), xexp2_mag(z1)));
            if (m < kExp2FastMax) {
              kf0 = xexp2_fast(y0), kf1 = xexp2_fast(y1), kr0 = xexp2_fast(z0), kr1 = xexp2_fast(z1);
            } else {
              kf0 = xexp2_slow(y0), kf1 = xexp2_slow(y1), kr0 = xexp2_slow(z0), kr1 = xexp2_slow(z1);
            }
          } else {    // FALLOFF
            const double2 m01 = ldg2(b0 + 7 * 64 + slot16), m2f = ldg2(b0 + 8 * 64 + slot16);
            const double cN = ldg2(b0 + 9 * 64 + slot16).x;
            const double w0 = fma(m2f.x, iT0, fma(m01.y, lT0, m01.x)) + cLM[l2];
            const double w1 = fma(m2f.x, iT1, fma(m01.y, lT1, m01.x)) + cLM[l2 + 1];
            const double lp0 = w0 - y0, lp1 = w1 - y1;             // log2 Pr
            const double x0 = lp0 * cN, x1 = lp1 * cN;
            const double lF0 = m2f.y / fma(x0, x0, 1.0), lF1 = m2f.y / fma(x1, x1, 1.0);
            const double d0 = 1.0 / (1.0 + xexp2(-fabs(lp0))), d1 = 1.0 / (1.0 + xexp2(-fabs(lp1)));
            const double ym0 = fmin(w0, y0) + lF0, ym1 = fmin(w1, y1) + lF1;
            kf0 = xexp2(ym0) * d0, kf1 = xexp2(ym1) * d1;
            kr0 = xexp2(ym0 + z0) * d0, kr1 = xexp2(ym1 + z1) * d1;
          }
        } else {                  // PHOTO
          const unsigned char *b0 = f.blk + XOD_IDX((size_t)f.blk_ph_off + (size_t)((ppw - f.fo_end) >> 2) * kFBlkPh, (size_t)f.blk_stride);
          sa = __ldg(reinterpret_cast<const int4 *>(b0 + slot16));
          const size_t jrow = (size_t)XOD_IDX(sa.w, a.n_photo);
          kf0 = a.J[jrow * a.ld + gc0], kf1 = a.J[jrow * a.ld + gc1];
          kr0 = kr1 = 0.0;
        }
        // a7: rates of progress (absent slots read the row of ones)
        const int r0 = XOD_IDX(sa.x & 0xffff, ns + 1), r1 = XOD_IDX((int)((unsigned)sa.x >> 16), ns + 1), r2 = XOD_IDX(sa.y & 0xffff, ns + 1);
        const int p0 = XOD_IDX((int)((unsigned)sa.y >> 16), ns + 1), p1 = XOD_IDX(sa.z & 0xffff, ns + 1), p2 = XOD_IDX((int)((unsigned)sa.z >> 16), ns + 1);
        double2 v = lds2(n_l + r0 * kFW);
        double qf0 = kf0 * v.x, qf1 = kf1 * v.y;
        if (r1 != ns) { v = lds2(n_l + r1 * kFW); qf0 *= v.x, qf1 *= v.y; }
        if (r2 != ns) { v = lds2(n_l + r2 * kFW); qf0 *= v.x, qf1 *= v.y; }
        v = lds2(n_l + p0 * kFW);
        double qr0 = kr0 * v.x, qr1 = kr1 * v.y;
        if (p1 != ns) { v = lds2(n_l + p1 * kFW); qr0 *= v.x, qr1 *= v.y; }
        if (p2 != ns) { v = lds2(n_l + p2 * kFW); qr0 *= v.x, qr1 *= v.y; }
        *reinterpret_cast<double2 *>(qb + (size_t)(rbase + grp) * kFW + l2) = make_double2(qf0 - qr0, qf1 - qr1);
      }
      cp_async_wait_all();
      __syncthreads();
      // ------------------------------------------------------------ phase B
      sched_reduce(mb, qb, acc_s, warp, grp, l2, qrows, f.n_acc, f.meta_cap);
    }
    __syncthreads();
    // ---- extra rows of hub species -> their species row, in row order (fixed order)
    if (tid < kFW) {
      for (int x = 0; x < f.n_extra; ++x) {
        const int er = __ldg(f.extra + 2 * x), sp = __ldg(f.extra + 2 * x + 1);
        acc_s[XOD_IDX(sp, ns) * kFW + tid] += acc_s[XOD_IDX(er, f.n_acc) * kFW + tid];
      }
    }
    __syncthreads();
    // ---- write the tile
    {
      const int c = tid & (kFW - 1);
      if (col0 + c < a.ncol) {
        double *o = a.nsplit == 1 ? a.out + col0 + c : a.out + (size_t)split * ns * a.ldp + col0 + c;
        const int64_t pitch = a.nsplit == 1 ? a.ldo : a.ldp;
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
