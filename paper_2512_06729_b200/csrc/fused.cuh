// fused.cuh -- k_fused: the whole source term a1-a8 of one column tile in ONE kernel (sm_100a).
//
// A CTA (kFWarps = 20 warps, one per SM, persistent over tiles) owns a tile of kFW = 16
// consecutive columns and a range of reaction chunks.
// Shared memory holds, as [row][16] fp64 rows of 128 bytes (= all 32 banks, so gathers of whole
// rows by different lane groups never conflict):
//   n_s   [ns + 2]      number densities of the tile, a row of ones (absent species slots) and a row of zeros
//                       (first product slot of an irreversible reaction: q_r = 0 exactly)
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

// log2 k_r (UNI/BI) or z (FALLOFF) of one reaction; b = its 16-byte column in the block of the column's interval
__device__ __forceinline__ double rev_eval(const unsigned char *b, double c0r /*C0*/, double T, double l2T, double invT) {
  const double2 c12 = ldg2(b + 4 * 64), d23 = ldg2(b + 5 * 64), d45 = ldg2(b + 6 * 64);
  const double poly = fma(T, fma(T, fma(T, d45.y, d45.x), d23.y), d23.x);
  return fma(c12.y, invT, fma(c12.x, l2T, fma(-T, poly, c0r)));
}
// the same for the second column of a thread when it sits in another thermo interval than the first (a tile that
// straddles a t_mid breakpoint: rare).  Out of line, so that the common path carries no predicated copy of it.
__device__ __noinline__ double rev_eval_other(const unsigned char *b, double T, double l2T, double invT) {
  return rev_eval(b, ldg2(b + 3 * 64).y, T, l2T, invT);
}

// a7: q = k_f prod n_reactants - k_r prod n_products for the thread's two columns.  sa = the six species slots as
// 16-bit rows of the n tile (r0 r1 | r2 p0 | p1 p2); row ns = ones (absent slot), row ns + 1 = zeros (first
// product slot of an irreversible reaction, so that q_r = 0 exactly whatever k_r holds).
__device__ __forceinline__ void rates_of_progress(const int4 sa, int ns, const double *n_l, double kf0, double kf1,
                                                  double kr0, double kr1, double *qdst) {
  const int r0 = XOD_IDX(sa.x & 0xffff, ns + 2), r1 = XOD_IDX((int)((unsigned)sa.x >> 16), ns + 2), r2 = XOD_IDX(sa.y & 0xffff, ns + 2);
  const int p0 = XOD_IDX((int)((unsigned)sa.y >> 16), ns + 2), p1 = XOD_IDX(sa.z & 0xffff, ns + 2), p2 = XOD_IDX((int)((unsigned)sa.z >> 16), ns + 2);
  double2 v = lds2(n_l + r0 * kFW);
  double qf0 = kf0 * v.x, qf1 = kf1 * v.y;
  if (r1 != ns) { v = lds2(n_l + r1 * kFW); qf0 *= v.x, qf1 *= v.y; }
  if (r2 != ns) { v = lds2(n_l + r2 * kFW); qf0 *= v.x, qf1 *= v.y; }
  v = lds2(n_l + p0 * kFW);
  double qr0 = kr0 * v.x, qr1 = kr1 * v.y;
  if (p1 != ns) { v = lds2(n_l + p1 * kFW); qr0 *= v.x, qr1 *= v.y; }
  if (p2 != ns) { v = lds2(n_l + p2 * kFW); qr0 *= v.x, qr1 *= v.y; }
  *reinterpret_cast<double2 *>(qdst) = make_double2(qf0 - qr0, qf1 - qr1);
}

// FROMK = false: xod_source_fused (coefficients evaluated here, a1-a8).
// FROMK = true : xod_source (a7-a8): k_f, k_r are read from the caller's arrays (USER reaction order).
template <bool FROMK>
__global__ void __launch_bounds__(kFWarps * 32, 1) k_fused(FusedDev f, int ns, FusedArgs a) {
  unsigned char *smem_raw = cta_dyn_smem();
  double *n_s = reinterpret_cast<double *>(smem_raw);
  double *acc_s = n_s + (size_t)(ns + 2) * kFW;
  double *q_s = acc_s + (size_t)f.n_acc * kFW;
  int4 *meta_s = reinterpret_cast<int4 *>(q_s + (size_t)2 * (f.chunk + 1) * kFW);
  double *cT = reinterpret_cast<double *>(meta_s + 2 * f.meta_cap);
  double *cL2T = cT + kFW, *cInvT = cL2T + kFW, *cLM = cInvT + kFW;
  int *cG = reinterpret_cast<int *>(cLM + kFW);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int grp = lane >> 3, l2 = (lane & 7) * 2;  // lane group (reaction slot) and first column
  const int slot16 = grp * 16;
  const int qrows = f.chunk + 1;
  const int npass = f.chunk / kFPass;
  constexpr int kArrStep = kFPass / kFRxnPerWarp * kFBlkArr, kFoStep = kFPass / kFRxnPerWarp * kFBlkFo,
                kPhStep = kFPass / kFRxnPerWarp * kFBlkPh;   // bytes between the blocks of consecutive passes of a warp

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
    // ---- n tile, ones and zeros rows, zeroed accumulators and zero rows of q
    {
      const int c = tid & (kFW - 1);
      const int64_t gc = min(col0 + c, a.ncol - 1);
      // all loads of the tile in flight at once (cp.async), not one round trip per row
      if (col0 + kFW <= a.ncol && ((reinterpret_cast<uintptr_t>(a.n) | ((size_t)a.ld * sizeof(double))) & 15) == 0) {
        // a full tile whose rows are 16-byte aligned: two columns per copy
        for (int u = tid; u < ns * (kFW / 2); u += kFWarps * 32)
          cp_async16(n_s + u * 2, a.n + (size_t)(u >> 3) * a.ld + col0 + (u & 7) * 2);
      } else {
        for (int i = tid >> 4; i < ns; i += (kFWarps * 32) >> 4) cp_async8(n_s + i * kFW + c, a.n + (size_t)i * a.ld + gc);
      }
      for (int i = tid; i < f.n_acc * kFW; i += kFWarps * 32) acc_s[i] = 0.0;
      if (tid < kFW) {
        n_s[ns * kFW + tid] = 1.0;
        n_s[(ns + 1) * kFW + tid] = 0.0;
        q_s[(size_t)f.chunk * kFW + tid] = 0.0;
        q_s[(size_t)(qrows + f.chunk) * kFW + tid] = 0.0;
      }
    }
    cp_async_wait_all();
    __syncthreads();
    const double T0 = cT[l2], T1 = cT[l2 + 1], lT0 = cL2T[l2], lT1 = cL2T[l2 + 1];
    const double iT0 = cInvT[l2], iT1 = cInvT[l2 + 1];
    const int64_t gc0 = min(col0 + l2, a.ncol - 1), gc1 = min(col0 + l2 + 1, a.ncol - 1);
    // the thread's 16-byte column (reaction slot grp) in the blocks of its first column's thermo interval, and the
    // distance to the same place in the interval of its second column (0 unless the tile straddles a breakpoint)
    const unsigned char *blk0 = f.blk + (size_t)cG[l2] * f.blk_stride + slot16;
    const int64_t dblk = ((int64_t)cG[l2 + 1] - cG[l2]) * f.blk_stride;
    const bool same_g = dblk == 0;
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
      // Pass p of this warp evaluates the 4 padded reactions ppw0 + p kFPass .. + 3, which lie in one code segment
      // (segments are padded to multiples of 4): the passes are three runs UNI/BI | FALLOFF | PHOTO, each a loop
      // of its own whose block pointer advances by a constant; passes past ph_end are padding and skipped.
      const int ppw0 = k * f.chunk + warp * kFRxnPerWarp;
      auto passes_below = [&](int end) { const int d = end - ppw0; return d <= 0 ? 0 : min(npass, (d + kFPass - 1) / kFPass); };
      double *qdst = qb + (size_t)(warp * kFRxnPerWarp + grp) * kFW + l2;
      const int p_ph = passes_below(f.ph_end);
      if (FROMK) {   // k_f, k_r from the caller's rows; the blocks supply the species slots only (any interval)
        const int p_arr = passes_below(f.arr_end), p_fo = passes_below(f.fo_end);
        const int *up = f.pp_user + ppw0 + grp;
        auto run = [&](int pass_end, const unsigned char *b, int step, int &pass) {
#pragma unroll 1
          for (; pass < pass_end; ++pass, b += step, up += kFPass, qdst += kFPass * kFW) {
            const int4 sa = __ldg(reinterpret_cast<const int4 *>(b));
            const int user = XOD_IDX(max(__ldg(up), 0), a.nr);  // padding slots read row 0 (their q is never used)
            const double *kfr = a.kf + (size_t)user * a.ld, *krr = a.kr + (size_t)user * a.ld;
            rates_of_progress(sa, ns, n_l, __ldg(kfr + gc0), __ldg(kfr + gc1), __ldg(krr + gc0), __ldg(krr + gc1), qdst);
          }
        };
        int pass = 0;
        const unsigned char *b0 = f.blk + slot16;
        if (p_arr > 0) run(p_arr, b0 + XOD_IDX((size_t)(ppw0 >> 2) * kFBlkArr, (size_t)f.blk_stride), kArrStep, pass);
        if (pass < p_fo)
          run(p_fo, b0 + XOD_IDX((size_t)f.blk_fo_off + (size_t)((ppw0 + pass * kFPass - f.arr_end) >> 2) * kFBlkFo, (size_t)f.blk_stride), kFoStep, pass);
        if (pass < p_ph)
          run(p_ph, b0 + XOD_IDX((size_t)f.blk_ph_off + (size_t)((ppw0 + pass * kFPass - f.fo_end) >> 2) * kFBlkPh, (size_t)f.blk_stride), kPhStep, pass);
      } else {
        const int p_arr = passes_below(f.arr_end), p_fo = passes_below(f.fo_end);
        int pass = 0;
        if (p_arr > 0) {     // UNI, BI
          const unsigned char *b = blk0 + XOD_IDX((size_t)(ppw0 >> 2) * kFBlkArr, (size_t)f.blk_stride);
          (void)XOD_IDX((size_t)((ppw0 + (p_arr - 1) * kFPass) >> 2) * kFBlkArr, (size_t)f.blk_stride);
#pragma unroll 1
          for (; pass < p_arr; ++pass, b += kArrStep, qdst += kFPass * kFW) {
            const int4 sa = __ldg(reinterpret_cast<const int4 *>(b));
            const double2 c01 = ldg2(b + 2 * 64), c2C = ldg2(b + 3 * 64);
            const double y0 = fma(c2C.x, iT0, fma(c01.y, lT0, c01.x)), y1 = fma(c2C.x, iT1, fma(c01.y, lT1, c01.x));
            const double z0 = rev_eval(b, c2C.y, T0, lT0, iT0);
            const double z1 = same_g ? rev_eval(b, c2C.y, T1, lT1, iT1) : rev_eval_other(b + dblk, T1, lT1, iT1);
            const unsigned m = max(max(xexp2_mag(y0), xexp2_mag(y1)), max(xexp2_mag(z0), xexp2_mag(z1)));
            double kf0, kf1, kr0, kr1;
            if (m < kExp2FastMax) {
              kf0 = xexp2_fast(y0), kf1 = xexp2_fast(y1), kr0 = xexp2_fast(z0), kr1 = xexp2_fast(z1);
            } else {
              kf0 = xexp2_slow(y0), kf1 = xexp2_slow(y1), kr0 = xexp2_slow(z0), kr1 = xexp2_slow(z1);
            }
            rates_of_progress(sa, ns, n_l, kf0, kf1, kr0, kr1, qdst);
          }
        }
        if (pass < p_fo) {   // FALLOFF
          const unsigned char *b = blk0 + XOD_IDX((size_t)f.blk_fo_off + (size_t)((ppw0 + pass * kFPass - f.arr_end) >> 2) * kFBlkFo, (size_t)f.blk_stride);
          (void)XOD_IDX((size_t)f.blk_fo_off + (size_t)((ppw0 + (p_fo - 1) * kFPass - f.arr_end) >> 2) * kFBlkFo, (size_t)f.blk_stride);
          const double lM0 = cLM[l2], lM1 = cLM[l2 + 1];
#pragma unroll 1
          for (; pass < p_fo; ++pass, b += kFoStep, qdst += kFPass * kFW) {
            const int4 sa = __ldg(reinterpret_cast<const int4 *>(b));
            const double2 c01 = ldg2(b + 2 * 64), c2C = ldg2(b + 3 * 64);
            const double y0 = fma(c2C.x, iT0, fma(c01.y, lT0, c01.x)), y1 = fma(c2C.x, iT1, fma(c01.y, lT1, c01.x));
            const double z0 = rev_eval(b, c2C.y, T0, lT0, iT0);
            const double z1 = same_g ? rev_eval(b, c2C.y, T1, lT1, iT1) : rev_eval_other(b + dblk, T1, lT1, iT1);
            const double2 m01 = ldg2(b + 7 * 64), m2f = ldg2(b + 8 * 64);
            const double cN = ldg2(b + 9 * 64).x;
            const double w0 = fma(m2f.x, iT0, fma(m01.y, lT0, m01.x)) + lM0;
            const double w1 = fma(m2f.x, iT1, fma(m01.y, lT1, m01.x)) + lM1;
            const double lp0 = w0 - y0, lp1 = w1 - y1;             // log2 Pr
            const double x0 = lp0 * cN, x1 = lp1 * cN;
            const double lF0 = m2f.y / fma(x0, x0, 1.0), lF1 = m2f.y / fma(x1, x1, 1.0);
            const double d0 = 1.0 / (1.0 + xexp2(-fabs(lp0))), d1 = 1.0 / (1.0 + xexp2(-fabs(lp1)));
            const double ym0 = fmin(w0, y0) + lF0, ym1 = fmin(w1, y1) + lF1;
            rates_of_progress(sa, ns, n_l, xexp2(ym0) * d0, xexp2(ym1) * d1, xexp2(ym0 + z0) * d0, xexp2(ym1 + z1) * d1, qdst);
          }
        }
        if (pass < p_ph) {   // PHOTO: k_f = J (the blocks hold species slots and the J row only; any interval)
          const unsigned char *b = f.blk + slot16 + XOD_IDX((size_t)f.blk_ph_off + (size_t)((ppw0 + pass * kFPass - f.fo_end) >> 2) * kFBlkPh, (size_t)f.blk_stride);
          (void)XOD_IDX((size_t)f.blk_ph_off + (size_t)((ppw0 + (p_ph - 1) * kFPass - f.fo_end) >> 2) * kFBlkPh, (size_t)f.blk_stride);
#pragma unroll 1
          for (; pass < p_ph; ++pass, b += kPhStep, qdst += kFPass * kFW) {
            const int4 sa = __ldg(reinterpret_cast<const int4 *>(b));
            const double *jr = a.J + (size_t)XOD_IDX(sa.w, a.n_photo) * a.ld;
            rates_of_progress(sa, ns, n_l, jr[gc0], jr[gc1], 0.0, 0.0, qdst);
          }
        }
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
