// rates2.cuh -- k_rate_coeffs: xod_rate_coeffs (a1, a3-a6) from the per-interval parameter blocks
// of pack_fused.cpp: no G/RT tile, no workspace, one kernel.  thread = column; a CTA covers 256
// columns x a slice of padded reactions (sized by the caller so the grid fills the chip); reaction parameters are warp-uniform 16-byte loads
// (lanes of one thermo interval read the same address); every store is a coalesced 256-byte row
// segment of k_f / k_r in USER reaction order.  Bound: HBM writes, 16 B per evaluation.
//   UNI/BI   k_f = 2^(c0 + c1 log2 T + c2/T)                                       (Eq. 7)
//            k_r = 2^(C0 + C1 log2 T + C2/T - T (D2 + T (D3 + T (D4 + T D5))))     (Eq. 15)
//   FALLOFF  Eq. 10-12 with Troe F (reading F1)
//   PHOTO    k_f = J, k_r = 0
#pragma once
#include <cuda_runtime.h>

#include "xod_internal.h"
#include "xod_math.cuh"
#include <xod_cta.cuh>

namespace xod {


__global__ void __launch_bounds__(256) k_rate_coeffs(FusedDev f, int64_t ncol, int64_t ld, const double *__restrict__ T,
                                                     const double *__restrict__ P, const double *__restrict__ J,
                                                     double *__restrict__ kf, double *__restrict__ kr, double log2_kb, int slice,
                                                     int nr, int n_photo /* rows of kf/kr and of J: bounds of the -DXOD_CHECK build */) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c - (threadIdx.x & 31) >= ncol) return;  // whole warp past the end
  const bool valid = c < ncol;
  const int64_t gc = valid ? c : ncol - 1;
  const double Tc = T[gc];
  const double l2T = log2(Tc), iT = 1.0 / Tc;
  const double lM = log2(P[gc]) - log2_kb - l2T;  // log2 [M], [M] = P/(k_B T)
  int g = 0;
  for (int k = 0; k < f.n_bp; ++k) g += __ldg(f.bp + k) < Tc;
  const unsigned char *blkg = f.blk + (size_t)XOD_IDX(g, f.n_bp + 1) * f.blk_stride;
  // The slice [p0, p1) is made of whole parameter blocks (4 reactions; slice and the segment ends are multiples
  // of 4), so it is three runs of blocks, UNI/BI | FALLOFF | PHOTO, each a loop whose block pointer advances by a
  // constant and whose four reaction slots sit at immediate offsets.
  const int p0 = blockIdx.y * slice, p1 = min(p0 + slice, f.ph_end);
  auto store = [&](int user, double vf, double vr) {
    if (valid && user >= 0) {  // user < 0: padding slot
      const size_t row = (size_t)XOD_IDX(user, nr);
      if (kf) kf[row * ld + c] = vf;
      if (kr) kr[row * ld + c] = vr;
    }
  };
  // log2 k_f (or log2 k_inf) and the reverse exponent of the reaction at b (its 16-byte column of the block)
  auto exponents = [&](const unsigned char *b, double &y, double &z) {
    const double2 c01 = __ldg(reinterpret_cast<const double2 *>(b + 2 * 64));
    const double2 c2C = __ldg(reinterpret_cast<const double2 *>(b + 3 * 64));
    const double2 c12 = __ldg(reinterpret_cast<const double2 *>(b + 4 * 64));
    const double2 d23 = __ldg(reinterpret_cast<const double2 *>(b + 5 * 64));
    const double2 d45 = __ldg(reinterpret_cast<const double2 *>(b + 6 * 64));
    y = fma(c2C.x, iT, fma(c01.y, l2T, c01.x));
    const double poly = fma(Tc, fma(Tc, fma(Tc, d45.y, d45.x), d23.y), d23.x);
    z = fma(c12.y, iT, fma(c12.x, l2T, fma(-Tc, poly, c2C.y)));
  };
  {  // UNI, BI
    const int q0 = min(p0, f.arr_end), q1 = min(p1, f.arr_end);
    const unsigned char *b = blkg + (size_t)(q0 >> 2) * kFBlkArr;
    if (q1 > q0) (void)XOD_IDX((size_t)((q1 - 1) >> 2) * kFBlkArr, (size_t)f.blk_stride);
#pragma unroll 1
    for (int pp = q0; pp < q1; pp += 4, b += kFBlkArr) {
      const int4 users = __ldg(reinterpret_cast<const int4 *>(f.pp_user + pp));
      const int4 flags = make_int4(__ldg(reinterpret_cast<const int *>(b + 64 + 12)), __ldg(reinterpret_cast<const int *>(b + 64 + 28)),
                                   __ldg(reinterpret_cast<const int *>(b + 64 + 44)), __ldg(reinterpret_cast<const int *>(b + 64 + 60)));
#pragma unroll
      for (int sl = 0; sl < 4; ++sl) {
        double y, z;
        exponents(b + 16 * sl, y, z);
        const int fl = sl == 0 ? flags.x : sl == 1 ? flags.y : sl == 2 ? flags.z : flags.w;
        const int user = sl == 0 ? users.x : sl == 1 ? users.y : sl == 2 ? users.z : users.w;
        store(user, xexp2(y), (fl & 1) ? xexp2(z) : 0.0);   // irreversible: k_r = 0 (the blocks hold z = 0)
      }
    }
  }
  {  // FALLOFF
    const int q0 = min(max(p0, f.arr_end), f.fo_end), q1 = min(max(p1, f.arr_end), f.fo_end);
    const unsigned char *b = blkg + (size_t)f.blk_fo_off + (size_t)((q0 - f.arr_end) >> 2) * kFBlkFo;
    if (q1 > q0) (void)XOD_IDX((size_t)f.blk_fo_off + (size_t)((q1 - 1 - f.arr_end) >> 2) * kFBlkFo, (size_t)f.blk_stride);
#pragma unroll 1
    for (int pp = q0; pp < q1; pp += 4, b += kFBlkFo) {
      const int4 users = __ldg(reinterpret_cast<const int4 *>(f.pp_user + pp));
#pragma unroll 2
      for (int sl = 0; sl < 4; ++sl) {
        const unsigned char *bs = b + 16 * sl;
        double y, z;
        exponents(bs, y, z);
        const bool rev = __ldg(reinterpret_cast<const int *>(bs + 64) + 3) & 1;
        const double2 m01 = __ldg(reinterpret_cast<const double2 *>(bs + 7 * 64));
        const double2 m2f = __ldg(reinterpret_cast<const double2 *>(bs + 8 * 64));
        const double cN = __ldg(reinterpret_cast<const double *>(bs + 9 * 64));
        const double w = fma(m2f.x, iT, fma(m01.y, l2T, m01.x)) + lM;
        const double lp = w - y, x = lp * cN;  // log2 Pr
        const double lF = m2f.y / fma(x, x, 1.0);
        const double den = 1.0 / (1.0 + xexp2(-fabs(lp)));
        const double ym = fmin(w, y) + lF;
        const int user = sl == 0 ? users.x : sl == 1 ? users.y : sl == 2 ? users.z : users.w;
        store(user, xexp2(ym) * den, rev ? xexp2(ym + z) * den : 0.0);
      }
    }
  }
  {  // PHOTO: k_f = J, k_r = 0
    const int q0 = min(max(p0, f.fo_end), f.ph_end), q1 = min(max(p1, f.fo_end), f.ph_end);
    const unsigned char *b = blkg + (size_t)f.blk_ph_off + (size_t)((q0 - f.fo_end) >> 2) * kFBlkPh;
    if (q1 > q0) (void)XOD_IDX((size_t)f.blk_ph_off + (size_t)((q1 - 1 - f.fo_end) >> 2) * kFBlkPh, (size_t)f.blk_stride);
#pragma unroll 1
    for (int pp = q0; pp < q1; pp += 4, b += kFBlkPh) {
      const int4 users = __ldg(reinterpret_cast<const int4 *>(f.pp_user + pp));
#pragma unroll
      for (int sl = 0; sl < 4; ++sl) {
        const int jrow = XOD_IDX(__ldg(reinterpret_cast<const int *>(b + 16 * sl) + 3), n_photo);
        const int user = sl == 0 ? users.x : sl == 1 ? users.y : sl == 2 ? users.z : users.w;
        store(user, J[(size_t)jrow * ld + gc], 0.0);
      }
    }
  }
}

}  // namespace xod
