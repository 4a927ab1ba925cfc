// xod_math.cuh -- device math shared by the kernels: a branch-light fp64 2^y.
// Part of libxodiac (CUDA product path); the oracle uses libm's expl/powl instead.
#pragma once
#include <cuda_runtime.h>

namespace xod {

// 2^y for any double y.  Rate coefficients are assembled in the log2 domain
// (log2 k = c0 + c1 log2 T + c2/T, Eq. 7 of the paper), so a single exp2 per
// coefficient is the only transcendental on the hot path.
//   fast path, |y| < 1020 (decided on the exponent field with integer compares, so NaN and
//   infinities leave it too): m = rint(y) via the 1.5*2^52 trick, f = y - m exactly,
//   |f| <= 1/2; 2^f by a degree-9 polynomial (gen_exp2_coeffs.py beside this file: maximum
//   relative error 3.7e-14, against the 1e-12 tolerance of k_f, k_r); scale by 2^m through the
//   exponent field.  12 FP64-pipe instructions (3 DADD + 9 DFMA).
//   slow path: clamp, then a two-step scaling that gives correctly scaled subnormals and
//   overflow to +inf (reading R5); NaN propagates.
__device__ __forceinline__ double xexp2_poly(double f) {
  double p = 1.0203121063391729e-07;
  p = fma(p, f, 1.3255224878668817e-06);
  p = fma(p, f, 1.525268684626772e-05);
  p = fma(p, f, 0.00015403455852453838);
  p = fma(p, f, 0.0013333558179043112);
  p = fma(p, f, 0.009618129159402558);
  p = fma(p, f, 0.055504108664760424);
  p = fma(p, f, 0.2402265069581299);
  p = fma(p, f, 0.6931471805599453);
  p = fma(p, f, 1.0);
  return p;
}

__device__ __forceinline__ double xexp2(double y) {
  const double kMagic = 6755399441055744.0;  // 1.5 * 2^52
  const unsigned ahi = (unsigned)__double2hiint(y) & 0x7fffffffu;
  if (ahi < 0x408fe000u) {  // |y| < 1020
    const double t = y + kMagic;
    const int mi = __double2loint(t);
    const double p = xexp2_poly(y - (t - kMagic));
    return __hiloint2double(__double2hiint(p) + (mi << 20), __double2loint(p));
  }
  if (y != y) return y;
  const double yc = fmin(fmax(y, -1100.0), 1100.0);
  const double t = yc + kMagic;
  const int mi = __double2loint(t);
  const double p = xexp2_poly(yc - (t - kMagic));
  const int a = mi >> 1, b = mi - a;  // |a|, |b| <= 551
  return p * __hiloint2double((1023 + a) << 20, 0) * __hiloint2double((1023 + b) << 20, 0);
}

}  // namespace xod
