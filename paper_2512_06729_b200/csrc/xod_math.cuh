// xod_math.cuh -- device math shared by the kernels: a branch-light fp64 2^y.
// Part of libxodiac (CUDA product path); the oracle uses libm's expl/powl instead.
#pragma once
#include <cuda_runtime.h>

namespace xod {

// 2^y for any double y.  Rate coefficients are assembled in the log2 domain
// (log2 k = c0 + c1 log2 T + c2/T, Eq. 7 of the paper), so a single exp2 per
// coefficient is the only transcendental on the hot path.
//   m = rint(y) via the 1.5*2^52 trick, f = y - m exactly, |f| <= 1/2
//   2^f by a degree-11 polynomial: near-minimax (Chebyshev fit, mpmath 50 digits, see
//   gen_exp2_coeffs.py beside this file); max relative error 2.0e-17 before rounding
//   scale by 2^m through the exponent field; |m| >= 1020 takes a two-step scaling that gives
//   correctly rounded subnormals and overflow to +inf (reading R5).
__device__ __forceinline__ double xexp2(double y) {
  const double kMagic = 6755399441055744.0;  // 1.5 * 2^52
  double yc = fmin(fmax(y, -1100.0), 1100.0);
  double t = yc + kMagic;
  int mi = __double2loint(t);
  double f = yc - (t - kMagic);
  double p = 4.45581790833606449e-10;
  p = fma(p, f, 7.07419429728852106e-09);
  p = fma(p, f, 1.01780570877339407e-07);
  p = fma(p, f, 1.32154325359123753e-06);
  p = fma(p, f, 1.52527338415567733e-05);
  p = fma(p, f, 1.54035304637243530e-04);
  p = fma(p, f, 1.33335581464064708e-03);
  p = fma(p, f, 9.61812910758725638e-03);
  p = fma(p, f, 5.55041086648216248e-02);
  p = fma(p, f, 2.40226506959101582e-01);
  p = fma(p, f, 6.93147180559945286e-01);
  p = fma(p, f, 1.0);
  double r;
  if (abs(mi) < 1020) {
    r = __hiloint2double(__double2hiint(p) + (mi << 20), __double2loint(p));
  } else {
    int a = mi >> 1, b = mi - a;  // |a|, |b| <= 551
    r = p * __hiloint2double((1023 + a) << 20, 0) * __hiloint2double((1023 + b) << 20, 0);
  }
  return (y != y) ? y : r;
}

}  // namespace xod
