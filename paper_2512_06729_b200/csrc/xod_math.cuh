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
// polynomial coefficients in constant memory: FP64 instructions take them as constant-bank
// operands, so no instruction is spent materialising 64-bit immediates
__constant__ double kExp2C[10] = {1.0, 0.6931471805599453, 0.2402265069581299, 0.055504108664760424,
                                  0.009618129159402558, 0.0013333558179043112, 0.00015403455852453838,
                                  1.525268684626772e-05, 1.3255224878668817e-06, 1.0203121063391729e-07};

__device__ __forceinline__ double xexp2_poly(double f) {
  double p = kExp2C[9];
#pragma unroll
  for (int k = 8; k >= 0; --k) p = fma(p, f, kExp2C[k]);
  return p;
}

// exponent-field magnitude of y: xexp2_fast is valid iff xexp2_mag(y) < kExp2FastMax (|y| < 1020)
constexpr unsigned kExp2FastMax = 0x408fe000u;
__device__ __forceinline__ unsigned xexp2_mag(double y) { return (unsigned)__double2hiint(y) & 0x7fffffffu; }

// 2^y for |y| < 1020: no range check
__device__ __forceinline__ double xexp2_fast(double y) {
  const double kMagic = 6755399441055744.0;  // 1.5 * 2^52
  const double t = y + kMagic;
  const int mi = __double2loint(t);
  const double p = xexp2_poly(y - (t - kMagic));
  return __hiloint2double(__double2hiint(p) + (mi << 20), __double2loint(p));
}

// 2^y for any y (NaN propagates; overflow to +inf, gradual underflow to 0)
__device__ __noinline__ double xexp2_slow(double y) {
  const double kMagic = 6755399441055744.0;
  if (y != y) return y;
  const double yc = fmin(fmax(y, -1100.0), 1100.0);
  const double t = yc + kMagic;
  const int mi = __double2loint(t);
  const double p = xexp2_poly(yc - (t - kMagic));
  const int a = mi >> 1, b = mi - a;  // |a|, |b| <= 551
  return p * __hiloint2double((1023 + a) << 20, 0) * __hiloint2double((1023 + b) << 20, 0);
}

__device__ __forceinline__ double xexp2(double y) {
  return xexp2_mag(y) < kExp2FastMax ? xexp2_fast(y) : xexp2_slow(y);
}

}  // namespace xod
