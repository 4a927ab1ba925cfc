// Host shim for compiling the CUDA kernel SOURCE of libxodiac as plain C++ (tests/kernel_emu): TEST
// INFRASTRUCTURE ONLY.  It lets `-m "not gpu"` tests execute the very kernel text (indexing,
// schedules, table decoding, arithmetic) on CPU threads, one std::thread per CUDA thread with a
// std::barrier as __syncthreads.  Nothing here is part of the product; the library is always
// built by nvcc from the same sources without this directory on its include path.
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>

#define __global__
#define __device__
#define __host__
#define __forceinline__ inline
#define __noinline__
#define __constant__
#define __shared__ static   /* blocks run one after another, so one copy per kernel is the CTA's */
#define __launch_bounds__(...)
#define __align__(n) __attribute__((aligned(n)))

struct alignas(8) int2 { int x, y; };
struct alignas(16) int4 { int x, y, z, w; };
struct uint2 { unsigned x, y; };
struct alignas(16) double2 { double x, y; };
struct emu_dim { unsigned x = 1, y = 1, z = 1; };
inline double2 make_double2(double x, double y) { return double2{x, y}; }
inline int4 make_int4(int x, int y, int z, int w) { return int4{x, y, z, w}; }

extern thread_local emu_dim threadIdx, blockIdx;
extern emu_dim gridDim, blockDim;
void emu_syncthreads();
int emu_syncthreads_or(int predicate);
#define __syncthreads() emu_syncthreads()
#define __syncthreads_or(p) emu_syncthreads_or((p) ? 1 : 0)
#define __syncwarp()

template <class T> inline T __ldg(const T *p) { return *p; }
inline double __hiloint2double(int hi, int lo) {
  const uint64_t b = ((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo;
  double d;
  std::memcpy(&d, &b, 8);
  return d;
}
inline int __double2hiint(double d) { uint64_t b; std::memcpy(&b, &d, 8); return (int)(b >> 32); }
inline int __double2loint(double d) { uint64_t b; std::memcpy(&b, &d, 8); return (int)(uint32_t)b; }
inline double __longlong_as_double(long long v) { double d; std::memcpy(&d, &v, 8); return d; }
inline float __int_as_float(int i) { float f; std::memcpy(&f, &i, 4); return f; }
inline size_t __cvta_generic_to_shared(const void *p) { return (size_t)p; }

// CUDA's overloaded min/max for the argument mixes the kernels use
inline int min(int a, int b) { return a < b ? a : b; }
inline int max(int a, int b) { return a > b ? a : b; }
inline unsigned max(unsigned a, unsigned b) { return a > b ? a : b; }
inline long min(long a, long b) { return a < b ? a : b; }
inline long max(long a, long b) { return a > b ? a : b; }
inline long long min(long long a, long long b) { return a < b ? a : b; }
inline long long max(long long a, long long b) { return a > b ? a : b; }
using std::exp; using std::fabs; using std::fma; using std::fmax; using std::fmin; using std::log; using std::log2;
