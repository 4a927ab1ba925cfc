// Host stand-in for csrc/xod_cta.cuh (tests/kernel_emu only; see cuda_runtime.h beside this file):
// the CTA's dynamic shared memory is one static buffer (blocks run one after another), a cp.async
// copy completes at once, and XOD_IDX always checks (an out-of-range table index aborts the test).
#pragma once
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "cuda_runtime.h"

namespace xod {
extern unsigned char smem_raw[];
inline unsigned char *cta_dyn_smem() { return smem_raw; }
inline void cp_async16(void *smem, const void *gmem) { std::memcpy(smem, gmem, 16); }
inline void cp_async8(void *smem, const void *gmem) { std::memcpy(smem, gmem, 8); }
inline void cp_async_wait_all() {}
inline long long xod_chk(long long i, long long n, int line) {
  if (i < 0 || i >= n) {
    std::fprintf(stderr, "kernel_emu: index %lld outside [0, %lld) at kernel source line %d\n", i, n, line);
    std::abort();
  }
  return i;
}
#define XOD_IDX(i, n) ((decltype(i))::xod::xod_chk((long long)(i), (long long)(n), __LINE__))
}  // namespace xod
