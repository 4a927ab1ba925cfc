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
// explicit shared-memory accesses: an address is the byte offset in the one static buffer
typedef unsigned smem_addr;
#define XOD_KEEP(r) ((void)(r))
inline smem_addr smem_addr_of(const void *p) {
  const long long off = (const unsigned char *)p - smem_raw;
  if (off < 0 || off > 256 * 1024) {
    std::fprintf(stderr, "kernel_emu: smem_addr_of a pointer outside shared memory\n");
    std::abort();
  }
  return (smem_addr)off;
}
template <class T> inline T emu_lds(smem_addr a) {
  if (a % alignof(T) != 0 || (size_t)a + sizeof(T) > 256 * 1024) {
    std::fprintf(stderr, "kernel_emu: misaligned or out-of-range shared access at %u\n", a);
    std::abort();
  }
  T v;
  std::memcpy(&v, smem_raw + a, sizeof(T));
  return v;
}
inline unsigned lds_u32(smem_addr a) { return emu_lds<unsigned>(a); }
inline unsigned lds_u16(smem_addr a) { return emu_lds<unsigned short>(a); }
inline int2 lds_i2(smem_addr a) { return emu_lds<int2>(a); }
inline double2 lds_d2(smem_addr a) { return emu_lds<double2>(a); }
inline void sts_d2(smem_addr a, double2 v) {
  (void)emu_lds<double2>(a);
  std::memcpy(smem_raw + a, &v, sizeof v);
}
inline long long xod_chk(long long i, long long n, int line) {
  if (i < 0 || i >= n) {
    std::fprintf(stderr, "kernel_emu: index %lld outside [0, %lld) at kernel source line %d\n", i, n, line);
    std::abort();
  }
  return i;
}
#define XOD_IDX(i, n) ((decltype(i))::xod::xod_chk((long long)(i), (long long)(n), __LINE__))
}  // namespace xod
