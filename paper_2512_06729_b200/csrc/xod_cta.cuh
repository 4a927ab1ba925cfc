// xod_cta.cuh -- CTA-level primitives of the libxodiac kernels (sm_100a): the dynamic shared
// memory base, cp.async copies, and the opt-in index checks of the -DXOD_CHECK build.
// Included as <xod_cta.cuh> (the build passes -I csrc) so that tests/kernel_emu, which compiles
// the kernel text as host C++, can put its own header of the same name first on the include path;
// the product sources themselves carry no test branches.
#pragma once
#include <cuda_runtime.h>

namespace xod {

__device__ __forceinline__ unsigned char *cta_dyn_smem() {
  extern __shared__ __align__(16) unsigned char xod_dyn_smem[];
  return xod_dyn_smem;
}
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async8(void *smem, const void *gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// ---- explicit shared-memory accesses by 32-bit address in the CTA's shared window.  The scheduled row
// reduction (sched.cuh) lives entirely in shared memory; with plain pointers the compiler rebuilt generic
// addresses (window base, kernel parameters) inside its inner loops.  ld/st.shared on an address register
// leaves it nothing to rematerialise.
typedef unsigned smem_addr;
// an opaque "mov r, r": the value now comes out of an instruction the compiler cannot recompute elsewhere, so a
// loop invariant stays in its register instead of being rebuilt from the thread index and kernel parameters
#define XOD_KEEP(r) asm volatile("mov.b32 %0, %0;\n" : "+r"(r))
__device__ __forceinline__ smem_addr smem_addr_of(const void *p) { return (smem_addr)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned lds_u32(smem_addr a) {
  unsigned v;
  asm volatile("ld.shared.u32 %0, [%1];\n" : "=r"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ unsigned lds_u16(smem_addr a) {
  unsigned short v;
  asm volatile("ld.shared.u16 %0, [%1];\n" : "=h"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ int2 lds_i2(smem_addr a) {
  int2 v;
  asm volatile("ld.shared.v2.s32 {%0, %1}, [%2];\n" : "=r"(v.x), "=r"(v.y) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ double2 lds_d2(smem_addr a) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void sts_d2(smem_addr a, double2 v) {
  asm volatile("st.shared.v2.f64 [%0], {%1, %2};\n" ::"r"(a), "d"(v.x), "d"(v.y) : "memory");
}

// ---- XOD_IDX(i, n): a table-derived index i that must lie in [0, n).
// Default build: the identity (no code).  -DXOD_CHECK build (debugging only, `XOD_CHECK=1 python -m
// paper_2512_06729_b200.build`): an out-of-range index records the source line in a device flag
// and is clamped to 0, so a bad table shows up as XOD_ERR_CUDA from xod_check_status() instead of
// faulting the GPU.
#ifdef XOD_CHECK
__device__ int g_xod_check_line = 0;
__device__ __forceinline__ long long xod_chk(long long i, long long n, int line) {
  if (i < 0 || i >= n) {
    g_xod_check_line = line;
    return 0;
  }
  return i;
}
#define XOD_IDX(i, n) ((decltype(i))::xod::xod_chk((long long)(i), (long long)(n), __LINE__))
#else
#define XOD_IDX(i, n) (i)
#endif

}  // namespace xod
