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
