// emu.cpp -- runs the CUDA kernel SOURCE of libxodiac on CPU threads.  TEST INFRASTRUCTURE ONLY
// (see shim/cuda_runtime.h).  Exports C functions the `-m "not gpu"` tests call through ctypes:
// the host packer builds the tables exactly as xod_network_create does, then k_fused /
// k_fused_combine / k_rate_coeffs are executed with one std::thread per CUDA thread of a block
// (blocks one after another) and a std::barrier as __syncthreads.
#include <barrier>
#include <memory>
#include <thread>
#include <vector>

#include "cuda_runtime.h"

thread_local emu_dim threadIdx, blockIdx;
emu_dim gridDim, blockDim;
static std::unique_ptr<std::barrier<>> g_barrier;
void emu_syncthreads() { g_barrier->arrive_and_wait(); }

#include "../../paper_2512_06729_b200/csrc/fused.cuh"
#include "../../paper_2512_06729_b200/csrc/rates2.cuh"

namespace xod {
alignas(16) unsigned char smem_raw[256 * 1024];  // the CTA's dynamic shared memory
}

using namespace xod;

namespace {

// every CUDA thread of every block; blocks sequentially, threads of a block concurrently
template <class Body>
void run_grid(unsigned gx, unsigned gy, unsigned block, bool needs_barrier, Body body) {
  gridDim = emu_dim{gx, gy, 1};
  blockDim = emu_dim{block, 1, 1};
  for (unsigned by = 0; by < gy; ++by)
    for (unsigned bx = 0; bx < gx; ++bx) {
      if (!needs_barrier) {
        for (unsigned t = 0; t < block; ++t) {
          threadIdx = emu_dim{t, 0, 0};
          blockIdx = emu_dim{bx, by, 0};
          body();
        }
        continue;
      }
      g_barrier = std::make_unique<std::barrier<>>((std::ptrdiff_t)block);
      std::vector<std::thread> th;
      for (unsigned t = 0; t < block; ++t)
        th.emplace_back([=] {
          threadIdx = emu_dim{t, 0, 0};
          blockIdx = emu_dim{bx, by, 0};
          body();
        });
      for (auto &x : th) x.join();
    }
}

constexpr size_t kSmemMax = 227 * 1024;
const double kLog2Kb = (double)std::log2(1.380649e-16L);

bool pack(const xod_network_desc *d, HostTables &h, FusedDev &fd) {
  std::string err;
  if (pack_network(d, h, err) != XOD_OK) return false;
  for (int chunk : {4 * kFPass, 3 * kFPass, 2 * kFPass, kFPass}) {
    pack_fused(d, h, chunk);
    if (h.f.enabled && fused_smem_bytes(h.ns, h.f.n_acc, chunk, h.f.meta_cap) <= kSmemMax) break;
    h.f.enabled = false;
  }
  if (!h.f.enabled || !check_fused(h, err)) return false;
  const FusedHost &f = h.f;
  fd = FusedDev{};
  fd.enabled = 1;
  fd.npad = f.npad, fd.arr_end = f.arr_end, fd.fo_end = f.fo_end, fd.ph_end = f.ph_end;
  fd.chunk = f.chunk, fd.nchunk = f.nchunk, fd.n_acc = f.n_acc, fd.n_bp = f.n_bp;
  fd.n_extra = (int32_t)(f.extra.size() / 2);
  fd.meta_cap = f.meta_cap;
  fd.blk_stride = f.blk_stride, fd.blk_fo_off = f.blk_fo_off, fd.blk_ph_off = f.blk_ph_off;
  fd.bp = f.bp.data(), fd.blk = f.blk.data(), fd.meta_ptr = f.meta_ptr.data();
  fd.meta = reinterpret_cast<const int4 *>(f.meta.data());
  fd.extra = f.extra.data(), fd.pp_user = f.pp_user.data();
  return true;
}

}  // namespace

extern "C" {

// dn/dt [ns][ld] by k_fused (kf == NULL: coefficients evaluated in the kernel; else read from kf, kr),
// on `grid` blocks (the persistent tile loop is exercised when grid < tiles x nsplit)
int emu_source_fused(const xod_network_desc *d, int64_t ncol, int64_t ld, const double *T, const double *P,
                     const double *J, const double *kf, const double *kr, const double *n, double *dndt, int grid,
                     int nsplit) {
  HostTables h;
  FusedDev fd;
  if (!pack(d, h, fd) || ncol <= 0) return 1;
  FusedArgs a{};
  a.ncol = ncol, a.ld = ld, a.T = T, a.P = P, a.J = J, a.n = n, a.kf = kf, a.kr = kr;
  a.ntiles = (int32_t)((ncol + kFW - 1) / kFW);
  a.nsplit = std::max(1, std::min(nsplit, (int)fd.nchunk));
  a.log2_kb = kLog2Kb;
  a.ldp = (ncol + 31) / 32 * 32;
  std::vector<double> part((size_t)a.nsplit * h.ns * a.ldp);
  a.out = a.nsplit == 1 ? dndt : part.data();
  const int ns = h.ns;
  if (kf)
    run_grid((unsigned)grid, 1, kFWarps * 32, true, [&] { k_fused<true>(fd, ns, a); });
  else
    run_grid((unsigned)grid, 1, kFWarps * 32, true, [&] { k_fused<false>(fd, ns, a); });
  if (a.nsplit > 1)
    run_grid((unsigned)((ncol + 127) / 128), (unsigned)ns, 128, false,
             [&] { k_fused_combine(ns, ncol, ld, a.ldp, a.nsplit, part.data(), dndt); });
  return 0;
}

int emu_rate_coeffs(const xod_network_desc *d, int64_t ncol, int64_t ld, const double *T, const double *P,
                    const double *J, double *kf, double *kr, int slice) {
  HostTables h;
  FusedDev fd;
  if (!pack(d, h, fd) || ncol <= 0) return 1;
  run_grid((unsigned)((ncol + 255) / 256), (unsigned)((fd.ph_end + slice - 1) / slice), 256, false,
           [&] { k_rate_coeffs(fd, ncol, ld, T, P, J, kf, kr, kLog2Kb, slice); });
  return 0;
}

}  // extern "C"
