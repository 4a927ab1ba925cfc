// emu.cpp -- runs the CUDA kernel SOURCE of libxodiac on CPU threads.  TEST INFRASTRUCTURE ONLY
// (see shim/cuda_runtime.h).  Exports C functions the `-m "not gpu"` tests call through ctypes:
// the host packer builds the tables exactly as xod_network_create does, then k_fused /
// k_fused_combine / k_rate_coeffs are executed with one std::thread per CUDA thread of a block
// (blocks one after another) and a std::barrier as __syncthreads.
#include <atomic>
#include <barrier>
#include <memory>
#include <thread>
#include <vector>

#include "cuda_runtime.h"

thread_local emu_dim threadIdx, blockIdx;
emu_dim gridDim, blockDim;
static std::unique_ptr<std::barrier<>> g_barrier;
void emu_syncthreads() { g_barrier->arrive_and_wait(); }
static std::atomic<int> g_or{0};
int emu_syncthreads_or(int predicate) {   // barrier with an OR reduction over the block
  if (predicate) g_or.fetch_or(1);
  g_barrier->arrive_and_wait();
  const int r = g_or.load();
  g_barrier->arrive_and_wait();
  if (threadIdx.x == 0) g_or.store(0);
  g_barrier->arrive_and_wait();
  return r;
}

#include "../../paper_2512_06729_b200/csrc/fused.cuh"
#include "../../paper_2512_06729_b200/csrc/rates2.cuh"
#include "../../paper_2512_06729_b200/csrc/jac_tiled.cuh"
#include "../../paper_2512_06729_b200/csrc/newton.cuh"
#include "../../paper_2512_06729_b200/csrc/photo.cuh"
#include "../../paper_2512_06729_b200/csrc/transport.cuh"
#include "../../paper_2512_06729_b200/csrc/pathway.cuh"
#include "../../paper_2512_06729_b200/csrc/equil.cuh"
#include "../../paper_2512_06729_b200/csrc/kernels.cuh"

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
  a.ldo = ld;
  a.nr = h.nr, a.n_photo = h.n_photo;
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
           [&] { k_rate_coeffs(fd, ncol, ld, T, P, J, kf, kr, kLog2Kb, slice, h.nr, h.n_photo); });
  return 0;
}

// ---- the multi-kernel entry points (kernels.cuh): thermo, Jacobian, and the prologue -> rates -> source
// pipeline that serves the prod/loss variants and the fallback of the fused path
static DevTables dev_tables(const HostTables &h) {
  DevTables d{};
  d.ns = h.ns, d.nr = h.nr, d.n_photo = h.n_photo;
  d.uni_begin = h.uni_begin, d.bi_begin = h.bi_begin, d.fo_begin = h.fo_begin, d.ph_begin = h.ph_begin;
  d.c0 = h.c0.data(), d.c1 = h.c1.data(), d.c2 = h.c2.data();
  d.l0 = h.l0.data(), d.l1 = h.l1.data(), d.l2 = h.l2.data(), d.fcl = h.fcl.data(), d.cN = h.cN.data();
  d.sp = h.sp.data(), d.flags = h.flags.data(), d.user = h.packed_to_user.data(), d.photo_row = h.photo_row.data();
  d.nasa = h.nasa.data(), d.nasa_l2 = h.nasa_l2.data(), d.tmid = h.tmid.data();
  d.src_rxn = h.src_rxn_packed.data(), d.src_nu = h.src_nu_f.data(), d.src_seg = h.src_seg.data();
  d.n_src_tasks = (int32_t)(h.src_seg.size() / kSrcWarpsPerCta);
  d.jac_term_ptr = h.jac_term_ptr.data(), d.jac_terms = h.jac_terms.data();
  d.nnz_jac = (int64_t)h.jac_col.size();
  return d;
}

int emu_thermo(const xod_network_desc *desc, int64_t ncol, int64_t ld, const double *T, double *cp, double *hh,
               double *ss, double *gg, int spb) {
  HostTables h;
  std::string err;
  if (pack_network(desc, h, err) != XOD_OK) return 1;
  const DevTables d = dev_tables(h);
  run_grid((unsigned)((ncol + 127) / 128), (unsigned)((h.ns + spb - 1) / spb), 128, false,
           [&] { k_thermo(d, ncol, ld, T, cp, hh, ss, gg, spb); });
  return 0;
}

int emu_jacobian(const xod_network_desc *desc, int64_t ncol, int64_t ld, const double *kf, const double *kr,
                 const double *n, double *jac, int gx) {
  HostTables h;
  std::string err;
  if (pack_network(desc, h, err) != XOD_OK) return 1;
  const DevTables d = dev_tables(h);
  run_grid((unsigned)gx, (unsigned)((ncol + 31) / 32), 256, false, [&] { k_jacobian(d, ncol, ld, kf, kr, n, jac); });
  return 0;
}

// Jacobian values by k_jac_tiled on `grid` blocks, each tile's units split over `nsplit` work items
int emu_jacobian_tiled(const xod_network_desc *desc, int64_t ncol, int64_t ld, const double *kf, const double *kr,
                       const double *n, double *jac, int grid, int nsplit) {
  HostTables h;
  std::string err;
  if (pack_network(desc, h, err) != XOD_OK || ncol <= 0) return 1;
  for (int chunk : {4 * kFPass, 3 * kFPass, 2 * kFPass, kFPass}) {
    const int64_t fixed = ((int64_t)(h.ns + 1) + 2 * (chunk + 1)) * kFW * 8 + 2 * 12 * 1024;
    const int64_t budget = ((int64_t)kSmemMax - fixed) / (kFW * 8);
    if (budget < 1) continue;
    pack_jac_tiled(h, chunk, (int)std::min<int64_t>(budget, 0xfff0));
    if (h.jt.enabled && jac_tiled_smem_bytes(h.ns, h.jt.acc_rows, chunk, h.jt.meta_cap) <= kSmemMax) break;
    h.jt.enabled = false;
  }
  if (!h.jt.enabled || !check_jac_tiled(h, err)) return 2;
  const JacTiledHost &t = h.jt;
  JacTiledDev jd{};
  jd.enabled = 1, jd.chunk = t.chunk, jd.nchunk = t.nchunk, jd.acc_rows = t.acc_rows, jd.meta_cap = t.meta_cap;
  jd.n_flush = (int32_t)(t.flush.size() / 4);
  jd.meta_ptr = t.meta_ptr.data();
  jd.meta = reinterpret_cast<const int4 *>(t.meta.data());
  jd.slots = reinterpret_cast<const int4 *>(t.slots.data());
  jd.chunk_info = reinterpret_cast<const int4 *>(t.chunk_info.data());
  jd.flush = reinterpret_cast<const int4 *>(t.flush.data());
  JacArgs a{};
  a.ncol = ncol, a.ld = ld, a.ldo = ld, a.kf = kf, a.kr = kr, a.n = n, a.jac = jac;
  a.ntiles = (int32_t)((ncol + kFW - 1) / kFW);
  a.nsplit = std::max(1, std::min(nsplit, (int)t.n_units));
  a.nr = h.nr, a.nnz = (int64_t)h.jac_col.size();
  const int ns = h.ns;
  run_grid((unsigned)grid, 1, kFWarps * 32, true, [&] { k_jac_tiled(jd, ns, a); });
  return 0;
}

// f1: one Newton iteration of the backward-Euler step, composed as xod_newton_step composes it: k_fused<true>
// (f), k_jac_tiled (Jac), k_newton_assemble, k_lu_factor, k_lu_solve; workspace pitch ldw != ld on purpose
int emu_newton_step(const xod_network_desc *desc, int64_t ncol, int64_t ld, const double *kf, const double *kr,
                    const double *n_old, const double *dt, double *y, double *delta) {
  HostTables h;
  FusedDev fd;
  std::string err;
  if (!pack(desc, h, fd) || ncol <= 0) return 1;
  for (int chunk : {4 * kFPass, 3 * kFPass, 2 * kFPass, kFPass}) {
    const int64_t fixed = ((int64_t)(h.ns + 1) + 2 * (chunk + 1)) * kFW * 8 + 2 * 12 * 1024;
    const int64_t budget = ((int64_t)kSmemMax - fixed) / (kFW * 8);
    if (budget < 1) continue;
    pack_jac_tiled(h, chunk, (int)std::min<int64_t>(budget, 0xfff0));
    if (h.jt.enabled && jac_tiled_smem_bytes(h.ns, h.jt.acc_rows, chunk, h.jt.meta_cap) <= kSmemMax) break;
    h.jt.enabled = false;
  }
  pack_lu(h);
  if (!h.jt.enabled || !h.lu.enabled || (size_t)h.lu.block_rows * h.lu.max_row * kLuCols * 8 > kSmemMax) return 2;
  const int ns = h.ns;
  const int64_t ldw = (ncol + 31) / 32 * 32 + 32, nnzj = (int64_t)h.jac_col.size();
  std::vector<double> f((size_t)ns * ldw, NAN), rhs((size_t)ns * ldw, NAN), jac((size_t)nnzj * ldw, NAN), lu((size_t)h.lu.nnz * ldw, NAN);
  {  // f(y)
    FusedArgs a{};
    a.ncol = ncol, a.ld = ld, a.ldo = ldw, a.n = y, a.kf = kf, a.kr = kr;
    a.ntiles = (int32_t)((ncol + kFW - 1) / kFW), a.nsplit = 1, a.log2_kb = kLog2Kb, a.ldp = ldw;
    a.nr = h.nr, a.n_photo = h.n_photo, a.out = f.data();
    run_grid(2, 1, kFWarps * 32, true, [&] { k_fused<true>(fd, ns, a); });
  }
  {  // Jac(y)
    const JacTiledHost &t = h.jt;
    JacTiledDev jd{};
    jd.enabled = 1, jd.chunk = t.chunk, jd.nchunk = t.nchunk, jd.acc_rows = t.acc_rows, jd.meta_cap = t.meta_cap;
    jd.n_flush = (int32_t)(t.flush.size() / 4);
    jd.meta_ptr = t.meta_ptr.data();
    jd.meta = reinterpret_cast<const int4 *>(t.meta.data());
    jd.slots = reinterpret_cast<const int4 *>(t.slots.data());
    jd.chunk_info = reinterpret_cast<const int4 *>(t.chunk_info.data());
    jd.flush = reinterpret_cast<const int4 *>(t.flush.data());
    JacArgs a{};
    a.ncol = ncol, a.ld = ld, a.ldo = ldw, a.kf = kf, a.kr = kr, a.n = y, a.jac = jac.data();
    a.ntiles = (int32_t)((ncol + kFW - 1) / kFW), a.nsplit = 1, a.nr = h.nr, a.nnz = nnzj;
    run_grid(2, 1, kFWarps * 32, true, [&] { k_jac_tiled(jd, ns, a); });
  }
  const LuHost &u = h.lu;
  LuDev ud{};
  ud.enabled = 1, ud.n = u.n, ud.max_row = u.max_row, ud.nnz = u.nnz;
  ud.perm = u.perm.data(), ud.diag = u.diag.data(), ud.src = u.src.data(), ud.col = u.col.data();
  ud.row_ptr = u.row_ptr.data(), ud.rows = u.rows.data(), ud.pairs = u.pairs.data(), ud.tgt = u.tgt.data();
  ud.block_rows = u.block_rows, ud.n_blocks = (int32_t)u.blocks.size();
  ud.blocks = u.blocks.data(), ud.steps = u.steps.data(), ud.items = u.items.data();
  NewtonArgs a{};
  a.ncol = ncol, a.ld = ld, a.ldw = ldw, a.n_old = n_old, a.dt = dt, a.f = f.data(), a.jac = jac.data();
  a.y = y, a.delta = delta, a.lu = lu.data(), a.rhs = rhs.data(), a.nnz_jac = nnzj;
  run_grid((unsigned)((ncol + 127) / 128), 3, 128, false, [&] { k_newton_assemble(ud, a); });
  run_grid((unsigned)((ncol + kLuCols - 1) / kLuCols), 1, 32 * kLuWarps, true, [&] { k_lu_factor(ud, lu.data(), ldw, ncol); });
  run_grid((unsigned)((ncol + 127) / 128), 1, 128, false, [&] { k_lu_solve(ud, a); });
  return 0;
}

// f2: photolysis rate constants, composed as xod_photo_rates composes them: k_photo_gemm (kappa), k_photo_flux,
// k_photo_gemm (quadrature)
int emu_photo_rates(int ns, int n_photo, int n_bins, int n_abs, const int32_t *abs_species, const double *sigma_ext,
                    const double *sigma_ph, const double *dlambda, int64_t n_atm, int64_t n_layers, int64_t ld,
                    const double *n, const double *dz, const double *j0, const double *j_diff, const double *mu,
                    const double *t_f, double *J) {
  const int64_t ncol = n_atm * n_layers, ldw = (ncol + 31) / 32 * 32;
  if (ncol <= 0 || (size_t)32 * (n_layers | 1) * 8 > sizeof(smem_raw)) return 1;
  std::vector<double> F((size_t)n_bins * ldw, NAN);
  {
    GemmArgs g{};
    g.M = n_bins, g.N = ncol, g.K = n_abs, g.A = sigma_ext, g.lda = n_bins, g.B = n, g.brow = abs_species, g.ldb = ld;
    g.n_brows = ns, g.C = F.data(), g.ldc = ldw, g.scale_atm = nullptr, g.n_layers = 1;
    run_grid((unsigned)((ncol + kGemmBN - 1) / kGemmBN), (unsigned)((n_bins + kGemmBM - 1) / kGemmBM), 256, true,
             [&] { k_photo_gemm<false>(g); });
  }
  {
    FluxArgs f{};
    f.n_bins = n_bins, f.n_atm = n_atm, f.n_layers = n_layers, f.ld = ld, f.ldw = ldw;
    f.F = F.data(), f.dz = dz, f.j0 = j0, f.j_diff = j_diff, f.mu = mu, f.dlambda = dlambda;
    run_grid((unsigned)((n_bins + 31) / 32), (unsigned)n_atm, 256, true, [&] { k_photo_flux(f); });
  }
  {
    GemmArgs g{};
    g.M = n_photo, g.N = ncol, g.K = n_bins, g.A = sigma_ph, g.lda = n_bins, g.B = F.data(), g.brow = nullptr, g.ldb = ldw;
    g.n_brows = n_bins, g.C = J, g.ldc = ld, g.scale_atm = t_f, g.n_layers = n_layers;
    run_grid((unsigned)((ncol + kGemmBN - 1) / kGemmBN), (unsigned)((n_photo + kGemmBM - 1) / kGemmBM), 256, true,
             [&] { k_photo_gemm<true>(g); });
  }
  return 0;
}

// f3: transport terms by k_transport (thread = column, species blocks over blockIdx.y)
int emu_transport(int ns, int64_t n_atm, int64_t n_layers, int64_t ld, const double *n, const double *T, const double *n_gas,
                  const double *D, const double *mass, const double *alpha_T, const double *mbar, const double *grav,
                  const double *dz, double *tr, int spb) {
  TransportArgs a{};
  a.ncol = n_atm * n_layers, a.n_layers = n_layers, a.ld = ld, a.ns = ns;
  a.n = n, a.T = T, a.n_gas = n_gas, a.D = D, a.mass = mass, a.alpha_T = alpha_T, a.mbar = mbar, a.grav = grav, a.dz = dz, a.tr = tr;
  a.spb = spb;
  if (a.ncol <= 0) return 1;
  run_grid((unsigned)((a.ncol + 127) / 128), (unsigned)((ns + spb - 1) / spb), 128, false, [&] { k_transport(a); });
  return 0;
}

// f4: pathway analyser: k_path_weights, then k_pathway on `grid` blocks
int emu_pathway(const xod_network_desc *desc, int64_t ncol, int64_t ld, const double *kf, const double *kr, const double *n,
                int source, double *dist, int32_t *pred, int32_t *via, int grid) {
  HostTables h;
  std::string err;
  if (pack_network(desc, h, err) != XOD_OK || ncol <= 0) return 1;
  pack_path(desc, h);
  if (!h.path.enabled || path_smem_bytes(h.ns) > sizeof(smem_raw)) return 2;
  const DevTables d = dev_tables(h);
  PathDev pd{};
  pd.enabled = 1, pd.n_steps = h.path.n_steps, pd.n_edges = h.path.n_edges;
  pd.in_u = h.path.in_u.data(), pd.in_rd = h.path.in_rd.data(), pd.sched = h.path.sched.data();
  PathArgs a{};
  a.ncol = ncol, a.ld = ld, a.ldw = (ncol + 31) / 32 * 32, a.kf = kf, a.kr = kr, a.n = n;
  std::vector<double> w((size_t)2 * h.nr * a.ldw, NAN);
  a.w = w.data(), a.dist = dist, a.pred = pred, a.via = via, a.source = source, a.ns = h.ns, a.nr = h.nr;
  a.ntiles = (int32_t)((ncol + kFW - 1) / kFW);
  run_grid((unsigned)((ncol + 127) / 128), 3, 128, false, [&] { k_path_weights(d, a, (h.nr + 2) / 3); });
  run_grid((unsigned)grid, 1, kFWarps * 32, true, [&] { k_pathway(pd, a); });
  return 0;
}

// f4: equilibrium composition: k_equilibrium (thread = column, no barrier: threads run one after another)
int emu_equilibrium(const xod_network_desc *desc, int64_t ncol, int64_t ld, const double *T, const double *P, const double *b,
                    int max_iter, double tol, double *n, double *pi, int32_t *iters) {
  HostTables h;
  std::string err;
  if (pack_network(desc, h, err) != XOD_OK || ncol <= 0 || h.ne <= 0 || h.ne > kEqMaxElem) return 1;
  if ((size_t)equil_smem_doubles(h.ne) * kEqThreads * sizeof(double) > sizeof(smem_raw)) return 2;
  EquilDev d{};
  d.ns = h.ns, d.ne = h.ne, d.sp_ptr = h.eq_ptr.data(), d.sp_ea = h.eq_ea.data(), d.el_neg = h.eq_neg.data();
  d.nasa = h.nasa.data(), d.tmid = h.tmid.data();
  EquilArgs a{};
  a.ncol = ncol, a.ld = ld, a.T = T, a.P = P, a.b = b, a.n = n, a.pi = pi, a.iters = iters;
  a.max_iter = max_iter > 0 ? max_iter : 500, a.tol = tol > 0 ? tol : 1e-13;
  run_grid((unsigned)((ncol + kEqThreads - 1) / kEqThreads), 1, kEqThreads, false, [&] { k_equilibrium(d, a); });
  return 0;
}

// (T, P, J, n) -> dn/dt [, P, L] through k_prologue + k_rates + k_source; with kf_in/kr_in given, through
// k_rates_from_k + k_source instead (xod_source with prod/loss).  One chunk holds all columns.
int emu_source_pipeline(const xod_network_desc *desc, int64_t ncol, int64_t ld, const double *T, const double *P,
                        const double *J, const double *kf_in, const double *kr_in, const double *n, double *dndt,
                        double *prod, double *loss, int rw) {
  HostTables h;
  std::string err;
  if (pack_network(desc, h, err) != XOD_OK) return 1;
  const DevTables d = dev_tables(h);
  const int64_t ldw = (ncol + 31) / 32 * 32, ncg = ldw / 32;
  const bool pl = prod != nullptr;
  std::vector<double> buf((size_t)(3 + h.ns + 2 * (size_t)h.nr) * ldw);
  ChunkScratch w{};
  w.ldw = ldw;
  w.l2T = buf.data(), w.invT = w.l2T + ldw, w.lM = w.invT + ldw, w.u = w.lM + ldw;
  w.q = w.u + (size_t)h.ns * ldw, w.qr = w.q + (size_t)h.nr * ldw;
  const int64_t nslices = (h.nr + rw - 1) / rw, ntasks = nslices * ncg;
  const unsigned blocks = (unsigned)((ntasks + 3) / 4);
  if (!kf_in) {
    run_grid((unsigned)ncg, 2, 256, false, [&] { k_prologue(d, ncol, 0, T, P, w, kLog2Kb); });
    if (pl)
      run_grid(blocks, 1, 128, false, [&] { k_rates<MODE_QSEP>(d, ncol, 0, ld, w, J, n, nullptr, nullptr, rw, (int)ncg, ntasks); });
    else
      run_grid(blocks, 1, 128, false, [&] { k_rates<MODE_QNET>(d, ncol, 0, ld, w, J, n, nullptr, nullptr, rw, (int)ncg, ntasks); });
  } else if (pl) {
    run_grid(blocks, 1, 128, false, [&] { k_rates_from_k<MODE_QSEP>(d, ncol, 0, ld, w, kf_in, kr_in, n, rw, (int)ncg, ntasks); });
  } else {
    run_grid(blocks, 1, 128, false, [&] { k_rates_from_k<MODE_QNET>(d, ncol, 0, ld, w, kf_in, kr_in, n, rw, (int)ncg, ntasks); });
  }
  if (pl)
    run_grid((unsigned)d.n_src_tasks, (unsigned)ncg, 256, true, [&] { k_source<true>(d, ncol, 0, ld, w, dndt, prod, loss); });
  else
    run_grid((unsigned)d.n_src_tasks, (unsigned)ncg, 256, true, [&] { k_source<false>(d, ncol, 0, ld, w, dndt, prod, loss); });
  return 0;
}

// k_f, k_r in USER order through k_prologue + k_rates<MODE_K> (the fallback of xod_rate_coeffs)
int emu_rate_coeffs_pipeline(const xod_network_desc *desc, int64_t ncol, int64_t ld, const double *T, const double *P,
                             const double *J, double *kf, double *kr, int rw) {
  HostTables h;
  std::string err;
  if (pack_network(desc, h, err) != XOD_OK) return 1;
  const DevTables d = dev_tables(h);
  const int64_t ldw = (ncol + 31) / 32 * 32, ncg = ldw / 32;
  std::vector<double> buf((size_t)(3 + h.ns) * ldw);
  ChunkScratch w{};
  w.ldw = ldw;
  w.l2T = buf.data(), w.invT = w.l2T + ldw, w.lM = w.invT + ldw, w.u = w.lM + ldw;
  const int64_t ntasks = (int64_t)((h.nr + rw - 1) / rw) * ncg;
  run_grid((unsigned)ncg, 1, 256, false, [&] { k_prologue(d, ncol, 0, T, P, w, kLog2Kb); });
  run_grid((unsigned)((ntasks + 3) / 4), 1, 128, false,
           [&] { k_rates<MODE_K>(d, ncol, 0, ld, w, J, nullptr, kf, kr, rw, (int)ncg, ntasks); });
  return 0;
}

}  // extern "C"
