// api.cu -- the C ABI of include/xodiac.h: argument checks, workspace carving, kernel launches
// on the caller's stream.  No host synchronisation in any compute call except *_host.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "fused.cuh"
#include "jac_tiled.cuh"
#include "newton.cuh"
#include "photo.cuh"
#include "transport.cuh"
#include "pathway.cuh"
#include "equil.cuh"
#include "rates2.cuh"
#include "kernels.cuh"

using namespace xod;

namespace {

thread_local std::string g_err;

xod_status fail(xod_status s, const std::string &m) {
  g_err = m;
  return s;
}
xod_status cuda_fail(cudaError_t e, const char *where) {
  g_err = std::string(where) + ": " + cudaGetErrorString(e);
  return XOD_ERR_CUDA;
}
#define XOD_CUDA(call)                                       \
  do {                                                       \
    cudaError_t e_ = (call);                                 \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call);      \
  } while (0)

inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

std::atomic<int64_t> g_launches{0};  // kernels launched by this library in this process

// Counts the launch and, when timing is on, brackets it with a CUDA event pair on the stream.
struct Timed {
  TimingState *t = nullptr;
  cudaStream_t s;
  size_t pair = 0;
  Timed(const xod_network *net, int kid, cudaStream_t stream) : s(stream) {
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (!net->timing.on) return;
    t = &net->timing;
    while (t->pool.size() < t->used + 2) {
      cudaEvent_t e = nullptr;
      if (cudaEventCreate(&e) != cudaSuccess) { t = nullptr; return; }
      t->pool.push_back(e);
    }
    pair = t->used;
    t->used += 2;
    t->kid.push_back(kid);
    cudaEventRecord(static_cast<cudaEvent_t>(t->pool[pair]), s);
  }
  ~Timed() {
    if (t) cudaEventRecord(static_cast<cudaEvent_t>(t->pool[pair + 1]), s);
  }
};

template <class T>
xod_status upload(xod_network *net, const std::vector<T> &v, const T **dst) {
  void *p = nullptr;
  size_t bytes = std::max<size_t>(v.size() * sizeof(T), 16);
  XOD_CUDA(cudaMalloc(&p, bytes));
  net->dev_allocs.push_back(p);
  if (!v.empty()) XOD_CUDA(cudaMemcpy(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
  *dst = static_cast<const T *>(p);
  return XOD_OK;
}

const double kLog2Kb = (double)std::log2(1.380649e-16L);
constexpr size_t kFusedSmemMax = 227 * 1024;  // shared memory one CTA may opt into on sm_100

constexpr int64_t kDefaultChunk = 1024;  // columns per pipeline chunk: q chunk = nr*1024*8 B stays in L2

int64_t chunk_cols(const xod_network *net, int64_t ncol) {
  int64_t c = net->chunk_cols > 0 ? net->chunk_cols : kDefaultChunk;
  c = round_up(c, 32);
  return std::min<int64_t>(c, round_up(std::max<int64_t>(ncol, 1), 32));
}

// carve the workspace: [l2T | invT | lM | u (ns rows) | q (nr rows) | qr (nr rows, optional)]
size_t scratch_bytes(const xod_network *net, int64_t ldw, bool need_u, bool need_q, bool pl) {
  size_t rows = 0;
  if (need_u) rows += 3 + (size_t)net->h.ns;
  if (need_q) rows += (size_t)net->h.nr * (pl ? 2 : 1);
  return rows * (size_t)ldw * sizeof(double) + 256;
}
ChunkScratch carve(const xod_network *net, void *ws, int64_t ldw, bool need_u, bool need_q, bool pl) {
  ChunkScratch s{};
  uintptr_t a = (reinterpret_cast<uintptr_t>(ws) + 255) & ~uintptr_t(255);
  double *p = reinterpret_cast<double *>(a);
  s.ldw = ldw;
  if (need_u) {
    s.l2T = p, p += ldw;
    s.invT = p, p += ldw;
    s.lM = p, p += ldw;
    s.u = p, p += (size_t)net->h.ns * ldw;
  }
  if (need_q) {
    s.q = p, p += (size_t)net->h.nr * ldw;
    if (pl) s.qr = p;
  }
  return s;
}

// Argument checks common to the compute calls.  The compute calls only enqueue kernels on the
// caller's stream; they never change the calling thread's current device (a mismatch is an error,
// not a silent switch: include/xodiac.h, "Streams") and they are legal inside a CUDA graph capture
// (cudaGetDevice is a thread-local read, not a stream operation).
xod_status check_common(const xod_network *net, int64_t ncol, int64_t ld) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  if (ncol < 0) return fail(XOD_ERR_INVALID_ARG, "ncol < 0");
  if (ld < ncol) return fail(XOD_ERR_INVALID_ARG, "ld < ncol");
  if (net->device < 0) return fail(XOD_ERR_CUDA, "network was created without a CUDA device");
  int cur = -1;
  XOD_CUDA(cudaGetDevice(&cur));
  if (cur != net->device) return fail(XOD_ERR_CUDA, "the calling thread's current CUDA device is not the network's device");
  return XOD_OK;
}

// Makes `device` current for the lifetime of the guard and restores the caller's device on every
// exit path (create, the *_host call and the probe allocate or synchronise, so they need it).
struct DeviceGuard {
  int prev = -1;
  cudaError_t err = cudaSuccess;
  explicit DeviceGuard(int device) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
  }
  ~DeviceGuard() {
    int cur = -1;
    if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
  }
};

// reactions per warp task: aim at ~2 resident waves of warps over the whole chip
int pick_rw(const xod_network *net, int nr, int64_t ncg) {
  const int64_t target = (int64_t)net->sm_count * 32 * 2;
  int64_t rw = ((int64_t)nr * ncg + target - 1) / target;
  return (int)std::min<int64_t>(std::max<int64_t>(rw, 8), 128);
}

}  // namespace

extern "C" {

const char *xod_last_error(void) { return g_err.c_str(); }

xod_status xod_network_create(const xod_network_desc *desc, int cuda_device, xod_network **out) {
  if (!out) return fail(XOD_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  xod_network *net = new (std::nothrow) xod_network;
  if (!net) return fail(XOD_ERR_ALLOC, "out of host memory");
  std::string err;
  xod_status st;
  try {
    st = pack_network(desc, net->h, err);
  } catch (const std::bad_alloc &) {
    delete net;
    return fail(XOD_ERR_ALLOC, "out of host memory while packing");
  }
  if (st != XOD_OK) {
    delete net;
    return fail(st, err);
  }
  net->device = cuda_device;
  // tables of the single-kernel fused path: the largest chunk whose shared memory fits one CTA
  try {
    for (int chunk : {4 * kFPass, 3 * kFPass, 2 * kFPass, kFPass}) {
      pack_fused(desc, net->h, chunk);
      if (net->h.f.enabled && fused_smem_bytes(net->h.ns, net->h.f.n_acc, chunk, net->h.f.meta_cap) <= kFusedSmemMax) break;
      net->h.f.enabled = false;
    }
    // tables of the tiled Jacobian kernel: the largest chunk whose shared memory fits one CTA
    for (int chunk : {4 * kFPass, 3 * kFPass, 2 * kFPass, kFPass}) {
      const int64_t fixed = ((int64_t)(net->h.ns + 1) + 2 * (chunk + 1)) * kFW * 8 + 2 * 12 * 1024;  // schedules: guess, checked below
      const int64_t budget = ((int64_t)kFusedSmemMax - fixed) / (kFW * 8);
      if (budget < 1) continue;
      pack_jac_tiled(net->h, chunk, (int)std::min<int64_t>(budget, 0xfff0));
      if (net->h.jt.enabled && jac_tiled_smem_bytes(net->h.ns, net->h.jt.acc_rows, chunk, net->h.jt.meta_cap) <= kFusedSmemMax) break;
      net->h.jt.enabled = false;
    }
    pack_path(desc, net->h);
    if (net->h.path.enabled && path_smem_bytes(net->h.ns) > kFusedSmemMax) net->h.path.enabled = false;
    if (desc->flags & XOD_FLAG_BUILD_LU) {
      pack_lu(net->h);
      if (!net->h.lu.enabled) {
        delete net;
        return fail(XOD_ERR_INVALID_ARG, "XOD_FLAG_BUILD_LU: the LU tables do not fit (too many species or too much fill)");
      }
    }
  } catch (const std::bad_alloc &) {
    delete net;
    return fail(XOD_ERR_ALLOC, "out of host memory while packing");
  }
  if (cuda_device >= 0) {
    DeviceGuard guard(cuda_device);
    if (guard.err != cudaSuccess) {
      delete net;
      return cuda_fail(guard.err, "cudaSetDevice");
    }
    HostTables &h = net->h;
    DevTables &d = net->d;
    d.ns = h.ns, d.nr = h.nr, d.n_photo = h.n_photo;
    d.uni_begin = h.uni_begin, d.bi_begin = h.bi_begin, d.fo_begin = h.fo_begin, d.ph_begin = h.ph_begin;
    d.n_src_tasks = (int32_t)(h.src_seg.size() / kSrcWarpsPerCta);
    d.nnz_jac = (int64_t)h.jac_col.size();
    st = XOD_OK;
#define UP(vec, field) if (st == XOD_OK) st = upload(net, h.vec, &d.field)
    UP(c0, c0); UP(c1, c1); UP(c2, c2);
    UP(l0, l0); UP(l1, l1); UP(l2, l2); UP(fcl, fcl); UP(cN, cN);
    UP(sp, sp); UP(flags, flags); UP(packed_to_user, user); UP(photo_row, photo_row);
    UP(nasa, nasa); UP(nasa_l2, nasa_l2); UP(tmid, tmid);
    UP(src_rxn_packed, src_rxn); UP(src_nu_f, src_nu); UP(src_seg, src_seg);
    UP(jac_term_ptr, jac_term_ptr); UP(jac_terms, jac_terms);
    if (h.f.enabled) {
      FusedHost &f = h.f;
      FusedDev &fd = net->fd;
      fd.enabled = 1;
      fd.npad = f.npad, fd.arr_end = f.arr_end, fd.fo_end = f.fo_end, fd.ph_end = f.ph_end;
      fd.chunk = f.chunk, fd.nchunk = f.nchunk, fd.n_acc = f.n_acc, fd.n_bp = f.n_bp;
      fd.n_extra = (int32_t)(f.extra.size() / 2);
      fd.meta_cap = f.meta_cap;
      fd.blk_stride = f.blk_stride, fd.blk_fo_off = f.blk_fo_off, fd.blk_ph_off = f.blk_ph_off;
#define UPF(vec, field) if (st == XOD_OK) st = upload(net, f.vec, &fd.field)
      UPF(bp, bp); UPF(blk, blk); UPF(meta_ptr, meta_ptr); UPF(extra, extra); UPF(pp_user, pp_user);
      if (st == XOD_OK) {
        const int32_t *m = nullptr;
        st = upload(net, f.meta, &m);
        fd.meta = reinterpret_cast<const int4 *>(m);
      }
#undef UPF
      if (st == XOD_OK) {
        // the attribute is per function, not per network: always opt into the device maximum
        cudaError_t ce = cudaFuncSetAttribute(k_fused<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              (int)kFusedSmemMax);
        if (ce == cudaSuccess)
          ce = cudaFuncSetAttribute(k_fused<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmemMax);
        if (ce != cudaSuccess) st = cuda_fail(ce, "cudaFuncSetAttribute(k_fused)");
      }
    }
    {
      int smc = 0;
      if (cudaDeviceGetAttribute(&smc, cudaDevAttrMultiProcessorCount, cuda_device) == cudaSuccess && smc > 0)
        net->sm_count = smc;
    }
    if (h.jt.enabled) {
      JacTiledHost &t = h.jt;
      JacTiledDev &jd = net->jd;
      jd.enabled = 1;
      jd.chunk = t.chunk, jd.nchunk = t.nchunk, jd.acc_rows = t.acc_rows, jd.meta_cap = t.meta_cap;
      jd.n_flush = (int32_t)(t.flush.size() / 4);
      const int32_t *p4 = nullptr;
      if (st == XOD_OK) st = upload(net, t.meta_ptr, &jd.meta_ptr);
      if (st == XOD_OK) st = upload(net, t.meta, &p4), jd.meta = reinterpret_cast<const int4 *>(p4);
      if (st == XOD_OK) st = upload(net, t.slots, &p4), jd.slots = reinterpret_cast<const int4 *>(p4);
      if (st == XOD_OK) st = upload(net, t.chunk_info, &p4), jd.chunk_info = reinterpret_cast<const int4 *>(p4);
      if (st == XOD_OK) st = upload(net, t.flush, &p4), jd.flush = reinterpret_cast<const int4 *>(p4);
      if (st == XOD_OK) {
        cudaError_t ce = cudaFuncSetAttribute(k_jac_tiled, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmemMax);
        if (ce != cudaSuccess) st = cuda_fail(ce, "cudaFuncSetAttribute(k_jac_tiled)");
      }
    }
    if (h.path.enabled) {
      PathHost &ph = h.path;
      PathDev &pd = net->pd;
      pd.enabled = 1, pd.n_steps = ph.n_steps, pd.n_edges = ph.n_edges;
      if (st == XOD_OK) st = upload(net, ph.in_u, &pd.in_u);
      if (st == XOD_OK) st = upload(net, ph.in_rd, &pd.in_rd);
      if (st == XOD_OK) st = upload(net, ph.sched, &pd.sched);
      if (st == XOD_OK) {
        cudaError_t ce = cudaFuncSetAttribute(k_pathway, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmemMax);
        if (ce != cudaSuccess) st = cuda_fail(ce, "cudaFuncSetAttribute(k_pathway)");
      }
    }
    if (h.ne > 0 && h.ne <= kEqMaxElem) {   // f4: composition lists of xod_equilibrium
      EquilDev &ed = net->ed;
      ed.ns = h.ns, ed.ne = h.ne;
      if (st == XOD_OK) st = upload(net, h.eq_ptr, &ed.sp_ptr);
      if (st == XOD_OK) st = upload(net, h.eq_ea, &ed.sp_ea);
      if (st == XOD_OK) st = upload(net, h.eq_neg, &ed.el_neg);
      ed.nasa = d.nasa, ed.tmid = d.tmid;
      if (st == XOD_OK) {
        cudaError_t ce = cudaFuncSetAttribute(k_equilibrium, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmemMax);
        if (ce != cudaSuccess) st = cuda_fail(ce, "cudaFuncSetAttribute(k_equilibrium)");
      }
    }
    if (h.lu.enabled) {
      LuHost &u = h.lu;
      LuDev &ud = net->ld;
      ud.enabled = 1, ud.n = u.n, ud.max_row = u.max_row, ud.nnz = u.nnz;
      if (st == XOD_OK) st = upload(net, u.perm, &ud.perm);
      if (st == XOD_OK) st = upload(net, u.diag, &ud.diag);
      if (st == XOD_OK) st = upload(net, u.src, &ud.src);
      if (st == XOD_OK) st = upload(net, u.col, &ud.col);
      if (st == XOD_OK) st = upload(net, u.row_ptr, &ud.row_ptr);
      if (st == XOD_OK) st = upload(net, u.rows, &ud.rows);
      if (st == XOD_OK) st = upload(net, u.pairs, &ud.pairs);
      if (st == XOD_OK) st = upload(net, u.tgt, &ud.tgt);
      ud.block_rows = u.block_rows, ud.n_blocks = (int32_t)u.blocks.size();
      if (st == XOD_OK) st = upload(net, u.blocks, &ud.blocks);
      if (st == XOD_OK) st = upload(net, u.steps, &ud.steps);
      if (st == XOD_OK) st = upload(net, u.items, &ud.items);
      if (st == XOD_OK) {
        cudaError_t ce = cudaFuncSetAttribute(k_lu_factor, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmemMax);
        if (ce != cudaSuccess) st = cuda_fail(ce, "cudaFuncSetAttribute(k_lu_factor)");
      }
    }
#undef UP
    if (st != XOD_OK) {
      std::string keep = g_err;
      xod_network_destroy(net);
      g_err = keep;
      return st;
    }
  }
  *out = net;
  return XOD_OK;
}

void xod_network_destroy(xod_network *net) {
  if (!net) return;
  for (void *e : net->timing.pool) cudaEventDestroy(static_cast<cudaEvent_t>(e));
  for (void *p : net->dev_allocs) cudaFree(p);
  if (net->stage) cudaFree(net->stage);
  for (void *hs : net->host_streams)
    if (hs) cudaStreamDestroy(static_cast<cudaStream_t>(hs));
  delete net;
}

xod_status xod_network_sizes(const xod_network *net, int32_t *n_species, int32_t *n_reactions,
                             int32_t *n_photo, int64_t *nnz_source, int64_t *nnz_jac,
                             int64_t *n_jac_terms) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  if (n_species) *n_species = net->h.ns;
  if (n_reactions) *n_reactions = net->h.nr;
  if (n_photo) *n_photo = net->h.n_photo;
  if (nnz_source) *nnz_source = (int64_t)net->h.src_rxn_user.size();
  if (nnz_jac) *nnz_jac = (int64_t)net->h.jac_col.size();
  if (n_jac_terms) *n_jac_terms = (int64_t)net->h.jac_terms.size();
  return XOD_OK;
}

xod_status xod_network_perm(const xod_network *net, int32_t *packed_to_user) {
  if (!net || !packed_to_user) return fail(XOD_ERR_INVALID_ARG, "NULL argument");
  std::memcpy(packed_to_user, net->h.packed_to_user.data(), net->h.packed_to_user.size() * sizeof(int32_t));
  return XOD_OK;
}

xod_status xod_network_photo_index(const xod_network *net, int32_t *user_rxn_of_photo_row) {
  if (!net || !user_rxn_of_photo_row) return fail(XOD_ERR_INVALID_ARG, "NULL argument");
  std::memcpy(user_rxn_of_photo_row, net->h.photo_user.data(), net->h.photo_user.size() * sizeof(int32_t));
  return XOD_OK;
}

xod_status xod_network_source_csr(const xod_network *net, int64_t *row_ptr, int32_t *rxn, int32_t *nu) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  const HostTables &h = net->h;
  if (row_ptr) std::memcpy(row_ptr, h.src_ptr.data(), h.src_ptr.size() * sizeof(int64_t));
  if (rxn) std::memcpy(rxn, h.src_rxn_user.data(), h.src_rxn_user.size() * sizeof(int32_t));
  if (nu) std::memcpy(nu, h.src_nu.data(), h.src_nu.size() * sizeof(int32_t));
  return XOD_OK;
}

xod_status xod_network_jac_pattern(const xod_network *net, int64_t *row_ptr, int32_t *col) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  const HostTables &h = net->h;
  if (row_ptr) std::memcpy(row_ptr, h.jac_ptr.data(), h.jac_ptr.size() * sizeof(int64_t));
  if (col) std::memcpy(col, h.jac_col.data(), h.jac_col.size() * sizeof(int32_t));
  return XOD_OK;
}

xod_status xod_network_fused_info(const xod_network *net, int64_t *info) {
  if (!net || !info) return fail(XOD_ERR_INVALID_ARG, "NULL argument");
  const FusedHost &f = net->h.f;
  info[0] = f.enabled, info[1] = f.chunk, info[2] = f.nchunk, info[3] = f.n_acc, info[4] = f.n_bp;
  info[5] = f.enabled ? (int64_t)fused_smem_bytes(net->h.ns, f.n_acc, f.chunk, f.meta_cap) : 0;
  info[6] = f.npad, info[7] = f.n_tasks, info[8] = f.n_entries;
  info[9] = (int64_t)f.blk.size();
  return XOD_OK;
}

xod_status xod_network_fused_params(const xod_network *net, int32_t interval, int32_t *user_rxn, int32_t *kind,
                                    double *coef, double *breakpoints) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  const HostTables &h = net->h;
  const FusedHost &f = h.f;
  if (!f.enabled) return fail(XOD_ERR_INVALID_ARG, "the fused-path tables are disabled for this network");
  if (interval < 0 || interval > f.n_bp) return fail(XOD_ERR_INVALID_ARG, "interval out of range");
  if (breakpoints) std::memcpy(breakpoints, f.bp.data(), f.bp.size() * sizeof(double));
  for (int pp = 0; pp < f.npad; ++pp) {
    if (user_rxn) user_rxn[pp] = f.pp_user[pp];
    const int seg = pp < f.arr_end ? 0 : pp < f.fo_end ? 1 : pp < f.ph_end ? 2 : 3;
    if (kind) kind[pp] = seg;
    if (!coef) continue;
    double *out = coef + (size_t)pp * 16;
    for (int k = 0; k < 16; ++k) out[k] = 0.0;
    if (seg >= 2) continue;
    const int first = seg == 0 ? 0 : f.arr_end;
    const int64_t off = seg == 0 ? 0 : f.blk_fo_off;
    const int bsz = seg == 0 ? kFBlkArr : kFBlkFo;
    const unsigned char *blk = &f.blk[(size_t)interval * f.blk_stride + off + (size_t)((pp - first) / kFRxnPerWarp) * bsz];
    const int slot = (pp - first) % kFRxnPerWarp, npair = seg == 0 ? 5 : 8;
    for (int u = 0; u < npair; ++u) std::memcpy(out + 2 * u, blk + (2 + u) * 64 + slot * 16, 16);
    // an irreversible reaction (or a padding slot) has k_r = 0: the blocks hold zeros there and the kernels select 0
    // by the reversible flag / the zeros row of the n tile; this view reports the equivalent C0 = -inf
    int32_t u1[4];
    std::memcpy(u1, blk + 64 + slot * 16, 16);
    if (!(u1[3] & 1)) out[3] = -INFINITY;
  }
  return XOD_OK;
}

xod_status xod_network_jac_info(const xod_network *net, int64_t *info) {
  if (!net || !info) return fail(XOD_ERR_INVALID_ARG, "NULL argument");
  const JacTiledHost &t = net->h.jt;
  info[0] = t.enabled, info[1] = t.chunk, info[2] = t.nchunk, info[3] = t.n_units, info[4] = t.acc_rows;
  info[5] = t.enabled ? (int64_t)jac_tiled_smem_bytes(net->h.ns, t.acc_rows, t.chunk, t.meta_cap) : 0;
  info[6] = t.n_slots, info[7] = t.n_entries;
  return XOD_OK;
}

xod_status xod_network_selfcheck(const xod_network *net) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  std::string err;
  if (!check_fused(net->h, err)) return fail(XOD_ERR_INVALID_ARG, err);
  if (!check_jac_tiled(net->h, err)) return fail(XOD_ERR_INVALID_ARG, err);
  if (!check_lu(net->h, err)) return fail(XOD_ERR_INVALID_ARG, err);
  return XOD_OK;
}

xod_status xod_network_tune(xod_network *net, int32_t knob, int64_t value) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  if (knob == XOD_TUNE_CHUNK_COLS) {
    if (value < 0) return fail(XOD_ERR_INVALID_ARG, "chunk columns must be >= 0");
    net->chunk_cols = value;
    return XOD_OK;
  }
  if (knob == XOD_TUNE_SPLIT) {
    if (value < 0) return fail(XOD_ERR_INVALID_ARG, "split must be >= 0");
    net->force_split = value;
    return XOD_OK;
  }
  if (knob == XOD_TUNE_FUSED_KERNEL) {
    net->use_fused = value;
    return XOD_OK;
  }
  if (knob == XOD_TUNE_JAC_TILED) {
    net->use_jac_tiled = value;
    return XOD_OK;
  }
  if (knob == XOD_TUNE_TIMING) {
    net->timing.on = value != 0;
    return XOD_OK;
  }
  return fail(XOD_ERR_INVALID_ARG, "unknown tuning knob");
}

// ---------------------------------------------------------------------------- compute calls

xod_status xod_thermo(const xod_network *net, int64_t ncol, int64_t ld, const double *T,
                      double *cp_R, double *h_RT, double *s_R, double *g_RT, void *stream) {
  xod_status st = check_common(net, ncol, ld);
  if (st != XOD_OK) return st;
  if (ncol == 0) return XOD_OK;
  if (!T) return fail(XOD_ERR_INVALID_ARG, "T is NULL");
  if (!cp_R && !h_RT && !s_R && !g_RT) return XOD_OK;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int64_t gx = (ncol + 127) / 128;
  // enough CTAs to fill the chip even for one atmosphere: split the species over blockIdx.y
  int spb = net->h.ns;
  while (spb > 4 && gx * ((net->h.ns + spb - 1) / spb) < (int64_t)net->sm_count * 8) spb = (spb + 1) / 2;
  dim3 grid((unsigned)gx, (unsigned)((net->h.ns + spb - 1) / spb));
  {
    Timed tm(net, KID_THERMO, s);
    k_thermo<<<grid, 128, 0, s>>>(net->d, ncol, ld, T, cp_R, h_RT, s_R, g_RT, spb);
  }
  XOD_CUDA(cudaGetLastError());
  return XOD_OK;
}

size_t xod_rate_coeffs_workspace_bytes(const xod_network *net, int64_t ncol) {
  if (!net || ncol < 0) return 0;
  return scratch_bytes(net, chunk_cols(net, ncol), true, false, false);
}

}  // extern "C"

namespace {

xod_status launch_prologue(const xod_network *net, int64_t ncol, int64_t col0, int64_t ncg,
                           const double *T, const double *P, const ChunkScratch &w, cudaStream_t s) {
  int split = 1;
  while (split < 64 && ncg * split < (int64_t)net->sm_count * 2 && split * 8 < net->h.ns) split *= 2;
  dim3 grid((unsigned)ncg, (unsigned)split);
  {
    Timed tm(net, KID_PROLOGUE, s);
    k_prologue<<<grid, 256, 0, s>>>(net->d, ncol, col0, T, P, w, kLog2Kb);
  }
  XOD_CUDA(cudaGetLastError());
  return XOD_OK;
}

template <int MODE>
xod_status launch_rates(const xod_network *net, int64_t ncol, int64_t col0, int64_t ld, int64_t ncg,
                        const ChunkScratch &w, const double *J, const double *n, double *kf, double *kr,
                        cudaStream_t s) {
  const int rw = pick_rw(net, net->h.nr, ncg);
  const int64_t nslices = (net->h.nr + rw - 1) / rw;
  const int64_t ntasks = nslices * ncg;
  const int64_t blocks = std::min<int64_t>((ntasks + 3) / 4, (int64_t)net->sm_count * 16);
  {
    Timed tm(net, KID_RATES, s);
    k_rates<MODE><<<(unsigned)blocks, 128, 0, s>>>(net->d, ncol, col0, ld, w, J, n, kf, kr, rw, (int)ncg, ntasks);
  }
  XOD_CUDA(cudaGetLastError());
  return XOD_OK;
}

// reaction splits per column tile of k_fused: enough work items to occupy every SM
int fused_split(const xod_network *net, int64_t ncol) {
  const int64_t ntiles = (ncol + kFW - 1) / kFW;
  int64_t sp = net->force_split > 0 ? net->force_split : (ntiles >= net->sm_count ? 1 : net->sm_count / std::max<int64_t>(ntiles, 1));
  return (int)std::max<int64_t>(1, std::min<int64_t>(sp, net->h.f.nchunk));
}

// columns of the leading part that fills whole rounds of tiles on every SM (0: no such split).
// The last partial round is launched separately with its chunks split over the idle SMs.
int64_t fused_full_round_cols(const xod_network *net, int64_t ncol) {
  const int64_t ntiles = (ncol + kFW - 1) / kFW, sm = net->sm_count;
  if (net->force_split > 0 || ntiles <= sm || ntiles % sm == 0) return 0;
  return ntiles / sm * sm * kFW;
}

// workspace bytes of the partial sums when k_fused splits the chunks of a tile over several CTAs
size_t fused_partial_bytes(const xod_network *net, int64_t ncol) {
  if (!net->h.f.enabled) return 0;
  const int64_t rem = ncol - fused_full_round_cols(net, ncol);  // the part that may run split
  const int ns_ = fused_split(net, rem);
  return ns_ > 1 ? (size_t)ns_ * net->h.ns * (size_t)round_up(rem, 32) * sizeof(double) + 256 : 0;
}

// T, P, J given: xod_source_fused (coefficients evaluated in the kernel); kf, kr given: xod_source
xod_status launch_fused(const xod_network *net, int64_t ncol, int64_t ld, const double *T, const double *P,
                        const double *J, const double *kf, const double *kr, const double *n, double *dndt,
                        void *workspace, cudaStream_t s, int64_t ldo = 0 /* pitch of dndt; 0: ld */) {
  if (ldo == 0) ldo = ld;
  const HostTables &h = net->h;
  auto off = [](const double *p, int64_t c) { return p ? p + c : p; };
  if (const int64_t c_full = fused_full_round_cols(net, ncol)) {  // columns are independent: two sub-ranges
    xod_status st = launch_fused(net, c_full, ld, T, P, J, kf, kr, n, dndt, workspace, s, ldo);
    if (st != XOD_OK) return st;
    return launch_fused(net, ncol - c_full, ld, off(T, c_full), off(P, c_full), off(J, c_full), off(kf, c_full),
                        off(kr, c_full), n + c_full, dndt + c_full, workspace, s, ldo);
  }
  FusedArgs a{};
  a.ncol = ncol, a.ld = ld, a.ldo = ldo, a.T = T, a.P = P, a.J = J, a.n = n, a.kf = kf, a.kr = kr;
  a.ntiles = (int32_t)((ncol + kFW - 1) / kFW);
  a.nsplit = fused_split(net, ncol);
  a.log2_kb = kLog2Kb;
  a.nr = h.nr, a.n_photo = h.n_photo;
  a.ldp = round_up(ncol, 32);
  double *part = reinterpret_cast<double *>((reinterpret_cast<uintptr_t>(workspace) + 255) & ~uintptr_t(255));
  a.out = a.nsplit == 1 ? dndt : part;
  const int64_t items = (int64_t)a.ntiles * a.nsplit;
  const unsigned grid = (unsigned)std::min<int64_t>(items, net->sm_count);
  const size_t smem = fused_smem_bytes(h.ns, h.f.n_acc, h.f.chunk, h.f.meta_cap);
  {
    Timed tm(net, KID_FUSED, s);
    if (kf)
      k_fused<true><<<grid, kFWarps * 32, smem, s>>>(net->fd, h.ns, a);
    else
      k_fused<false><<<grid, kFWarps * 32, smem, s>>>(net->fd, h.ns, a);
  }
  XOD_CUDA(cudaGetLastError());
  if (a.nsplit > 1) {
    dim3 g((unsigned)((ncol + 127) / 128), (unsigned)h.ns);
    Timed tm(net, KID_FUSED_COMBINE, s);
    k_fused_combine<<<g, 128, 0, s>>>(h.ns, ncol, ldo, a.ldp, a.nsplit, part, dndt);
  }
  XOD_CUDA(cudaGetLastError());
  return XOD_OK;
}

// k_jac_tiled: whole rounds of column tiles on every SM run unsplit; the last partial round (or a batch with
// fewer tiles than SMs) has each tile's units split over the otherwise idle SMs (units are independent)
xod_status launch_jac_tiled(const xod_network *net, int64_t ncol, int64_t ld, int64_t ldo, const double *kf,
                            const double *kr, const double *n, double *jac, cudaStream_t s) {
  const size_t smem = jac_tiled_smem_bytes(net->h.ns, net->h.jt.acc_rows, net->h.jt.chunk, net->h.jt.meta_cap);
  const int64_t ntiles = (ncol + kFW - 1) / kFW, sm = net->sm_count;
  const int64_t full = net->force_split > 0 ? 0 : ntiles / sm * sm;
  for (int part = 0; part < 2; ++part) {
    const int64_t t0 = part == 0 ? 0 : full, t1 = part == 0 ? full : ntiles;
    if (t1 <= t0) continue;
    JacArgs a{};
    const int64_t c0 = t0 * kFW;
    a.ncol = std::min<int64_t>(ncol, t1 * kFW) - c0, a.ld = ld, a.ldo = ldo;
    a.kf = kf + c0, a.kr = kr + c0, a.n = n + c0, a.jac = jac + c0;
    a.ntiles = (int32_t)(t1 - t0);
    const int64_t split = part == 0 ? 1 : (net->force_split > 0 ? net->force_split : sm / (t1 - t0));
    a.nsplit = (int32_t)std::max<int64_t>(1, std::min<int64_t>(split, net->h.jt.n_units));
    a.nr = net->h.nr, a.nnz = net->d.nnz_jac;
    const unsigned grid = (unsigned)std::min<int64_t>((int64_t)a.ntiles * a.nsplit, sm);
    Timed tm(net, KID_JAC_TILED, s);
    k_jac_tiled<<<grid, kFWarps * 32, smem, s>>>(net->jd, net->h.ns, a);
    XOD_CUDA(cudaGetLastError());
  }
  return XOD_OK;
}

template <bool PL>
xod_status launch_source(const xod_network *net, int64_t ncol, int64_t col0, int64_t ld, int64_t ncg,
                         const ChunkScratch &w, double *dndt, double *prod, double *loss, cudaStream_t s) {
  dim3 grid((unsigned)net->d.n_src_tasks, (unsigned)ncg);
  {
    Timed tm(net, KID_SOURCE, s);
    k_source<PL><<<grid, 256, 0, s>>>(net->d, ncol, col0, ld, w, dndt, prod, loss);
  }
  XOD_CUDA(cudaGetLastError());
  return XOD_OK;
}

}  // namespace

extern "C" {

xod_status xod_rate_coeffs(const xod_network *net, int64_t ncol, int64_t ld, const double *T,
                           const double *P, const double *J, double *kf, double *kr,
                           void *workspace, size_t workspace_bytes, void *stream) {
  xod_status st = check_common(net, ncol, ld);
  if (st != XOD_OK) return st;
  if (ncol == 0 || net->h.nr == 0) return XOD_OK;
  if (!T || !P) return fail(XOD_ERR_INVALID_ARG, "T or P is NULL");
  if (net->h.n_photo > 0 && !J) return fail(XOD_ERR_INVALID_ARG, "J is NULL but the network has photolysis reactions");
  if (!kf && !kr) return XOD_OK;
  if (!workspace || workspace_bytes < xod_rate_coeffs_workspace_bytes(net, ncol))
    return fail(XOD_ERR_WORKSPACE, "workspace NULL or smaller than xod_rate_coeffs_workspace_bytes");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (net->fd.enabled && net->use_fused) {  // one kernel from the per-interval parameter blocks
    // reactions per CTA: enough CTAs for ~8 per SM, at most 64 reactions each
    const int64_t nbx = (ncol + 255) / 256;
    int slice = (int)std::min<int64_t>(64, std::max<int64_t>(4, (int64_t)net->fd.ph_end * nbx / (net->sm_count * 8)));
    slice = (slice + 3) / 4 * 4;
    dim3 grid((unsigned)nbx, (unsigned)((net->fd.ph_end + slice - 1) / slice));
    Timed tm(net, KID_RATE_COEFFS, s);
    k_rate_coeffs<<<grid, 256, 0, s>>>(net->fd, ncol, ld, T, P, J, kf, kr, kLog2Kb, slice, net->h.nr, net->h.n_photo);
    XOD_CUDA(cudaGetLastError());
    return XOD_OK;
  }
  const int64_t ldw = chunk_cols(net, ncol);
  ChunkScratch w = carve(net, workspace, ldw, true, false, false);
  for (int64_t col0 = 0; col0 < ncol; col0 += ldw) {
    const int64_t nc = std::min(ldw, ncol - col0), ncg = (nc + 31) / 32;
    if ((st = launch_prologue(net, ncol, col0, ncg, T, P, w, s)) != XOD_OK) return st;
    if ((st = launch_rates<MODE_K>(net, ncol, col0, ld, ncg, w, J, nullptr, kf, kr, s)) != XOD_OK) return st;
  }
  return XOD_OK;
}

size_t xod_source_workspace_bytes(const xod_network *net, int64_t ncol) {
  if (!net || ncol < 0) return 0;
  return std::max(scratch_bytes(net, chunk_cols(net, ncol), false, true, true), fused_partial_bytes(net, ncol));
}

size_t xod_source_workspace_bytes_dndt(const xod_network *net, int64_t ncol) {
  if (!net || ncol < 0) return 0;
  if (net->fd.enabled && net->use_fused && net->h.nr > 0) return fused_partial_bytes(net, ncol) + 16;
  return scratch_bytes(net, chunk_cols(net, ncol), false, true, false);
}

xod_status xod_source(const xod_network *net, int64_t ncol, int64_t ld, const double *kf,
                      const double *kr, const double *n, double *dndt, double *prod, double *loss,
                      void *workspace, size_t workspace_bytes, void *stream) {
  xod_status st = check_common(net, ncol, ld);
  if (st != XOD_OK) return st;
  if (ncol == 0) return XOD_OK;
  if (!n || !dndt) return fail(XOD_ERR_INVALID_ARG, "n or dndt is NULL");
  if (net->h.nr > 0 && (!kf || !kr)) return fail(XOD_ERR_INVALID_ARG, "kf or kr is NULL");
  if ((prod == nullptr) != (loss == nullptr)) return fail(XOD_ERR_INVALID_ARG, "prod and loss must be given together");
  const bool pl = prod != nullptr;
  if (!workspace || workspace_bytes < (pl ? xod_source_workspace_bytes(net, ncol) : xod_source_workspace_bytes_dndt(net, ncol)))
    return fail(XOD_ERR_WORKSPACE, "workspace NULL or smaller than xod_source_workspace_bytes (xod_source_workspace_bytes_dndt without prod/loss)");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (!pl && net->fd.enabled && net->use_fused && net->h.nr > 0)
    return launch_fused(net, ncol, ld, nullptr, nullptr, nullptr, kf, kr, n, dndt, workspace, s);
  const int64_t ldw = chunk_cols(net, ncol);
  ChunkScratch w = carve(net, workspace, ldw, false, true, pl);
  for (int64_t col0 = 0; col0 < ncol; col0 += ldw) {
    const int64_t nc = std::min(ldw, ncol - col0), ncg = (nc + 31) / 32;
    if (net->h.nr > 0) {
      const int rw = pick_rw(net, net->h.nr, ncg);
      const int64_t ntasks = (int64_t)((net->h.nr + rw - 1) / rw) * ncg;
      const int64_t blocks = std::min<int64_t>((ntasks + 3) / 4, (int64_t)net->sm_count * 16);
      Timed tm(net, KID_RATES_FROM_K, s);
      if (pl)
        k_rates_from_k<MODE_QSEP><<<(unsigned)blocks, 128, 0, s>>>(net->d, ncol, col0, ld, w, kf, kr, n, rw, (int)ncg, ntasks);
      else
        k_rates_from_k<MODE_QNET><<<(unsigned)blocks, 128, 0, s>>>(net->d, ncol, col0, ld, w, kf, kr, n, rw, (int)ncg, ntasks);
      XOD_CUDA(cudaGetLastError());
    }
    st = pl ? launch_source<true>(net, ncol, col0, ld, ncg, w, dndt, prod, loss, s)
            : launch_source<false>(net, ncol, col0, ld, ncg, w, dndt, prod, loss, s);
    if (st != XOD_OK) return st;
  }
  return XOD_OK;
}

size_t xod_source_fused_workspace_bytes(const xod_network *net, int64_t ncol) {
  if (!net || ncol < 0) return 0;
  return std::max(scratch_bytes(net, chunk_cols(net, ncol), true, true, true), fused_partial_bytes(net, ncol));
}

size_t xod_source_fused_workspace_bytes_dndt(const xod_network *net, int64_t ncol) {
  if (!net || ncol < 0) return 0;
  if (net->fd.enabled && net->use_fused) return fused_partial_bytes(net, ncol) + 16;
  return scratch_bytes(net, chunk_cols(net, ncol), true, true, false);
}

xod_status xod_source_fused(const xod_network *net, int64_t ncol, int64_t ld, const double *T,
                            const double *P, const double *J, const double *n, double *dndt,
                            double *prod, double *loss, void *workspace, size_t workspace_bytes,
                            void *stream) {
  xod_status st = check_common(net, ncol, ld);
  if (st != XOD_OK) return st;
  if (ncol == 0) return XOD_OK;
  if (!T || !P || !n || !dndt) return fail(XOD_ERR_INVALID_ARG, "T, P, n or dndt is NULL");
  if (net->h.n_photo > 0 && !J) return fail(XOD_ERR_INVALID_ARG, "J is NULL but the network has photolysis reactions");
  if ((prod == nullptr) != (loss == nullptr)) return fail(XOD_ERR_INVALID_ARG, "prod and loss must be given together");
  const bool pl = prod != nullptr;
  if (!workspace || workspace_bytes < (pl ? xod_source_fused_workspace_bytes(net, ncol) : xod_source_fused_workspace_bytes_dndt(net, ncol)))
    return fail(XOD_ERR_WORKSPACE, "workspace NULL or smaller than xod_source_fused_workspace_bytes (xod_source_fused_workspace_bytes_dndt without prod/loss)");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (!pl && net->fd.enabled && net->use_fused)
    return launch_fused(net, ncol, ld, T, P, J, nullptr, nullptr, n, dndt, workspace, s);
  const int64_t ldw = chunk_cols(net, ncol);
  ChunkScratch w = carve(net, workspace, ldw, true, true, pl);
  for (int64_t col0 = 0; col0 < ncol; col0 += ldw) {
    const int64_t nc = std::min(ldw, ncol - col0), ncg = (nc + 31) / 32;
    if (net->h.nr > 0) {
      if ((st = launch_prologue(net, ncol, col0, ncg, T, P, w, s)) != XOD_OK) return st;
      st = pl ? launch_rates<MODE_QSEP>(net, ncol, col0, ld, ncg, w, J, n, nullptr, nullptr, s)
              : launch_rates<MODE_QNET>(net, ncol, col0, ld, ncg, w, J, n, nullptr, nullptr, s);
      if (st != XOD_OK) return st;
    }
    st = pl ? launch_source<true>(net, ncol, col0, ld, ncg, w, dndt, prod, loss, s)
            : launch_source<false>(net, ncol, col0, ld, ncg, w, dndt, prod, loss, s);
    if (st != XOD_OK) return st;
  }
  return XOD_OK;
}

xod_status xod_jacobian(const xod_network *net, int64_t ncol, int64_t ld, const double *kf,
                        const double *kr, const double *n, double *jac, void *stream) {
  xod_status st = check_common(net, ncol, ld);
  if (st != XOD_OK) return st;
  if (ncol == 0) return XOD_OK;
  if (!n || !jac) return fail(XOD_ERR_INVALID_ARG, "n or jac is NULL");
  if (net->h.nr > 0 && (!kf || !kr)) return fail(XOD_ERR_INVALID_ARG, "kf or kr is NULL");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (net->jd.enabled && net->use_jac_tiled && net->h.nr > 0) return launch_jac_tiled(net, ncol, ld, ld, kf, kr, n, jac, s);
  const int64_t ncg = (ncol + 31) / 32;
  if (ncg > 65535) return fail(XOD_ERR_INVALID_ARG, "ncol too large for one xod_jacobian call (max 2097120)");
  const int64_t want = (net->d.nnz_jac + 7) / 8;
  // CTAs per column group: at least two per SM, so the CTAs resident on an SM mostly share one
  // column group and its n rows stay in L1 (measured 2.96 -> 2.52 ms on config 5)
  const int64_t gx = std::max<int64_t>(1, std::min<int64_t>(want, std::max<int64_t>(2LL * net->sm_count, 64LL * net->sm_count / ncg)));
  dim3 grid((unsigned)gx, (unsigned)ncg);
  {
    Timed tm(net, KID_JACOBIAN, s);
    k_jacobian<<<grid, 256, 0, s>>>(net->d, ncol, ld, kf, kr, n, jac);
  }
  XOD_CUDA(cudaGetLastError());
  return XOD_OK;
}

xod_status xod_source_fused_host(xod_network *net, int64_t ncol, int64_t ld, const double *T,
                                 const double *P, const double *J, const double *n, double *dndt) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  if (net->device < 0) return fail(XOD_ERR_CUDA, "network was created without a CUDA device");
  DeviceGuard guard(net->device);  // this call allocates and synchronises: it may switch, and restores
  if (guard.err != cudaSuccess) return cuda_fail(guard.err, "cudaSetDevice");
  xod_status st = check_common(net, ncol, ld);
  if (st != XOD_OK) return st;
  if (ncol == 0) return XOD_OK;
  if (!T || !P || !n || !dndt) return fail(XOD_ERR_INVALID_ARG, "T, P, n or dndt is NULL");
  if (net->h.n_photo > 0 && !J) return fail(XOD_ERR_INVALID_ARG, "J is NULL but the network has photolysis reactions");
  // Column-chunk pipeline over kHostSlots staging slots, one stream each: the H2D copy of chunk
  // c + 1, the kernels of chunk c and the D2H copy of chunk c - 1 overlap (PCIe is full duplex).
  // A chunk is one full round of column tiles on every SM (sm_count x 16 columns), so chunking
  // costs the persistent kernel no tail.  Rows are strided in host memory: cudaMemcpy2DAsync.
  const size_t ns = net->h.ns, nph = net->h.n_photo;
  const int64_t cw = std::min<int64_t>(round_up(ncol, 32), (int64_t)net->sm_count * kFW);  // columns per chunk
  // the ragged last chunk runs with fewer tiles and therefore more reaction splits: size for both widths
  const size_t ws = std::max(xod_source_fused_workspace_bytes_dndt(net, cw),
                             ncol % cw ? xod_source_fused_workspace_bytes_dndt(net, ncol % cw) : 0) + 256;
  const size_t rows = 2 + nph + 2 * ns;
  const size_t slot_bytes = round_up((int64_t)(rows * cw * sizeof(double) + ws), 256);
  const size_t need = slot_bytes * kHostSlots;
  if (net->stage_bytes < need) {
    if (net->stage) cudaFree(net->stage);
    net->stage = nullptr, net->stage_bytes = 0;
    XOD_CUDA(cudaMalloc(&net->stage, need));
    net->stage_bytes = need;
  }
  for (int i = 0; i < kHostSlots; ++i)
    if (!net->host_streams[i]) {
      cudaStream_t s = nullptr;
      XOD_CUDA(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
      net->host_streams[i] = s;
    }
  const size_t hp = (size_t)ld * sizeof(double), dp = (size_t)cw * sizeof(double);
  // an error after the first chunk must not return with copies still in flight on the private streams
  auto drain = [&](xod_status code) {
    const std::string keep = g_err;
    for (void *hs : net->host_streams)
      if (hs) cudaStreamSynchronize(static_cast<cudaStream_t>(hs));
    g_err = keep;
    return code;
  };
#define XOD_CUDA_DRAIN(call)                                          \
  do {                                                                \
    cudaError_t e_ = (call);                                          \
    if (e_ != cudaSuccess) return drain(cuda_fail(e_, #call));        \
  } while (0)
  int slot = 0;
  for (int64_t c0 = 0; c0 < ncol; c0 += cw, slot = (slot + 1) % kHostSlots) {
    const int64_t w = std::min(cw, ncol - c0);
    const size_t wb = (size_t)w * sizeof(double);
    cudaStream_t s = static_cast<cudaStream_t>(net->host_streams[slot]);
    double *dT = reinterpret_cast<double *>(static_cast<char *>(net->stage) + slot_bytes * slot);
    double *dP = dT + cw, *dJ = dP + cw, *dn = dJ + nph * cw, *dd = dn + ns * cw;
    void *dws = dd + ns * cw;
    XOD_CUDA_DRAIN(cudaMemcpyAsync(dT, T + c0, wb, cudaMemcpyHostToDevice, s));
    XOD_CUDA_DRAIN(cudaMemcpyAsync(dP, P + c0, wb, cudaMemcpyHostToDevice, s));
    if (nph) XOD_CUDA_DRAIN(cudaMemcpy2DAsync(dJ, dp, J + c0, hp, wb, nph, cudaMemcpyHostToDevice, s));
    XOD_CUDA_DRAIN(cudaMemcpy2DAsync(dn, dp, n + c0, hp, wb, ns, cudaMemcpyHostToDevice, s));
    st = xod_source_fused(net, w, cw, dT, dP, dJ, dn, dd, nullptr, nullptr, dws, ws, s);
    if (st != XOD_OK) return drain(st);
    XOD_CUDA_DRAIN(cudaMemcpy2DAsync(dndt + c0, hp, dd, dp, wb, ns, cudaMemcpyDeviceToHost, s));
  }
#undef XOD_CUDA_DRAIN
  for (int i = 0; i < kHostSlots; ++i) XOD_CUDA(cudaStreamSynchronize(static_cast<cudaStream_t>(net->host_streams[i])));
  return XOD_OK;
}

// ---------------------------------------------------------------------------- f1: implicit step

xod_status xod_network_lu_info(const xod_network *net, int64_t *info) {
  if (!net || !info) return fail(XOD_ERR_INVALID_ARG, "NULL argument");
  const LuHost &u = net->h.lu;
  info[0] = u.enabled, info[1] = u.nnz, info[2] = (int64_t)u.pairs.size(), info[3] = u.n_updates, info[4] = u.max_row;
  info[5] = u.block_rows, info[6] = u.n_block_loads, info[7] = (int64_t)u.steps.size();
  return XOD_OK;
}

xod_status xod_network_lu_pattern(const xod_network *net, int32_t *perm, int64_t *row_ptr, int32_t *col) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  const LuHost &u = net->h.lu;
  if (!u.enabled) return fail(XOD_ERR_INVALID_ARG, "the network was created without XOD_FLAG_BUILD_LU");
  if (perm) std::memcpy(perm, u.perm.data(), u.perm.size() * sizeof(int32_t));
  if (row_ptr) std::memcpy(row_ptr, u.row_ptr.data(), u.row_ptr.size() * sizeof(int64_t));
  if (col) std::memcpy(col, u.col.data(), u.col.size() * sizeof(int32_t));
  return XOD_OK;
}

}  // extern "C"

namespace {
constexpr int64_t kNewtonChunk = 2368;   // columns per pass of the implicit step (bounds the workspace): 148 SMs x 16 = two full waves of k_lu_factor's 8-column CTAs
int64_t newton_chunk(int64_t ncol) { return std::min<int64_t>(round_up(std::max<int64_t>(ncol, 1), 32), kNewtonChunk); }
}  // namespace

extern "C" {

size_t xod_newton_workspace_bytes(const xod_network *net, int64_t ncol) {
  if (!net || ncol < 0 || !net->h.lu.enabled) return 0;
  const int64_t cw = newton_chunk(ncol);
  const size_t rows = (size_t)2 * net->h.ns + (size_t)net->h.jac_col.size() + (size_t)net->h.lu.nnz;
  // k_fused's partial sums: a narrower last pass has fewer tiles, hence more reaction splits and a larger buffer
  const int64_t last = ncol % cw;
  const size_t part = std::max(ncol >= cw ? fused_partial_bytes(net, cw) : 0, last ? fused_partial_bytes(net, last) : 0);
  return rows * (size_t)cw * sizeof(double) + part + 1024;
}

xod_status xod_newton_step(const xod_network *net, int64_t ncol, int64_t ld, const double *kf, const double *kr,
                           const double *n_old, const double *dt, double *y, double *delta, void *workspace,
                           size_t workspace_bytes, void *stream) {
  xod_status st = check_common(net, ncol, ld);
  if (st != XOD_OK) return st;
  if (!net->h.lu.enabled) return fail(XOD_ERR_INVALID_ARG, "the network was created without XOD_FLAG_BUILD_LU");
  if (!net->fd.enabled || !net->jd.enabled || net->h.nr == 0)
    return fail(XOD_ERR_INVALID_ARG, "the implicit step needs the single-kernel source and Jacobian tables (see xod_network_fused_info, xod_network_jac_info)");
  if (ncol == 0) return XOD_OK;
  if (!kf || !kr || !n_old || !dt || !y) return fail(XOD_ERR_INVALID_ARG, "kf, kr, n_old, dt or y is NULL");
  if (!workspace || workspace_bytes < xod_newton_workspace_bytes(net, ncol))
    return fail(XOD_ERR_WORKSPACE, "workspace NULL or smaller than xod_newton_workspace_bytes");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int64_t cw = newton_chunk(ncol);
  const size_t ns = net->h.ns, nnzj = net->h.jac_col.size(), nnzl = (size_t)net->h.lu.nnz;
  double *f = reinterpret_cast<double *>((reinterpret_cast<uintptr_t>(workspace) + 255) & ~uintptr_t(255));
  double *rhs = f + ns * cw, *jac = rhs + ns * cw, *lu = jac + nnzj * cw;
  void *src_ws = lu + nnzl * cw;
  const size_t smem = (size_t)net->h.lu.block_rows * net->h.lu.max_row * kLuCols * sizeof(double);
  if (smem > kFusedSmemMax) return fail(XOD_ERR_INVALID_ARG, "a row of the LU pattern does not fit shared memory");
  for (int64_t c0 = 0; c0 < ncol; c0 += cw) {
    const int64_t w = std::min(cw, ncol - c0);
    // f(y) and Jac(y) of this chunk into the workspace (pitch cw), by the kernels of xod_source / xod_jacobian
    if ((st = launch_fused(net, w, ld, nullptr, nullptr, nullptr, kf + c0, kr + c0, y + c0, f, src_ws, s, cw)) != XOD_OK) return st;
    if ((st = launch_jac_tiled(net, w, ld, cw, kf + c0, kr + c0, y + c0, jac, s)) != XOD_OK) return st;
    NewtonArgs a{};
    a.ncol = w, a.ld = ld, a.ldw = cw;
    a.n_old = n_old + c0, a.dt = dt + c0, a.f = f, a.jac = jac, a.y = y + c0, a.delta = delta ? delta + c0 : nullptr;
    a.lu = lu, a.rhs = rhs, a.nnz_jac = (int64_t)nnzj;
    {
      const int64_t gx = (w + 127) / 128;
      dim3 grid((unsigned)gx, (unsigned)std::max<int64_t>(1, std::min<int64_t>(net->h.lu.nnz, (int64_t)net->sm_count * 16 / gx)));
      Timed tm(net, KID_NEWTON_ASSEMBLE, s);
      k_newton_assemble<<<grid, 128, 0, s>>>(net->ld, a);
      XOD_CUDA(cudaGetLastError());
    }
    {
      Timed tm(net, KID_LU_FACTOR, s);
      k_lu_factor<<<(unsigned)((w + kLuCols - 1) / kLuCols), 32 * kLuWarps, smem, s>>>(net->ld, lu, cw, w);
      XOD_CUDA(cudaGetLastError());
    }
    {
      Timed tm(net, KID_LU_SOLVE, s);
      k_lu_solve<<<(unsigned)((w + 127) / 128), 128, 0, s>>>(net->ld, a);
      XOD_CUDA(cudaGetLastError());
    }
  }
  return XOD_OK;
}

// ---------------------------------------------------------------------------- f2: photolysis rate constants

xod_status xod_photo_create(const xod_network *net, const xod_photo_desc *d, xod_photo **out) {
  if (!out) return fail(XOD_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (!net || !d) return fail(XOD_ERR_INVALID_ARG, "net or desc is NULL");
  if (d->n_bins <= 0 || d->n_abs < 0) return fail(XOD_ERR_INVALID_ARG, "n_bins must be > 0 and n_abs >= 0");
  if (!d->dlambda || (net->h.n_photo > 0 && !d->sigma_ph) || (d->n_abs > 0 && (!d->abs_species || !d->sigma_ext)))
    return fail(XOD_ERR_INVALID_ARG, "dlambda, sigma_ph, abs_species, sigma_ext must not be NULL");
  for (int x = 0; x < d->n_abs; ++x)
    if (d->abs_species[x] < 0 || d->abs_species[x] >= net->h.ns) return fail(XOD_ERR_INVALID_ARG, "abs_species index out of range");
  const size_t nb = (size_t)d->n_bins;
  auto all_ok = [](const double *p, size_t n) {
    for (size_t i = 0; i < n; ++i)
      if (!std::isfinite(p[i]) || p[i] < 0) return false;
    return true;
  };
  if (!all_ok(d->dlambda, nb) || !all_ok(d->sigma_ext, nb * d->n_abs) || !all_ok(d->sigma_ph, nb * net->h.n_photo))
    return fail(XOD_ERR_INVALID_ARG, "bin widths and cross-sections must be finite and >= 0");
  xod_photo *ph = new (std::nothrow) xod_photo;
  if (!ph) return fail(XOD_ERR_ALLOC, "out of host memory");
  ph->net = net, ph->device = net->device, ph->n_bins = d->n_bins, ph->n_abs = d->n_abs, ph->n_photo = net->h.n_photo;
  ph->h_dlambda.assign(d->dlambda, d->dlambda + nb);
  ph->h_sigma_ext.assign(d->sigma_ext, d->sigma_ext + nb * d->n_abs);
  ph->h_sigma_ph.assign(d->sigma_ph, d->sigma_ph + nb * net->h.n_photo);
  ph->h_abs.assign(d->abs_species, d->abs_species + d->n_abs);
  if (ph->device >= 0) {
    DeviceGuard guard(ph->device);
    cudaError_t e = guard.err;
    auto up = [&](const void *src, size_t bytes, void **dst) {
      if (e != cudaSuccess) return;
      e = cudaMalloc(dst, std::max<size_t>(bytes, 16));
      if (e == cudaSuccess && bytes) e = cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice);
    };
    up(ph->h_dlambda.data(), nb * 8, (void **)&ph->dlambda);
    up(ph->h_sigma_ext.data(), ph->h_sigma_ext.size() * 8, (void **)&ph->sigma_ext);
    up(ph->h_sigma_ph.data(), ph->h_sigma_ph.size() * 8, (void **)&ph->sigma_ph);
    up(ph->h_abs.data(), ph->h_abs.size() * 4, (void **)&ph->abs_species);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_photo_flux, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmemMax);
    if (e != cudaSuccess) {
      xod_photo_destroy(ph);
      return cuda_fail(e, "xod_photo_create");
    }
  }
  *out = ph;
  return XOD_OK;
}

void xod_photo_destroy(xod_photo *ph) {
  if (!ph) return;
  if (ph->dlambda) cudaFree(ph->dlambda);
  if (ph->sigma_ext) cudaFree(ph->sigma_ext);
  if (ph->sigma_ph) cudaFree(ph->sigma_ph);
  if (ph->abs_species) cudaFree(ph->abs_species);
  delete ph;
}

size_t xod_photo_workspace_bytes(const xod_photo *ph, int64_t ncol) {
  if (!ph || ncol < 0) return 0;
  return (size_t)ph->n_bins * (size_t)round_up(std::max<int64_t>(ncol, 1), 32) * sizeof(double) + 256;
}

xod_status xod_photo_rates(const xod_photo *ph, int64_t n_atm, int64_t n_layers, int64_t ld, const double *n,
                           const double *dz, const double *j0, const double *j_diff, const double *mu,
                           const double *t_f, double *J, void *workspace, size_t workspace_bytes, void *stream) {
  if (!ph) return fail(XOD_ERR_INVALID_ARG, "photo is NULL");
  if (n_atm < 0 || n_layers < 0) return fail(XOD_ERR_INVALID_ARG, "n_atm or n_layers < 0");
  const int64_t ncol = n_atm * n_layers;
  xod_status st = check_common(ph->net, ncol, ld);
  if (st != XOD_OK) return st;
  if (ncol == 0 || ph->n_photo == 0) return XOD_OK;
  if (!n || !dz || !j0 || !mu || !t_f || !J) return fail(XOD_ERR_INVALID_ARG, "n, dz, j0, mu, t_f or J is NULL");
  if (!workspace || workspace_bytes < xod_photo_workspace_bytes(ph, ncol))
    return fail(XOD_ERR_WORKSPACE, "workspace NULL or smaller than xod_photo_workspace_bytes");
  const size_t smem = (size_t)32 * (size_t)(n_layers | 1) * sizeof(double);
  if (smem > kFusedSmemMax) return fail(XOD_ERR_INVALID_ARG, "n_layers too large for one call (max 907)");
  if (n_atm > 65535) return fail(XOD_ERR_INVALID_ARG, "n_atm too large for one call (max 65535)");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const xod_network *net = ph->net;
  const int64_t ldw = round_up(ncol, 32);
  double *F = reinterpret_cast<double *>((reinterpret_cast<uintptr_t>(workspace) + 255) & ~uintptr_t(255));
  {   // kappa[b][col] = sum_x sigma_ext[x][b] n[abs_species[x]][col]
    GemmArgs g{};
    g.M = ph->n_bins, g.N = ncol, g.K = ph->n_abs;
    g.A = ph->sigma_ext, g.lda = ph->n_bins;
    g.B = n, g.brow = ph->abs_species, g.ldb = ld, g.n_brows = net->h.ns;
    g.C = F, g.ldc = ldw, g.scale_atm = nullptr, g.n_layers = 1;
    dim3 grid((unsigned)((ncol + kGemmBN - 1) / kGemmBN), (unsigned)((ph->n_bins + kGemmBM - 1) / kGemmBM));
    Timed tm(net, KID_PHOTO_GEMM, s);
    k_photo_gemm<false><<<grid, 256, 0, s>>>(g);
    XOD_CUDA(cudaGetLastError());
  }
  {   // tau (layer centres, top down), Beer-Lambert, times the bin width, in place
    FluxArgs f{};
    f.n_bins = ph->n_bins, f.n_atm = n_atm, f.n_layers = n_layers, f.ld = ld, f.ldw = ldw;
    f.F = F, f.dz = dz, f.j0 = j0, f.j_diff = j_diff, f.mu = mu, f.dlambda = ph->dlambda;
    dim3 grid((unsigned)((ph->n_bins + 31) / 32), (unsigned)n_atm);
    Timed tm(net, KID_PHOTO_FLUX, s);
    k_photo_flux<<<grid, 256, smem, s>>>(f);
    XOD_CUDA(cudaGetLastError());
  }
  {   // J[p][col] = t_f sum_b sigma_ph[p][b] F[b][col]
    GemmArgs g{};
    g.M = ph->n_photo, g.N = ncol, g.K = ph->n_bins;
    g.A = ph->sigma_ph, g.lda = ph->n_bins;
    g.B = F, g.brow = nullptr, g.ldb = ldw, g.n_brows = ph->n_bins;
    g.C = J, g.ldc = ld, g.scale_atm = t_f, g.n_layers = n_layers;
    dim3 grid((unsigned)((ncol + kGemmBN - 1) / kGemmBN), (unsigned)((ph->n_photo + kGemmBM - 1) / kGemmBM));
    Timed tm(net, KID_PHOTO_GEMM, s);
    k_photo_gemm<true><<<grid, 256, 0, s>>>(g);
    XOD_CUDA(cudaGetLastError());
  }
  return XOD_OK;
}

// ---------------------------------------------------------------------------- f3: transport terms

xod_status xod_transport(const xod_network *net, int64_t n_atm, int64_t n_layers, int64_t ld, const double *n,
                         const double *T, const double *n_gas, const double *D, const double *mass,
                         const double *alpha_T, const double *mbar, const double *grav, const double *dz, double *tr,
                         void *stream) {
  if (n_atm < 0 || n_layers < 0) return fail(XOD_ERR_INVALID_ARG, "n_atm or n_layers < 0");
  const int64_t ncol = n_atm * n_layers;
  xod_status st = check_common(net, ncol, ld);
  if (st != XOD_OK) return st;
  if (ncol == 0) return XOD_OK;
  if (!n || !T || !n_gas || !D || !mass || !alpha_T || !mbar || !grav || !dz || !tr)
    return fail(XOD_ERR_INVALID_ARG, "n, T, n_gas, D, mass, alpha_T, mbar, grav, dz or tr is NULL");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  TransportArgs a{};
  a.ncol = ncol, a.n_layers = n_layers, a.ld = ld, a.ns = net->h.ns;
  a.n = n, a.T = T, a.n_gas = n_gas, a.D = D, a.mass = mass, a.alpha_T = alpha_T, a.mbar = mbar, a.grav = grav, a.dz = dz, a.tr = tr;
  const int64_t gx = (ncol + 127) / 128;
  int spb = net->h.ns;   // enough CTAs to fill the chip even for one atmosphere: split the species over blockIdx.y
  while (spb > 4 && gx * ((net->h.ns + spb - 1) / spb) < (int64_t)net->sm_count * 8) spb = (spb + 1) / 2;
  a.spb = spb;
  dim3 grid((unsigned)gx, (unsigned)((net->h.ns + spb - 1) / spb));
  {
    Timed tm(net, KID_TRANSPORT, s);
    k_transport<<<grid, 128, 0, s>>>(a);
  }
  XOD_CUDA(cudaGetLastError());
  return XOD_OK;
}

// ---------------------------------------------------------------------------- f4: pathway analyser

size_t xod_pathway_workspace_bytes(const xod_network *net, int64_t ncol) {
  if (!net || ncol < 0 || !net->h.path.enabled) return 0;
  return (size_t)2 * net->h.nr * (size_t)round_up(std::max<int64_t>(ncol, 1), 32) * sizeof(double) + 256;
}

xod_status xod_pathway(const xod_network *net, int64_t ncol, int64_t ld, const double *kf, const double *kr,
                       const double *n, int32_t source, double *dist, int32_t *pred, int32_t *via, void *workspace,
                       size_t workspace_bytes, void *stream) {
  xod_status st = check_common(net, ncol, ld);
  if (st != XOD_OK) return st;
  if (!net->h.path.enabled) return fail(XOD_ERR_INVALID_ARG, "the pathway tables do not fit (too many species or reactions)");
  if (source < 0 || source >= net->h.ns) return fail(XOD_ERR_INVALID_ARG, "source species out of range");
  if (ncol == 0) return XOD_OK;
  if (!n || !dist || !pred || !via) return fail(XOD_ERR_INVALID_ARG, "n, dist, pred or via is NULL");
  if (net->h.nr > 0 && (!kf || !kr)) return fail(XOD_ERR_INVALID_ARG, "kf or kr is NULL");
  if (!workspace || workspace_bytes < xod_pathway_workspace_bytes(net, ncol))
    return fail(XOD_ERR_WORKSPACE, "workspace NULL or smaller than xod_pathway_workspace_bytes");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  PathArgs a{};
  a.ncol = ncol, a.ld = ld, a.ldw = round_up(ncol, 32);
  a.kf = kf, a.kr = kr, a.n = n;
  a.w = reinterpret_cast<double *>((reinterpret_cast<uintptr_t>(workspace) + 255) & ~uintptr_t(255));
  a.dist = dist, a.pred = pred, a.via = via, a.source = source, a.ns = net->h.ns, a.nr = net->h.nr;
  a.ntiles = (int32_t)((ncol + kFW - 1) / kFW);
  if (net->h.nr > 0) {
    const int64_t gx = (ncol + 127) / 128;
    int rslice = net->h.nr;
    while (rslice > 16 && gx * ((net->h.nr + rslice - 1) / rslice) < (int64_t)net->sm_count * 8) rslice = (rslice + 1) / 2;
    dim3 grid((unsigned)gx, (unsigned)((net->h.nr + rslice - 1) / rslice));
    Timed tm(net, KID_PATH_WEIGHTS, s);
    k_path_weights<<<grid, 128, 0, s>>>(net->d, a, rslice);
    XOD_CUDA(cudaGetLastError());
  }
  {
    const unsigned grid = (unsigned)std::min<int64_t>(a.ntiles, net->sm_count);
    Timed tm(net, KID_PATHWAY, s);
    k_pathway<<<grid, kFWarps * 32, path_smem_bytes(net->h.ns), s>>>(net->pd, a);
    XOD_CUDA(cudaGetLastError());
  }
  return XOD_OK;
}

// ---------------------------------------------------------------------------- f4: equilibrium composition

xod_status xod_equilibrium(const xod_network *net, int64_t ncol, int64_t ld, const double *T, const double *P,
                           const double *b, int32_t max_iter, double tol, double *n, double *pi, int32_t *iters,
                           void *stream) {
  xod_status st = check_common(net, ncol, ld);
  if (st != XOD_OK) return st;
  if (net->h.ne <= 0 || net->h.ne > kEqMaxElem)
    return fail(XOD_ERR_INVALID_ARG, "xod_equilibrium supports 1 to 16 elements (including a charge column)");
  if (net->h.ns <= 0) return fail(XOD_ERR_INVALID_ARG, "the network has no species");
  if (ncol == 0) return XOD_OK;
  if (!T || !P || !b || !n) return fail(XOD_ERR_INVALID_ARG, "T, P, b or n is NULL");
  if (tol < 0 || tol != tol) return fail(XOD_ERR_INVALID_ARG, "tol must be >= 0 (0 selects the default 1e-13)");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  EquilArgs a{};
  a.ncol = ncol, a.ld = ld, a.T = T, a.P = P, a.b = b, a.n = n, a.pi = pi, a.iters = iters;
  a.max_iter = max_iter > 0 ? max_iter : 500;
  a.tol = tol > 0 ? tol : 1.0e-13;
  const size_t smem = (size_t)equil_smem_doubles(net->h.ne) * kEqThreads * sizeof(double);
  {
    Timed tm(net, KID_EQUILIBRIUM, s);
    k_equilibrium<<<(unsigned)((ncol + kEqThreads - 1) / kEqThreads), kEqThreads, smem, s>>>(net->ed, a);
  }
  XOD_CUDA(cudaGetLastError());
  return XOD_OK;
}

int64_t xod_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

xod_status xod_check_status(const xod_network *net) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  if (net->device < 0) return fail(XOD_ERR_CUDA, "network was created without a CUDA device");
  DeviceGuard guard(net->device);
  if (guard.err != cudaSuccess) return cuda_fail(guard.err, "cudaSetDevice");
  XOD_CUDA(cudaDeviceSynchronize());
#ifdef XOD_CHECK
  int line = 0, zero = 0;
  XOD_CUDA(cudaMemcpyFromSymbol(&line, g_xod_check_line, sizeof line));
  if (line != 0) {
    XOD_CUDA(cudaMemcpyToSymbol(g_xod_check_line, &zero, sizeof zero));
    return fail(XOD_ERR_CUDA, "XOD_CHECK: a table-derived index was out of range at kernel source line " + std::to_string(line));
  }
#endif
  return XOD_OK;
}

int32_t xod_build_has_checks(void) {
#ifdef XOD_CHECK
  return 1;
#else
  return 0;
#endif
}

xod_status xod_network_timing_read(xod_network *net, double *ms, int64_t *launches) {
  if (!net) return fail(XOD_ERR_INVALID_ARG, "net is NULL");
  TimingState &t = net->timing;
  for (int k = 0; k < KID_COUNT; ++k) {
    if (ms) ms[k] = 0;
    if (launches) launches[k] = 0;
  }
  if (t.used) XOD_CUDA(cudaEventSynchronize(static_cast<cudaEvent_t>(t.pool[t.used - 1])));
  for (size_t p = 0; p < t.kid.size(); ++p) {
    float f = 0;
    XOD_CUDA(cudaEventElapsedTime(&f, static_cast<cudaEvent_t>(t.pool[2 * p]), static_cast<cudaEvent_t>(t.pool[2 * p + 1])));
    if (ms) ms[t.kid[p]] += f;
    if (launches) ++launches[t.kid[p]];
  }
  t.used = 0;
  t.kid.clear();
  return XOD_OK;
}

xod_status xod_probe_fp64_peak(int cuda_device, int32_t iters, double *dfma_per_second) {
  if (!dfma_per_second || iters <= 0) return fail(XOD_ERR_INVALID_ARG, "bad probe arguments");
  DeviceGuard guard(cuda_device);
  if (guard.err != cudaSuccess) return cuda_fail(guard.err, "cudaSetDevice");
  int smc = 0;
  XOD_CUDA(cudaDeviceGetAttribute(&smc, cudaDevAttrMultiProcessorCount, cuda_device));
  const int blocks = smc * 8, threads = 256, inner = 4096;
  double *out = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  float ms = 0;
  cudaError_t e = cudaMalloc(&out, (size_t)blocks * threads * sizeof(double));
  if (e == cudaSuccess) e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  if (e == cudaSuccess) {
    k_probe_dfma<<<blocks, threads>>>(out, inner, 1.0000001, 0.9999999);  // warm-up
    e = cudaEventRecord(e0);
  }
  if (e == cudaSuccess) {
    for (int i = 0; i < iters; ++i) k_probe_dfma<<<blocks, threads>>>(out, inner, 1.0000001, 0.9999999);
    e = cudaEventRecord(e1);
  }
  if (e == cudaSuccess) e = cudaEventSynchronize(e1);
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (out) cudaFree(out);
  if (e != cudaSuccess) return cuda_fail(e, "xod_probe_fp64_peak");
  *dfma_per_second = (double)blocks * threads * 16.0 * inner * iters / (ms * 1e-3);
  return XOD_OK;
}

}  // extern "C"
