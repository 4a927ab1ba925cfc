// sched.cuh -- the scheduled, atomic-free row reduction shared by k_fused (production/loss, a8) and
// k_jac_tiled (Jacobian values, a9).
//
// A chunk's values v[r][16 columns] (net rates of progress, or Jacobian derivative slots) sit in
// shared memory as 128-byte rows.  The packer (build_chunk_schedule, pack_fused.cpp) cut the sums
//     acc[row][col] += sum_e coef_e * v[r_e][col]
// into row tasks of at most kFSegMax entries, no two tasks of a chunk sharing an accumulator row; four
// similar-length row tasks form a warp task whose entries are interleaved [step][lane group].  A lane
// group (8 lanes x 2 columns) owns one row task; a warp keeps two warp tasks in flight because the
// dependent chain header -> entry -> value -> FMA is the latency that matters, not the instruction
// count.  An entry is one 32-bit word: low 16 bits = value row, high 16 bits = the top half of the
// coefficient as an fp64 (small integers are exact there).  No atomics, fixed order: deterministic.
#pragma once
#include <cuda_runtime.h>

#include "xod_internal.h"
#include <xod_cta.cuh>

namespace xod {

__device__ __forceinline__ double2 lds2(const double *p) { return *reinterpret_cast<const double2 *>(p); }

// mb: the chunk's schedule blob in shared memory (header | tasks | entries); vb: the chunk's value rows
// (vrows of them, the last one all zero); acc_s: accumulator rows (n_acc of them); meta_cap: 16-byte
// units a blob may occupy (bounds of the -DXOD_CHECK build).
__device__ __forceinline__ void sched_reduce(const int4 *mb, const double *vb, double *acc_s, int warp, int grp, int l2,
                                             int vrows, int n_acc, int meta_cap) {
  const int *hdr = reinterpret_cast<const int *>(mb);
  const int max_tasks = meta_cap - kFMetaHdr / 4 + 1;
  const int t_begin = hdr[warp], t_end = XOD_IDX(hdr[warp + 1], max_tasks);
  const int n_tasks = XOD_IDX(hdr[kFWarps + 1], max_tasks);
  const unsigned *ent = reinterpret_cast<const unsigned *>(mb + kFMetaHdr / 4 + n_tasks) + grp;
  const int ent_words = (meta_cap - kFMetaHdr / 4 - n_tasks) * 4;  // words of the entry section (XOD_CHECK bound)
  (void)ent_words;
  const double *v_l = vb + l2;
  auto row_of = [&](const int4 &tk) {
    const unsigned rows = (grp & 2) ? (unsigned)tk.w : (unsigned)tk.z;
    return (int)((grp & 1) ? rows >> 16 : rows & 0xffffu);
  };
  auto add_row = [&](int row, double s0, double s1) {
    if (row != 0xffff) {
      double2 *dst = reinterpret_cast<double2 *>(acc_s + (size_t)XOD_IDX(row, n_acc) * kFW + l2);
      double2 cur = *dst;
      cur.x += s0, cur.y += s1;
      *dst = cur;
    }
  };
  // entry word `st` of the lane group's row task that starts at word `off` of the entry section
  auto entry = [&](int off, int st) { return ent[XOD_IDX(off + st * 4 + grp, ent_words) - grp]; };
  auto value = [&](unsigned x) { return lds2(v_l + XOD_IDX(x & 0xffffu, vrows) * kFW); };
  auto coef = [](unsigned x) { return __hiloint2double((int)(x & 0xffff0000u), 0); };
  int t = t_begin;
#pragma unroll 1
  for (; t + 1 < t_end; t += 2) {
    const int4 ta = mb[kFMetaHdr / 4 + t], tb = mb[kFMetaHdr / 4 + t + 1];
    double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
    const int nmin = min(ta.y, tb.y);
    int st = 0;
#pragma unroll 1
    for (; st < nmin; ++st) {
      const unsigned xa = entry(ta.x, st), xb = entry(tb.x, st);
      const double2 qa = value(xa), qc = value(xb);
      const double na = coef(xa), nb = coef(xb);
      a0 = fma(na, qa.x, a0), a1 = fma(na, qa.y, a1);
      b0 = fma(nb, qc.x, b0), b1 = fma(nb, qc.y, b1);
    }
#pragma unroll 1
    for (int s2 = st; s2 < ta.y; ++s2) {
      const unsigned xa = entry(ta.x, s2);
      const double2 qa = value(xa);
      const double na = coef(xa);
      a0 = fma(na, qa.x, a0), a1 = fma(na, qa.y, a1);
    }
#pragma unroll 1
    for (int s2 = st; s2 < tb.y; ++s2) {
      const unsigned xb = entry(tb.x, s2);
      const double2 qc = value(xb);
      const double nb = coef(xb);
      b0 = fma(nb, qc.x, b0), b1 = fma(nb, qc.y, b1);
    }
    add_row(row_of(ta), a0, a1);
    add_row(row_of(tb), b0, b1);
  }
  if (t < t_end) {
    const int4 ta = mb[kFMetaHdr / 4 + t];
    double a0 = 0.0, a1 = 0.0;
#pragma unroll 1
    for (int st = 0; st < ta.y; ++st) {
      const unsigned xa = entry(ta.x, st);
      const double2 qa = value(xa);
      const double na = coef(xa);
      a0 = fma(na, qa.x, a0), a1 = fma(na, qa.y, a1);
    }
    add_row(row_of(ta), a0, a1);
  }
}

}  // namespace xod
