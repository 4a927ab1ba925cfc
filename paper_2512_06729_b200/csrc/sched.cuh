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
// units a blob may occupy (bounds of the -DXOD_CHECK build).  All three live in shared memory and are
// addressed by 32-bit shared-window addresses (xod_cta.cuh): a task descriptor is read as (entry offset,
// steps) plus the lane group's own 16-bit accumulator row, an entry as one word, a value row and an
// accumulator row as the thread's 16 bytes of a 128-byte row.
__device__ __forceinline__ void sched_reduce(const int4 *mb, const double *vb, double *acc_s, int warp, int grp, int l2,
                                             int vrows, int n_acc, int meta_cap) {
  const smem_addr hdr = smem_addr_of(mb);
  const int max_tasks = meta_cap - kFMetaHdr / 4 + 1;
  (void)max_tasks;
  const int t_begin = (int)lds_u32(hdr + 4 * warp), t_end = XOD_IDX((int)lds_u32(hdr + 4 * warp + 4), max_tasks);
  const int n_tasks = XOD_IDX((int)lds_u32(hdr + 4 * (kFWarps + 1)), max_tasks);
  const smem_addr tasks = hdr + 4 * kFMetaHdr;                 // 16 bytes per warp task
  const smem_addr ent = tasks + 16 * n_tasks + 4 * grp;        // the lane group's column of the entry section
  const int ent_words = (meta_cap - kFMetaHdr / 4 - n_tasks) * 4;  // words of the entry section (XOD_CHECK bound)
  (void)ent_words;
  smem_addr v_l = smem_addr_of(vb) + 8 * l2, acc_l = smem_addr_of(acc_s) + 8 * l2;
  smem_addr row_hw = 8 + 2 * grp;                              // the lane group's accumulator row inside a descriptor
  XOD_KEEP(v_l);                                               // loop invariants: keep them in registers
  XOD_KEEP(acc_l);
  XOD_KEEP(row_hw);
  auto add_row = [&](unsigned row, double s0, double s1) {
    if (row != 0xffffu) {
      const smem_addr dst = acc_l + ((smem_addr)XOD_IDX((int)row, n_acc) << 7);
      double2 cur = lds_d2(dst);
      cur.x += s0, cur.y += s1;
      sts_d2(dst, cur);
    }
  };
  // address of the first entry word of the lane group's row task whose entries start at word `off` of the entry
  // section; the following steps are 16 bytes apart (entries are interleaved [step][lane group])
  auto first = [&](int off, int nsteps) {
    (void)XOD_IDX(off + grp, ent_words), (void)XOD_IDX(off + grp + 4 * (nsteps > 0 ? nsteps - 1 : 0), ent_words);
    return ent + 4 * (smem_addr)off;
  };
  // value row of an entry: its low 16 bits are the row, a row is kFW doubles = 128 bytes
  auto value = [&](unsigned x) { return lds_d2(v_l + ((smem_addr)XOD_IDX((int)(x & 0xffffu), vrows) << 7)); };
  auto coef = [](unsigned x) { return __hiloint2double((int)(x & 0xffff0000u), 0); };
  smem_addr ta = tasks + 16 * (smem_addr)t_begin;
  const smem_addr ta_end = tasks + 16 * (smem_addr)t_end;
#pragma unroll 1
  for (; ta + 16 < ta_end; ta += 32) {   // two warp tasks in flight
    const int2 da = lds_i2(ta), db = lds_i2(ta + 16);
    const unsigned ra = lds_u16(ta + row_hw), rb = lds_u16(ta + 16 + row_hw);
    double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
    smem_addr pa = first(da.x, da.y), pb = first(db.x, db.y);
    const smem_addr pa_end = pa + 16 * (smem_addr)da.y, pb_end = pb + 16 * (smem_addr)db.y;
    const smem_addr pa_min = pa + 16 * (smem_addr)min(da.y, db.y);
#pragma unroll 1
    for (; pa != pa_min; pa += 16, pb += 16) {
      const unsigned xa = lds_u32(pa), xb = lds_u32(pb);
      const double2 qa = value(xa), qc = value(xb);
      const double na = coef(xa), nb = coef(xb);
      a0 = fma(na, qa.x, a0), a1 = fma(na, qa.y, a1);
      b0 = fma(nb, qc.x, b0), b1 = fma(nb, qc.y, b1);
    }
#pragma unroll 1
    for (; pa != pa_end; pa += 16) {
      const unsigned xa = lds_u32(pa);
      const double2 qa = value(xa);
      const double na = coef(xa);
      a0 = fma(na, qa.x, a0), a1 = fma(na, qa.y, a1);
    }
#pragma unroll 1
    for (; pb != pb_end; pb += 16) {
      const unsigned xb = lds_u32(pb);
      const double2 qc = value(xb);
      const double nb = coef(xb);
      b0 = fma(nb, qc.x, b0), b1 = fma(nb, qc.y, b1);
    }
    add_row(ra, a0, a1);
    add_row(rb, b0, b1);
  }
  if (ta < ta_end) {
    const int2 da = lds_i2(ta);
    const unsigned ra = lds_u16(ta + row_hw);
    double a0 = 0.0, a1 = 0.0;
    smem_addr pa = first(da.x, da.y);
    const smem_addr pa_end = pa + 16 * (smem_addr)da.y;
#pragma unroll 1
    for (; pa != pa_end; pa += 16) {
      const unsigned xa = lds_u32(pa);
      const double2 qa = value(xa);
      const double na = coef(xa);
      a0 = fma(na, qa.x, a0), a1 = fma(na, qa.y, a1);
    }
    add_row(ra, a0, a1);
  }
}

}  // namespace xod
