// jac_tiled.cuh -- k_jac_tiled: Jacobian values (a9) with each derivative evaluated once (sm_100a).
//
// jac[e = (i, j)][col] = sum_r nu_ir (d q_f,r / d n_j - d q_r,r / d n_j)     (BASELINE.json config 5)
// with d q / d n_j = m k n_j^(m-1) prod_{l != j} n_l^(m_l), never formed as q / n_j (reading Q2), and
// k_f, k_r, [M], J independent of n (reading J3).
//
// A CTA (kFWarps warps) owns a tile of kFW = 16 columns and a range of units (pack_jac.cpp).  Shared
// memory holds [row][16] fp64 rows of 128 bytes, as in k_fused:
//   n_s   [ns + 1]      number densities of the tile (+ a row of ones for absent factors)
//   acc_s [acc_rows]    accumulator rows of the current unit's entries
//   v_s   [2][chunk+1]  slot values k n[o1] n[o2] of the current / next chunk (+ a zero row)
//   meta_s[2][meta_cap] the row schedule of the current / next chunk (cp.async)
// Per chunk: phase A evaluates the chunk's slots (a lane group of 8 lanes x 2 columns per slot; k is
// read from global memory ONCE per slot, n from the tile); one __syncthreads; phase B is the scheduled
// row reduction of sched.cuh.  At the end of a unit the entries' accumulator rows are added in row order,
// written to jac[e][col0 .. col0+15] and zeroed.  Atomic-free, fixed order.
// HBM traffic per column: 8 B per slot (k) + 8 B per species (n) + 8 B per entry (jac): config 3 network
// 28 k slots, 594 species, 37 k entries.
#pragma once
#include <cuda_runtime.h>

#include "xod_internal.h"
#include <xod_cta.cuh>
#include "sched.cuh"

namespace xod {

struct JacArgs {
  int64_t ncol, ld;
  int64_t ldo;                 // row pitch of jac (= ld in the public call)
  const double *kf, *kr, *n;   // [n_reactions][ld] x 2 (USER order), [ns][ld]
  double *jac;                 // [nnz_jac][ldo]
  int32_t ntiles, nsplit;      // column tiles; CTAs a tile's chunks are split over (at unit boundaries)
  int32_t nr;                  // rows of kf / kr
  int64_t nnz;                 // rows of jac
};

__global__ void __launch_bounds__(kFWarps * 32, 1) k_jac_tiled(JacTiledDev f, int ns, JacArgs a) {
  unsigned char *smem_raw = cta_dyn_smem();
  double *n_s = reinterpret_cast<double *>(smem_raw);
  double *acc_s = n_s + (size_t)(ns + 1) * kFW;
  double *v_s = acc_s + (size_t)f.acc_rows * kFW;
  int4 *meta_s = reinterpret_cast<int4 *>(v_s + (size_t)2 * (f.chunk + 1) * kFW);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int grp = lane >> 3, l2 = (lane & 7) * 2;
  const int vrows = f.chunk + 1;

  for (int item = blockIdx.x; item < a.ntiles * a.nsplit; item += gridDim.x) {
    const int tile = item / a.nsplit, split = item - tile * a.nsplit;
    // chunk range of this split, cut at unit boundaries (a unit's accumulators live in one CTA)
    const int cut0 = (int)((int64_t)f.nchunk * split / a.nsplit), cut1 = (int)((int64_t)f.nchunk * (split + 1) / a.nsplit);
    const int k_begin = split == 0 ? 0 : __ldg(f.chunk_info + XOD_IDX(cut0, f.nchunk)).x;
    const int k_end = split + 1 == a.nsplit ? f.nchunk : __ldg(f.chunk_info + XOD_IDX(cut1, f.nchunk)).x;
    const int64_t col0 = (int64_t)tile * kFW;

    __syncthreads();  // the previous item's readers are done with shared memory
    {
      const int c = tid & (kFW - 1);
      const int64_t gc = min(col0 + c, a.ncol - 1);   // idle columns of a ragged tile reuse the last valid column
      if (col0 + kFW <= a.ncol && ((reinterpret_cast<uintptr_t>(a.n) | ((size_t)a.ld * sizeof(double))) & 15) == 0) {
        // a full tile whose rows are 16-byte aligned: two columns per copy
        for (int u = tid; u < ns * (kFW / 2); u += kFWarps * 32)
          cp_async16(n_s + u * 2, a.n + (size_t)(u >> 3) * a.ld + col0 + (u & 7) * 2);
      } else {
        for (int i = tid >> 4; i < ns; i += (kFWarps * 32) >> 4) cp_async8(n_s + i * kFW + c, a.n + (size_t)i * a.ld + gc);
      }
      for (int i = tid; i < f.acc_rows * kFW; i += kFWarps * 32) acc_s[i] = 0.0;
      if (tid < kFW) {
        n_s[ns * kFW + tid] = 1.0;
        v_s[(size_t)f.chunk * kFW + tid] = 0.0;
        v_s[(size_t)(vrows + f.chunk) * kFW + tid] = 0.0;
      }
    }
    cp_async_wait_all();
    __syncthreads();
    const int64_t gc0 = min(col0 + l2, a.ncol - 1), gc1 = min(col0 + l2 + 1, a.ncol - 1);
    const double *n_l = n_s + l2;

    for (int k = k_begin; k < k_end; ++k) {
      const int buf = (k - k_begin) & 1;
      double *vb = v_s + (size_t)buf * vrows * kFW;
      int4 *mb = meta_s + (size_t)buf * f.meta_cap;
      {
        const int m0 = __ldg(f.meta_ptr + k), m1 = __ldg(f.meta_ptr + k + 1);
        for (int u = m0 + tid; u < m1; u += kFWarps * 32) cp_async16(mb + XOD_IDX(u - m0, f.meta_cap), f.meta + u);
      }
      const int4 info = __ldg(f.chunk_info + k);   // first chunk of the unit, flush begin, flush end, slots used
      // ------------------------------------------------------------ phase A: slot values
      const int4 *sd = f.slots + (size_t)k * f.chunk;
#pragma unroll 1
      for (int s = warp * kFRxnPerWarp + grp; s - grp < info.w; s += kFPass) {
        const int4 d = __ldg(sd + XOD_IDX(s, f.chunk));   // padded to the chunk with dummies (k row 0, ones row)
        const double *kk = (d.x < 0 ? a.kr : a.kf) + (size_t)XOD_IDX(d.x & 0x7fffffff, a.nr) * a.ld;
        const double k0 = __ldg(kk + gc0), k1 = __ldg(kk + gc1);
        const double2 u = lds2(n_l + XOD_IDX(d.y, ns + 1) * kFW), w = lds2(n_l + XOD_IDX(d.z, ns + 1) * kFW);
        *reinterpret_cast<double2 *>(vb + (size_t)s * kFW + l2) = make_double2(k0 * u.x * w.x, k1 * u.y * w.y);
      }
      cp_async_wait_all();
      __syncthreads();
      // ------------------------------------------------------------ phase B: coef * value into the entries' rows
      sched_reduce(mb, vb, acc_s, warp, grp, l2, vrows, f.acc_rows, f.meta_cap);
      if (info.z > info.y) {   // last chunk of a unit: flush its entries (CTA-uniform branch)
        __syncthreads();
        const int c = tid & (kFW - 1);
        const bool valid = col0 + c < a.ncol;
        for (int fl = info.y + (tid >> 4); fl < info.z; fl += (kFWarps * 32) >> 4) {
          const int4 e = __ldg(f.flush + XOD_IDX(fl, f.n_flush));   // entry, first row, rows
          double *r = acc_s + (size_t)XOD_IDX(e.y, f.acc_rows) * kFW + c;
          (void)XOD_IDX(e.y + e.z - 1, f.acc_rows);
          double sum = r[0];
          r[0] = 0.0;
          for (int x = 1; x < e.z; ++x) sum += r[x * kFW], r[x * kFW] = 0.0;
          if (valid) a.jac[(size_t)XOD_IDX((int64_t)e.x, a.nnz) * a.ldo + col0 + c] = sum;
        }
        // no barrier needed here: the next chunk's phase B touches these rows only after its own barrier
      }
    }
  }
}

}  // namespace xod
