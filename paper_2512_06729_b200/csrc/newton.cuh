// newton.cuh -- kernels of the batched implicit step, sm_100a.
//
// One Newton iteration of a backward-Euler step for every column at once:
//     (I - dt Jac(y)) delta = -(y - n_old - dt f(y)),      y <- y + delta
// f comes from xod_source, Jac from xod_jacobian; this file holds the linear algebra, one system of
// order n_species per column, all with the SAME pattern (pack_lu.cpp: minimum-degree order, filled
// pattern, update schedule), lanes = columns, values in [position][column] arrays:
//   k_newton_assemble  A = I - dt Jac scattered into the filled LU storage (fill = 0); rhs = -F permuted
//   k_lu_factor        LU without pivoting (the order is fixed by the pattern, as in DLSODES' sparse solver), blocks
//                      of rows at a time: CTA = 8 columns x 64 entry slices; the rows of a block sit in shared
//                      memory while the updates a_ij -= l_ik a_kj of each pivot k are shared by the threads and
//                      the pivot's U row is read once per block
//   k_lu_solve         forward / backward substitution, delta scattered back to species order, y += delta
// Atomic-free and deterministic.  Division by a zero pivot gives IEEE inf/NaN, not an error.
#pragma once
#include <cuda_runtime.h>

#include "xod_internal.h"
#include <xod_cta.cuh>

namespace xod {

struct NewtonArgs {
  int64_t ncol;        // columns of this chunk
  int64_t ld;          // pitch of the caller's arrays (n_old, y, delta, dt)
  int64_t ldw;         // pitch of the workspace arrays (f, jac, lu, rhs)
  const double *n_old, *dt, *f, *jac;
  double *y, *delta;   // delta may be NULL
  double *lu, *rhs;
  int64_t nnz_jac;
};

// grid (ceil(ncol / 128), position slices); thread = column
__global__ void __launch_bounds__(128) k_newton_assemble(LuDev u, NewtonArgs a) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= a.ncol) return;
  const double h = a.dt[c];
  for (int64_t x = blockIdx.y; x < u.nnz; x += gridDim.y) {
    const int32_t s = __ldg(u.src + x);
    double v = 0.0;   // fill
    if (s >= 0) {
      const double one = (s & kLuDiagBit) ? 1.0 : 0.0;
      v = fma(-h, a.jac[(size_t)XOD_IDX((int64_t)(s & ~kLuDiagBit), a.nnz_jac) * a.ldw + c], one);
    }
    a.lu[(size_t)x * a.ldw + c] = v;
  }
  for (int p = blockIdx.y; p < u.n; p += gridDim.y) {
    const size_t sp = (size_t)XOD_IDX(__ldg(u.perm + p), u.n);
    const double yv = a.y[sp * a.ld + c];
    a.rhs[(size_t)p * a.ldw + c] = -(yv - a.n_old[sp * a.ld + c] - h * a.f[sp * a.ldw + c]);
  }
}

// grid ceil(ncol / kLuCols); block 32 x kLuWarps = 64 entry slices x kLuCols columns; dynamic shared memory
// block_rows x max_row x kLuCols doubles.  Blocks of consecutive rows (pack_lu.cpp) are factorised together: the
// rows sit in shared memory as [slot][column] while the pivots of the union of their L parts are applied in
// ascending order, one barrier per pivot; the pivot's U row is read once (global memory, or the block's own rows
// when the pivot lies inside the block) and applied to every row of the block that holds a_ik.  On write-back the
// L part is stored as l_ik = a_ik / a_kk and the DIAGONAL AS ITS RECIPROCAL (so that neither later blocks nor
// k_lu_solve divide).  Idle column lanes of a ragged last CTA only take part in the barriers.
__global__ void __launch_bounds__(32 * kLuWarps) k_lu_factor(LuDev u, double *lu, int64_t ldw, int64_t ncol) {
  double *w = reinterpret_cast<double *>(cta_dyn_smem());
  const int c = threadIdx.x & (kLuCols - 1), es = threadIdx.x / kLuCols;
  constexpr int kSlices = 32 * kLuWarps / kLuCols;
  const int64_t gc = (int64_t)blockIdx.x * kLuCols + c;
  const bool valid = gc < ncol;
  double *col = lu + (valid ? gc : 0);
  double *wc = w + c;
  const int wslots = u.block_rows * u.max_row;
  (void)wslots;
  for (int bi = 0; bi < u.n_blocks; ++bi) {
    const LuBlock blk = u.blocks[bi];
    if (valid)
      for (int b = 0; b < blk.nrows; ++b) {
        const LuRow row = u.rows[XOD_IDX(blk.row0 + b, u.n)];
        for (int t = es; t < row.len; t += kSlices)
          wc[(size_t)XOD_IDX(b * u.max_row + t, wslots) * kLuCols] = col[(size_t)XOD_IDX((int64_t)row.begin + t, u.nnz) * ldw];
      }
    __syncthreads();
    for (int si = blk.step_begin; si < blk.step_end; ++si) {
      const LuStep st = u.steps[si];
      if (valid) {
        // a_ik of every item is final here: pivots below k have been applied (barrier), pivots >= k never touch it
        const double rd = st.src >= 0 ? 1.0 / wc[(size_t)XOD_IDX(st.src - 1, wslots) * kLuCols]
                                      : col[(size_t)XOD_IDX((int64_t)st.diag_k, u.nnz) * ldw];
        double l[kLuMaxBlockRows];
        int base[kLuMaxBlockRows];
        const uint16_t *tg[kLuMaxBlockRows];
#pragma unroll
        for (int x = 0; x < kLuMaxBlockRows; ++x) {
          l[x] = 0.0, base[x] = 0, tg[x] = u.tgt;
          if (x < st.n_items) {
            const LuItem item = u.items[st.item_begin + x];
            l[x] = wc[(size_t)XOD_IDX(item.slot_ik, wslots) * kLuCols] * rd;
            base[x] = item.base, tg[x] = u.tgt + item.tgt_off;
          }
        }
        const double *urow = col + (size_t)(st.diag_k + 1) * ldw;
        for (int jj = es; jj < st.cnt; jj += kSlices) {
          (void)XOD_IDX((int64_t)st.diag_k + 1 + jj, u.nnz);
          const double uv = st.src >= 0 ? wc[(size_t)XOD_IDX(st.src + jj, wslots) * kLuCols] : urow[(size_t)jj * ldw];
#pragma unroll
          for (int x = 0; x < kLuMaxBlockRows; ++x)
            if (x < st.n_items) {
              double *dst = wc + (size_t)XOD_IDX(base[x] + (int)tg[x][jj], wslots) * kLuCols;
              *dst = fma(-l[x], uv, *dst);
            }
        }
      }
      __syncthreads();
    }
    if (valid)
      for (int b = 0; b < blk.nrows; ++b) {
        const int i = blk.row0 + b;
        const LuRow row = u.rows[i];
        const int n_l = row.pair_end - row.pair_begin;
        for (int t = es; t < row.len; t += kSlices) {
          double v = wc[(size_t)(b * u.max_row + t) * kLuCols];
          if (t < n_l) {        // L part: l_ik = a_ik / a_kk; the pivot row is an earlier block's (reciprocal stored) or this block's
            const int k = XOD_IDX(__ldg(u.col + row.begin + t), u.n);
            const int dslot = __ldg(u.diag + k) - (int)__ldg(u.row_ptr + k);
            v *= k >= blk.row0 ? 1.0 / wc[(size_t)XOD_IDX((k - blk.row0) * u.max_row + dslot, wslots) * kLuCols]
                               : col[(size_t)__ldg(u.diag + k) * ldw];
          } else if (t == n_l) {
            v = 1.0 / v;        // the diagonal is stored as its reciprocal
          }
          col[(size_t)(row.begin + t) * ldw] = v;
        }
      }
    __syncthreads();   // the block is in global memory before later blocks read it; w may be overwritten
  }
}

// thread = column; rhs is overwritten by the permuted solution
__global__ void __launch_bounds__(128) k_lu_solve(LuDev u, NewtonArgs a) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= a.ncol) return;
  const double *lu = a.lu + c;
  double *x = a.rhs + c;
  for (int p = 0; p < u.n; ++p) {          // L z = b, unit diagonal
    double s = x[(size_t)p * a.ldw];
    const int64_t b = __ldg(u.row_ptr + p), d = __ldg(u.diag + p);
    for (int64_t e = b; e < d; ++e) s = fma(-lu[(size_t)e * a.ldw], x[(size_t)XOD_IDX(__ldg(u.col + e), u.n) * a.ldw], s);
    x[(size_t)p * a.ldw] = s;
  }
  for (int p = u.n - 1; p >= 0; --p) {     // U x = z
    double s = x[(size_t)p * a.ldw];
    const int64_t d = __ldg(u.diag + p), e1 = __ldg(u.row_ptr + p + 1);
    for (int64_t e = d + 1; e < e1; ++e) s = fma(-lu[(size_t)e * a.ldw], x[(size_t)XOD_IDX(__ldg(u.col + e), u.n) * a.ldw], s);
    x[(size_t)p * a.ldw] = s * lu[(size_t)d * a.ldw];   // k_lu_factor stores the reciprocal of the diagonal
  }
  for (int p = 0; p < u.n; ++p) {
    const size_t sp = (size_t)XOD_IDX(__ldg(u.perm + p), u.n);
    const double dv = x[(size_t)p * a.ldw];
    if (a.delta) a.delta[sp * a.ld + c] = dv;
    a.y[sp * a.ld + c] += dv;
  }
}

}  // namespace xod
