// newton.cuh -- kernels of the batched implicit step, sm_100a.
//
// One Newton iteration of a backward-Euler step for every column at once:
//     (I - dt Jac(y)) delta = -(y - n_old - dt f(y)),      y <- y + delta
// f comes from xod_source, Jac from xod_jacobian; this file holds the linear algebra, one system of
// order n_species per column, all with the SAME pattern (pack_lu.cpp: minimum-degree order, filled
// pattern, update schedule), lanes = columns, values in [position][column] arrays:
//   k_newton_assemble  A = I - dt Jac scattered into the filled LU storage (fill = 0); rhs = -F permuted
//   k_lu_factor        row-by-row LU without pivoting (the order is fixed by the pattern, as in DLSODES'
//                      sparse solver); CTA = 32 columns x kLuWarps warps; row i sits in shared memory
//                      while the warps share the updates a_ij -= l_ik a_kj of each pivot k in L(i)
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

// grid ceil(ncol / 32); block 32 x kLuWarps; dynamic shared memory max_row x 32 doubles
__global__ void __launch_bounds__(32 * kLuWarps) k_lu_factor(LuDev u, double *lu, int64_t ldw, int64_t ncol) {
  double *w = reinterpret_cast<double *>(cta_dyn_smem());
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t c = (int64_t)blockIdx.x * 32 + lane;
  const bool valid = c < ncol;   // idle lanes of a ragged group only take part in the barriers
  double *col = lu + (valid ? c : 0);
  for (int i = 0; i < u.n; ++i) {
    const LuRow row = u.rows[i];
    if (valid)
      for (int t = warp; t < row.len; t += kLuWarps)
        w[XOD_IDX(t, u.max_row) * 32 + lane] = col[(size_t)XOD_IDX((int64_t)row.begin + t, u.nnz) * ldw];
    __syncthreads();
    for (int pi = row.pair_begin; pi < row.pair_end; ++pi) {
      const LuPair pr = u.pairs[pi];
      if (valid) {
        // a_ik is final here: pivots k' < k have been applied (barrier below), pivots >= k never touch it
        const double l = w[XOD_IDX(pr.t_k, row.len) * 32 + lane] / col[(size_t)XOD_IDX((int64_t)pr.diag_k, u.nnz) * ldw];
        const double *urow = col + (size_t)(pr.diag_k + 1) * ldw;
        const uint16_t *tg = u.tgt + pr.tgt_off;
        for (int jj = warp; jj < pr.cnt; jj += kLuWarps) {
          (void)XOD_IDX((int64_t)pr.diag_k + 1 + jj, u.nnz);
          double *dst = w + XOD_IDX((int)tg[jj], row.len) * 32 + lane;
          *dst = fma(-l, urow[(size_t)jj * ldw], *dst);
        }
      }
      __syncthreads();
    }
    const int n_l = row.pair_end - row.pair_begin;   // the L part: store l_ik = a_ik / a_kk
    if (valid)
      for (int t = warp; t < row.len; t += kLuWarps) {
        double v = w[t * 32 + lane];
        if (t < n_l) v /= col[(size_t)u.pairs[row.pair_begin + t].diag_k * ldw];
        col[(size_t)(row.begin + t) * ldw] = v;
      }
    __syncthreads();   // row i is in global memory before later rows read it; w may be overwritten
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
    x[(size_t)p * a.ldw] = s / lu[(size_t)d * a.ldw];
  }
  for (int p = 0; p < u.n; ++p) {
    const size_t sp = (size_t)XOD_IDX(__ldg(u.perm + p), u.n);
    const double dv = x[(size_t)p * a.ldw];
    if (a.delta) a.delta[sp * a.ld + c] = dv;
    a.y[sp * a.ld + c] += dv;
  }
}

}  // namespace xod
