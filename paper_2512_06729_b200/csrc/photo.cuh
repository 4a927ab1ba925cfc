// photo.cuh -- kernels of the photolysis rate constants, sm_100a.
//
//   kappa[b][col] = sum_x sigma_ext[x][b] n[abs_species[x]][col]              (extinction per unit length)
//   tau[b][col]   = sum over the layers above col of kappa dz + kappa dz / 2   (layer centre)
//   F[b][col]     = (J0[a][b] exp(-tau / mu_a) + J_diff[b][col]) dlambda_b
//   k_ph[p][col]  = t_f,a sum_b sigma_ph[p][b] F[b][col]
// The first and last lines are dense contractions over absorbers / over the 10 000 wavelength bins -- the one
// GEMM-shaped step near the path -- done here by a register-tiled fp64 DFMA kernel (k_photo_gemm, 64 x 64 x 16
// tiles, 4 x 4 outputs per thread, operands staged in shared memory).  fp64 tensor-core MMA has the same
// peak as the FP64 pipe on this part, so it would not raise the roofline; the contraction binds on the FP64 pipe
// either way.  The middle two lines are one kernel (k_photo_flux): a CTA takes 32 bins of one atmosphere, stages
// kappa in shared memory, 32 threads run the top-down prefix sums, all threads apply Beer-Lambert and write F
// over kappa in place.  Columns stay the contiguous dimension throughout.
#pragma once
#include <cuda_runtime.h>

#include "xod_internal.h"
#include "xod_math.cuh"
#include <xod_cta.cuh>

namespace xod {

constexpr int kGemmBM = 64, kGemmBN = 64, kGemmBK = 16;

struct GemmArgs {
  int64_t M, N, K;
  const double *A;
  int64_t lda;          // A_KMAJOR: A[m * lda + k]; else A[k * lda + m]
  const double *B;      // row k of B = B + (brow ? brow[k] : k) * ldb, N contiguous
  const int32_t *brow;
  int64_t ldb, n_brows; // n_brows: rows B may address (bound of the -DXOD_CHECK build)
  double *C;            // C[m * ldc + n]
  int64_t ldc;
  const double *scale_atm;  // optional: C *= scale_atm[n / n_layers]
  int64_t n_layers;
};

template <bool A_KMAJOR>
__global__ void __launch_bounds__(256) k_photo_gemm(GemmArgs g) {
  __shared__ double As[kGemmBK][kGemmBM + 1];
  __shared__ double Bs[kGemmBK][kGemmBN];
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int64_t m0 = (int64_t)blockIdx.y * kGemmBM, n0 = (int64_t)blockIdx.x * kGemmBN;
  double acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
  for (int64_t k0 = 0; k0 < g.K; k0 += kGemmBK) {
    // A tile: 64 x 16 values, 4 per thread along the contiguous direction of A
    if (A_KMAJOR) {
      const int m = tid >> 2, kq = (tid & 3) * 4;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int64_t gm = m0 + m, gk = k0 + kq + q;
        As[kq + q][m] = (gm < g.M && gk < g.K) ? g.A[gm * g.lda + gk] : 0.0;
      }
    } else {
      const int k = tid >> 4, mq = (tid & 15) * 4;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int64_t gm = m0 + mq + q, gk = k0 + k;
        As[k][mq + q] = (gm < g.M && gk < g.K) ? g.A[gk * g.lda + gm] : 0.0;
      }
    }
    {
      const int k = tid >> 4, nq = (tid & 15) * 4;
      const int64_t gk = k0 + k;
      const double *brow = nullptr;
      if (gk < g.K) brow = g.B + (size_t)XOD_IDX(g.brow ? (int64_t)g.brow[gk] : gk, g.n_brows) * g.ldb;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int64_t gn = n0 + nq + q;
        Bs[k][nq + q] = (brow && gn < g.N) ? brow[gn] : 0.0;
      }
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < kGemmBK; ++kk) {
      double a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t gm = m0 + ty * 4 + i;
    if (gm >= g.M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int64_t gn = n0 + tx * 4 + j;
      if (gn >= g.N) continue;
      const double s = g.scale_atm ? g.scale_atm[gn / g.n_layers] : 1.0;
      g.C[gm * g.ldc + gn] = s * acc[i][j];
    }
  }
}

struct FluxArgs {
  int64_t n_bins, n_atm, n_layers, ld, ldw;
  double *F;                 // in: kappa [n_bins][ldw]; out: F
  const double *dz;          // [ld]
  const double *j0;          // [n_atm][n_bins]
  const double *j_diff;      // [n_bins][ld] or NULL
  const double *mu;          // [n_atm]
  const double *dlambda;     // [n_bins]
};

// grid (ceil(n_bins / 32), n_atm); block 256; dynamic shared memory 32 x (n_layers | 1) doubles
__global__ void __launch_bounds__(256) k_photo_flux(FluxArgs f) {
  double *tile = reinterpret_cast<double *>(cta_dyn_smem());
  const int tid = threadIdx.x;
  const int64_t b0 = (int64_t)blockIdx.x * 32, a = blockIdx.y, L = f.n_layers, col0 = a * L;
  const int64_t Ls = L | 1;   // odd row pitch: the 32 scanning threads hit 32 different banks
  for (int64_t idx = tid; idx < 32 * L; idx += 256) {
    const int64_t bb = idx / L, k = idx - bb * L, b = b0 + bb;
    tile[bb * Ls + k] = b < f.n_bins ? f.F[b * f.ldw + col0 + k] : 0.0;
  }
  __syncthreads();
  if (tid < 32 && b0 + tid < f.n_bins) {
    double above = 0.0;   // optical depth of everything above the current layer
    for (int64_t k = L - 1; k >= 0; --k) {
      const double slab = tile[tid * Ls + k] * f.dz[col0 + k];
      tile[tid * Ls + k] = above + 0.5 * slab;
      above += slab;
    }
  }
  __syncthreads();
  const double c = -1.4426950408889634 / f.mu[a];   // exp(-tau/mu) = 2^(tau c)
  for (int64_t idx = tid; idx < 32 * L; idx += 256) {
    const int64_t bb = idx / L, k = idx - bb * L, b = b0 + bb;
    if (b >= f.n_bins) continue;
    double flux = f.j0[a * f.n_bins + b] * xexp2(tile[bb * Ls + k] * c);
    if (f.j_diff) flux += f.j_diff[b * f.ld + col0 + k];
    f.F[b * f.ldw + col0 + k] = flux * f.dlambda[b];
  }
}

}  // namespace xod
