// pathway.cuh -- kernels of the reaction pathway analyser, sm_100a.
//
// "identifies the kinetically fastest reaction pathway by minimizing the cumulative sum of inverse reaction rates"
// (PAPER.md:318).  Per column: nodes = species, a directed edge u -> v of weight 1 / q for every reaction direction
// that consumes u and forms v (reading W1), single-source shortest paths from `source`.
//   k_path_weights   w[2 r + dir][col] = 1 / q (thread = column; q = k prod n as in a7; +inf where the direction has
//                    no positive finite rate), rows in USER reaction order
//   k_pathway        Bellman-Ford by destination ("pull"), which needs no priority queue and no atomics: a CTA owns a
//                    tile of 16 columns; two distance tiles [species][16] and a predecessor-edge tile live in shared
//                    memory; a round runs the packer's step schedule (pack_path.cpp): in a step every warp takes one
//                    part of one node's incoming edges, its four lane groups (8 lanes x 2 columns) every fourth edge,
//                    and keeps min (dist[u] + w) and the first edge that attains it; after a barrier the node's first
//                    warp combines the parts in part order and writes the next tile.  Rounds repeat until no distance
//                    changed (at most n_species).  Distances are unique; ties between equally short routes are broken
//                    by edge order (the oracle's Dijkstra may break them differently: tests compare dist and check that
//                    pred/via form a valid tight tree).
#pragma once
#include <cuda_runtime.h>

#include "xod_internal.h"
#include <xod_cta.cuh>

namespace xod {

struct PathArgs {
  int64_t ncol, ld, ldw;
  const double *kf, *kr, *n;   // [nr][ld] x 2 (USER order), [ns][ld]
  double *w;                   // [2 nr][ldw]
  double *dist;                // [ns][ld]
  int32_t *pred, *via;         // [ns][ld]
  int32_t source, ns, nr, ntiles;
};

// grid ceil(ncol / 128) x reaction slices; thread = column
__global__ void __launch_bounds__(128) k_path_weights(DevTables d, PathArgs a, int rslice) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= a.ncol) return;
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  const int p0 = blockIdx.y * rslice, p1 = min(d.nr, p0 + rslice);
  for (int p = p0; p < p1; ++p) {   // packed order; rows of w and k in USER order
    const int32_t *sp = d.sp + (size_t)p * 6;
    const size_t user = (size_t)XOD_IDX(__ldg(d.user + p), d.nr);
    double qf = a.kf[user * a.ld + c], qr = 0.0;
    for (int s = 0; s < 3; ++s) {
      const int i = __ldg(sp + s);
      if (i >= 0) qf *= a.n[(size_t)XOD_IDX(i, d.ns) * a.ld + c];
    }
    if (p < d.ph_begin && (__ldg(d.flags + p) & 1)) {
      qr = a.kr[user * a.ld + c];
      for (int s = 3; s < 6; ++s) {
        const int i = __ldg(sp + s);
        if (i >= 0) qr *= a.n[(size_t)XOD_IDX(i, d.ns) * a.ld + c];
      }
    }
    const double wf = 1.0 / qf, wr = 1.0 / qr;
    a.w[(2 * user) * a.ldw + c] = (qf > 0.0 && wf > 0.0 && wf < inf) ? wf : inf;
    a.w[(2 * user + 1) * a.ldw + c] = (qr > 0.0 && wr > 0.0 && wr < inf) ? wr : inf;
  }
}

// grid = column tiles (persistent loop); block kFWarps x 32; dynamic shared memory path_smem_bytes(ns)
__global__ void __launch_bounds__(kFWarps * 32, 1) k_pathway(PathDev f, PathArgs a) {
  unsigned char *smem_raw = cta_dyn_smem();
  const int ns = a.ns;
  double *dist_s = reinterpret_cast<double *>(smem_raw);                       // [2][ns][16]
  int32_t *pred_s = reinterpret_cast<int32_t *>(dist_s + (size_t)2 * ns * kFW);  // [ns][16] edge index or -1
  double *pmin_s = reinterpret_cast<double *>(pred_s + (size_t)ns * kFW);        // [kFWarps][4][16]
  int32_t *parg_s = reinterpret_cast<int32_t *>(pmin_s + (size_t)kFWarps * 4 * kFW);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, grp = lane >> 3, l2 = (lane & 7) * 2;
  const double inf = __longlong_as_double(0x7ff0000000000000LL);

  for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
    const int64_t col0 = (int64_t)tile * kFW;
    const int64_t gc0 = min(col0 + l2, a.ncol - 1), gc1 = min(col0 + l2 + 1, a.ncol - 1);   // idle columns repeat the last one
    __syncthreads();
    for (int i = tid; i < ns * kFW; i += kFWarps * 32) {
      const double v = (i / kFW == a.source) ? 0.0 : inf;
      dist_s[i] = v, dist_s[(size_t)ns * kFW + i] = v, pred_s[i] = -1;
    }
    __syncthreads();
    int cur = 0;
    for (int round = 0; round < ns; ++round) {
      const double *dc = dist_s + (size_t)cur * ns * kFW;
      double *dn = dist_s + (size_t)(cur ^ 1) * ns * kFW;
      bool ch = false;   // did this thread lower a distance in this round
      for (int step = 0; step < f.n_steps; ++step) {
        const PathTask t = f.sched[(size_t)step * kFWarps + warp];
        double m0 = inf, m1 = inf;
        int e0 = -1, e1 = -1;
        if (t.node >= 0) {
          for (int e = t.begin + grp; e < t.end; e += 4) {
            (void)XOD_IDX((int64_t)e, f.n_edges);
            const int u = XOD_IDX((int)__ldg(f.in_u + e), ns);
            const size_t rd = (size_t)XOD_IDX((int)__ldg(f.in_rd + e), 2 * a.nr);
            const double2 du = *reinterpret_cast<const double2 *>(dc + (size_t)u * kFW + l2);
            const double c0 = du.x + __ldg(a.w + rd * a.ldw + gc0), c1 = du.y + __ldg(a.w + rd * a.ldw + gc1);
            if (c0 < m0) m0 = c0, e0 = e;
            if (c1 < m1) m1 = c1, e1 = e;
          }
          double *pm = pmin_s + ((size_t)warp * 4 + grp) * kFW + l2;
          int32_t *pa = parg_s + ((size_t)warp * 4 + grp) * kFW + l2;
          pm[0] = m0, pm[1] = m1, pa[0] = e0, pa[1] = e1;
        }
        __syncthreads();
        if (t.node >= 0 && (t.first_warp_parts & 0xffff) == warp && grp == 0) {   // the node's first warp combines, part by part
          const int parts = t.first_warp_parts >> 16;
          const size_t o = (size_t)XOD_IDX(t.node, ns) * kFW + l2;
          double b0 = dc[o], b1 = dc[o + 1];
          int a0 = pred_s[o], a1 = pred_s[o + 1];
          for (int q = 0; q < parts * 4; ++q) {   // parts in warp order, lane groups in order: a fixed order, first minimum kept
            const size_t po = ((size_t)XOD_IDX(warp + q / 4, kFWarps) * 4 + (q & 3)) * kFW + l2;
            if (pmin_s[po] < b0) b0 = pmin_s[po], a0 = parg_s[po], ch = true;
            if (pmin_s[po + 1] < b1) b1 = pmin_s[po + 1], a1 = parg_s[po + 1], ch = true;
          }
          dn[o] = b0, dn[o + 1] = b1, pred_s[o] = a0, pred_s[o + 1] = a1;
        }
        __syncthreads();   // the partial minima may be overwritten; dn is complete after the last step
      }
      cur ^= 1;
      if (!__syncthreads_or(ch)) break;      // CTA-uniform: no distance changed anywhere in the tile
    }
    __syncthreads();
    const double *dfin = dist_s + (size_t)cur * ns * kFW;
    {
      const int c = tid & (kFW - 1);
      if (col0 + c < a.ncol)
        for (int i = tid >> 4; i < ns; i += (kFWarps * 32) >> 4) {
          const size_t o = (size_t)i * a.ld + col0 + c;
          a.dist[o] = dfin[i * kFW + c];
          const int e = pred_s[i * kFW + c];
          (void)XOD_IDX((int64_t)(e < 0 ? 0 : e), f.n_edges);
          a.pred[o] = e < 0 ? -1 : (int32_t)__ldg(f.in_u + e);
          const int rd = e < 0 ? 0 : (int)__ldg(f.in_rd + e);
          a.via[o] = e < 0 ? -1 : ((rd >> 1) | ((rd & 1) << 30));
        }
    }
  }
}

}  // namespace xod
