// pack_lu.cpp -- symbolic factorisation for the batched implicit step.
//
// The chemistry is a stiff ODE integrated implicitly; each Newton iteration of a
// backward-Euler / BDF step solves (I - gamma Jac) delta = -F with the SAME sparsity for every
// column, so the elimination order, the filled pattern and the whole update schedule are built once
// here, on the host, and shared by all columns (the kernels of newton.cuh only stream values).
//   * order: greedy minimum degree on the symmetric pattern of xod_network_jac_pattern (ties -> the
//     lowest species index), which keeps hub species (H, H2, OH-like) for last;
//   * pattern: the elimination graph with fill; row p = L part | diagonal | U part in permuted indices;
//   * schedule (row-by-row "up-looking" LU without pivoting, as DLSODES' sparse solver does): for row i
//     and every k in L(i) ascending,  l = a_ik / a_kk;  a_ij -= l a_kj for j in U(k);  the slots of
//     those j inside row i are precomputed (tgt);
//   * block schedule: consecutive rows are factorised together, as many as shared memory holds; the pivots of the
//     union of their L parts are applied in ascending order, so that a pivot's U row is read once per block and
//     not once per row (for a trailing block that is dense, that divides the traffic by the rows per block).
#include <algorithm>
#include <cstring>

#include "xod_internal.h"

namespace xod {

void pack_lu(HostTables &h) {
  LuHost &u = h.lu;
  u = LuHost();
  const int n = h.ns;
  if (n <= 0 || n >= 0xffff) return;
  // adjacency as a dense bit matrix (n <= 65534: at most 512 MB, the configs need 44 KB)
  const size_t W = ((size_t)n + 63) / 64;
  if ((double)W * n * 8 > 1.0e9) return;
  std::vector<uint64_t> adj(W * n, 0);
  auto set = [&](int a, int b) { adj[(size_t)a * W + (b >> 6)] |= 1ull << (b & 63); };
  auto get = [&](int a, int b) { return (adj[(size_t)a * W + (b >> 6)] >> (b & 63)) & 1ull; };
  auto clr = [&](int a, int b) { adj[(size_t)a * W + (b >> 6)] &= ~(1ull << (b & 63)); };
  for (int i = 0; i < n; ++i)
    for (int64_t e = h.jac_ptr[i]; e < h.jac_ptr[i + 1]; ++e) {
      const int j = h.jac_col[e];
      if (j != i) set(i, j), set(j, i);
    }
  std::vector<int> deg(n);
  for (int i = 0; i < n; ++i) {
    int d = 0;
    for (size_t w = 0; w < W; ++w) d += __builtin_popcountll(adj[(size_t)i * W + w]);
    deg[i] = d;
  }
  std::vector<char> alive(n, 1);
  u.perm.resize(n), u.pos_of.resize(n);
  std::vector<std::vector<int>> urow(n);  // U(p) as species indices, filled at elimination time
  for (int p = 0; p < n; ++p) {
    int best = -1;
    for (int i = 0; i < n; ++i)
      if (alive[i] && (best < 0 || deg[i] < deg[best])) best = i;
    u.perm[p] = best, u.pos_of[best] = p;
    alive[best] = 0;
    std::vector<int> &nb = urow[p];
    for (size_t w = 0; w < W; ++w) {
      uint64_t bits = adj[(size_t)best * W + w];
      while (bits) {
        const int b = __builtin_ctzll(bits);
        bits &= bits - 1;
        nb.push_back((int)(w * 64 + b));
      }
    }
    for (int a : nb) clr(a, best), --deg[a];
    for (size_t x = 0; x < nb.size(); ++x)
      for (size_t y = x + 1; y < nb.size(); ++y)
        if (!get(nb[x], nb[y])) set(nb[x], nb[y]), set(nb[y], nb[x]), ++deg[nb[x]], ++deg[nb[y]];
  }
  // rows in permuted indices: U(p) from the elimination, L(p) = {q < p : p in U(q)} by symmetry
  std::vector<std::vector<int>> U(n), L(n);
  for (int p = 0; p < n; ++p) {
    for (int s : urow[p]) U[p].push_back(u.pos_of[s]);
    std::sort(U[p].begin(), U[p].end());
    for (int q : U[p]) L[q].push_back(p);   // p ascending, so every L row comes out sorted
  }
  u.n = n;
  u.row_ptr.assign(n + 1, 0);
  u.diag.resize(n);
  for (int p = 0; p < n; ++p) {
    u.diag[p] = (int32_t)(u.row_ptr[p] + (int64_t)L[p].size());
    u.row_ptr[p + 1] = u.row_ptr[p] + (int64_t)L[p].size() + 1 + (int64_t)U[p].size();
    u.max_row = std::max<int32_t>(u.max_row, (int32_t)(u.row_ptr[p + 1] - u.row_ptr[p]));
  }
  u.nnz = u.row_ptr[n];
  if (u.nnz >= 0x7fffffff || u.max_row > 0xffff) {
    u = LuHost();
    return;
  }
  u.col.resize(u.nnz), u.src.assign(u.nnz, -1);
  for (int p = 0; p < n; ++p) {
    int64_t x = u.row_ptr[p];
    for (int q : L[p]) u.col[x++] = q;
    u.col[x++] = p;
    for (int q : U[p]) u.col[x++] = q;
  }
  // where the Jacobian entries land (the rest is fill)
  {
    std::vector<int32_t> slot(n, -1);   // permuted column -> storage position, for the current row
    for (int p = 0; p < n; ++p) {
      for (int64_t x = u.row_ptr[p]; x < u.row_ptr[p + 1]; ++x) slot[u.col[x]] = (int32_t)x;
      const int i = u.perm[p];
      for (int64_t e = h.jac_ptr[i]; e < h.jac_ptr[i + 1]; ++e)   // bit 30 marks the diagonal (the "I" of I - gamma Jac)
        u.src[slot[u.pos_of[h.jac_col[e]]]] = (int32_t)e | (h.jac_col[e] == i ? kLuDiagBit : 0);
      for (int64_t x = u.row_ptr[p]; x < u.row_ptr[p + 1]; ++x) slot[u.col[x]] = -1;
    }
  }
  // update schedule
  u.rows.resize(n);
  {
    std::vector<int32_t> slot(n, -1);   // permuted column -> slot inside row i
    for (int i = 0; i < n; ++i) {
      const int64_t b = u.row_ptr[i], len = u.row_ptr[i + 1] - b;
      for (int64_t x = 0; x < len; ++x) slot[u.col[b + x]] = (int32_t)x;
      LuRow r;
      r.begin = (int32_t)b, r.len = (int32_t)len, r.pair_begin = (int32_t)u.pairs.size();
      for (size_t a = 0; a < L[i].size(); ++a) {
        const int k = L[i][a];
        LuPair pr;
        pr.t_k = (int32_t)a, pr.diag_k = u.diag[k], pr.cnt = (int32_t)U[k].size(), pr.tgt_off = (int32_t)u.tgt.size();
        if (u.tgt.size() + U[k].size() >= 0x7fffffffu) {
          u = LuHost();
          return;
        }
        for (int j : U[k]) {
          if (slot[j] < 0) {   // cannot happen: (i, j) is in the filled pattern whenever k is in L(i) and j in U(k)
            u = LuHost();
            return;
          }
          u.tgt.push_back((uint16_t)slot[j]);
        }
        u.n_updates += pr.cnt;
        u.pairs.push_back(pr);
      }
      r.pair_end = (int32_t)u.pairs.size();
      u.rows[i] = r;
      for (int64_t x = 0; x < len; ++x) slot[u.col[b + x]] = -1;
    }
  }
  // block schedule: as many rows per block as shared memory holds (kLuCols columns of max_row slots each)
  u.block_rows = (int32_t)std::min<int64_t>(kLuMaxBlockRows, (int64_t)(227 * 1024) / ((int64_t)u.max_row * kLuCols * 8));
  if (u.block_rows < 1) {
    u = LuHost();
    return;
  }
  for (int row0 = 0; row0 < n; row0 += u.block_rows) {
    const int nrows = std::min(u.block_rows, n - row0);
    LuBlock blk;
    blk.row0 = row0, blk.nrows = nrows, blk.step_begin = (int32_t)u.steps.size();
    std::vector<size_t> cur(nrows);   // next pair of every row of the block (pairs ascend in k)
    for (int b = 0; b < nrows; ++b) cur[b] = (size_t)u.rows[row0 + b].pair_begin;
    for (;;) {
      int k = -1;
      for (int b = 0; b < nrows; ++b)
        if (cur[b] < (size_t)u.rows[row0 + b].pair_end) {
          const int kb = L[row0 + b][cur[b] - (size_t)u.rows[row0 + b].pair_begin];
          if (k < 0 || kb < k) k = kb;
        }
      if (k < 0) break;
      LuStep st;
      st.diag_k = u.diag[k], st.cnt = (int32_t)U[k].size(), st.item_begin = (int32_t)u.items.size(), st.n_items = 0, st.pad = 0;
      st.src = k >= row0 ? (k - row0) * u.max_row + (int32_t)(u.diag[k] - u.row_ptr[k]) + 1 : -1;
      for (int b = 0; b < nrows; ++b) {
        if (cur[b] >= (size_t)u.rows[row0 + b].pair_end) continue;
        const size_t a = cur[b] - (size_t)u.rows[row0 + b].pair_begin;
        if (L[row0 + b][a] != k) continue;
        const LuPair &pr = u.pairs[cur[b]];
        LuItem it2;
        it2.base = b * u.max_row, it2.slot_ik = it2.base + pr.t_k, it2.tgt_off = pr.tgt_off, it2.pad = 0;
        u.items.push_back(it2);
        ++st.n_items, ++cur[b];
      }
      u.n_block_loads += st.cnt;
      u.steps.push_back(st);
    }
    blk.step_end = (int32_t)u.steps.size();
    u.blocks.push_back(blk);
  }
  u.enabled = true;
}

}  // namespace xod

namespace xod {

// Host-only self-check of the implicit-step tables, decoding them exactly as the kernels of newton.cuh do:
//  * rows tile the value array; the diagonal sits after the L part; columns ascend; L(i) < i < U(i);
//  * every pair (i, k) names a slot of row i that holds column k, the diagonal of row k, |U(k)| targets, and every
//    target slot of row i holds the column of the matching entry of U(k);
//  * the block schedule covers the rows in order, at most block_rows at a time, within shared memory; every pair
//    of a block's rows appears exactly once as an item, under a step of its own pivot, steps ascending in the pivot;
//    a pivot inside the block is read from the shared slot right after that row's diagonal, a pivot before the
//    block from global memory.
bool check_lu(const HostTables &h, std::string &err) {
  const LuHost &u = h.lu;
  if (!u.enabled) return true;
  auto fail = [&](const std::string &m) { err = "LU tables: " + m; return false; };
  const int n = u.n;
  if ((int)u.rows.size() != n || (int)u.diag.size() != n || (int)u.row_ptr.size() != n + 1) return fail("sizes");
  std::vector<int32_t> row_of_diag(u.nnz, -1);
  for (int i = 0; i < n; ++i) {
    const LuRow &r = u.rows[i];
    if (r.begin != u.row_ptr[i] || r.len != u.row_ptr[i + 1] - u.row_ptr[i] || r.len > u.max_row) return fail("row range");
    const int n_l = r.pair_end - r.pair_begin;
    if (u.diag[i] != r.begin + n_l || u.col[u.diag[i]] != i) return fail("diagonal position");
    for (int t = 0; t < r.len; ++t) {
      const int c = u.col[r.begin + t];
      if (c < 0 || c >= n || (t > 0 && c <= u.col[r.begin + t - 1])) return fail("columns not ascending");
      if ((t < n_l) != (c < i)) return fail("L / U split");
    }
    row_of_diag[u.diag[i]] = i;
  }
  for (int i = 0; i < n; ++i) {
    const LuRow &r = u.rows[i];
    for (int p = r.pair_begin; p < r.pair_end; ++p) {
      const LuPair &pr = u.pairs[p];
      if (pr.t_k != p - r.pair_begin || pr.diag_k < 0 || pr.diag_k >= u.nnz || row_of_diag[pr.diag_k] < 0) return fail("pair");
      const int k = row_of_diag[pr.diag_k];
      if (u.col[r.begin + pr.t_k] != k) return fail("pair slot does not hold its pivot column");
      const int64_t ub = (int64_t)u.diag[k] + 1, ue = u.row_ptr[k + 1];
      if (pr.cnt != ue - ub || (int64_t)pr.tgt_off + pr.cnt > (int64_t)u.tgt.size()) return fail("pair count");
      for (int jj = 0; jj < pr.cnt; ++jj) {
        const int slot = u.tgt[(size_t)pr.tgt_off + jj];
        if (slot >= r.len || u.col[r.begin + slot] != u.col[ub + jj]) return fail("target slot holds another column");
      }
    }
  }
  if (u.block_rows < 1 || u.block_rows > kLuMaxBlockRows || (int64_t)u.block_rows * u.max_row * kLuCols * 8 > 227 * 1024)
    return fail("block rows");
  int next_row = 0;
  std::vector<char> seen(u.pairs.size(), 0);
  for (const LuBlock &b : u.blocks) {
    if (b.row0 != next_row || b.nrows < 1 || b.nrows > u.block_rows || b.row0 + b.nrows > n) return fail("block range");
    next_row += b.nrows;
    int last_k = -1;
    for (int si = b.step_begin; si < b.step_end; ++si) {
      const LuStep &st = u.steps[(size_t)si];
      if (st.diag_k < 0 || st.diag_k >= u.nnz || row_of_diag[st.diag_k] < 0) return fail("step pivot");
      const int k = row_of_diag[st.diag_k];
      if (k <= last_k) return fail("steps not ascending in the pivot");
      last_k = k;
      if (st.cnt != u.row_ptr[k + 1] - u.diag[k] - 1 || st.n_items < 1 || st.n_items > b.nrows) return fail("step");
      const int want_src = k >= b.row0 ? (k - b.row0) * u.max_row + (int)(u.diag[k] - u.row_ptr[k]) + 1 : -1;
      if (st.src != want_src || k >= b.row0 + b.nrows) return fail("step source");
      for (int x = 0; x < st.n_items; ++x) {
        const LuItem &it = u.items[(size_t)st.item_begin + x];
        if (it.base % u.max_row != 0) return fail("item base");
        const int brow = it.base / u.max_row;
        if (brow < 0 || brow >= b.nrows) return fail("item row");
        const int i = b.row0 + brow;
        if (i <= k) return fail("item row does not lie below its pivot");
        const LuRow &r = u.rows[i];
        const int t_k = it.slot_ik - it.base;
        if (t_k < 0 || t_k >= r.pair_end - r.pair_begin) return fail("item slot");
        const int p = r.pair_begin + t_k;
        if (u.pairs[p].diag_k != st.diag_k || u.pairs[p].tgt_off != it.tgt_off || seen[p]) return fail("item does not match its pair");
        seen[p] = 1;
      }
    }
  }
  if (next_row != n) return fail("blocks do not cover the rows");
  for (char c : seen)
    if (!c) return fail("a (row, pivot) pair is missing from the block schedule");
  return true;
}

}  // namespace xod
