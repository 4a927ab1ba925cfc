// pack_path.cpp -- host tables of the reaction pathway analyser.
//
// The analyser finds, per column, the route from a source species to every other species that minimises the
// cumulative sum of inverse reaction rates.  Graph (reading W1): a directed edge from every distinct
// species a reaction direction consumes to every distinct species it forms, u != v, weight 1 / q of that direction.
// The kernel relaxes edges by destination (atomic-free: one owner per node), so this packer builds the
// incoming-edge list of every species (reactions in ascending USER order, forward before reverse) and a step
// schedule for one CTA: nodes with many incoming edges (hub species) are cut into parts that run on consecutive
// warps of one step and are combined in part order.
#include <algorithm>

#include "xod_internal.h"

namespace xod {

size_t path_smem_bytes(int ns) {
  // two distance tiles | predecessor edge per (node, column) | partial minima and their edges of one step
  return (size_t)2 * ns * kFW * sizeof(double) + (size_t)ns * kFW * sizeof(int32_t) +
         (size_t)kFWarps * 4 * kFW * (sizeof(double) + sizeof(int32_t));
}

void pack_path(const xod_network_desc *d, HostTables &h) {
  PathHost &p = h.path;
  p = PathHost();
  const int ns = h.ns, nr = h.nr;
  if (ns >= 0xffff || 2 * (int64_t)nr >= 0xffff) return;
  struct E { int32_t v; uint16_t u, rd; };
  std::vector<E> edges;
  for (int r = 0; r < nr; ++r)
    for (int dir = 0; dir < 2; ++dir) {
      if (dir == 1 && (!d->reversible[r] || d->type[r] == XOD_PHOTO)) continue;
      const int32_t *from = (dir ? d->products : d->reactants) + 3 * r, *to = (dir ? d->reactants : d->products) + 3 * r;
      for (int a = 0; a < 3; ++a) {
        if (from[a] < 0 || std::find(from, from + a, from[a]) != from + a) continue;   // each distinct species once
        for (int b = 0; b < 3; ++b) {
          if (to[b] < 0 || to[b] == from[a] || std::find(to, to + b, to[b]) != to + b) continue;
          edges.push_back({to[b], (uint16_t)from[a], (uint16_t)(2 * r + dir)});
        }
      }
    }
  std::stable_sort(edges.begin(), edges.end(), [](const E &a, const E &b) { return a.v < b.v; });
  p.n_edges = (int64_t)edges.size();
  if (p.n_edges >= 0x7fffffff) return;
  p.in_ptr.assign(ns + 1, 0);
  for (const E &e : edges) ++p.in_ptr[e.v + 1];
  for (int i = 0; i < ns; ++i) p.in_ptr[i + 1] += p.in_ptr[i];
  p.in_u.resize(edges.size()), p.in_rd.resize(edges.size());
  for (size_t k = 0; k < edges.size(); ++k) p.in_u[k] = edges[k].u, p.in_rd[k] = edges[k].rd;

  // parts: at most kFWarps per node, about 256 edges each; every node gets at least one (possibly empty) part so
  // that its distance is carried into the next buffer every round
  struct Node { int v, parts; int64_t per; };
  std::vector<Node> nodes;
  for (int v = 0; v < ns; ++v) {
    const int64_t deg = p.in_ptr[v + 1] - p.in_ptr[v];
    const int parts = (int)std::max<int64_t>(1, std::min<int64_t>(kFWarps, (deg + 255) / 256));
    nodes.push_back({v, parts, (deg + parts - 1) / parts});
  }
  std::stable_sort(nodes.begin(), nodes.end(), [](const Node &a, const Node &b) { return a.per > b.per; });
  std::vector<int> used;   // warp slots used per step
  for (const Node &nd : nodes) {
    int step = -1;
    for (size_t s = 0; s < used.size(); ++s)   // first fit; steps are filled with parts of similar length (sorted)
      if (used[s] + nd.parts <= kFWarps) { step = (int)s; break; }
    if (step < 0) {
      step = (int)used.size();
      used.push_back(0);
      p.sched.resize((size_t)(step + 1) * kFWarps, PathTask{-1, 0, 0, 0});
    }
    const int w0 = used[step];
    const int64_t b = p.in_ptr[nd.v], e = p.in_ptr[nd.v + 1];
    for (int q = 0; q < nd.parts; ++q) {
      PathTask t;
      t.node = nd.v;
      t.begin = (int32_t)std::min(e, b + q * nd.per), t.end = (int32_t)std::min(e, b + (q + 1) * nd.per);
      t.first_warp_parts = w0 | (nd.parts << 16);
      p.sched[(size_t)step * kFWarps + w0 + q] = t;
    }
    used[step] += nd.parts;
  }
  p.n_steps = (int32_t)used.size();
  p.enabled = true;
}

}  // namespace xod
