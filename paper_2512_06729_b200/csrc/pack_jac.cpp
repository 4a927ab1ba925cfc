// pack_jac.cpp -- host tables of the tiled Jacobian kernel (k_jac_tiled in jac_tiled.cuh), step a9.
//
// jac[e = (i, j)] = sum_r nu_ir (d q_f,r / d n_j - d q_r,r / d n_j)   (BASELINE.json config 5; the
// rate-of-progress law is north_star's k prod n; nothing here depends on n through k, reading J3).
// The per-entry term lists of pack.cpp hold coef * k[dir][r] * n[o1] * n[o2]; the same product
// k n[o1] n[o2] ("slot") appears in up to six entries of one Jacobian column j (one per species i
// with nu_ir != 0).  This packer groups the terms by column j, so a slot is evaluated once per
// (column tile, slot) and k is read once per slot instead of once per term:
//   * unit  = a run of consecutive columns j whose slots fit one chunk, or one hub column with
//             several chunks; all terms of an entry lie inside its unit;
//   * chunk = up to `chunk` slots + the production/loss-style row schedule (build_chunk_schedule)
//             that sums coef * slot value into the accumulator rows of the unit's entries;
//   * flush = at the end of a unit, every entry's accumulator rows are added in row order and
//             written to jac[e][col].
#include <algorithm>
#include <array>
#include <cmath>
#include <cstring>
#include <map>
#include <tuple>

#include "xod_internal.h"

namespace xod {

size_t jac_tiled_smem_bytes(int ns, int acc_rows, int chunk, int meta_cap) {
  // n tile (+ ones row) | accumulator rows | two slot-value buffers (+ zero row each) | two chunk schedules
  return ((size_t)(ns + 1) + (size_t)acc_rows + 2 * (size_t)(chunk + 1)) * kFW * sizeof(double) + 2 * (size_t)meta_cap * 16;
}

void pack_jac_tiled(HostTables &h, int chunk, int acc_budget) {
  JacTiledHost &t = h.jt;
  t = JacTiledHost();
  const int ns = h.ns;
  const int64_t nnz = (int64_t)h.jac_col.size();
  if (chunk <= 0 || chunk % kFPass != 0 || chunk > 0xfffe || ns >= 0xffff || h.jac_terms.empty()) return;

  // ---- per Jacobian column j: its entries (ascending i), its slots, and each entry's (slot, coef) list
  struct Term { int32_t slot; float coef; };
  struct Col {
    std::vector<int64_t> entries;                                 // pattern entries e of this column
    std::vector<std::array<int32_t, 3>> slots;                    // rk, o1, o2
    std::vector<std::vector<Term>> terms;                         // per entry
  };
  std::vector<Col> cols(ns);
  for (int i = 0; i < ns; ++i)
    for (int64_t e = h.jac_ptr[i]; e < h.jac_ptr[i + 1]; ++e) cols[h.jac_col[e]].entries.push_back(e);
  for (int j = 0; j < ns; ++j) {
    Col &c = cols[j];
    std::map<std::tuple<int32_t, int32_t, int32_t>, int32_t> id;
    c.terms.resize(c.entries.size());
    for (size_t x = 0; x < c.entries.size(); ++x) {
      const int64_t e = c.entries[x];
      for (int64_t q = h.jac_term_ptr[e]; q < h.jac_term_ptr[e + 1]; ++q) {
        const JacTerm &jt = h.jac_terms[q];
        const auto key = std::make_tuple(jt.rk, jt.o1, jt.o2);
        auto it = id.find(key);
        if (it == id.end()) {
          it = id.emplace(key, (int32_t)c.slots.size()).first;
          c.slots.push_back({jt.rk, jt.o1 < 0 ? ns : jt.o1, jt.o2 < 0 ? ns : jt.o2});
        }
        c.terms[x].push_back({it->second, jt.coef});
      }
    }
  }

  // ---- units: consecutive columns while slots <= chunk and accumulator rows <= budget; a column with
  // more slots than a chunk is a unit of its own
  auto rows_of = [&](const Col &c) {   // accumulator rows if the column sits in ONE chunk
    int r = 0;
    for (const auto &tl : c.terms) r += std::max(1, ((int)tl.size() + kFSegMax - 1) / kFSegMax);
    return r;
  };
  struct Unit { int j0, j1; };
  std::vector<Unit> units;
  {
    int j = 0;
    while (j < ns) {
      if ((int)cols[j].slots.size() > chunk) {
        units.push_back({j, j + 1});
        ++j;
        continue;
      }
      int slots = 0, rows = 0, j1 = j;
      while (j1 < ns && (int)cols[j1].slots.size() <= chunk && slots + (int)cols[j1].slots.size() <= chunk &&
             rows + rows_of(cols[j1]) <= acc_budget) {
        slots += (int)cols[j1].slots.size();
        rows += rows_of(cols[j1]);
        ++j1;
      }
      if (j1 == j) return;  // a single column does not fit the accumulator budget: tiled path disabled
      units.push_back({j, j1});
      j = j1;
    }
  }
  t.n_units = (int32_t)units.size();

  const uint32_t zero_entry = (uint32_t)chunk;  // coefficient bits 0, the zero row of the value buffer
  auto enc = [](int slot_local, float coef) {
    const double c = (double)coef;
    uint64_t bits;
    std::memcpy(&bits, &c, 8);
    return (uint32_t)((bits >> 48) << 16) | (uint32_t)slot_local;
  };
  t.meta_ptr.assign(1, 0);
  t.chunk = chunk;
  for (const Unit &u : units) {
    // unit-local slot numbering: column by column; chunk = slot / chunk
    std::vector<int> base(u.j1 - u.j0 + 1, 0);
    for (int j = u.j0; j < u.j1; ++j) base[j - u.j0 + 1] = base[j - u.j0] + (int)cols[j].slots.size();
    const int nslots = base.back(), nck = std::max(1, (nslots + chunk - 1) / chunk);
    const int first_chunk = t.nchunk;
    // per entry, per chunk: encoded terms
    struct Ent { int64_t e; std::vector<std::vector<uint32_t>> per_chunk; int row0 = 0, rows = 1; };
    std::vector<Ent> ents;
    for (int j = u.j0; j < u.j1; ++j) {
      const Col &c = cols[j];
      for (size_t x = 0; x < c.entries.size(); ++x) {
        Ent en;
        en.e = c.entries[x];
        en.per_chunk.resize(nck);
        for (const Term &tm : c.terms[x]) {
          const int s = base[j - u.j0] + tm.slot;
          en.per_chunk[s / chunk].push_back(enc(s % chunk, tm.coef));
        }
        for (const auto &v : en.per_chunk) en.rows = std::max(en.rows, ((int)v.size() + kFSegMax - 1) / kFSegMax);
        ents.push_back(std::move(en));
      }
    }
    int rows = 0;
    for (Ent &en : ents) en.row0 = rows, rows += en.rows;
    if (rows > acc_budget || rows >= 0xffff) {
      t = JacTiledHost();
      return;
    }
    t.acc_rows = std::max(t.acc_rows, rows);
    const int flush_begin = (int)(t.flush.size() / 4);
    for (const Ent &en : ents) {
      t.flush.push_back((int32_t)en.e), t.flush.push_back(en.row0), t.flush.push_back(en.rows), t.flush.push_back(0);
    }
    const int flush_end = (int)(t.flush.size() / 4);
    for (int ck = 0; ck < nck; ++ck) {
      // slot descriptors of this chunk (padded with harmless dummies: k row 0 times the ones row)
      const int s0 = ck * chunk, s1 = std::min(nslots, s0 + chunk);
      for (int s = s0; s < s0 + chunk; ++s) {
        std::array<int32_t, 3> d = {0, ns, ns};
        if (s < s1) {
          const int jj = (int)(std::upper_bound(base.begin(), base.end(), s) - base.begin()) - 1;
          d = cols[u.j0 + jj].slots[s - base[jj]];
        }
        t.slots.push_back(d[0]), t.slots.push_back(d[1]), t.slots.push_back(d[2]), t.slots.push_back(0);
      }
      std::vector<SchedSeg> segs;
      for (const Ent &en : ents) {
        const auto &v = en.per_chunk[ck];
        const int len = (int)v.size(), nseg = (len + kFSegMax - 1) / kFSegMax;
        if (!len) continue;
        const int per = (len + nseg - 1) / nseg;
        for (int s = 0; s < nseg; ++s) {
          const int b = s * per, e2 = std::min(len, b + per);
          if (e2 > b) segs.push_back({en.row0 + s, v.data() + b, e2 - b});
        }
      }
      std::vector<int32_t> blob;
      int64_t nt = 0, nent = 0;
      build_chunk_schedule(segs, zero_entry, blob, nt, nent);
      t.n_tasks += nt, t.n_entries += nent;
      t.meta.insert(t.meta.end(), blob.begin(), blob.end());
      t.meta_ptr.push_back((int32_t)(t.meta.size() / 4));
      t.meta_cap = std::max<int32_t>(t.meta_cap, (int32_t)(blob.size() / 4));
      const bool last = ck == nck - 1;
      t.chunk_info.push_back(first_chunk), t.chunk_info.push_back(last ? flush_begin : 0);
      t.chunk_info.push_back(last ? flush_end : 0), t.chunk_info.push_back(s1 - s0);
      ++t.nchunk;
    }
    t.n_slots += nslots;
  }
  t.enabled = true;
}

// Host-only self-check, decoding the tables exactly as k_jac_tiled does: every term of pack.cpp's
// per-entry lists appears exactly once (same k row, same other species, same coefficient) under an
// accumulator row that is flushed into its own entry; every entry is flushed exactly once; no
// accumulator row is written by two row tasks of one chunk or owned by two entries of a unit.
bool check_jac_tiled(const HostTables &h, std::string &err) {
  const JacTiledHost &t = h.jt;
  if (!t.enabled) return true;
  auto fail = [&](const std::string &m) { err = "tiled Jacobian tables: " + m; return false; };
  const int ns = h.ns;
  const int64_t nnz = (int64_t)h.jac_col.size();
  using Key = std::tuple<int64_t, int32_t, int32_t, int32_t, int32_t>;  // entry, rk, o1, o2, coef
  std::vector<Key> want, got;
  for (int64_t e = 0; e < nnz; ++e)
    for (int64_t q = h.jac_term_ptr[e]; q < h.jac_term_ptr[e + 1]; ++q) {
      const JacTerm &jt = h.jac_terms[q];
      want.emplace_back(e, jt.rk, jt.o1 < 0 ? ns : jt.o1, jt.o2 < 0 ? ns : jt.o2, (int32_t)jt.coef);
    }
  std::vector<char> flushed(nnz, 0);
  if ((int)t.meta_ptr.size() != t.nchunk + 1 || (int)t.chunk_info.size() != 4 * t.nchunk ||
      (int64_t)t.slots.size() != (int64_t)4 * t.nchunk * t.chunk)
    return fail("table sizes");
  std::vector<int64_t> row_entry;  // accumulator row -> entry, for the current unit
  for (int k = 0; k < t.nchunk; ++k) {
    const int32_t *ci = &t.chunk_info[(size_t)4 * k];
    const int first = ci[0];
    if (first < 0 || first > k) return fail("bad first chunk of unit");
    if (first == k) {
      // the unit's flush list sits on its last chunk: find it
      int last = k;
      while (last + 1 < t.nchunk && t.chunk_info[(size_t)4 * (last + 1)] == first) ++last;
      const int fb = t.chunk_info[(size_t)4 * last + 1], fe = t.chunk_info[(size_t)4 * last + 2];
      if (fb < 0 || fe < fb || (size_t)fe * 4 > t.flush.size()) return fail("bad flush range");
      row_entry.assign(t.acc_rows, -1);
      for (int f = fb; f < fe; ++f) {
        const int64_t e = t.flush[(size_t)4 * f];
        const int r0 = t.flush[(size_t)4 * f + 1], nr = t.flush[(size_t)4 * f + 2];
        if (e < 0 || e >= nnz || flushed[e]) return fail("entry flushed twice or out of range");
        flushed[e] = 1;
        if (r0 < 0 || nr < 1 || r0 + nr > t.acc_rows) return fail("flush rows out of range");
        for (int r = r0; r < r0 + nr; ++r) {
          if (row_entry[r] >= 0) return fail("accumulator row owned by two entries");
          row_entry[r] = e;
        }
      }
    }
    if ((ci[1] != 0 || ci[2] != 0) && k + 1 < t.nchunk && t.chunk_info[(size_t)4 * (k + 1)] == first)
      return fail("flush on a chunk that is not the unit's last");
    const int32_t *blob = &t.meta[(size_t)t.meta_ptr[k] * 4];
    const int64_t blob_words = ((int64_t)t.meta_ptr[k + 1] - t.meta_ptr[k]) * 4;
    if (blob_words / 4 > t.meta_cap) return fail("schedule larger than meta_cap");
    const int nt = blob[kFWarps + 1];
    if (blob[0] != 0 || blob[kFWarps] != nt) return fail("bad warp offsets");
    const int32_t *tasks = blob + kFMetaHdr, *ent = tasks + 4 * nt;
    const int64_t nent = blob_words - kFMetaHdr - 4 * nt;
    std::vector<char> row_used(t.acc_rows, 0);
    for (int w = 0; w < kFWarps; ++w) {
      if (blob[w] > blob[w + 1]) return fail("warp offsets not monotone");
      for (int q = blob[w]; q < blob[w + 1]; ++q) {
        const int32_t off = tasks[4 * q], nsteps = tasks[4 * q + 1];
        if (off < 0 || nsteps < 0 || nsteps > kFSegMax || (int64_t)off + 4 * nsteps > nent) return fail("task out of range");
        for (int g = 0; g < 4; ++g) {
          const uint32_t rows = (uint32_t)tasks[4 * q + 2 + (g >> 1)];
          const int row = (g & 1) ? rows >> 16 : rows & 0xffffu;
          for (int st = 0; st < nsteps; ++st) {
            const uint32_t en = (uint32_t)ent[off + st * 4 + g];
            const int sl = en & 0xffffu;
            uint64_t bits = (uint64_t)(en & 0xffff0000u) << 32;
            double coef;
            std::memcpy(&coef, &bits, 8);
            if (sl > t.chunk) return fail("value row beyond the chunk");
            if (sl == t.chunk) {
              if (coef != 0.0) return fail("padding entry with nonzero coefficient");
              continue;
            }
            if (row == 0xffff || row >= t.acc_rows || row_entry[row] < 0) return fail("entry under an idle or unowned row");
            if (sl >= ci[3]) return fail("entry refers to an unused slot");
            if (coef != std::floor(coef) || coef == 0.0 || std::fabs(coef) > 9) return fail("bad coefficient encoding");
            const int32_t *d = &t.slots[((size_t)k * t.chunk + sl) * 4];
            got.emplace_back(row_entry[row], d[0], d[1], d[2], (int32_t)coef);
          }
          if (row != 0xffff) {
            if (row >= t.acc_rows) return fail("accumulator row out of range");
            if (row_used[row]) return fail("accumulator row written by two row tasks of one chunk");
            row_used[row] = 1;
          }
        }
      }
    }
    for (int s = 0; s < t.chunk; ++s) {
      const int32_t *d = &t.slots[((size_t)k * t.chunk + s) * 4];
      if ((d[0] & 0x7fffffff) >= std::max(h.nr, 1) || d[1] < 0 || d[1] > ns || d[2] < 0 || d[2] > ns) return fail("slot descriptor out of range");
    }
  }
  for (int64_t e = 0; e < nnz; ++e)
    if (!flushed[e]) return fail("entry never flushed");
  std::sort(want.begin(), want.end());
  std::sort(got.begin(), got.end());
  if (want != got) return fail("scheduled terms differ from the per-entry term lists");
  return true;
}

}  // namespace xod
