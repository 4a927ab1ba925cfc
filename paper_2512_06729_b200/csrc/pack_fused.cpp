// pack_fused.cpp -- host tables of the single-kernel fused source path (k_fused in kernels.cuh).
//
// (1) Reverse coefficients without per-species gathers.  With u_i(T) the scaled NASA-7 Gibbs
//     polynomial of species i (pack.cpp), detailed balance (Eq. 15)
//     gives  log2 k_r = log2 k_f + sum_products u_i - sum_reactants u_i.  Every u_i is piecewise
//     in T (low/high set at t_mid,i), so between two consecutive values of the sorted distinct
//     t_mid list ("breakpoints") the right-hand side is ONE seven-coefficient expression per
//     reaction:  log2 k_r = C0 + C1 log2 T + C2/T - T (D2 + T (D3 + T (D4 + T D5))).
//     The packer sums the coefficients in long double per (interval, reaction).
// (2) Production/loss schedule.  Reactions are processed in chunks; a chunk's net rates q sit
//     in shared memory and are summed into per-species accumulator rows by "row tasks" of at
//     most kFSegMax entries.  A species with more entries in one chunk gets extra accumulator
//     rows (combined in a fixed order at the end), so no two tasks of a chunk ever touch the
//     same row: atomic-free and deterministic (north_star).
#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

#include "xod_internal.h"

namespace xod {

namespace {
constexpr long double kLog2e = 1.442695040888963407359924681001892137L;
constexpr long double kBoltz = 1.380649e-16L;
constexpr long double kPref = 1.0e6L;

// b-coefficients of u_i = b0 - b1 log2 T - T (b2 + T (b3 + T (b4 + T b5))) + b6 / T  (pack.cpp)
void scaled_nasa(const double *a, long double b[7]) {
  const long double lpk = std::log2(kPref / kBoltz);
  b[0] = ((long double)a[0] - (long double)a[6]) * kLog2e - lpk;
  b[1] = (long double)a[0] - 1.0L;
  b[2] = (long double)a[1] * kLog2e / 2;
  b[3] = (long double)a[2] * kLog2e / 6;
  b[4] = (long double)a[3] * kLog2e / 12;
  b[5] = (long double)a[4] * kLog2e / 20;
  b[6] = (long double)a[5] * kLog2e;
}
}  // namespace

size_t fused_smem_bytes(int ns, int n_acc, int chunk, int meta_cap) {
  // n tile (+ ones row, zeros row) | accumulator rows | two q buffers (+ zero row each) | two chunk
  // schedules | column scalars
  return ((size_t)(ns + 2) + (size_t)n_acc + 2 * (size_t)(chunk + 1)) * kFW * sizeof(double) +
         2 * (size_t)meta_cap * 16 + (size_t)kFW * (4 * sizeof(double) + sizeof(int32_t));
}

// The production/loss schedule of one chunk (shared by k_fused and k_jac_tiled): row tasks (an
// accumulator row and <= kFSegMax entries) are sorted by length, four similar-length ones form a
// warp task whose entries are interleaved [step][lane group], and warp tasks are dealt to the
// least-loaded warp, longest first.  blob = header (kFWarps + 1 task offsets, task count, two
// spare words) | tasks | entries, in 16-byte units.
void build_chunk_schedule(std::vector<SchedSeg> segs, uint32_t zero_entry, std::vector<int32_t> &blob,
                          int64_t &n_tasks, int64_t &n_entries) {
  std::stable_sort(segs.begin(), segs.end(), [](const SchedSeg &a, const SchedSeg &b) { return a.len > b.len; });
  std::vector<std::vector<FusedTask>> per_warp(kFWarps);
  std::vector<int> load(kFWarps, 0);
  std::vector<uint32_t> entries;
  for (size_t s0 = 0; s0 < segs.size(); s0 += 4) {
    const int cnt = (int)std::min<size_t>(4, segs.size() - s0), nsteps = segs[s0].len;
    FusedTask t;
    t.entry_off = (int32_t)entries.size();
    t.nsteps = nsteps;
    uint32_t r[4] = {0xffffu, 0xffffu, 0xffffu, 0xffffu};
    for (int g = 0; g < cnt; ++g) r[g] = (uint32_t)segs[s0 + g].row;
    t.rows01 = (int32_t)(r[0] | (r[1] << 16));
    t.rows23 = (int32_t)(r[2] | (r[3] << 16));
    for (int st = 0; st < nsteps; ++st)
      for (int g = 0; g < 4; ++g)
        entries.push_back(g < cnt && st < segs[s0 + g].len ? segs[s0 + g].ent[st] : zero_entry);
    const int w = (int)(std::min_element(load.begin(), load.end()) - load.begin());
    load[w] += nsteps + 2;
    per_warp[w].push_back(t);
  }
  blob.assign(kFMetaHdr, 0);
  int nt = 0;
  for (int w = 0; w < kFWarps; ++w) {
    blob[w] = nt;
    nt += (int)per_warp[w].size();
  }
  blob[kFWarps] = nt, blob[kFWarps + 1] = nt;
  for (int w = 0; w < kFWarps; ++w)
    for (const FusedTask &t : per_warp[w]) {
      blob.push_back(t.entry_off), blob.push_back(t.nsteps), blob.push_back(t.rows01), blob.push_back(t.rows23);
    }
  for (uint32_t e : entries) blob.push_back((int32_t)e);
  while (blob.size() % 4) blob.push_back((int32_t)zero_entry);
  n_tasks = nt, n_entries = (int64_t)entries.size();
}

void pack_fused(const xod_network_desc *d, HostTables &h, int chunk) {
  FusedHost &f = h.f;
  f = FusedHost();
  const int ns = h.ns, nr = h.nr;
  if (nr == 0 || chunk <= 0 || chunk % kFPass != 0 || chunk > 0xfffe) return;

  // ---- breakpoints: sorted distinct t_mid.  Interval g of a column = #{bp < T}; species i with
  // t_mid,i = bp[k] uses its low set iff T <= bp[k] iff g <= k  (reading T3).
  f.bp.assign(h.tmid.begin(), h.tmid.end());
  std::sort(f.bp.begin(), f.bp.end());
  f.bp.erase(std::unique(f.bp.begin(), f.bp.end()), f.bp.end());
  f.n_bp = (int32_t)f.bp.size();
  if (f.n_bp + 1 > kFMaxIntervals || ns >= 0xffff) return;
  std::vector<int> bp_of(ns);
  for (int i = 0; i < ns; ++i)
    bp_of[i] = (int)(std::lower_bound(f.bp.begin(), f.bp.end(), h.tmid[i]) - f.bp.begin());

  // ---- padded packed order
  auto pad = [](int x, int m) { return (x + m - 1) / m * m; };
  const int n_arr = h.fo_begin, n_fo = h.ph_begin - h.fo_begin, n_ph = nr - h.ph_begin;
  f.arr_end = pad(n_arr, kFRxnPerWarp);
  f.fo_end = f.arr_end + pad(n_fo, kFRxnPerWarp);
  f.ph_end = f.fo_end + pad(n_ph, kFRxnPerWarp);
  f.npad = pad(f.ph_end, chunk);
  f.chunk = chunk;
  f.nchunk = f.npad / chunk;
  f.pp_to_packed.assign(f.npad, -1);
  for (int p = 0; p < n_arr; ++p) f.pp_to_packed[p] = p;
  for (int p = 0; p < n_fo; ++p) f.pp_to_packed[f.arr_end + p] = h.fo_begin + p;
  for (int p = 0; p < n_ph; ++p) f.pp_to_packed[f.fo_end + p] = h.ph_begin + p;
  f.pp_user.assign(f.npad, -1);
  for (int pp = 0; pp < f.npad; ++pp)
    if (f.pp_to_packed[pp] >= 0) f.pp_user[pp] = h.packed_to_user[f.pp_to_packed[pp]];
  std::vector<int32_t> packed_to_pp(nr);
  for (int pp = 0; pp < f.npad; ++pp)
    if (f.pp_to_packed[pp] >= 0) packed_to_pp[f.pp_to_packed[pp]] = pp;

  // ---- parameter blocks [interval][group], see xod_internal.h
  //   reverse coefficients, per interval (seven numbers per reaction):
  //   UNI/BI : C0 = c0 + dB0, C1 = c1 - dB1, C2 = c2 + dB6   (k_f folded in: one exp2 gives k_r)
  //   FALLOFF: C0 = dB0, C1 = -dB1, C2 = dB6                 (pure z; added to log2 k_f in the kernel)
  //   irreversible: all seven 0 (k_r = 1 or k_f, finite) and the first product slot points at the zeros row of
  //   the n tile, so q_r = 0 exactly without a special case on the kernel's fast path; k_rate_coeffs, which
  //   stores k_r itself, selects 0 by the reversible flag (word 3 of unit 1).  Padding slots: all 0, ones rows.
  const int ng = f.n_bp + 1;
  const int64_t n_arr_g = f.arr_end / kFRxnPerWarp, n_fo_g = (f.fo_end - f.arr_end) / kFRxnPerWarp,
                n_ph_g = (f.ph_end - f.fo_end) / kFRxnPerWarp;
  f.blk_fo_off = n_arr_g * kFBlkArr;
  f.blk_ph_off = f.blk_fo_off + n_fo_g * kFBlkFo;
  f.blk_stride = f.blk_ph_off + n_ph_g * kFBlkPh;
  f.blk.assign((size_t)ng * f.blk_stride, 0);
  std::vector<long double> blo((size_t)ns * 7), bhi((size_t)ns * 7);
  for (int i = 0; i < ns; ++i) {
    scaled_nasa(d->nasa_lo + (size_t)7 * i, &blo[(size_t)i * 7]);
    scaled_nasa(d->nasa_hi + (size_t)7 * i, &bhi[(size_t)i * 7]);
  }
  for (int g = 0; g < ng; ++g)
    for (int pp = 0; pp < f.ph_end; ++pp) {
      const int seg = pp < f.arr_end ? 0 : pp < f.fo_end ? 1 : 2;
      const int first = seg == 0 ? 0 : seg == 1 ? f.arr_end : f.fo_end;
      const int64_t off = seg == 0 ? 0 : seg == 1 ? f.blk_fo_off : f.blk_ph_off;
      const int bsz = seg == 0 ? kFBlkArr : seg == 1 ? kFBlkFo : kFBlkPh;
      unsigned char *blk = &f.blk[(size_t)g * f.blk_stride + off + (size_t)((pp - first) / kFRxnPerWarp) * bsz];
      const int slot = (pp - first) % kFRxnPerWarp;
      const int p = f.pp_to_packed[pp];
      int32_t sp8[8] = {ns, ns, ns, ns, ns, ns, 0, 0};  // absent species -> the ones row of the n tile
      double v[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
      if (p >= 0) {
        for (int a = 0; a < 6; ++a)
          if (h.sp[(size_t)p * 6 + a] >= 0) sp8[a] = h.sp[(size_t)p * 6 + a];
        sp8[7] = h.flags[p];
        if (p < h.ph_begin && !(h.flags[p] & 1)) sp8[3] = ns + 1, sp8[4] = ns, sp8[5] = ns;   // irreversible: zeros row
        if (p >= h.ph_begin) sp8[6] = h.photo_row[p - h.ph_begin];
        v[0] = h.c0[p], v[1] = h.c1[p], v[2] = h.c2[p];
        if (p < h.ph_begin && (h.flags[p] & 1)) {
          long double db[7] = {0, 0, 0, 0, 0, 0, 0};
          for (int a = 0; a < 6; ++a) {
            const int i = h.sp[(size_t)p * 6 + a];
            if (i < 0) continue;
            const long double *b = (g <= bp_of[i] ? &blo[(size_t)i * 7] : &bhi[(size_t)i * 7]);
            for (int k = 0; k < 7; ++k) db[k] += a < 3 ? -b[k] : b[k];
          }
          const bool fold = p < h.fo_begin;
          v[3] = (double)((fold ? (long double)h.c0[p] : 0.0L) + db[0]);
          v[4] = (double)((fold ? (long double)h.c1[p] : 0.0L) - db[1]);
          v[5] = (double)((fold ? (long double)h.c2[p] : 0.0L) + db[6]);
          v[6] = (double)db[2], v[7] = (double)db[3], v[8] = (double)db[4], v[9] = (double)db[5];
        }
        if (seg == 1) {
          const int fo = p - h.fo_begin;
          v[10] = h.l0[fo], v[11] = h.l1[fo], v[12] = h.l2[fo], v[13] = h.fcl[fo], v[14] = h.cN[fo];
        }
      }
      // unit 0: the six species slots as 16-bit indices (r0 r1 | r2 p0 | p1 p2) and the J row; unit 1 spare
      const int32_t packed[4] = {sp8[0] | (sp8[1] << 16), sp8[2] | (sp8[3] << 16), sp8[4] | (sp8[5] << 16), sp8[6]};
      std::memcpy(blk + 0 * 64 + slot * 16, packed, 16);
      std::memcpy(blk + 1 * 64 + slot * 16, sp8 + 4, 16);
      const int npair = seg == 0 ? 5 : seg == 1 ? 8 : 0;
      for (int u = 0; u < npair; ++u) std::memcpy(blk + (2 + u) * 64 + slot * 16, v + 2 * u, 16);
    }

  // ---- production/loss schedule
  // entries of chunk k grouped by species (source CSR order inside a species)
  struct Row { int32_t species; std::vector<uint32_t> ent; };
  const int nchunk = f.nchunk;
  std::vector<std::vector<Row>> rows(nchunk);
  std::vector<int> max_seg(ns, 1);
  {
    std::vector<std::vector<std::vector<uint32_t>>> tmp(nchunk);  // [chunk][species] lazily sized
    std::vector<std::vector<int32_t>> touched(nchunk);
    for (int k = 0; k < nchunk; ++k) tmp[k].resize(ns);
    for (int i = 0; i < ns; ++i)
      for (int64_t e = h.src_ptr[i]; e < h.src_ptr[i + 1]; ++e) {
        const int pp = packed_to_pp[h.src_rxn_packed[e]];
        const int k = pp / chunk, rloc = pp % chunk;
        const double nu = (double)h.src_nu[e];
        uint64_t bits;
        std::memcpy(&bits, &nu, 8);
        if (tmp[k][i].empty()) touched[k].push_back(i);
        tmp[k][i].push_back((uint32_t)((bits >> 48) << 16) | (uint32_t)rloc);
      }
    for (int k = 0; k < nchunk; ++k)
      for (int i : touched[k]) {
        const int nseg = ((int)tmp[k][i].size() + kFSegMax - 1) / kFSegMax;
        max_seg[i] = std::max(max_seg[i], nseg);
        rows[k].push_back({i, std::move(tmp[k][i])});
      }
  }
  // extra accumulator rows of hub species: segment s > 0 of species i -> row extra_base[i] + s - 1
  std::vector<int32_t> extra_base(ns, -1);
  f.n_acc = ns;
  f.extra.clear();
  for (int i = 0; i < ns; ++i)
    if (max_seg[i] > 1) {
      extra_base[i] = f.n_acc;
      for (int s = 1; s < max_seg[i]; ++s) {
        f.extra.push_back(f.n_acc++);
        f.extra.push_back(i);
      }
    }
  if (f.n_acc >= 0xffff) return;

  const uint32_t zero_entry = (uint32_t)chunk;  // nu bits 0 (= +0.0), the zero row of q
  f.meta_ptr.assign((size_t)nchunk + 1, 0);
  f.meta.clear();
  f.meta_cap = 0, f.n_tasks = 0, f.n_entries = 0;
  for (int k = 0; k < nchunk; ++k) {
    std::vector<SchedSeg> segs;
    for (const Row &r : rows[k]) {
      const int len = (int)r.ent.size(), nseg = (len + kFSegMax - 1) / kFSegMax, per = (len + nseg - 1) / nseg;
      for (int s = 0; s < nseg; ++s) {
        const int b = s * per, e = std::min(len, b + per);
        if (e > b) segs.push_back({s == 0 ? r.species : extra_base[r.species] + s - 1, r.ent.data() + b, e - b});
      }
    }
    std::vector<int32_t> blob;
    int64_t nt = 0, nent = 0;
    build_chunk_schedule(segs, zero_entry, blob, nt, nent);
    f.n_tasks += nt, f.n_entries += nent;
    f.meta.insert(f.meta.end(), blob.begin(), blob.end());
    f.meta_ptr[k + 1] = (int32_t)(f.meta.size() / 4);
    f.meta_cap = std::max<int32_t>(f.meta_cap, (int32_t)(blob.size() / 4));
  }
  f.enabled = true;
}

}  // namespace xod

namespace xod {

// Host-only self-check of the fused-path tables, decoding them exactly as k_fused does:
//  * every (species, reaction, nu) entry of the source CSR appears exactly once in the chunk
//    schedules, under its own species' accumulator row or one of that species' extra rows;
//  * no accumulator row is written by two row tasks of one chunk (the atomic-free guarantee);
//  * entry offsets, step counts and q-row indices stay inside their chunk;
//  * the species slots and photolysis rows stored in the parameter blocks match the packed tables.
// Returns true when consistent; otherwise err names the first violation.
bool check_fused(const HostTables &h, std::string &err) {
  const FusedHost &f = h.f;
  if (!f.enabled) return true;
  const int ns = h.ns;
  auto fail = [&](const std::string &m) { err = "fused tables: " + m; return false; };
  std::vector<int32_t> row_species(f.n_acc, -1);
  for (int i = 0; i < ns; ++i) row_species[i] = i;
  for (size_t x = 0; x + 1 < f.extra.size(); x += 2) {
    if (f.extra[x] < ns || f.extra[x] >= f.n_acc || f.extra[x + 1] < 0 || f.extra[x + 1] >= ns) return fail("bad extra row");
    row_species[f.extra[x]] = f.extra[x + 1];
  }
  for (int r = ns; r < f.n_acc; ++r)
    if (row_species[r] < 0) return fail("unmapped extra row");
  // expected multiset of (species, padded reaction, nu)
  std::vector<int32_t> packed_to_pp(h.nr, -1);
  for (int pp = 0; pp < f.npad; ++pp)
    if (f.pp_to_packed[pp] >= 0) packed_to_pp[f.pp_to_packed[pp]] = pp;
  std::vector<int64_t> want, got;
  auto key = [&](int sp, int pp, int nu) { return ((int64_t)sp * f.npad + pp) * 8 + (nu + 4); };
  for (int i = 0; i < ns; ++i)
    for (int64_t e = h.src_ptr[i]; e < h.src_ptr[i + 1]; ++e)
      want.push_back(key(i, packed_to_pp[h.src_rxn_packed[e]], h.src_nu[e]));
  for (int k = 0; k < f.nchunk; ++k) {
    const int32_t *blob = &f.meta[(size_t)f.meta_ptr[k] * 4];
    const int64_t blob_words = ((int64_t)f.meta_ptr[k + 1] - f.meta_ptr[k]) * 4;
    if (blob_words / 4 > f.meta_cap) return fail("schedule larger than meta_cap");
    const int nt = blob[kFWarps + 1];
    if (blob[0] != 0 || blob[kFWarps] != nt) return fail("bad warp offsets");
    const int32_t *tasks = blob + kFMetaHdr;
    const int32_t *ent = tasks + 4 * nt;
    const int64_t nent = blob_words - kFMetaHdr - 4 * nt;
    std::vector<char> row_used(f.n_acc, 0);
    for (int w = 0; w < kFWarps; ++w) {
      if (blob[w] > blob[w + 1]) return fail("warp offsets not monotone");
      for (int t = blob[w]; t < blob[w + 1]; ++t) {
        const int32_t off = tasks[4 * t], nsteps = tasks[4 * t + 1];
        if (off < 0 || nsteps < 0 || nsteps > kFSegMax || (int64_t)off + 4 * nsteps > nent) return fail("task out of range");
        for (int g = 0; g < 4; ++g) {
          const uint32_t rows = (uint32_t)tasks[4 * t + 2 + (g >> 1)];
          const int row = (g & 1) ? rows >> 16 : rows & 0xffffu;
          for (int st = 0; st < nsteps; ++st) {
            const uint32_t en = (uint32_t)ent[off + st * 4 + g];
            const int rloc = en & 0xffffu;
            uint64_t bits = (uint64_t)(en & 0xffff0000u) << 32;
            double nu;
            std::memcpy(&nu, &bits, 8);
            if (rloc > f.chunk) return fail("q row beyond the chunk");
            if (rloc == f.chunk) {
              if (nu != 0.0) return fail("padding entry with nonzero nu");
              continue;
            }
            if (row == 0xffff) return fail("entry under an idle lane group");
            if (nu != std::floor(nu) || std::fabs(nu) > 3 || nu == 0.0) return fail("bad nu encoding");
            got.push_back(key(row_species[row], k * f.chunk + rloc, (int)nu));
          }
          if (row != 0xffff) {
            if (row >= f.n_acc) return fail("accumulator row out of range");
            if (row_used[row]) return fail("accumulator row written by two row tasks of one chunk");
            row_used[row] = 1;
          }
        }
      }
    }
  }
  std::sort(want.begin(), want.end());
  std::sort(got.begin(), got.end());
  if (want != got) return fail("schedule entries differ from the source CSR");
  // parameter blocks: species slots and J rows, every interval
  for (int g = 0; g <= f.n_bp; ++g)
    for (int pp = 0; pp < f.ph_end; ++pp) {
      const int seg = pp < f.arr_end ? 0 : pp < f.fo_end ? 1 : 2;
      const int first = seg == 0 ? 0 : seg == 1 ? f.arr_end : f.fo_end;
      const int64_t off = seg == 0 ? 0 : seg == 1 ? f.blk_fo_off : f.blk_ph_off;
      const int bsz = seg == 0 ? kFBlkArr : seg == 1 ? kFBlkFo : kFBlkPh;
      const unsigned char *blk = &f.blk[(size_t)g * f.blk_stride + off + (size_t)((pp - first) / kFRxnPerWarp) * bsz];
      int32_t u[4];
      std::memcpy(u, blk + ((pp - first) % kFRxnPerWarp) * 16, 16);
      const int p = f.pp_to_packed[pp];
      const int slots[6] = {u[0] & 0xffff, (int)((uint32_t)u[0] >> 16), u[1] & 0xffff, (int)((uint32_t)u[1] >> 16),
                            u[2] & 0xffff, (int)((uint32_t)u[2] >> 16)};
      const bool irrev = p >= 0 && p < h.ph_begin && !(h.flags[p] & 1);   // products: zeros row, ones, ones
      for (int a = 0; a < 6; ++a) {
        int expect = p >= 0 && h.sp[(size_t)p * 6 + a] >= 0 ? h.sp[(size_t)p * 6 + a] : ns;
        if (irrev && a >= 3) expect = a == 3 ? ns + 1 : ns;
        if (slots[a] != expect) return fail("species slot mismatch in a parameter block");
      }
      {
        int32_t u1[4];
        std::memcpy(u1, blk + 64 + ((pp - first) % kFRxnPerWarp) * 16, 16);
        if (p >= 0 && u1[3] != h.flags[p]) return fail("reversible flag mismatch in a parameter block");
      }
      if (p >= h.ph_begin && u[3] != h.photo_row[p - h.ph_begin]) return fail("J row mismatch in a parameter block");
      if (u[3] < 0 || (h.n_photo > 0 && u[3] >= h.n_photo) ) return fail("J row out of range");
    }
  return true;
}

}  // namespace xod
