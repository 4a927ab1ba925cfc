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

size_t fused_smem_bytes(int ns, int n_acc, int chunk) {
  // n tile (+ ones row) | accumulator rows | two q buffers (+ zero row each) | column scalars
  return ((size_t)(ns + 1) + (size_t)n_acc + 2 * (size_t)(chunk + 1)) * kFW * sizeof(double) +
         (size_t)kFW * (4 * sizeof(double) + sizeof(int32_t));
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
  if (f.n_bp + 1 > kFMaxIntervals) return;
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
  std::vector<int32_t> packed_to_pp(nr);
  for (int pp = 0; pp < f.npad; ++pp)
    if (f.pp_to_packed[pp] >= 0) packed_to_pp[f.pp_to_packed[pp]] = pp;

  // ---- forward coefficients, falloff extras, species slots
  const size_t np = (size_t)f.npad, nfo_pad = (size_t)(f.fo_end - f.arr_end);
  f.c.assign(3 * np, 0.0);
  f.l.assign(5 * std::max<size_t>(nfo_pad, 1), 0.0);
  f.sp.assign(8 * np, ns);  // absent species -> the ones row of the n tile
  for (int pp = 0; pp < f.npad; ++pp) {
    int32_t *s = &f.sp[(size_t)pp * 8];
    s[6] = 0, s[7] = 0;  // padding slots of the PHOTO segment read row 0 of J (result unused)
    const int p = f.pp_to_packed[pp];
    if (p < 0) continue;
    for (int a = 0; a < 6; ++a)
      if (h.sp[(size_t)p * 6 + a] >= 0) s[a] = h.sp[(size_t)p * 6 + a];
    s[7] = h.flags[p];
    f.c[pp] = h.c0[p], f.c[np + pp] = h.c1[p], f.c[2 * np + pp] = h.c2[p];
    if (p >= h.ph_begin) s[6] = h.photo_row[p - h.ph_begin];
    if (p >= h.fo_begin && p < h.ph_begin) {
      const size_t q = (size_t)(pp - f.arr_end);
      const int fo = p - h.fo_begin;
      f.l[q] = h.l0[fo], f.l[nfo_pad + q] = h.l1[fo], f.l[2 * nfo_pad + q] = h.l2[fo];
      f.l[3 * nfo_pad + q] = h.fcl[fo], f.l[4 * nfo_pad + q] = h.cN[fo];
    }
  }

  // ---- reverse-coefficient table [interval][7][npad]
  //   UNI/BI : C0 = c0 + dB0, C1 = c1 - dB1, C2 = c2 + dB6   (k_f folded in: one exp2 gives k_r)
  //   FALLOFF: C0 = dB0, C1 = -dB1, C2 = dB6                 (pure z; added to log2 k_f in the kernel)
  //   irreversible, photolysis, padding: C0 = -inf, rest 0   (k_r = 0)
  const int ng = f.n_bp + 1;
  f.rev.assign((size_t)ng * 7 * np, 0.0);
  std::vector<long double> blo((size_t)ns * 7), bhi((size_t)ns * 7);
  for (int i = 0; i < ns; ++i) {
    scaled_nasa(d->nasa_lo + (size_t)7 * i, &blo[(size_t)i * 7]);
    scaled_nasa(d->nasa_hi + (size_t)7 * i, &bhi[(size_t)i * 7]);
  }
  for (int g = 0; g < ng; ++g)
    for (int pp = 0; pp < f.npad; ++pp) {
      double *out = &f.rev[((size_t)g * 7) * np + pp];
      const int p = f.pp_to_packed[pp];
      if (p < 0 || p >= h.ph_begin || !(h.flags[p] & 1)) {
        out[0] = -INFINITY;
        continue;
      }
      long double db[7] = {0, 0, 0, 0, 0, 0, 0};
      for (int a = 0; a < 6; ++a) {
        const int i = h.sp[(size_t)p * 6 + a];
        if (i < 0) continue;
        const long double *b = (g <= bp_of[i] ? &blo[(size_t)i * 7] : &bhi[(size_t)i * 7]);
        for (int k = 0; k < 7; ++k) db[k] += a < 3 ? -b[k] : b[k];
      }
      const bool fold = p < h.fo_begin;
      out[0] = (double)((fold ? (long double)h.c0[p] : 0.0L) + db[0]);
      out[1 * np] = (double)((fold ? (long double)h.c1[p] : 0.0L) - db[1]);
      out[2 * np] = (double)((fold ? (long double)h.c2[p] : 0.0L) + db[6]);
      out[3 * np] = (double)db[2];
      out[4 * np] = (double)db[3];
      out[5 * np] = (double)db[4];
      out[6 * np] = (double)db[5];
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

  struct Seg { int32_t row; const uint32_t *ent; int len; };
  const uint32_t zero_entry = (uint32_t)chunk;  // nu bits 0 (= +0.0), the zero row of q
  f.task_ptr.assign((size_t)nchunk * kFWarps + 1, 0);
  f.task.clear();
  f.entry.clear();
  for (int k = 0; k < nchunk; ++k) {
    std::vector<Seg> segs;
    for (const Row &r : rows[k]) {
      const int len = (int)r.ent.size(), nseg = (len + kFSegMax - 1) / kFSegMax, per = (len + nseg - 1) / nseg;
      for (int s = 0; s < nseg; ++s) {
        const int b = s * per, e = std::min(len, b + per);
        if (e > b) segs.push_back({s == 0 ? r.species : extra_base[r.species] + s - 1, r.ent.data() + b, e - b});
      }
    }
    std::stable_sort(segs.begin(), segs.end(), [](const Seg &a, const Seg &b) { return a.len > b.len; });
    // warp tasks of 4 similar-length segments, dealt to the least-loaded warp (longest first)
    std::vector<std::vector<FusedTask>> per_warp(kFWarps);
    std::vector<int> load(kFWarps, 0);
    for (size_t s0 = 0; s0 < segs.size(); s0 += 4) {
      const int cnt = (int)std::min<size_t>(4, segs.size() - s0), nsteps = segs[s0].len;
      FusedTask t;
      t.entry_base = (int32_t)f.entry.size();
      t.nsteps = nsteps;
      uint32_t r[4] = {0xffffu, 0xffffu, 0xffffu, 0xffffu};
      for (int g = 0; g < cnt; ++g) r[g] = (uint32_t)segs[s0 + g].row;
      t.rows01 = (int32_t)(r[0] | (r[1] << 16));
      t.rows23 = (int32_t)(r[2] | (r[3] << 16));
      for (int st = 0; st < nsteps; ++st)
        for (int g = 0; g < 4; ++g)
          f.entry.push_back(g < cnt && st < segs[s0 + g].len ? segs[s0 + g].ent[st] : zero_entry);
      const int w = (int)(std::min_element(load.begin(), load.end()) - load.begin());
      load[w] += nsteps + 2;
      per_warp[w].push_back(t);
    }
    for (int w = 0; w < kFWarps; ++w) {
      f.task.insert(f.task.end(), per_warp[w].begin(), per_warp[w].end());
      f.task_ptr[(size_t)k * kFWarps + w + 1] = (int32_t)f.task.size();
    }
  }
  f.enabled = true;
}

}  // namespace xod
