// pack.cpp -- step a0 of the path: validate the network description, sort the
// reactions by type (north_star: "a network packer that sorts reactions by type ... into SoA
// parameter tables"), pre-fold the Arrhenius/Kooij constants of PAPER.md:118-122 (Eq. 7) and
// 148-151 (Eq. 10-11) into the log2 domain, pre-scale the NASA-7 coefficients of PAPER.md:671,
// and build the source CSR, the Jacobian CSR pattern and the per-entry term lists.
// Host only; runs once per network.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <numeric>

#include "xod_internal.h"

namespace xod {

namespace {

constexpr long double kLog2e = 1.442695040888963407359924681001892137L;
constexpr long double kBoltz = 1.380649e-16L;  // erg/K
constexpr long double kPref = 1.0e6L;          // dyn/cm^2 (1 bar), reading T2

std::string fmt(const char *f, long a = 0, long b = 0, long c = 0) {
  char buf[256];
  std::snprintf(buf, sizeof buf, f, a, b, c);
  return buf;
}

// species of one side, compacted (the -1 padding may sit anywhere)
int side_of(const int32_t *s3, int32_t out[3]) {
  int k = 0;
  for (int a = 0; a < 3; ++a)
    if (s3[a] >= 0) out[k++] = s3[a];
  for (int a = k; a < 3; ++a) out[a] = -1;
  return k;
}

}  // namespace

xod_status pack_network(const xod_network_desc *d, HostTables &h, std::string &err) {
  if (!d) return err = "desc is NULL", XOD_ERR_INVALID_ARG;
  const int ns = d->n_species, ne = d->n_elements, nr = d->n_reactions;
  if (ns <= 0 || ne < 0 || nr < 0) return err = "n_species must be > 0, n_elements and n_reactions >= 0", XOD_ERR_INVALID_ARG;
  if (ns > 32767 * 2) return err = "n_species too large", XOD_ERR_INVALID_ARG;
  if (!d->nasa_lo || !d->nasa_hi || !d->t_mid) return err = "nasa_lo, nasa_hi, t_mid must not be NULL", XOD_ERR_INVALID_ARG;
  if (ne > 0 && !d->composition) return err = "composition is NULL", XOD_ERR_INVALID_ARG;
  if (nr > 0 && (!d->type || !d->reactants || !d->products || !d->reversible || !d->arrh))
    return err = "type, reactants, products, reversible, arrh must not be NULL", XOD_ERR_INVALID_ARG;

  // ---------------------------------------------------------------- validation
  int counts[4] = {0, 0, 0, 0};
  for (int r = 0; r < nr; ++r) {
    int t = d->type[r];
    if (t < XOD_UNI || t > XOD_PHOTO) return err = fmt("reaction %ld: bad type %ld", r, t), XOD_ERR_INVALID_ARG;
    ++counts[t];
    int32_t lhs[3], rhs[3];
    for (int a = 0; a < 3; ++a) {
      int32_t x = d->reactants[3 * r + a], y = d->products[3 * r + a];
      if (x < -1 || x >= ns || y < -1 || y >= ns)
        return err = fmt("reaction %ld: species index out of range", r), XOD_ERR_INVALID_ARG;
    }
    int nl = side_of(d->reactants + 3 * r, lhs), nrhs = side_of(d->products + 3 * r, rhs);
    if (nl == 0) return err = fmt("reaction %ld: no reactants", r), XOD_ERR_INVALID_ARG;
    if (nrhs == 0) return err = fmt("reaction %ld: no products", r), XOD_ERR_INVALID_ARG;
    if (t == XOD_PHOTO && d->reversible[r])
      return err = fmt("reaction %ld: photolysis cannot be reversible", r), XOD_ERR_INVALID_ARG;
    if (t != XOD_PHOTO) {
      if (!(d->arrh[3 * r] > 0) || !std::isfinite(d->arrh[3 * r]) || !std::isfinite(d->arrh[3 * r + 1]) ||
          !std::isfinite(d->arrh[3 * r + 2]))
        return err = fmt("reaction %ld: alpha must be finite and > 0, beta and gamma finite", r), XOD_ERR_INVALID_ARG;
      double tr = d->t_ref ? d->t_ref[r] : 1.0;
      if (!(tr > 0) || !std::isfinite(tr)) return err = fmt("reaction %ld: t_ref must be > 0", r), XOD_ERR_INVALID_ARG;
    }
    if (t == XOD_FALLOFF) {
      if (!d->arrh_low || !d->troe_fc) return err = "arrh_low and troe_fc are required for XOD_FALLOFF", XOD_ERR_INVALID_ARG;
      if (!(d->arrh_low[3 * r] > 0) || !std::isfinite(d->arrh_low[3 * r]) ||
          !std::isfinite(d->arrh_low[3 * r + 1]) || !std::isfinite(d->arrh_low[3 * r + 2]))
        return err = fmt("reaction %ld: alpha0 must be finite and > 0", r), XOD_ERR_INVALID_ARG;
      double fc = d->troe_fc[r];
      if (!(fc > 0.0 && fc <= 1.0)) return err = fmt("reaction %ld: Troe Fc must be in (0, 1]", r), XOD_ERR_INVALID_ARG;
    }
    if (!(d->flags & XOD_FLAG_SKIP_BALANCE_CHECK)) {
      for (int e = 0; e < ne; ++e) {
        long bal = 0;
        for (int a = 0; a < nl; ++a) bal -= d->composition[(size_t)lhs[a] * ne + e];
        for (int a = 0; a < nrhs; ++a) bal += d->composition[(size_t)rhs[a] * ne + e];
        if (bal != 0) return err = fmt("reaction %ld does not conserve element %ld (imbalance %ld)", r, e, bal), XOD_ERR_UNBALANCED;
      }
    }
  }
  for (int i = 0; i < ns; ++i)
    if (!std::isfinite(d->t_mid[i])) return err = fmt("species %ld: t_mid not finite", i), XOD_ERR_INVALID_ARG;

  h.ns = ns, h.ne = ne, h.nr = nr;
  // composition as short (element, count) lists per species (xod_equilibrium); which columns carry both signs
  h.eq_ptr.assign(1, 0), h.eq_ea.clear(), h.eq_neg.assign((size_t)ne, 0);
  for (int i = 0; i < ns; ++i) {
    for (int e = 0; e < ne; ++e) {
      const int32_t a = d->composition[(size_t)i * ne + e];
      if (a < 0) h.eq_neg[e] = 1;
      if (a != 0 && e < 256) h.eq_ea.push_back(a * 256 + e);
    }
    h.eq_ptr.push_back((int32_t)h.eq_ea.size());
  }
  h.uni_begin = 0;
  h.bi_begin = counts[XOD_UNI];
  h.fo_begin = h.bi_begin + counts[XOD_BI];
  h.ph_begin = h.fo_begin + counts[XOD_FALLOFF];
  h.n_photo = counts[XOD_PHOTO];
  const int nfo = counts[XOD_FALLOFF];

  // ---------------------------------------------------------------- stable sort by type (reading P1)
  h.packed_to_user.resize(nr);
  std::iota(h.packed_to_user.begin(), h.packed_to_user.end(), 0);
  std::stable_sort(h.packed_to_user.begin(), h.packed_to_user.end(),
                   [&](int a, int b) { return d->type[a] < d->type[b]; });
  h.user_to_packed.resize(nr);
  for (int p = 0; p < nr; ++p) h.user_to_packed[h.packed_to_user[p]] = p;
  // photolysis rows of J: p-th XOD_PHOTO reaction in user order
  h.photo_user.clear();
  std::vector<int32_t> photo_row_of_user(nr, -1);
  for (int r = 0; r < nr; ++r)
    if (d->type[r] == XOD_PHOTO) {
      photo_row_of_user[r] = (int32_t)h.photo_user.size();
      h.photo_user.push_back(r);
    }

  // ---------------------------------------------------------------- SoA parameter tables
  // k = alpha (T/t_ref)^beta exp(-gamma/T)  ->  log2 k = c0 + c1 log2 T + c2 / T
  //   c0 = log2 alpha - beta log2 t_ref,  c1 = beta,  c2 = -gamma log2 e
  h.c0.assign(nr, 0), h.c1.assign(nr, 0), h.c2.assign(nr, 0);
  h.l0.assign(nfo, 0), h.l1.assign(nfo, 0), h.l2.assign(nfo, 0), h.fcl.assign(nfo, 0), h.cN.assign(nfo, 0);
  h.sp.assign((size_t)nr * 6, -1);
  h.flags.assign(nr, 0);
  h.photo_row.assign(h.n_photo, 0);
  for (int p = 0; p < nr; ++p) {
    int r = h.packed_to_user[p], t = d->type[r];
    side_of(d->reactants + 3 * r, &h.sp[(size_t)p * 6]);
    side_of(d->products + 3 * r, &h.sp[(size_t)p * 6 + 3]);
    h.flags[p] = d->reversible[r] ? 1 : 0;
    if (t == XOD_PHOTO) {
      h.photo_row[p - h.ph_begin] = photo_row_of_user[r];
      continue;
    }
    long double ltr = std::log2((long double)(d->t_ref ? d->t_ref[r] : 1.0));
    h.c0[p] = (double)(std::log2((long double)d->arrh[3 * r]) - (long double)d->arrh[3 * r + 1] * ltr);
    h.c1[p] = d->arrh[3 * r + 1];
    h.c2[p] = (double)(-(long double)d->arrh[3 * r + 2] * kLog2e);
    if (t == XOD_FALLOFF) {
      int f = p - h.fo_begin;
      h.l0[f] = (double)(std::log2((long double)d->arrh_low[3 * r]) - (long double)d->arrh_low[3 * r + 1] * ltr);
      h.l1[f] = d->arrh_low[3 * r + 1];
      h.l2[f] = (double)(-(long double)d->arrh_low[3 * r + 2] * kLog2e);
      // Troe (reading F1): log2 F = log2 Fc / (1 + (log10 Pr / N)^2), N = 0.75 - 1.27 log10 Fc
      //   log10 Pr / N = log2 Pr * (log10 2 / N) = log2 Pr * cN
      long double fc = d->troe_fc[r];
      long double N = 0.75L - 1.27L * std::log10(fc);
      h.fcl[f] = (double)std::log2(fc);
      h.cN[f] = (double)(std::log10(2.0L) / N);
    }
  }

  // ---------------------------------------------------------------- thermo tables
  // raw: [ns][2][7].  scaled (for the reverse-coefficient exponent, k_thermo.cu):
  //   u_i = log2(e) G_i/RT - log2(P0/(k_B T))
  //       = b0 - b1 log2 T - T (b2 + T (b3 + T (b4 + T b5))) + b6 / T
  //   b0 = (a1 - a7) log2 e - log2(P0/k_B), b1 = a1 - 1, b2 = a2 log2e/2, b3 = a3 log2e/6,
  //   b4 = a4 log2e/12, b5 = a5 log2e/20, b6 = a6 log2e
  h.nasa.resize((size_t)ns * 14);
  h.nasa_l2.resize((size_t)ns * 14);
  h.tmid.assign(d->t_mid, d->t_mid + ns);
  const long double lpk = std::log2(kPref / kBoltz);
  for (int i = 0; i < ns; ++i)
    for (int s = 0; s < 2; ++s) {
      const double *a = (s ? d->nasa_hi : d->nasa_lo) + (size_t)7 * i;
      double *raw = &h.nasa[(size_t)i * 14 + 7 * s], *b = &h.nasa_l2[(size_t)i * 14 + 7 * s];
      for (int k = 0; k < 7; ++k) {
        if (!std::isfinite(a[k])) return err = fmt("species %ld: NASA coefficient not finite", i), XOD_ERR_INVALID_ARG;
        raw[k] = a[k];
      }
      b[0] = (double)(((long double)a[0] - (long double)a[6]) * kLog2e - lpk);
      b[1] = (double)((long double)a[0] - 1.0L);
      b[2] = (double)((long double)a[1] * kLog2e / 2);
      b[3] = (double)((long double)a[2] * kLog2e / 6);
      b[4] = (double)((long double)a[3] * kLog2e / 12);
      b[5] = (double)((long double)a[4] * kLog2e / 20);
      b[6] = (double)((long double)a[5] * kLog2e);
    }

  // ---------------------------------------------------------------- source CSR (reading S2)
  // triples (species, user reaction, nu) generated in user reaction order, then a stable
  // counting sort by species: rows come out sorted by ascending user reaction index.
  struct Trip { int32_t i, r, nu; };
  std::vector<Trip> trips;
  trips.reserve((size_t)nr * 4);
  for (int r = 0; r < nr; ++r) {
    int32_t sp6[6];
    side_of(d->reactants + 3 * r, sp6);
    side_of(d->products + 3 * r, sp6 + 3);
    for (int a = 0; a < 6; ++a) {
      int i = sp6[a];
      if (i < 0) continue;
      bool first = true;
      for (int b = 0; b < a; ++b) first &= sp6[b] != i;
      if (!first) continue;
      int nu = 0;
      for (int b = 0; b < 6; ++b)
        if (sp6[b] == i) nu += b < 3 ? -1 : +1;
      if (nu) trips.push_back({i, r, nu});
    }
  }
  h.src_ptr.assign(ns + 1, 0);
  for (auto &t : trips) ++h.src_ptr[t.i + 1];
  for (int i = 0; i < ns; ++i) h.src_ptr[i + 1] += h.src_ptr[i];
  const size_t nnz = trips.size();
  h.src_rxn_user.resize(nnz), h.src_nu.resize(nnz), h.src_rxn_packed.resize(nnz), h.src_nu_f.resize(nnz);
  {
    std::vector<int64_t> cur(h.src_ptr.begin(), h.src_ptr.end() - 1);
    for (auto &t : trips) {
      int64_t k = cur[t.i]++;
      h.src_rxn_user[k] = t.r;
      h.src_nu[k] = t.nu;
      h.src_rxn_packed[k] = h.user_to_packed[t.r];
      h.src_nu_f[k] = (float)t.nu;
    }
  }

  // schedule of the production/loss kernel (k_source.cu): every CTA task holds kSrcWarpsPerCta
  // warp slots; a row of up to kSrcSegMin entries is one slot, a longer row is cut into at
  // most kSrcWarpsPerCta equal segments that all sit in one task and are combined in order.
  h.src_seg.clear();
  {
    std::vector<SrcSeg> task;
    auto flush = [&]() {
      while ((int)task.size() < kSrcWarpsPerCta) task.push_back({-1, 0, 0, 0});
      h.src_seg.insert(h.src_seg.end(), task.begin(), task.end());
      task.clear();
    };
    // long rows first (they are the critical path), then the rest in species order
    std::vector<int> order(ns);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
      return h.src_ptr[a + 1] - h.src_ptr[a] > h.src_ptr[b + 1] - h.src_ptr[b];
    });
    for (int i : order) {
      int64_t b = h.src_ptr[i], e = h.src_ptr[i + 1], len = e - b;
      int nseg = len <= kSrcSegMin ? 1 : (int)std::min<int64_t>(kSrcWarpsPerCta, (len + kSrcSegMin - 1) / kSrcSegMin);
      if ((int)task.size() + nseg > kSrcWarpsPerCta) flush();
      int64_t per = (len + nseg - 1) / nseg;
      for (int s = 0; s < nseg; ++s) {
        int64_t sb = std::min(e, b + s * per), se = std::min(e, sb + per);
        task.push_back({i, (int32_t)sb, (int32_t)se, s == 0 ? nseg : 0});
      }
      if ((int)task.size() == kSrcWarpsPerCta) flush();
    }
    if (!task.empty()) flush();
  }

  // ---------------------------------------------------------------- Jacobian pattern (readings J1, J2)
  // sort-based: keys i*ns + j of every ordered pair of distinct species of each reaction, plus
  // the diagonal; sort + unique gives CSR rows with ascending columns.
  std::vector<int64_t> keys;
  keys.reserve((size_t)nr * 16 + ns);
  for (int i = 0; i < ns; ++i) keys.push_back((int64_t)i * ns + i);
  for (int r = 0; r < nr; ++r) {
    int32_t sp6[6];
    side_of(d->reactants + 3 * r, sp6);
    side_of(d->products + 3 * r, sp6 + 3);
    for (int a = 0; a < 6; ++a)
      for (int b = 0; b < 6; ++b)
        if (sp6[a] >= 0 && sp6[b] >= 0) keys.push_back((int64_t)sp6[a] * ns + sp6[b]);
  }
  std::sort(keys.begin(), keys.end());
  keys.erase(std::unique(keys.begin(), keys.end()), keys.end());
  const size_t nnzj = keys.size();
  h.jac_ptr.assign(ns + 1, 0);
  h.jac_col.resize(nnzj);
  for (size_t k = 0; k < nnzj; ++k) {
    ++h.jac_ptr[keys[k] / ns + 1];
    h.jac_col[k] = (int32_t)(keys[k] % ns);
  }
  for (int i = 0; i < ns; ++i) h.jac_ptr[i + 1] += h.jac_ptr[i];

  // term lists: d q_f,r / d n_j = k_f m_j n_j^(m_j - 1) prod_{l != j} n_l^(m_l): the product over
  // all reactant slots but one j-slot, times m_j.  Entry (i, j) collects nu_ir * that, forward
  // terms positive, reverse terms negative, in user reaction order (forward before reverse).
  struct RawTerm { int64_t key; JacTerm t; };
  std::vector<RawTerm> raw;
  raw.reserve((size_t)nr * 14);
  for (int r = 0; r < nr; ++r) {
    int32_t sp6[6];
    side_of(d->reactants + 3 * r, sp6);
    side_of(d->products + 3 * r, sp6 + 3);
    // net nu of the distinct species
    int32_t di[6], dnu[6];
    int nd = 0;
    for (int a = 0; a < 6; ++a) {
      int i = sp6[a];
      if (i < 0) continue;
      bool first = true;
      for (int b = 0; b < a; ++b) first &= sp6[b] != i;
      if (!first) continue;
      int nu = 0;
      for (int b = 0; b < 6; ++b)
        if (sp6[b] == i) nu += b < 3 ? -1 : +1;
      if (nu) di[nd] = i, dnu[nd] = nu, ++nd;
    }
    for (int dir = 0; dir < 2; ++dir) {
      if (dir == 1 && (!d->reversible[r] || d->type[r] == XOD_PHOTO)) continue;
      const int32_t *side = sp6 + 3 * dir;
      for (int a = 0; a < 3; ++a) {
        int j = side[a];
        if (j < 0) continue;
        bool first = true;
        int m = 0;
        for (int b = 0; b < 3; ++b) {
          if (side[b] == j) {
            ++m;
            if (b < a) first = false;
          }
        }
        if (!first) continue;
        int32_t others[2] = {-1, -1};
        int no = 0;
        for (int b = 0; b < 3; ++b)
          if (b != a && side[b] >= 0) others[no++] = side[b];
        for (int q = 0; q < nd; ++q) {
          JacTerm t;
          t.rk = r | (dir ? (int32_t)0x80000000u : 0);
          t.o1 = others[0], t.o2 = others[1];
          t.coef = (float)((dir ? -1 : 1) * dnu[q] * m);
          raw.push_back({(int64_t)di[q] * ns + j, t});
        }
      }
    }
  }
  std::stable_sort(raw.begin(), raw.end(), [](const RawTerm &a, const RawTerm &b) { return a.key < b.key; });
  h.jac_term_ptr.assign(nnzj + 1, 0);
  h.jac_terms.resize(raw.size());
  {
    size_t e = 0;
    for (size_t k = 0; k < raw.size(); ++k) {
      while (keys[e] < raw[k].key) ++e;  // every term key is in the pattern by construction
      if (keys[e] != raw[k].key) return err = "internal: Jacobian term outside the pattern", XOD_ERR_INVALID_ARG;
      ++h.jac_term_ptr[e + 1];
      h.jac_terms[k] = raw[k].t;
    }
    for (size_t k = 0; k < nnzj; ++k) h.jac_term_ptr[k + 1] += h.jac_term_ptr[k];
  }
  return XOD_OK;
}

}  // namespace xod
