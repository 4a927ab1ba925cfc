/* xodiac_oracle.c -- CPU ORACLE for the XODIAC chemical source term.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, single-threaded, obviously-correct evaluation of what the hot path
 * computes, written from the paper (arxiv 2512.06729, /root/reference/PAPER.md) and the
 * readings listed in DESIGN.md.  It shares no code, header, table or helper with the CUDA
 * library: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load it.  The product path never calls it.
 *
 * Method = direct evaluation of closed-form definitions, so the oracle is those
 * definitions written out, one column at a time, with direct powl/expl/log10l calls:
 * no log-domain folding, no type sorting, no precomputed per-reaction coefficients, no
 * blocking, no sparse tricks (the Jacobian is filled as a dense N_s x N_s matrix and the
 * pattern entries are read out of it).
 *
 * Precision: inputs and outputs are IEEE double (the path's arithmetic type).  Internal
 * values are `real_t` = long double (x86-64 80-bit extended) so that (i) the oracle's own
 * rounding error is far below the 1e-12 parity tolerance and (ii) K_c = exp(-dG/RT) never
 * overflows before k_r = k_f / K_c is rounded to double (reading R5).  Building
 * with -DXOD_ORACLE_DOUBLE makes real_t = double: the pure-fp64 variant that is timed as
 * the CPU baseline and cross-checked against the extended one in tests.
 *
 * Units: cgs.  T [K], P [dyn cm^-2], n [cm^-3], k [s^-1, cm^3 s^-1, cm^6 s^-1], J [s^-1].
 * Layout: every per-column array is [row][ld], column index contiguous, ld >= ncol.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Table 1 coefficients against textbook
 * thermochemistry of H2O, CO2 and a monatomic gas, G = H - TS, calculus
 * identities between cp, H and S, the n = 0, E = 0 => k = A case, Lindemann limits, Troe
 * symmetry, K_c recomputed from the thermo outputs by the test, element conservation, the
 * equilibrium fixed point, hand-expanded rate laws on a 3-species network, finite
 * differences of dn/dt against the Jacobian, and brute-force CSR construction.
 * Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifdef XOD_ORACLE_DOUBLE
typedef double real_t;
#define R_EXP exp
#define R_LOG log
#define R_LOG10 log10
#define R_POW pow
#define R_FABS fabs
#else
typedef long double real_t;
#define R_EXP expl
#define R_LOG logl
#define R_LOG10 log10l
#define R_POW powl
#define R_FABS fabsl
#endif

/* physical constants (cgs); BASELINE.json north_star: [M] = P/(k_B T); T2: P0 = 1 bar */
static const real_t K_BOLTZ = (real_t)1.380649e-16L; /* erg/K, exact SI 2019 value */
static const real_t P_REF = (real_t)1.0e6L;          /* dyn/cm^2 = 1 bar */

enum { ORC_UNI = 0, ORC_BI = 1, ORC_FALLOFF = 2, ORC_PHOTO = 3 };

/* The reaction record of PAPER.md:105-157: type, reactants, products, Arrhenius/Kooij
 * constants (alpha, beta, gamma) and, for three-body reactions, the low-pressure set. */
typedef struct {
  int n_species, n_elements, n_reactions;
  const int *composition;          /* [n_species][n_elements] */
  const double *nasa_lo, *nasa_hi; /* [n_species][7]  a1..a7 */
  const double *t_mid;             /* [n_species] */
  const int *type;                 /* [n_reactions] */
  const int *reactants, *products; /* [n_reactions][3], -1 padded, repeated index = coefficient 2 */
  const unsigned char *reversible; /* [n_reactions] */
  const double *arrh;              /* [n_reactions][3] alpha, beta, gamma   (k_inf for FALLOFF) */
  const double *arrh_low;          /* [n_reactions][3] alpha0, beta0, gamma0 (FALLOFF only) */
  const double *troe_fc;           /* [n_reactions] */
  const double *t_ref;             /* [n_reactions] 1 = modified Arrhenius, 300 = Kooij; NULL -> 1 */
} orc_network;

int orc_real_bits(void) { return (int)(sizeof(real_t) * 8); }
int orc_real_mant_dig(void) {
#ifdef XOD_ORACLE_DOUBLE
  return 53;
#else
  return __LDBL_MANT_DIG__;
#endif
}

/* ---------------------------------------------------------------- O1 thermo (NASA-7)
 * two coefficient sets, low- and high-temperature range.
 * PAPER.md:671  G/RT = a1(1 - ln T) - a2 T/2 - a3 T^2/6 - a4 T^3/12 - a5 T^4/20 + a6/T - a7
 * PAPER.md:673  cp/R = a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4
 * H/RT and S/R are not printed; the standard NASA-7 forms are used (reading T1):
 *   H/RT = a1 + a2 T/2 + a3 T^2/3 + a4 T^3/4 + a5 T^4/5 + a6/T
 *   S/R  = a1 ln T + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7
 * Range selection (reading T3): T <= t_mid -> low set, else high set; no clamping (T4). */
static const double *nasa_set(const orc_network *net, int i, real_t T) {
  return (T <= (real_t)net->t_mid[i]) ? net->nasa_lo + 7 * i : net->nasa_hi + 7 * i;
}
static real_t nasa_cp(const double *a, real_t T) {
  return a[0] + a[1] * T + a[2] * T * T + a[3] * T * T * T + a[4] * T * T * T * T;
}
static real_t nasa_h(const double *a, real_t T) {
  return a[0] + a[1] * T / 2 + a[2] * T * T / 3 + a[3] * T * T * T / 4 + a[4] * T * T * T * T / 5 +
         a[5] / T;
}
static real_t nasa_s(const double *a, real_t T) {
  return a[0] * R_LOG(T) + a[1] * T + a[2] * T * T / 2 + a[3] * T * T * T / 3 +
         a[4] * T * T * T * T / 4 + a[6];
}
static real_t nasa_g(const double *a, real_t T) {
  return a[0] * (1 - R_LOG(T)) - a[1] * T / 2 - a[2] * T * T / 6 - a[3] * T * T * T / 12 -
         a[4] * T * T * T * T / 20 + a[5] / T - a[6];
}

/* Any of cp_R, h_RT, s_R, g_RT may be NULL.  Each is [n_species][ld]. */
int orc_thermo(const orc_network *net, long ncol, long ld, const double *T, double *cp_R,
               double *h_RT, double *s_R, double *g_RT) {
  for (long c = 0; c < ncol; ++c) {
    real_t Tc = T[c];
    for (int i = 0; i < net->n_species; ++i) {
      const double *a = nasa_set(net, i, Tc);
      if (cp_R) cp_R[(long)i * ld + c] = (double)nasa_cp(a, Tc);
      if (h_RT) h_RT[(long)i * ld + c] = (double)nasa_h(a, Tc);
      if (s_R) s_R[(long)i * ld + c] = (double)nasa_s(a, Tc);
      if (g_RT) g_RT[(long)i * ld + c] = (double)nasa_g(a, Tc);
    }
  }
  return 0;
}

/* ---------------------------------------------------------------- O2 forward coefficients
 * PAPER.md:118-122 (Eq. 7): k = alpha T_b^beta exp(-gamma/T_c), T_b = T/300 (Kooij) or T
 * (modified Arrhenius), T_c = T. */
static real_t arrhenius(const double *abg, real_t T, real_t t_ref) {
  return (real_t)abg[0] * R_POW(T / t_ref, (real_t)abg[1]) * R_EXP(-(real_t)abg[2] / T);
}

/* PAPER.md:148-157 (Eq. 10-12): k0, k_inf as Eq. 7; k = k0[M] / (1 + k0[M]/k_inf).
 * [M] = P/(k_B T) (north_star).  Troe broadening is not in the paper; reading
 * F1: log10 F = log10 Fc / (1 + (log10 Pr / N)^2), N = 0.75 - 1.27 log10 Fc, Pr = k0[M]/k_inf;
 * Fc == 1 is pure Lindemann (Eq. 12). */
static real_t falloff(const double *inf_abg, const double *low_abg, double fc, real_t T, real_t P,
                      real_t t_ref) {
  real_t k0 = arrhenius(low_abg, T, t_ref);
  real_t kinf = arrhenius(inf_abg, T, t_ref);
  real_t M = P / (K_BOLTZ * T);
  real_t Pr = k0 * M / kinf;
  real_t kL = k0 * M / (1 + Pr);
  if (fc == 1.0) return kL;
  real_t lfc = R_LOG10((real_t)fc);
  real_t N = (real_t)0.75L - (real_t)1.27L * lfc;
  real_t x = R_LOG10(Pr) / N;
  real_t F = R_POW((real_t)fc, 1 / (1 + x * x));
  return kL * F;
}

/* ---------------------------------------------------------------- O3 reverse coefficients
 * PAPER.md:225-235 (Eq. 13-15): k_c = k_f / k_r, k_c from the Gibbs energy of reaction
 * (Tsai et al. 2017 App. E):  K_c = exp(-dG/RT) (P0 / (k_B T))^dnu,
 *   dG/RT = sum_products G_i/RT - sum_reactants G_i/RT,  dnu = #products - #reactants,
 * the third body M excluded from both (reading R1).  Photolysis has no reverse (R2). */
static real_t forward_coeff(const orc_network *net, int r, real_t T, real_t P, const double *J,
                            int photo_row, long ld, long c) {
  real_t t_ref = net->t_ref ? (real_t)net->t_ref[r] : (real_t)1;
  switch (net->type[r]) {
    case ORC_UNI:
    case ORC_BI:
      return arrhenius(net->arrh + 3 * r, T, t_ref);
    case ORC_FALLOFF:
      return falloff(net->arrh + 3 * r, net->arrh_low + 3 * r, net->troe_fc[r], T, P, t_ref);
    default: /* ORC_PHOTO: J supplied by the caller */
      return (real_t)J[(long)photo_row * ld + c];
  }
}

static real_t reverse_coeff(const orc_network *net, int r, real_t kf, real_t T) {
  if (!net->reversible[r] || net->type[r] == ORC_PHOTO) return 0;
  real_t dG = 0;
  int dnu = 0;
  for (int s = 0; s < 3; ++s) {
    int i = net->products[3 * r + s];
    if (i >= 0) {
      dG += nasa_g(nasa_set(net, i, T), T);
      ++dnu;
    }
  }
  for (int s = 0; s < 3; ++s) {
    int i = net->reactants[3 * r + s];
    if (i >= 0) {
      dG -= nasa_g(nasa_set(net, i, T), T);
      --dnu;
    }
  }
  real_t Kc = R_EXP(-dG) * R_POW(P_REF / (K_BOLTZ * T), (real_t)dnu);
  return kf / Kc;
}

/* kf, kr: [n_reactions][ld] in USER reaction order.  J: [n_photo][ld]. */
int orc_rate_coeffs(const orc_network *net, long ncol, long ld, const double *T, const double *P,
                    const double *J, double *kf, double *kr) {
  for (long c = 0; c < ncol; ++c) {
    real_t Tc = T[c], Pc = P[c];
    int photo_row = 0; /* row p of J is the p-th PHOTO reaction in user order */
    for (int r = 0; r < net->n_reactions; ++r) {
      real_t f = forward_coeff(net, r, Tc, Pc, J, photo_row, ld, c);
      if (net->type[r] == ORC_PHOTO) ++photo_row;
      real_t b = reverse_coeff(net, r, f, Tc);
      if (kf) kf[(long)r * ld + c] = (double)f;
      if (kr) kr[(long)r * ld + c] = (double)b;
    }
  }
  return 0;
}

/* ---------------------------------------------------------------- O4 rates of progress
 * q_f = k_f prod_{reactants} n_l, q_r = k_r prod_{products} n_l  (north_star: "k . prod n_reactant";
 * a repeated index gives n^2, e.g. 2 SO -> SO2 + S). */
static real_t rate_of(const int *side, real_t k, const double *n, long ld, long c) {
  real_t q = k;
  for (int s = 0; s < 3; ++s)
    if (side[s] >= 0) q *= (real_t)n[(long)side[s] * ld + c];
  return q;
}

int orc_rates(const orc_network *net, long ncol, long ld, const double *kf, const double *kr,
              const double *n, double *qf, double *qr) {
  for (long c = 0; c < ncol; ++c)
    for (int r = 0; r < net->n_reactions; ++r) {
      qf[(long)r * ld + c] = (double)rate_of(net->reactants + 3 * r, kf[(long)r * ld + c], n, ld, c);
      qr[(long)r * ld + c] = (double)rate_of(net->products + 3 * r, kr[(long)r * ld + c], n, ld, c);
    }
  return 0;
}

/* net stoichiometric coefficient nu_ir = (#i in products) - (#i in reactants) */
static int nu_of(const orc_network *net, int i, int r) {
  int v = 0;
  for (int s = 0; s < 3; ++s) {
    if (net->products[3 * r + s] == i) ++v;
    if (net->reactants[3 * r + s] == i) --v;
  }
  return v;
}

/* ---------------------------------------------------------------- O5 production and loss
 * PAPER.md:53 (Eq. 1): dn_i/dt = P_i - L_i.  dn_i/dt = sum_r nu_ir (q_f,r - q_r,r), summed
 * in user reaction order, forward term then reverse term.  P_i = sum of the positive terms,
 * L_i = sum of |negative terms| (a rate, reading S1).  prod, loss may be NULL. */
/* distinct species of reaction r (both sides), in slot order; returns how many */
static int distinct_species(const orc_network *net, int r, int *out) {
  int k = 0;
  for (int s = 0; s < 6; ++s) {
    int i = s < 3 ? net->reactants[3 * r + s] : net->products[3 * r + s - 3];
    if (i < 0) continue;
    int seen = 0;
    for (int t = 0; t < k; ++t)
      if (out[t] == i) seen = 1;
    if (!seen) out[k++] = i;
  }
  return k;
}

int orc_source(const orc_network *net, long ncol, long ld, const double *kf, const double *kr,
               const double *n, double *dndt, double *prod, double *loss) {
  int ns = net->n_species;
  real_t *sum = (real_t *)malloc(sizeof(real_t) * ns * 3), *sp = sum + ns, *sl = sum + 2 * ns;
  if (!sum) return -1;
  for (long c = 0; c < ncol; ++c) {
    for (int i = 0; i < 3 * ns; ++i) sum[i] = 0;
    for (int r = 0; r < net->n_reactions; ++r) { /* user reaction order */
      real_t qf = rate_of(net->reactants + 3 * r, kf[(long)r * ld + c], n, ld, c);
      real_t qr = rate_of(net->products + 3 * r, kr[(long)r * ld + c], n, ld, c);
      int sp_r[6], k = distinct_species(net, r, sp_r);
      for (int t = 0; t < k; ++t) {
        int i = sp_r[t], nu = nu_of(net, i, r);
        if (!nu) continue;
        real_t tf = nu * qf, tr = -nu * qr; /* forward term, then reverse term */
        sum[i] += tf;
        sum[i] += tr;
        if (tf > 0) sp[i] += tf; else sl[i] += -tf;
        if (tr > 0) sp[i] += tr; else sl[i] += -tr;
      }
    }
    for (int i = 0; i < ns; ++i) {
      if (dndt) dndt[(long)i * ld + c] = (double)sum[i];
      if (prod) prod[(long)i * ld + c] = (double)sp[i];
      if (loss) loss[(long)i * ld + c] = (double)sl[i];
    }
  }
  free(sum);
  return 0;
}

/* ---------------------------------------------------------------- O6 Jacobian
 * d q_f,r / d n_j = k_f,r m_jr n_j^(m_jr - 1) prod_{l != j} n_l^(m_lr), m = multiplicity among the
 * reactants (never q/n_j: exact at n_j = 0).  k_f, k_r, [M], J do not depend on n (reading J3).
 * Jac_ij = sum_r nu_ir (d q_f,r/d n_j - d q_r,r/d n_j);
 * scale_ij = sum_r |nu_ir| (|d q_f,r/d n_j| + |d q_r,r/d n_j|)  (the parity tolerance scale).
 * dense, scale: [n_species][n_species] row-major for ONE column c. */
static void add_side_derivatives(const orc_network *net, int r, const int *side, real_t k,
                                 real_t sign, const double *n, long ld, long c, real_t *dense,
                                 real_t *scale) {
  long ns = net->n_species;
  for (int a = 0; a < 3; ++a) {
    int j = side[a];
    if (j < 0) continue;
    int first = 1, m = 0;
    for (int b = 0; b < 3; ++b) {
      if (side[b] == j) {
        ++m;
        if (b < a) first = 0;
      }
    }
    if (!first) continue; /* each distinct species j once */
    real_t d = k * m;     /* k m_j n_j^(m_j-1) prod_{l!=j} n_l^m_l = k m_j prod over all slots but one j-slot */
    for (int b = 0; b < 3; ++b)
      if (b != a && side[b] >= 0) d *= (real_t)n[(long)side[b] * ld + c];
    int sp_r[6], k = distinct_species(net, r, sp_r);
    for (int t = 0; t < k; ++t) {
      int i = sp_r[t], nu = nu_of(net, i, r);
      if (!nu) continue;
      dense[(long)i * ns + j] += sign * nu * d;
      scale[(long)i * ns + j] += R_FABS(nu * d);
    }
  }
}

static void jacobian_dense_real(const orc_network *net, long ld, const double *kf, const double *kr,
                                const double *n, long c, real_t *dense, real_t *scale) {
  long ns = net->n_species;
  for (long e = 0; e < ns * ns; ++e) dense[e] = scale[e] = 0;
  for (int r = 0; r < net->n_reactions; ++r) {
    add_side_derivatives(net, r, net->reactants + 3 * r, kf[(long)r * ld + c], +1, n, ld, c, dense, scale);
    add_side_derivatives(net, r, net->products + 3 * r, kr[(long)r * ld + c], -1, n, ld, c, dense, scale);
  }
}

int orc_jacobian_dense(const orc_network *net, long ld, const double *kf, const double *kr,
                       const double *n, long c, double *dense, double *scale) {
  long ns = net->n_species;
  real_t *d = (real_t *)malloc(sizeof(real_t) * ns * ns), *s = (real_t *)malloc(sizeof(real_t) * ns * ns);
  if (!d || !s) return -1;
  jacobian_dense_real(net, ld, kf, kr, n, c, d, s);
  for (long e = 0; e < ns * ns; ++e) {
    dense[e] = (double)d[e];
    if (scale) scale[e] = (double)s[e];
  }
  free(d);
  free(s);
  return 0;
}

/* Pattern values: jac, scale are [nnz][ld].  Returns the number of (entry, column) pairs
 * OUTSIDE the pattern whose dense value or scale is not exactly 0 (must be 0), or -1. */
long orc_jacobian(const orc_network *net, long ncol, long ld, const double *kf, const double *kr,
                  const double *n, const long *row_ptr, const int *col, double *jac, double *scale) {
  long ns = net->n_species, bad = 0;
  real_t *d = (real_t *)malloc(sizeof(real_t) * ns * ns), *s = (real_t *)malloc(sizeof(real_t) * ns * ns);
  unsigned char *in = (unsigned char *)calloc(ns * ns, 1);
  if (!d || !s || !in) return -1;
  for (long i = 0; i < ns; ++i)
    for (long e = row_ptr[i]; e < row_ptr[i + 1]; ++e) in[i * ns + col[e]] = 1;
  for (long c = 0; c < ncol; ++c) {
    jacobian_dense_real(net, ld, kf, kr, n, c, d, s);
    for (long e = 0; e < ns * ns; ++e)
      if (!in[e] && (d[e] != 0 || s[e] != 0)) ++bad;
    for (long i = 0; i < ns; ++i)
      for (long e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
        jac[e * ld + c] = (double)d[i * ns + col[e]];
        if (scale) scale[e * ld + c] = (double)s[i * ns + col[e]];
      }
  }
  free(d);
  free(s);
  free(in);
  return bad;
}

/* ---------------------------------------------------------------- CSR layouts (readings S2, J1, J2)
 * Source CSR: row i = species i; entries = all reactions with nu_ir != 0 in ascending user
 * reaction index; nu in -3..3.  Pass rxn = nu = NULL to get only row_ptr (sizes). */
long orc_source_csr(const orc_network *net, long *row_ptr, int *rxn, int *nu) {
  long k = 0;
  for (int i = 0; i < net->n_species; ++i) {
    row_ptr[i] = k;
    for (int r = 0; r < net->n_reactions; ++r) {
      int v = nu_of(net, i, r);
      if (!v) continue;
      if (rxn) rxn[k] = r;
      if (nu) nu[k] = v;
      ++k;
    }
  }
  row_ptr[net->n_species] = k;
  return k;
}

/* Jacobian pattern: union over reactions of S_r x S_r (S_r = distinct species of reaction r,
 * both sides) plus the diagonal; rows = species, column indices ascending.  Built from a
 * dense boolean matrix.  Pass col = NULL to get only row_ptr. */
long orc_jac_pattern(const orc_network *net, long *row_ptr, int *col) {
  long ns = net->n_species, k = 0;
  unsigned char *m = (unsigned char *)calloc(ns * ns, 1);
  if (!m) return -1;
  for (long i = 0; i < ns; ++i) m[i * ns + i] = 1;
  for (int r = 0; r < net->n_reactions; ++r) {
    int sp[6];
    for (int s = 0; s < 3; ++s) {
      sp[s] = net->reactants[3 * r + s];
      sp[3 + s] = net->products[3 * r + s];
    }
    for (int a = 0; a < 6; ++a)
      for (int b = 0; b < 6; ++b)
        if (sp[a] >= 0 && sp[b] >= 0) m[(long)sp[a] * ns + sp[b]] = 1;
  }
  for (long i = 0; i < ns; ++i) {
    row_ptr[i] = k;
    for (long j = 0; j < ns; ++j)
      if (m[i * ns + j]) {
        if (col) col[k] = (int)j;
        ++k;
      }
  }
  row_ptr[ns] = k;
  free(m);
  return k;
}

/* ---------------------------------------------------------------- f1: implicit (backward-Euler) Newton step
 * The paper's continuity equation "is a stiff ordinary differential equation (ODE), implicit solvers
 * are the most suitable choice ... the lower-order backward Euler method (Hu et al. 2012), the
 * higher-order DLSODES solver".  One backward-Euler step of size dt from n_old solves
 *     F(y) = y - n_old - dt f(y) = 0,        f = dn/dt of O5 (chemistry only; transport is off the path)
 * and one Newton iteration from the iterate y is
 *     (I - dt Jac(y)) delta = -F(y),          y_new = y + delta,      Jac of O6.
 * The oracle is that definition written out for ONE column at a time: f from orc_source (rounded to
 * double, as the library's xod_source returns it), Jac as the dense matrix of O6 in real_t, and the
 * linear system solved by plain dense Gaussian elimination with partial pivoting in real_t.  No
 * sparsity, no ordering, no reuse of factors.
 * Pins (tests/test_oracle_newton.py): the closed form n0/(1 + dt k) of a first-order decay; a 2 x 2
 * reversible pair solved by hand; numpy's solver on the exported system; a^T delta = -a^T (y - n_old)
 * for every element; delta = 0 at the equilibrium fixed point; delta/dt -> f as dt -> 0; quadratic
 * convergence of the iteration to F = 0. */

/* A [ns][ns] row-major and b [ns] of column c:  A = I - dt Jac(y), b = -(y - n_old - dt f(y)) */
static int newton_system_real(const orc_network *net, long ld, const double *kf, const double *kr,
                              const double *n_old, const double *dt, const double *y, long c,
                              real_t *A, real_t *b, real_t *scratch /* ns*ns */) {
  long ns = net->n_species;
  double *col = (double *)malloc(sizeof(double) * (size_t)(ns * 2 + 2 * net->n_reactions + 1));
  if (!col) return -1;
  double *yc = col, *fc = col + ns, *kfc = fc + ns, *krc = kfc + net->n_reactions;
  for (long i = 0; i < ns; ++i) yc[i] = y[i * ld + c];
  for (long r = 0; r < net->n_reactions; ++r) kfc[r] = kf[r * ld + c], krc[r] = kr[r * ld + c];
  if (orc_source(net, 1, 1, kfc, krc, yc, fc, NULL, NULL) != 0) { free(col); return -1; }
  jacobian_dense_real(net, 1, kfc, krc, yc, 0, A, scratch);
  real_t h = (real_t)dt[c];
  for (long i = 0; i < ns; ++i) {
    for (long j = 0; j < ns; ++j) A[i * ns + j] = (i == j ? (real_t)1 : (real_t)0) - h * A[i * ns + j];
    b[i] = -((real_t)yc[i] - (real_t)n_old[i * ld + c] - h * (real_t)fc[i]);
  }
  free(col);
  return 0;
}

/* dense Gaussian elimination with partial pivoting; A is destroyed, x = A^-1 b.  Returns -1 if singular. */
static int solve_dense_real(long n, real_t *A, real_t *b, real_t *x) {
  for (long k = 0; k < n; ++k) {
    long p = k;
    for (long i = k + 1; i < n; ++i)
      if (R_FABS(A[i * n + k]) > R_FABS(A[p * n + k])) p = i;
    if (A[p * n + k] == 0) return -1;
    if (p != k) {
      for (long j = 0; j < n; ++j) { real_t t = A[k * n + j]; A[k * n + j] = A[p * n + j]; A[p * n + j] = t; }
      real_t t = b[k]; b[k] = b[p]; b[p] = t;
    }
    for (long i = k + 1; i < n; ++i) {
      real_t l = A[i * n + k] / A[k * n + k];
      if (l == 0) continue;
      for (long j = k + 1; j < n; ++j) A[i * n + j] -= l * A[k * n + j];
      b[i] -= l * b[k];
    }
  }
  for (long i = n - 1; i >= 0; --i) {
    real_t s = b[i];
    for (long j = i + 1; j < n; ++j) s -= A[i * n + j] * x[j];
    x[i] = s / A[i * n + i];
  }
  return 0;
}

/* The system of column c, rounded to double (tests form residuals and call a library solver on it). */
int orc_newton_system(const orc_network *net, long ld, const double *kf, const double *kr,
                      const double *n_old, const double *dt, const double *y, long c, double *A_out,
                      double *b_out) {
  long ns = net->n_species;
  real_t *A = (real_t *)malloc(sizeof(real_t) * (size_t)(2 * ns * ns + ns));
  if (!A) return -1;
  real_t *S = A + ns * ns, *b = S + ns * ns;
  int rc = newton_system_real(net, ld, kf, kr, n_old, dt, y, c, A, b, S);
  if (rc == 0) {
    for (long e = 0; e < ns * ns; ++e) A_out[e] = (double)A[e];
    for (long i = 0; i < ns; ++i) b_out[i] = (double)b[i];
  }
  free(A);
  return rc;
}

/* delta, y_new: [n_species][ld]; either may be NULL.  Returns 0, -1 (memory) or -2 (singular matrix). */
int orc_newton_step(const orc_network *net, long ncol, long ld, const double *kf, const double *kr,
                    const double *n_old, const double *dt, const double *y, double *delta, double *y_new) {
  long ns = net->n_species;
  real_t *A = (real_t *)malloc(sizeof(real_t) * (size_t)(2 * ns * ns + 2 * ns));
  if (!A) return -1;
  real_t *S = A + ns * ns, *b = S + ns * ns, *x = b + ns;
  int rc = 0;
  for (long c = 0; c < ncol && rc == 0; ++c) {
    rc = newton_system_real(net, ld, kf, kr, n_old, dt, y, c, A, b, S);
    if (rc == 0 && solve_dense_real(ns, A, b, x) != 0) rc = -2;
    if (rc != 0) break;
    for (long i = 0; i < ns; ++i) {
      if (delta) delta[i * ld + c] = (double)x[i];
      if (y_new) y_new[i * ld + c] = (double)((real_t)y[i * ld + c] + x[i]);
    }
  }
  free(A);
  return rc;
}

/* ---------------------------------------------------------------- f2: photolysis rate constants
 * PAPER.md:165-213 (section 2.3.3).  For every atmosphere and wavelength bin:
 *   optical depth   tau(z, lambda) = sum over the gas above z of (sigma_a,i + sigma_s,i) n_i dz
 *   actinic flux    J(z, lambda) = J0(lambda) exp(-tau / mu) + J_diff(z, lambda)
 *   rate constant   k_ph,i(z) = t_f * integral of J(z, lambda) sigma_i(lambda) d lambda
 * Discretisation (readings H1-H4; the paper gives none): layers are columns
 * a * n_layers + k with k = 0 at the bottom; tau is taken at the CENTRE of layer k, i.e. all layers above it
 * plus half of its own; the integral is the rectangle rule over the bins, sum_b J sigma dlambda_b (the paper's
 * bins are "approximately 1 A wide", uniform or not); J_diff = (J_up + J_down)/2 is an INPUT (the paper
 * names no transfer scheme for it), NULL = 0; sigma_ext rows are sigma_a + sigma_s of the absorbing species
 * abs_species[x]; sigma_ph rows are the reaction-specific cross-sections (molecular cross-section times
 * quantum yield already applied), in the row order of the library's J input.
 * Plain loops, one atmosphere and one bin at a time, top of the atmosphere downwards, in real_t.
 * tau_out (optional) [n_bins][ld] receives the layer-centre optical depths.
 * Pins (tests/test_oracle_photo.py): transparent atmosphere = t_f sum J0 sigma dlambda; a grey uniform slab
 * against the closed form exp(-kappa (depth + dz/2) / mu); a one-bin cross-section; the invariance
 * (sigma_ext, mu) -> (c sigma_ext, c mu); linearity in J0, sigma_ph and t_f; J_diff alone; monotone decrease downwards. */
int orc_photo_rates(int n_photo, int n_bins, int n_abs, const int *abs_species, const double *sigma_ext,
                    const double *sigma_ph, const double *dlambda, long n_atm, long n_layers, long ld,
                    const double *n, const double *dz, const double *j0, const double *j_diff,
                    const double *mu, const double *t_f, double *kph, double *tau_out) {
  real_t *acc = (real_t *)malloc(sizeof(real_t) * (size_t)n_photo * (size_t)n_layers);
  if (!acc) return -1;
  for (long a = 0; a < n_atm; ++a) {
    for (long e = 0; e < (long)n_photo * n_layers; ++e) acc[e] = 0;
    for (int b = 0; b < n_bins; ++b) {
      real_t above = 0; /* optical depth of everything above the current layer */
      for (long k = n_layers - 1; k >= 0; --k) {
        long c = a * n_layers + k;
        real_t kappa = 0;
        for (int x = 0; x < n_abs; ++x)
          kappa += (real_t)sigma_ext[(long)x * n_bins + b] * (real_t)n[(long)abs_species[x] * ld + c];
        real_t slab = kappa * (real_t)dz[c];
        real_t tau = above + slab / 2;
        above += slab;
        if (tau_out) tau_out[(long)b * ld + c] = (double)tau;
        real_t flux = (real_t)j0[a * n_bins + b] * R_EXP(-tau / (real_t)mu[a]);
        if (j_diff) flux += (real_t)j_diff[(long)b * ld + c];
        for (int p = 0; p < n_photo; ++p)
          acc[(long)p * n_layers + k] += flux * (real_t)sigma_ph[(long)p * n_bins + b] * (real_t)dlambda[b];
      }
    }
    for (int p = 0; p < n_photo; ++p)
      for (long k = 0; k < n_layers; ++k)
        kph[(long)p * ld + a * n_layers + k] = (double)((real_t)t_f[a] * acc[(long)p * n_layers + k]);
  }
  free(acc);
  return 0;
}

/* ---------------------------------------------------------------- f3: vertical (molecular-diffusion) transport terms
 * PAPER.md:73-83.  Eq. 4:
 *   d_{k+-1/2} = D_{k+-1/2} / (2 dz^2) * [ (mbar - m_y) g dz / (k_B T_{k+-1/2}) - alpha_T / T_{k+-1/2} * (T_{k+-1} - T_k) ]
 * "k +- 1/2 refers to the arithmetic mean of k and k +- 1".  Eq. 3, the part that is
 * not P - L:
 *   tr_{y,k} = - d_{k+1/2} (N_{k+1/2} / N_{k+1}) n_{y,k+1}
 *              - [ d_{k+1/2} (N_{k+1/2} / N_k) - d_{k-1/2} (N_{k-1/2} / N_k) ] n_{y,k}
 *              + d_{k-1/2} (N_{k-1/2} / N_k) n_{y,k-1}
 * with N = n_gas.  The printed equation is garbled in two places (reading V1): it carries an
 * index "n_gas,j" where only k makes sense and a stray "/2" under the first term; both are dropped, everything
 * else is taken literally.  Eddy diffusion does not appear ("the movement of the air parcel itself accounts for
 * this process").  Zero-flux boundaries: the half-level coefficients outside the
 * atmosphere are 0, so the terms that would reach below layer 0 or above the top layer vanish (reading V2).
 * mbar and g are per atmosphere, dz is the uniform layer spacing of an atmosphere (Eq. 4 has one dz), D is
 * given per (species, layer) (the paper computes it from Chapman-Enskog or binary-mixture theory, PAPER.md:67;
 * here it is an input, reading V3), alpha_T per species.
 * Layout: column = atmosphere * n_layers + layer, layer 0 at the bottom; tr [n_species][ld].
 * d_out (optional) [n_species][ld]: d_{k+1/2} of every layer (0 at the top layer).
 * Pins (tests/test_oracle_transport.py): Eq. 4 evaluated by hand; d = 0 for m_y = mbar in an isothermal column;
 * the uniform-N reduction -d+ n_{k+1} - (d+ - d-) n_k + d- n_{k-1}; linearity in n; a three-layer column
 * expanded by hand; zero-flux rows; independence of atmospheres. */
int orc_transport(int n_species, long n_atm, long n_layers, long ld, const double *n, const double *T,
                  const double *n_gas, const double *D, const double *mass, const double *alpha_T,
                  const double *mbar, const double *grav, const double *dz, double *tr, double *d_out) {
  for (long a = 0; a < n_atm; ++a) {
    real_t h = (real_t)dz[a];
    for (int y = 0; y < n_species; ++y) {
      const double *ny = n + (long)y * ld, *Dy = D + (long)y * ld;
      for (long k = 0; k < n_layers; ++k) {
        long c = a * n_layers + k;
        real_t dp = 0, dm = 0, Np = 0, Nm = 0; /* d_{k+1/2}, d_{k-1/2}, N_{k+1/2}, N_{k-1/2} */
        if (k + 1 < n_layers) {
          real_t Th = ((real_t)T[c] + (real_t)T[c + 1]) / 2, Dh = ((real_t)Dy[c] + (real_t)Dy[c + 1]) / 2;
          Np = ((real_t)n_gas[c] + (real_t)n_gas[c + 1]) / 2;
          dp = Dh / (2 * h * h) *
               (((real_t)mbar[a] - (real_t)mass[y]) * (real_t)grav[a] * h / (K_BOLTZ * Th) -
                (real_t)alpha_T[y] / Th * ((real_t)T[c + 1] - (real_t)T[c]));
        }
        if (k > 0) {
          real_t Th = ((real_t)T[c] + (real_t)T[c - 1]) / 2, Dh = ((real_t)Dy[c] + (real_t)Dy[c - 1]) / 2;
          Nm = ((real_t)n_gas[c] + (real_t)n_gas[c - 1]) / 2;
          dm = Dh / (2 * h * h) *
               (((real_t)mbar[a] - (real_t)mass[y]) * (real_t)grav[a] * h / (K_BOLTZ * Th) -
                (real_t)alpha_T[y] / Th * ((real_t)T[c - 1] - (real_t)T[c]));
        }
        real_t Nk = (real_t)n_gas[c], t = 0;
        if (k + 1 < n_layers) t -= dp * (Np / (real_t)n_gas[c + 1]) * (real_t)ny[c + 1];
        t -= (dp * (Np / Nk) - dm * (Nm / Nk)) * (real_t)ny[c];
        if (k > 0) t += dm * (Nm / Nk) * (real_t)ny[c - 1];
        tr[(long)y * ld + c] = (double)t;
        if (d_out) d_out[(long)y * ld + c] = (double)dp;
      }
    }
  }
  return 0;
}

/* ---------------------------------------------------------------- f4: reaction pathway analyser
 * "a reaction pathway analyzer designed to identify the most efficient conversion routes between any
 * two species ... built upon Dijkstra's classic algorithm (Dijkstra 1959), which identifies the kinetically fastest
 * reaction pathway by minimizing the cumulative sum of inverse reaction rates"; "The rate-limiting
 * step, defined as the slowest reaction in each pathway".
 * Graph of one column (reading W1; the paper does not spell it out): nodes are species; every listed
 * reaction contributes, for its forward direction with rate q_f = k_f prod n_reactant and (if reversible) its reverse
 * direction with q_r = k_r prod n_product (O4), a directed edge from each distinct species it consumes to each
 * distinct species it forms in that direction (u != v), of weight 1 / q.  A direction whose rate is not a positive
 * finite number offers no edge.  Parallel edges: the lighter one counts.
 * The oracle is Dijkstra's algorithm as in any textbook, one column and one source at a time, with a linear scan for
 * the closest unsettled node; distances are accumulated in real_t from the source outwards.
 * Outputs [n_species][ld]: dist (0 at the source, +inf if unreachable), pred (previous species on the path, -1 for
 * the source and for unreachable species), via (user reaction index of the last edge, bit 30 set for the reverse
 * direction; -1 likewise).  Ties between equally short paths are broken by the scan order (lowest species index
 * settled first, first edge found kept); only dist is unique.
 * Pins (tests/test_oracle_pathway.py): a hand graph where the two-step route beats the direct one exactly when
 * 1/q1 + 1/q2 < 1/q3; the min-plus closure (Floyd-Warshall in numpy) of the same edge weights from every source;
 * the optimality conditions dist[v] <= dist[u] + w on every edge with equality on the tree; dist scales as 1/c when
 * all rates are multiplied by c; unreachable species; the rate-limiting step of a path. */
int orc_pathway(const orc_network *net, long ncol, long ld, const double *kf, const double *kr, const double *n,
                int source, double *dist_out, int *pred_out, int *via_out) {
  int ns = net->n_species, nr = net->n_reactions;
  real_t *dist = (real_t *)malloc(sizeof(real_t) * (size_t)ns);
  real_t *w = (real_t *)malloc(sizeof(real_t) * (size_t)nr * 2);
  unsigned char *done = (unsigned char *)malloc((size_t)ns);
  int *pred = (int *)malloc(sizeof(int) * (size_t)ns * 2), *via = pred + ns;
  if (!dist || !w || !done || !pred) return -1;
  if (source < 0 || source >= ns) return -2;
  for (long c = 0; c < ncol; ++c) {
    for (int r = 0; r < nr; ++r) { /* edge weights of this column: 1 / rate of progress, per direction */
      /* the rates are rounded to double first: whether a direction "has a positive finite rate" is decided in the
       * path's arithmetic type (fp64), like every other quantity the library hands out (q beyond the double range is
       * +inf and offers no edge, exactly as a caller computing 1/q from xod's own outputs would see it) */
      double qf = (double)rate_of(net->reactants + 3 * r, kf[(long)r * ld + c], n, ld, c);
      double qr = net->reversible[r] ? (double)rate_of(net->products + 3 * r, kr[(long)r * ld + c], n, ld, c) : 0;
      double wf = 1 / qf, wr = 1 / qr;
      w[2 * r] = (qf > 0 && wf > 0 && wf < INFINITY) ? (real_t)1 / (real_t)qf : (real_t)INFINITY;
      w[2 * r + 1] = (qr > 0 && wr > 0 && wr < INFINITY) ? (real_t)1 / (real_t)qr : (real_t)INFINITY;
    }
    for (int i = 0; i < ns; ++i) dist[i] = (real_t)INFINITY, done[i] = 0, pred[i] = via[i] = -1;
    dist[source] = 0;
    for (;;) {
      int u = -1;
      for (int i = 0; i < ns; ++i)
        if (!done[i] && dist[i] < (real_t)INFINITY && (u < 0 || dist[i] < dist[u])) u = i;
      if (u < 0) break;
      done[u] = 1;
      for (int r = 0; r < nr; ++r)
        for (int d = 0; d < 2; ++d) {
          if (!(w[2 * r + d] < (real_t)INFINITY)) continue;
          const int *from = d ? net->products + 3 * r : net->reactants + 3 * r;
          const int *to = d ? net->reactants + 3 * r : net->products + 3 * r;
          int consumes = 0;
          for (int a = 0; a < 3; ++a) consumes |= from[a] == u;
          if (!consumes) continue;
          for (int b = 0; b < 3; ++b) {
            int v = to[b];
            if (v < 0 || v == u || done[v]) continue;
            real_t cand = dist[u] + w[2 * r + d];
            if (cand < dist[v]) dist[v] = cand, pred[v] = u, via[v] = r | (d ? (1 << 30) : 0);
          }
        }
    }
    for (int i = 0; i < ns; ++i) {
      dist_out[(long)i * ld + c] = (double)dist[i];
      if (pred_out) pred_out[(long)i * ld + c] = pred[i];
      if (via_out) via_out[(long)i * ld + c] = via[i];
    }
  }
  free(dist);
  free(w);
  free(done);
  free(pred);
  return 0;
}

/* ---------------------------------------------------------------- f4: thermochemical-equilibrium composition
 * PAPER.md:248 (section 2.5): "the initial atmospheric composition can be specified using ... (i) equilibrium
 * abundances from the built-in equilibrium chemistry solver NEXOCHEM"; a Gibbs-energy
 * minimisation that reuses the NASA-7 thermochemistry.  The paper names the solver and gives no method, so the
 * oracle computes the DEFINITION (reading E1): for a column at (T, P) with element abundances b_e, the
 * equilibrium composition of an ideal gas mixture is the n >= 0 that minimises
 *     G / RT = sum_i n_i ( G_i/RT (T) + ln (n_i / N) + ln (P / P0) ),   N = sum_i n_i,
 * subject to sum_i a_ie n_i = b_e for every element e (a_ie = the composition matrix; a column of it with entries of
 * both signs is the charge, b = 0 for a neutral gas).  Only the ratios of b matter; the result is returned as number
 * densities n_i = x_i P / (k_B T), x_i = n_i / N.  G is strictly convex on the feasible set, so the minimiser is
 * unique and is characterised by the Lagrange conditions
 *     G_i/RT + ln x_i + ln (P / P0) = sum_e a_ie pi_e  for every species,   sum_i x_i = 1,   sum_i a_ie x_i  ~  b_e,
 * pi_e = the element potentials (over RT).  These are also exactly the conditions under which every reversible
 * reaction of the kinetics has q_f = q_r (O3: K_c from the same G_i/RT), i.e. dn/dt = 0 without photolysis.
 * Method: the Lagrange conditions are solved by the damped Newton iteration of Gordon & McBride (NASA RP-1311, 1994,
 * section 2.3, gas phase only): unknowns ln n_i, ln N; each iteration solves the (n_e + 1) x (n_e + 1) system
 *     sum_e' ( sum_i a_ie a_ie' n_i ) pi_e' + ( sum_i a_ie n_i ) dlnN = b_e - sum_i a_ie n_i + sum_i a_ie n_i mu_i
 *     sum_e' ( sum_i a_ie' n_i ) pi_e'      + ( sum_i n_i - N ) dlnN  = N - sum_i n_i + sum_i n_i mu_i
 * with mu_i = G_i/RT + ln (n_i / N) + ln (P / P0), then dln n_i = -mu_i + sum_e a_ie pi_e + dlnN, and applies
 * lambda = min(1, 2 / max(5 |dlnN|, max over species with ln (n_i/N) > -18.42 of |dln n_i|),
 *              min over the other species with dln n_i > 0 of |(-ln (n_i/N) - 9.21) / (dln n_i - dlnN)|)
 * of the step.  Start: b scaled to sum 1, N = 0.1, n_i = 0.1 / n_species.  Converged when lambda = 1,
 * max_i n_i |dln n_i| / sum n <= tol, N |dlnN| / sum n <= tol and |sum_i a_ie n_i - b_e| <= tol max(b_e,
 * sum_i |a_ie| n_i) for every e (relative to the element's OWN abundance: a trace element carried by one inert
 * species is decoupled from all the others, and only this residual sees it);
 * then ln n_i = ln N + sum_e a_ie pi_e - G_i/RT - ln (P / P0) is taken for EVERY species (trace species sit exactly
 * on the Lagrange condition).  The linear system is solved by Gaussian elimination with partial pivoting after each
 * row is divided by its largest entry (a charge row is many orders below the element rows).  Plain loops, one
 * column at a time, real_t arithmetic.
 * Outputs: n [n_species][ld]; pi (optional) [n_elements][ld]; iters (optional) [ld] = iterations used, negated if
 * max_iter was reached first.  Returns 0, -1 (memory), -2 (singular system), -3 (an element with b_e <= 0 whose
 * composition column has no negative entry).
 * Pins (tests/test_oracle_equilibrium.py): A <=> B and A2 <=> 2 A in closed form; the Lagrange conditions rebuilt by
 * the test from orc_thermo (least squares over pi); element conservation and sum x = 1; the kinetic fixed point
 * (orc_source gives dn/dt = 0 at the returned composition when J = 0); G at the returned composition below G at
 * feasible perturbations; invariance under scaling b; a pressure shift moves A2 <=> 2 A the Le Chatelier way. */
static int solve_scaled_real(long n, real_t *A, real_t *b, real_t *x) {
  for (long i = 0; i < n; ++i) {
    real_t m = 0;
    for (long j = 0; j < n; ++j)
      if (R_FABS(A[i * n + j]) > m) m = R_FABS(A[i * n + j]);
    if (m == 0) return -1;
    for (long j = 0; j < n; ++j) A[i * n + j] /= m;
    b[i] /= m;
  }
  return solve_dense_real(n, A, b, x);
}

int orc_equilibrium(const orc_network *net, long ncol, long ld, const double *T, const double *P, const double *b_in,
                    int max_iter, double tol, double *n_out, double *pi_out, int *iters_out) {
  const int ns = net->n_species, ne = net->n_elements, m = ne + 1;
  real_t *lnn = (real_t *)malloc(sizeof(real_t) * (size_t)(4 * ns + 2 * m + 2 * m * m + ne));
  if (!lnn) return -1;
  real_t *c = lnn + ns, *dln = c + ns, *nn = dln + ns, *M = nn + ns, *rhs = M + m * m, *sol = rhs + m, *b = sol + m;
  int rc = 0;
  for (long col = 0; col < ncol && rc == 0; ++col) {
    const real_t Tc = (real_t)T[col], lnP = R_LOG((real_t)P[col] / P_REF);
    real_t bsum = 0;
    for (int e = 0; e < ne; ++e) {
      b[e] = (real_t)b_in[(long)e * ld + col];
      int has_neg = 0;
      for (int i = 0; i < ns; ++i) has_neg |= net->composition[i * ne + e] < 0;
      if (!(b[e] > 0) && !has_neg) rc = -3;
      if (b[e] > 0) bsum += b[e];
    }
    if (rc != 0) break;
    for (int e = 0; e < ne; ++e) b[e] /= bsum;
    for (int i = 0; i < ns; ++i) {
      c[i] = nasa_g(nasa_set(net, i, Tc), Tc) + lnP;
      lnn[i] = R_LOG((real_t)0.1 / (real_t)ns);
    }
    real_t lnN = R_LOG((real_t)0.1);
    int it = 0, done = 0;
    while (!done && it < max_iter) {
      ++it;
      const real_t N = R_EXP(lnN);
      for (int k = 0; k < m * m; ++k) M[k] = 0;
      for (int k = 0; k < m; ++k) rhs[k] = 0;
      real_t sumn = 0, sumnmu = 0;
      for (int i = 0; i < ns; ++i) {
        const real_t ni = R_EXP(lnn[i]), mu = c[i] + lnn[i] - lnN;
        nn[i] = ni;
        sumn += ni, sumnmu += ni * mu;
        for (int e = 0; e < ne; ++e) {
          const real_t ae = (real_t)net->composition[i * ne + e];
          if (ae == 0) continue;
          for (int f = 0; f < ne; ++f) M[e * m + f] += ae * (real_t)net->composition[i * ne + f] * ni;
          M[e * m + ne] += ae * ni;
          M[ne * m + e] += ae * ni;
          rhs[e] += ae * ni * mu;
        }
      }
      for (int e = 0; e < ne; ++e) rhs[e] += b[e] - M[e * m + ne];
      M[ne * m + ne] = sumn - N;
      rhs[ne] = N - sumn + sumnmu;
      if (solve_scaled_real(m, M, rhs, sol) != 0) { rc = -2; break; }
      const real_t dlnN = sol[ne];
      real_t big = 5 * R_FABS(dlnN), lam2 = 1;
      for (int i = 0; i < ns; ++i) {
        real_t d = -(c[i] + lnn[i] - lnN) + dlnN;
        for (int e = 0; e < ne; ++e) d += (real_t)net->composition[i * ne + e] * sol[e];
        dln[i] = d;
        const real_t lx = lnn[i] - lnN;
        if (lx > (real_t)-18.420681L) {
          if (R_FABS(d) > big) big = R_FABS(d);
        } else if (d > 0) {
          const real_t l = R_FABS((-lx - (real_t)9.2103404L) / (d - dlnN));
          if (l < lam2) lam2 = l;
        }
      }
      real_t lam = big > 2 ? 2 / big : 1;
      if (lam2 < lam) lam = lam2;
      real_t err = 0, newsum = 0;
      for (int i = 0; i < ns; ++i) lnn[i] += lam * dln[i], newsum += R_EXP(lnn[i]);
      lnN += lam * dlnN;
      for (int i = 0; i < ns; ++i) {
        const real_t w = R_EXP(lnn[i]) * R_FABS(dln[i]) / newsum;
        if (w > err) err = w;
      }
      if (R_EXP(lnN) * R_FABS(dlnN) / newsum > err) err = R_EXP(lnN) * R_FABS(dlnN) / newsum;
      real_t res = 0;   /* per element, relative to its own abundance (to the charge carried, for a signed column) */
      for (int e = 0; e < ne; ++e) {
        real_t s = -b[e], sa = 0;
        for (int i = 0; i < ns; ++i) {
          const real_t t = (real_t)net->composition[i * ne + e] * R_EXP(lnn[i]);
          s += t, sa += R_FABS(t);
        }
        const real_t ref = b[e] > sa ? b[e] : sa;
        if (R_FABS(s) > res * ref) res = R_FABS(s) / ref;
      }
      done = lam == 1 && err <= (real_t)tol && res <= (real_t)tol;
    }
    if (rc != 0) break;
    const real_t ntot = (real_t)P[col] / (K_BOLTZ * Tc);
    for (int i = 0; i < ns; ++i) {
      real_t lx = -c[i];   /* ln x_i = sum_e a_ie pi_e - G_i/RT - ln (P/P0), every species on the Lagrange condition */
      for (int e = 0; e < ne; ++e) lx += (real_t)net->composition[i * ne + e] * sol[e];
      n_out[(long)i * ld + col] = (double)(ntot * R_EXP(lx));
    }
    if (pi_out)
      for (int e = 0; e < ne; ++e) pi_out[(long)e * ld + col] = (double)sol[e];
    if (iters_out) iters_out[col] = done ? it : -it;
  }
  free(lnn);
  return rc;
}
