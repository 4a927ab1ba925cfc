/* xodiac.h -- C ABI of libxodiac: the batched fp64 chemical source term of the XODIAC 1-D
 * photochemical kinetics model (arxiv 2512.06729), hand-written CUDA for sm_100a (B200).
 *
 * The path (citations are /root/reference/PAPER.md lines):
 *   a2 NASA-7 thermochemistry  cp/R, H/RT, S/R, G/RT
 *   a3 forward coefficients    k = alpha T_b^beta exp(-gamma/T)      PAPER.md:116-124 (Eq. 7)
 *   a4 three-body falloff      Lindemann k0[M]/(1 + k0[M]/k_inf)     PAPER.md:146-159 (Eq. 10-12)
 *                              x Troe broadening (BASELINE.json north_star; reading F1)
 *   a5 photolysis              k_f = J (input), dn_A/dt = -k_ph n_A
 *   a6 reverse coefficients    k_r = k_f / K_c,                      PAPER.md:219-235 (Eq. 13-15)
 *                              K_c = exp(-dG/RT) (P0/(k_B T))^dnu
 *   a7 rates of progress       q_f = k_f prod n_reactant, q_r = k_r prod n_product
 *   a8 production and loss     dn_i/dt = P_i - L_i = sum_r nu_ir (q_f,r - q_r,r)   PAPER.md:53 (Eq. 1)
 *   a9 Jacobian values         d(dn_i/dt)/dn_j on a fixed CSR pattern (BASELINE.json config 5)
 *
 * Conventions
 *   Units       cgs: T [K], P [dyn cm^-2] (1 bar = 1e6), n [cm^-3], J [s^-1], E/R [K],
 *               k [s^-1 | cm^3 s^-1 | cm^6 s^-1].  k_B = 1.380649e-16 erg/K, P0 = 1e6 dyn cm^-2.
 *   Layout      every per-column array is [row][ld], the column index contiguous, ld >= ncol the
 *               row pitch in elements.  A column is one (atmosphere, layer) pair.
 *   Order       kf, kr rows are the USER's reaction order.  Row p of J is the p-th XOD_PHOTO
 *               reaction in user order.  The type-sorted order is internal (xod_network_perm).
 *   Memory      xod_network_desc pointers are HOST memory, copied by create.  Every pointer of a
 *               compute call is DEVICE memory owned by the caller, except in the *_host call.
 *   Streams     `stream` is a cudaStream_t passed as void* (NULL = default stream) of the network's
 *               device, which must be the calling thread's current device (otherwise XOD_ERR_CUDA;
 *               the library never switches the caller's device).  Compute calls only enqueue work,
 *               never synchronise and may be captured into a CUDA graph; the *_host call
 *               synchronises.
 *   Errors      argument problems return synchronously with nothing enqueued; xod_last_error()
 *               (thread-local) says what was wrong.  IEEE overflow/underflow in results (k_r
 *               beyond the double range, reading R5) is not an error.
 *   Threads     a network is immutable after create; concurrent calls on different streams are
 *               legal if each has its own workspace.
 *   No CPU fallback exists: without a CUDA device every compute call returns XOD_ERR_CUDA.
 */
#ifndef XODIAC_H
#define XODIAC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct xod_network xod_network; /* opaque; owns its device tables */

typedef enum {
  XOD_OK = 0,
  XOD_ERR_INVALID_ARG = 1, /* NULL pointer, bad size, index out of range, bad type, Fc not in (0,1] ... */
  XOD_ERR_UNBALANCED = 2,  /* a reaction does not conserve an element (names the reaction) */
  XOD_ERR_ALLOC = 3,
  XOD_ERR_CUDA = 4,        /* no device, or a launch / copy failed */
  XOD_ERR_WORKSPACE = 5    /* workspace NULL or smaller than xod_*_workspace_bytes */
} xod_status;

/* Reaction categories of PAPER.md:105; also the internal sort key (north_star: "sorts reactions by
 * type (unimolecular, bimolecular, three-body falloff, photolysis)").  XOD_UNI / XOD_BI are thermal
 * non-falloff reactions with one / two-or-three listed reactants. */
enum { XOD_UNI = 0, XOD_BI = 1, XOD_FALLOFF = 2, XOD_PHOTO = 3 };

enum {
  XOD_FLAG_SKIP_BALANCE_CHECK = 1u,
  XOD_FLAG_BUILD_LU = 2u /* also build the symbolic LU of the Jacobian pattern (needed by xod_newton_step) */
};

typedef struct {
  int32_t n_species, n_elements, n_reactions;
  const int32_t *composition; /* [n_species][n_elements] atoms per element; may be negative (charge
                                 carried as an extra "element", cf. C -> C+ + e-) */
  const double *nasa_lo;      /* [n_species][7] a1..a7, low-temperature range */
  const double *nasa_hi;      /* [n_species][7] a1..a7, high-temperature range */
  const double *t_mid;        /* [n_species]; T <= t_mid uses nasa_lo, else nasa_hi */
  const int32_t *type;        /* [n_reactions] XOD_* */
  const int32_t *reactants;   /* [n_reactions][3], -1 padded; a stoichiometric 2 is the index repeated */
  const int32_t *products;    /* [n_reactions][3], -1 padded; the third body M is never listed */
  const uint8_t *reversible;  /* [n_reactions]; must be 0 for XOD_PHOTO */
  const double *arrh;         /* [n_reactions][3] alpha, beta, gamma (Eq. 7); k_inf for XOD_FALLOFF
                                 (Eq. 11); ignored for XOD_PHOTO */
  const double *arrh_low;     /* [n_reactions][3] alpha0, beta0, gamma0 (Eq. 10); XOD_FALLOFF only */
  const double *troe_fc;      /* [n_reactions] Fc in (0,1]; 1 = pure Lindemann (Eq. 12); XOD_FALLOFF only */
  const double *t_ref;        /* [n_reactions] 1 = modified Arrhenius, 300 = Kooij (Eq. 7); NULL = all 1 */
  uint32_t flags;             /* XOD_FLAG_* */
} xod_network_desc;

/* a0: validate, sort by type, build the SoA parameter tables, the source CSR and the Jacobian CSR
 * with its term lists, and upload them to `cuda_device`.  With cuda_device < 0 only the host side
 * is built (introspection works, compute calls fail with XOD_ERR_CUDA). */
xod_status xod_network_create(const xod_network_desc *desc, int cuda_device, xod_network **out);
void xod_network_destroy(xod_network *net);
const char *xod_last_error(void);

/* ---- introspection: host outputs, caller-allocated; any output pointer may be NULL */
xod_status xod_network_sizes(const xod_network *net, int32_t *n_species, int32_t *n_reactions,
                             int32_t *n_photo, int64_t *nnz_source, int64_t *nnz_jac,
                             int64_t *n_jac_terms);
/* packed (type-sorted, stable) position -> user reaction index, [n_reactions] */
xod_status xod_network_perm(const xod_network *net, int32_t *packed_to_user);
/* row p of J -> user reaction index, [n_photo] */
xod_status xod_network_photo_index(const xod_network *net, int32_t *user_rxn_of_photo_row);
/* source CSR (reading S2): row i = species i; entries = reactions with nu_ir != 0 in
 * ascending USER reaction index; row_ptr [n_species+1], rxn and nu [nnz_source] */
xod_status xod_network_source_csr(const xod_network *net, int64_t *row_ptr, int32_t *rxn, int32_t *nu);
/* Jacobian pattern (readings J1, J2): union over reactions of (distinct species)^2 plus the
 * diagonal; rows = species, ascending column indices; row_ptr [n_species+1], col [nnz_jac] */
xod_status xod_network_jac_pattern(const xod_network *net, int64_t *row_ptr, int32_t *col);

/* layout of the single-kernel fused path (xod_source_fused), info[10]: enabled, reactions per chunk,
 * chunks, accumulator rows, thermo breakpoints, shared-memory bytes per CTA, padded reactions,
 * production/loss warp tasks, padded production/loss entries, bytes of the reverse-coefficient table */
xod_status xod_network_fused_info(const xod_network *net, int64_t *info);

/* host-only view of the fused path's parameter blocks for one thermo interval (0 .. breakpoints), for
 * tests of the packer's arithmetic.  Arrays of info[6] = npad padded reactions: user_rxn (-1 = padding
 * slot), kind (0 UNI/BI, 1 FALLOFF, 2 PHOTO, 3 padding), coef [npad][16] =
 * c0 c1 c2 | C0 C1 C2 D2 D3 D4 D5 | l0 l1 l2 log2Fc cN | 0  with
 *   log2 k_f (or log2 k_inf) = c0 + c1 log2 T + c2/T                                        (Eq. 7, 11)
 *   C0 + C1 log2 T + C2/T - T (D2 + T (D3 + T (D4 + T D5))) = log2 k_r (UNI/BI) or log2 (k_r/k_f) (FALLOFF)
 *   log2 k0 = l0 + l1 log2 T + l2/T                                                           (Eq. 10)
 * An irreversible reaction or a padding slot is reported with C0 = -inf (k_r = 0).
 * breakpoints [info[4]]: the sorted distinct t_mid values; a column with T is in interval #{bp < T}.
 * Any output may be NULL. */
xod_status xod_network_fused_params(const xod_network *net, int32_t interval, int32_t *user_rxn, int32_t *kind,
                                    double *coef, double *breakpoints);

/* layout of the tiled Jacobian kernel (xod_jacobian), info[8]: enabled, slots per chunk, chunks, units,
 * accumulator rows, shared-memory bytes per CTA, distinct derivative slots (k reads per column), padded
 * schedule entries.  A slot is one distinct d q_{r,dir} / d n_j; the pattern's terms share them. */
xod_status xod_network_jac_info(const xod_network *net, int64_t *info);

/* host-only consistency check of the internal tables of the fused path (decoded as the kernel
 * decodes them): every source-CSR entry and every Jacobian term scheduled exactly once, no
 * accumulator row shared by two row tasks of a chunk, species slots intact; with XOD_FLAG_BUILD_LU also the
 * implicit step's rows, target slots and block schedule (every (row, pivot) pair applied exactly once, pivots ascending).  XOD_OK, or XOD_ERR_INVALID_ARG with xod_last_error. */
xod_status xod_network_selfcheck(const xod_network *net);

/* ---- tuning knobs (optional; defaults are chosen for B200) */
enum {
  XOD_TUNE_CHUNK_COLS = 0, /* columns per pipeline chunk of the fused source call (0 = default) */
  XOD_TUNE_TIMING = 1,     /* != 0: bracket every kernel launch with a CUDA event pair (measurement) */
  XOD_TUNE_SPLIT = 2,      /* reaction splits per column tile of the single-kernel fused path (0 = auto) */
  XOD_TUNE_FUSED_KERNEL = 3, /* 0: xod_source_fused uses the multi-kernel pipeline instead (default 1) */
  XOD_TUNE_JAC_TILED = 4     /* 0: xod_jacobian uses the one-warp-per-entry gather kernel instead (default 1) */
};
xod_status xod_network_tune(xod_network *net, int32_t knob, int64_t value);

/* ---- measurement: per-kernel device time of the launches made since the last read while
 * XOD_TUNE_TIMING was on.  ms, launches: [XOD_KERNEL_COUNT], indexed by XOD_KERNEL_*; either may
 * be NULL.  Synchronises on the last recorded event, then clears the record. */
enum { XOD_KERNEL_THERMO = 0, XOD_KERNEL_PROLOGUE = 1, XOD_KERNEL_RATES = 2, XOD_KERNEL_RATES_FROM_K = 3,
       XOD_KERNEL_SOURCE = 4, XOD_KERNEL_JACOBIAN = 5, XOD_KERNEL_FUSED = 6, XOD_KERNEL_FUSED_COMBINE = 7,
       XOD_KERNEL_RATE_COEFFS = 8, XOD_KERNEL_JAC_TILED = 9, XOD_KERNEL_NEWTON_ASSEMBLE = 10,
       XOD_KERNEL_LU_FACTOR = 11, XOD_KERNEL_LU_SOLVE = 12, XOD_KERNEL_PHOTO_GEMM = 13, XOD_KERNEL_PHOTO_FLUX = 14,
       XOD_KERNEL_TRANSPORT = 15, XOD_KERNEL_PATH_WEIGHTS = 16, XOD_KERNEL_PATHWAY = 17, XOD_KERNEL_COUNT = 18 };
xod_status xod_network_timing_read(xod_network *net, double *ms, int64_t *launches);
/* kernels launched by this library in this process so far (all networks, all threads) */
int64_t xod_launch_count(void);

/* ---- a2: NASA-7 thermochemistry (PAPER.md:650-653 two coefficient sets; PAPER.md:671 G/RT, 673 cp/R;
 * H/RT, S/R standard forms, reading T1; set chosen by T <= t_mid, reading T3).  T [ld] device;
 * each output [n_species][ld] device, any may be NULL; columns >= ncol are not touched.
 * Errors: XOD_ERR_INVALID_ARG (NULL T, ncol < 0, ld < ncol), XOD_ERR_CUDA. */
xod_status xod_thermo(const xod_network *net, int64_t ncol, int64_t ld, const double *T,
                      double *cp_R, double *h_RT, double *s_R, double *g_RT, void *stream);

/* ---- a1, a3-a6: forward and reverse rate coefficients: Eq. 7, Eq. 10-12 with
 * [M] = P/(k_B T) and Troe F (reading F1), k_f = J for photolysis,
 * k_r = k_f/K_c, K_c = exp(-dG/RT)(P0/k_B T)^dnu (Eq. 13-15).  T, P [ld]; J
 * [n_photo][ld] (may be NULL if n_photo == 0); kf, kr [n_reactions][ld] in user order, either may be
 * NULL; all device memory owned by the caller.  kr rows of irreversible and photolysis reactions are
 * 0; values beyond the double range saturate as IEEE does (reading R5).  The workspace (device,
 * >= xod_rate_coeffs_workspace_bytes) is only used by the multi-kernel fallback.
 * Errors: XOD_ERR_INVALID_ARG, XOD_ERR_WORKSPACE, XOD_ERR_CUDA; nothing is enqueued on error. */
size_t xod_rate_coeffs_workspace_bytes(const xod_network *net, int64_t ncol);
xod_status xod_rate_coeffs(const xod_network *net, int64_t ncol, int64_t ld, const double *T,
                           const double *P, const double *J, double *kf, double *kr,
                           void *workspace, size_t workspace_bytes, void *stream);

/* ---- a7-a8: dn/dt from stored coefficients: q_f = k_f prod n_reactant, q_r = k_r prod n_product
 * (north_star; PAPER.md:211 for photolysis), dn_i/dt = P_i - L_i = sum_r nu_ir (q_f,r - q_r,r)
 * (Eq. 1).  kf, kr [n_reactions][ld] user order; n, dndt [n_species][ld]; prod, loss
 * optional (both or neither): P_i = sum of positive terms, L_i = sum of |negative terms|.  Device
 * memory owned by the caller; workspace >= xod_source_workspace_bytes(net, ncol).
 * Errors: XOD_ERR_INVALID_ARG, XOD_ERR_WORKSPACE, XOD_ERR_CUDA. */
size_t xod_source_workspace_bytes(const xod_network *net, int64_t ncol);
/* the (much smaller) requirement when prod and loss are NULL: only the partial sums of the single-kernel path */
size_t xod_source_workspace_bytes_dndt(const xod_network *net, int64_t ncol);
xod_status xod_source(const xod_network *net, int64_t ncol, int64_t ld, const double *kf,
                      const double *kr, const double *n, double *dndt, double *prod, double *loss,
                      void *workspace, size_t workspace_bytes, void *stream);

/* ---- a1-a8 fused: (T, P, J, n) -> dn/dt without k_f, k_r ever reaching HBM (the headline path).
 * Which code runs (also for xod_source): with prod and loss NULL, ONE kernel per call (k_fused; a second launch for
 * the last partial round of column tiles and a combine launch when tiles are split over SMs).  With prod and loss
 * given, a pipeline of three kernels per 1 024-column chunk with the rates of progress in an L2-resident scratch
 * (measured 2.3x the time of the dn/dt-only call in round 1): the single kernel keeps one accumulator tile per
 * species in shared memory and P, L would need two more.  Ask for P and L only where they
 * are needed (diagnostics); a solver needs dn/dt.  Results are the same on both paths to the stated tolerance. */
size_t xod_source_fused_workspace_bytes(const xod_network *net, int64_t ncol);
/* the requirement when prod and loss are NULL (0-few MB instead of the multi-kernel scratch of the P/L variant) */
size_t xod_source_fused_workspace_bytes_dndt(const xod_network *net, int64_t ncol);
xod_status xod_source_fused(const xod_network *net, int64_t ncol, int64_t ld, const double *T,
                            const double *P, const double *J, const double *n, double *dndt,
                            double *prod, double *loss, void *workspace, size_t workspace_bytes,
                            void *stream);

/* ---- a9: Jacobian values jac[e][col] = d(dn_i/dt)/dn_j for entry e = (i, j) of the pattern of
 * xod_network_jac_pattern (BASELINE.json config 5; k_f, k_r, [M], J do not depend on n, reading J3):
 * sum_r nu_ir (d q_f,r/d n_j - d q_r,r/d n_j), never formed as q/n_j, so n_j = 0 is exact (reading Q2).
 * kf, kr [n_reactions][ld], n [n_species][ld], jac [nnz_jac][ld]: device memory owned by the caller.
 * Errors: XOD_ERR_INVALID_ARG (NULL, sizes, ncol > 2097120), XOD_ERR_CUDA. */
xod_status xod_jacobian(const xod_network *net, int64_t ncol, int64_t ld, const double *kf,
                        const double *kr, const double *n, double *jac, void *stream);

/* ---- f1: one Newton iteration of a backward-Euler step, batched over columns.
 * "The discretized continuity equation is a stiff ordinary differential equation (ODE), implicit solvers are
 * the most suitable choice ... the lower-order backward Euler method ... the higher-order DLSODES solver"
 * (PAPER.md:85).  With f = dn/dt (Eq. 1 without transport) and Jac its Jacobian, a backward-Euler step of
 * size dt from n_old solves F(y) = y - n_old - dt f(y) = 0; this call performs
 *     (I - dt Jac(y)) delta = -F(y),     y <- y + delta
 * for every column: f(y) by the kernels of xod_source, Jac(y) by those of xod_jacobian, then a sparse LU
 * without pivoting in a fixed minimum-degree order (one symbolic factorisation per network, built at create
 * with XOD_FLAG_BUILD_LU; the numeric factorisation runs with columns as lanes) and the two triangular
 * solves.  Iterate the call until delta is small; with dt[c] = gamma it is also the Newton step of a BDF
 * formula whose history terms the caller folds into n_old.
 * kf, kr [n_reactions][ld] (xod_rate_coeffs; T, P are fixed during a step), n_old, y [n_species][ld], dt [ld]
 * (per column, seconds), delta [n_species][ld] optional (NULL to skip): device memory owned by the caller; y is
 * updated in place; workspace >= xod_newton_workspace_bytes(net, ncol) (columns are processed 2 048 at a time).
 * A zero pivot gives IEEE inf/NaN in that column (no pivoting, no error).
 * Errors: XOD_ERR_INVALID_ARG (NULL, sizes, network created without XOD_FLAG_BUILD_LU or without the
 * single-kernel tables), XOD_ERR_WORKSPACE, XOD_ERR_CUDA.
 * xod_network_lu_info: info[8] = enabled, nonzeros of L + U (with fill), (row, pivot) pairs, multiply-add
 * updates of one factorisation, longest row, rows factorised together per block, U values read per column by the
 * block schedule (its memory traffic / 8 bytes; without blocks it would equal the updates), pivot steps.  xod_network_lu_pattern: perm[p] = species eliminated p-th;
 * row p of the filled pattern = permuted column indices, ascending (L part, diagonal, U part). */
xod_status xod_network_lu_info(const xod_network *net, int64_t *info);
xod_status xod_network_lu_pattern(const xod_network *net, int32_t *perm, int64_t *row_ptr, int32_t *col);
size_t xod_newton_workspace_bytes(const xod_network *net, int64_t ncol);
xod_status xod_newton_step(const xod_network *net, int64_t ncol, int64_t ld, const double *kf, const double *kr,
                           const double *n_old, const double *dt, double *y, double *delta, void *workspace,
                           size_t workspace_bytes, void *stream);

/* ---- f2: photolysis rate constants, the J input of the calls above.
 *   tau(z, lambda) = sum over the gas above z of (sigma_a,i + sigma_s,i) n_i dz
 *   J(z, lambda)   = J0(lambda) exp(-tau / mu) + J_diff(z, lambda)
 *   k_ph,i(z)      = t_f * integral J(z, lambda) sigma_i(lambda) d lambda
 * Discretisation (readings H1-H4): column = atmosphere * n_layers + layer, layer 0 at the bottom;
 * tau at the CENTRE of a layer (everything above it plus half of its own kappa dz); rectangle rule over the
 * wavelength bins, sum_b J sigma dlambda_b (uniform or non-uniform widths); J_diff = (J_up + J_down)/2
 * is an input (NULL = 0).  t_f is the irradiated-time fraction.
 * xod_photo_desc (HOST pointers, copied): dlambda [n_bins] bin widths; abs_species [n_abs] species index of each
 * extinction row; sigma_ext [n_abs][n_bins] = sigma_a + sigma_s in cm^2; sigma_ph [n_photo][n_bins] = the
 * reaction-specific cross-section (PHIDRATES kind, or molecular cross-section times quantum yield)
 * of the p-th XOD_PHOTO reaction in user order, i.e. row p of J.  All values finite and >= 0.
 * xod_photo_rates: n [n_species][ld], dz [ld] layer thickness in cm, j0 [n_atm][n_bins] photons cm^-2 s^-1 per unit
 * of dlambda at the top of the atmosphere, j_diff [n_bins][ld] or NULL, mu [n_atm] cosine of the zenith angle (> 0),
 * t_f [n_atm], J [n_photo][ld] out: device memory owned by the caller; columns >= n_atm * n_layers are not touched;
 * workspace >= xod_photo_workspace_bytes(photo, n_atm * n_layers) (one [n_bins][columns] array).
 * Errors: XOD_ERR_INVALID_ARG (NULL, sizes, n_layers > 907, n_atm > 65535), XOD_ERR_WORKSPACE, XOD_ERR_CUDA.
 * The photo object keeps a pointer to `net`: destroy it before the network. */
typedef struct xod_photo xod_photo;
typedef struct {
  int32_t n_bins, n_abs;
  const double *dlambda;
  const int32_t *abs_species;
  const double *sigma_ext;
  const double *sigma_ph;
} xod_photo_desc;
xod_status xod_photo_create(const xod_network *net, const xod_photo_desc *desc, xod_photo **out);
void xod_photo_destroy(xod_photo *photo);
size_t xod_photo_workspace_bytes(const xod_photo *photo, int64_t ncol);
xod_status xod_photo_rates(const xod_photo *photo, int64_t n_atm, int64_t n_layers, int64_t ld, const double *n,
                           const double *dz, const double *j0, const double *j_diff, const double *mu,
                           const double *t_f, double *J, void *workspace, size_t workspace_bytes, void *stream);

/* ---- f3: the molecular-diffusion transport terms of the continuity equation
 * (PAPER.md:73-83).  Eq. 4, half levels k +- 1/2 being arithmetic means of k and k +- 1:
 *   d_{k+-1/2} = D_{k+-1/2} / (2 dz^2) [ (mbar - m_y) g dz / (k_B T_{k+-1/2}) - alpha_T / T_{k+-1/2} (T_{k+-1} - T_k) ]
 * and the part of Eq. 3 that is not P - L, with N = n_gas:
 *   tr_{y,k} = - d_{k+1/2} (N_{k+1/2}/N_{k+1}) n_{y,k+1} - [ d_{k+1/2} (N_{k+1/2}/N_k) - d_{k-1/2} (N_{k-1/2}/N_k) ] n_{y,k}
 *              + d_{k-1/2} (N_{k-1/2}/N_k) n_{y,k-1}
 * so that dn/dt of Eq. 1 = (xod_source's dn/dt) + tr.  Two extraction garbles of the printed Eq. 3 (an index
 * "n_gas,j" and a stray "/2") are dropped (reading V1); zero-flux boundaries: no term reaches
 * across the bottom or top layer of an atmosphere (V2); eddy diffusion does not appear.
 * Column = atmosphere * n_layers + layer, layer 0 at the bottom.  n, D [n_species][ld] (D: molecular diffusion
 * coefficient of each species in each layer, cm^2 s^-1, an input: reading V3), T, n_gas [ld], mass, alpha_T
 * [n_species] (g; thermal diffusion factor), mbar, grav, dz [n_atm] (mean molecular mass in g, gravity in cm s^-2,
 * uniform layer spacing in cm), tr [n_species][ld] out: device memory owned by the caller; columns >= n_atm *
 * n_layers are not touched.  Errors: XOD_ERR_INVALID_ARG, XOD_ERR_CUDA. */
xod_status xod_transport(const xod_network *net, int64_t n_atm, int64_t n_layers, int64_t ld, const double *n,
                         const double *T, const double *n_gas, const double *D, const double *mass,
                         const double *alpha_T, const double *mbar, const double *grav, const double *dz, double *tr,
                         void *stream);

/* ---- f4: the reaction pathway analyser.  "identifies the kinetically fastest reaction
 * pathway by minimizing the cumulative sum of inverse reaction rates" (after Dijkstra 1959); "the
 * rate-limiting step, defined as the slowest reaction in each pathway".
 * Graph of a column (reading W1): nodes = species; every reaction direction with a positive finite rate of
 * progress q (q_f = k_f prod n_reactant, q_r = k_r prod n_product, reversible reactions only) gives a directed edge of
 * weight 1/q from each distinct species it consumes to each distinct species it forms.  For every column the call
 * returns, for all species v, dist[v][col] = the smallest sum of weights over routes source -> v (0 for the source,
 * +inf if unreachable), pred[v][col] = the species before v on such a route and via[v][col] = the USER index of its
 * last reaction, bit 30 set for the reverse direction (both -1 for the source and for unreachable species).  Walking
 * pred back from a target lists the route; its largest 1/q step is the rate-limiting one.  dist is unique; when
 * several routes are equally short, pred/via name one of them (fixed, deterministic choice).
 * kf, kr [n_reactions][ld], n, dist [n_species][ld] fp64, pred, via [n_species][ld] int32: device memory owned by the
 * caller; workspace >= xod_pathway_workspace_bytes (the edge weights, [2 n_reactions][columns]).
 * Errors: XOD_ERR_INVALID_ARG (NULL, sizes, source out of range, tables unavailable: n_species or 2 n_reactions
 * >= 65535, or the tiles exceed shared memory), XOD_ERR_WORKSPACE, XOD_ERR_CUDA. */
size_t xod_pathway_workspace_bytes(const xod_network *net, int64_t ncol);
xod_status xod_pathway(const xod_network *net, int64_t ncol, int64_t ld, const double *kf, const double *kr,
                       const double *n, int32_t source, double *dist, int32_t *pred, int32_t *via, void *workspace,
                       size_t workspace_bytes, void *stream);

/* ---- f4: the thermochemical-equilibrium composition, the start the paper takes from its
 * "built-in equilibrium chemistry solver" (the paper names the solver, not a method).
 * Definition (reading E1): for every column the n >= 0 that minimises the Gibbs energy of an ideal gas
 * mixture, G/RT = sum_i n_i (G_i/RT(T) + ln(n_i/N) + ln(P/P0)), N = sum_i n_i, P0 = 1 bar, among the compositions
 * with sum_i a_ie n_i proportional to the element abundances b_e (a = the composition matrix given to
 * xod_network_create, G_i/RT = the NASA-7 polynomial of xod_thermo), returned as number densities with
 * sum_i n_i = P / (k_B T).  Equivalently (Lagrange conditions) G_i/RT + ln x_i + ln(P/P0) = sum_e a_ie pi_e for every
 * species; at this composition every reversible reaction of the network has equal forward and reverse rates.
 * Method: damped Newton iteration on the Lagrange conditions in (ln n_i, ln N) after Gordon & McBride, NASA RP-1311
 * (1994), gas phase only; trace species are taken from the element potentials, so they are exact however small.
 * b [n_elements][ld]: any positive scale, only ratios matter; an element whose composition column has entries of
 * both signs (the charge) may have b = 0, i.e. a neutral gas; every other element needs b > 0.
 * max_iter <= 0 selects 500, tol = 0 selects 1e-13 (largest abundance-weighted correction, and largest element residual relative to that
 * element's own abundance, accepted).
 * n [n_species][ld] out; pi [n_elements][ld] out, optional: the element potentials over RT; iters [ld] out, optional
 * (int32): iterations used, NEGATIVE if max_iter was reached first, 0 if the column's inputs were rejected (T, P or b
 * not positive and finite); in both failure cases the column of n and pi is NaN.  A numerically singular system (two
 * elements that only ever occur together) shows up as non-convergence, not as an error.
 * All arrays: device memory owned by the caller, column contiguous; no workspace (ln n_i is kept in n while the
 * iteration runs).  Errors: XOD_ERR_INVALID_ARG (NULL, sizes, more than 16 elements, tol < 0), XOD_ERR_CUDA. */
xod_status xod_equilibrium(const xod_network *net, int64_t ncol, int64_t ld, const double *T, const double *P,
                           const double *b, int32_t max_iter, double tol, double *n, double *pi, int32_t *iters,
                           void *stream);

/* ---- end-to-end convenience: the fused call on HOST buffers (pinned for overlap; pageable works
 * but serialises).  Columns are processed in chunks of one round of tiles per SM through three
 * staging slots on private streams, so the H2D copy of the next chunk, the kernels of this one and
 * the D2H copy of the previous one overlap; synchronises before returning.  Staging buffers and
 * streams are owned by the network and grown on demand (not thread-safe on one network). */
xod_status xod_source_fused_host(xod_network *net, int64_t ncol, int64_t ld, const double *T,
                                 const double *P, const double *J, const double *n, double *dndt);

/* ---- debugging: synchronises the network's device and returns XOD_OK, or XOD_ERR_CUDA if the
 * device reports an error.  In the bounds-checked build of the library (-DXOD_CHECK, built by
 * `XOD_CHECK=1 python -m paper_2512_06729_b200.build`; xod_build_has_checks() == 1) every index a
 * kernel derives from the packed tables is range-checked and clamped, and this call reports the
 * first violation (kernel source line in xod_last_error) instead of the GPU faulting.  The default
 * build has no such code in its kernels. */
xod_status xod_check_status(const xod_network *net);
int32_t xod_build_has_checks(void);

/* ---- measurement helper: sustained DFMA issue rate of the device (dependent-chain-free FMA
 * loop on every SM), used as the FP64 roofline denominator.  Returns fused multiply-adds per
 * second (flops = 2x) measured over `iters` launches with CUDA events; synchronises. */
xod_status xod_probe_fp64_peak(int cuda_device, int32_t iters, double *dfma_per_second);

#ifdef __cplusplus
}
#endif
#endif /* XODIAC_H */
