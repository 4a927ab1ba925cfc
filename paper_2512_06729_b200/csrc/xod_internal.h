// xod_internal.h -- host/device tables shared by the packer, the API layer and the kernels.
// Part of libxodiac (the CUDA product path).  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <vector_types.h>
#include <string>
#include <vector>

#include "../../include/xodiac.h"

namespace xod {

// One Jacobian term: coef * k[dir][rxn] * n[o1] * n[o2]   (o < 0: factor 1)
// (SURVEY §7.3 "Jacobian as gather"; never divides by n_j.)
struct JacTerm {
  int32_t rk;   // user reaction index; bit 31 set = reverse direction (uses kr)
  int32_t o1;   // other species or -1
  int32_t o2;   // other species or -1
  float coef;   // nu_ir * m_jr, signed (reverse terms negative); |coef| <= 9, exact in fp32
};

// One warp's share of a source-CSR row inside a CTA task (see pack.cpp: build_source_schedule)
struct SrcSeg {
  int32_t row;     // species index, or -1 for an idle warp slot
  int32_t begin;   // first CSR entry
  int32_t end;     // one past the last CSR entry
  int32_t nseg;    // >0 on the FIRST segment of a row: number of segments to combine; 0 otherwise
};

constexpr int kSrcWarpsPerCta = 8;
constexpr int kSrcSegMin = 48;  // rows up to this many entries are summed by a single warp

// Device-side view (plain pointers, passed to kernels by value)
struct DevTables {
  int32_t ns, nr, n_photo;
  int32_t uni_begin, bi_begin, fo_begin, ph_begin;  // packed ranges [uni_begin,bi_begin) ...
  // per packed reaction
  const double *c0, *c1, *c2;               // log2 A - beta log2 t_ref, beta, -gamma log2 e
  const double *l0, *l1, *l2, *fcl, *cN;    // falloff extras, indexed by p - fo_begin
  const int32_t *sp;                        // [nr][6] reactants r0 r1 r2, products p0 p1 p2 (-1 none)
  const int32_t *flags;                     // bit0 reversible
  const int32_t *user;                      // packed -> user reaction index
  const int32_t *photo_row;                 // packed photolysis p - ph_begin -> row of J
  // thermo
  const double *nasa;                       // [ns][2][7] raw a1..a7 (lo, hi)
  const double *nasa_l2;                    // [ns][2][7] pre-scaled for u_i = log2(e) G_i/RT (see k_thermo.cu)
  const double *tmid;                       // [ns]
  // source CSR (device copy uses packed reaction indices = rows of q)
  const int32_t *src_rxn;                   // [nnz_source] packed index
  const float *src_nu;                      // [nnz_source]
  const SrcSeg *src_seg;                    // [n_src_tasks][kSrcWarpsPerCta]
  int32_t n_src_tasks;
  // Jacobian
  const int64_t *jac_term_ptr;              // [nnz_jac + 1]
  const JacTerm *jac_terms;
  int64_t nnz_jac;
};

// ---- tables of the single-kernel fused source path (k_fused, kernels.cuh) -------------------
// Padded packed order: the type-sorted order with each code segment (UNI+BI | FALLOFF | PHOTO)
// padded to a multiple of kFRxnPerWarp and the total to a multiple of the chunk size; padding
// slots are dummy reactions without stoichiometry entries.
constexpr int kFW = 16;           // columns per tile (one 128-byte shared-memory row)
constexpr int kFWarps = 20;       // warps per CTA
constexpr int kFRxnPerWarp = 4;   // reactions a warp evaluates per pass (8 lanes x 2 columns each)
constexpr int kFPass = kFWarps * kFRxnPerWarp;  // reactions per CTA pass
constexpr int kFSegMax = 16;      // longest row task of the production/loss phase
constexpr int kFMaxIntervals = 32;  // distinct thermo temperature intervals the fused path supports

struct FusedTask {   // one warp task of the production/loss phase: 4 row tasks run side by side
  int32_t entry_off;   // first entry (in words from the start of the chunk's entry section);
                       // entries are interleaved [step][4]
  int32_t nsteps;
  int32_t rows01;      // accumulator rows of lane groups 0, 1 (low, high 16 bits); 0xffff = idle
  int32_t rows23;
};

// Parameter blocks: one block per (thermo interval, group of kFRxnPerWarp reactions), made of
// 16-byte units indexed [unit][reaction in group]: sa, sb (species slots as int4), then double2
// pairs (c0,c1) (c2,C0) (C1,C2) (D2,D3) (D4,D5) and, for FALLOFF, (m0,m1) (m2,fcl) (cN,-).
constexpr int kFBlkArr = 7 * 64;   // bytes of a UNI/BI block
constexpr int kFBlkFo = 10 * 64;   // bytes of a FALLOFF block
constexpr int kFBlkPh = 2 * 64;    // bytes of a PHOTO block (species slots only)
constexpr int kFMetaHdr = (kFWarps + 2 + 3) / 4 * 4;  // int32 words of a chunk's schedule header (kFWarps + 1 task offsets, task count)

struct FusedDev {
  int32_t enabled;            // 0: fall back to the multi-kernel path
  int32_t npad, arr_end, fo_end, ph_end;   // padded packed ranges
  int32_t chunk, nchunk;      // reactions per chunk (multiple of kFPass), number of chunks
  int32_t n_acc;              // accumulator rows: ns species rows + extra rows of hub species
  int32_t n_bp;               // thermo breakpoints (distinct t_mid), n_bp + 1 intervals
  int32_t n_extra;
  int32_t meta_cap;           // 16-byte units of the largest chunk schedule
  int64_t blk_stride;         // bytes of one interval's parameter blocks
  int64_t blk_fo_off, blk_ph_off;  // byte offsets of the FALLOFF and PHOTO blocks in an interval
  const double *bp;           // [n_bp] ascending
  const unsigned char *blk;   // [n_bp+1] x blk_stride
  const int32_t *meta_ptr;    // [nchunk + 1] in 16-byte units into meta
  const int4 *meta;           // per chunk: header | tasks | entries
  const int32_t *extra;       // [n_extra][2] (extra accumulator row, species), grouped by species
  const int32_t *pp_user;     // [npad] padded packed index -> USER reaction index, -1 for padding
};

struct FusedHost {
  bool enabled = false;
  int32_t npad = 0, arr_end = 0, fo_end = 0, ph_end = 0, chunk = 0, nchunk = 0, n_acc = 0, n_bp = 0;
  int32_t meta_cap = 0;
  int64_t blk_stride = 0, blk_fo_off = 0, blk_ph_off = 0;
  int64_t n_tasks = 0, n_entries = 0;
  std::vector<int32_t> pp_to_packed;   // [npad], -1 for padding
  std::vector<double> bp;
  std::vector<unsigned char> blk;
  std::vector<int32_t> meta_ptr, extra, pp_user;
  std::vector<int32_t> meta;           // 4 words per 16-byte unit
};

// ---- tables of the tiled Jacobian kernel (k_jac_tiled, jac_tiled.cuh; packed by pack_jac.cpp) ----
// A *slot* is one distinct derivative d q_{r,dir} / d n_j = m k[dir][r] n[o1] n[o2]; all terms of the
// entries (i, j) of one Jacobian column j draw on the slots of that column only.  Columns are grouped
// into *units* (several small columns, or one hub column); a unit is processed in chunks of `chunk`
// slots; its entries own accumulator rows that are flushed to jac[e][col] when the unit ends.
struct JacTiledHost {
  bool enabled = false;
  int32_t chunk = 0, nchunk = 0, n_units = 0, acc_rows = 0, meta_cap = 0;
  int64_t n_slots = 0, n_tasks = 0, n_entries = 0;
  std::vector<int32_t> meta_ptr;    // [nchunk + 1] in 16-byte units into meta
  std::vector<int32_t> meta;        // per chunk: header | tasks | entries (build_chunk_schedule)
  std::vector<int32_t> slots;       // [nchunk * chunk][4]: rk (user reaction, bit 31 = reverse), o1, o2 (ns = none), 0
  std::vector<int32_t> chunk_info;  // [nchunk][4]: first chunk of the unit, flush begin, flush end (last chunk of a unit only), slots used
  std::vector<int32_t> flush;       // [n_flush][4]: pattern entry e, first accumulator row, rows, 0
};

struct JacTiledDev {
  int32_t enabled;
  int32_t chunk, nchunk, acc_rows, meta_cap, n_flush;
  const int32_t *meta_ptr;
  const int4 *meta, *slots, *chunk_info, *flush;
};

// ---- tables of the batched implicit step (f1: xod_newton_step; pack_lu.cpp, newton.cuh) ---------
// Symbolic LU of the Jacobian pattern (symmetric, with diagonal) in a minimum-degree elimination order,
// shared by all columns; values live in a [nnz_lu][cols] array, rows in elimination order, each row
// stored as  L part (ascending) | diagonal | U part (ascending).
constexpr int32_t kLuDiagBit = 1 << 30;   // in LuHost::src: the position is a diagonal
constexpr int kLuWarps = 16;              // warps of a k_lu_factor CTA
constexpr int kLuCols = 8;                // columns per k_lu_factor CTA: a thread = (entry slice, column), 64 slices
constexpr int kLuMaxBlockRows = 6;        // rows factorised together, all resident in shared memory
struct LuRow { int32_t begin, len, pair_begin, pair_end; };           // storage range of the row, its (i, k) pairs
struct LuPair { int32_t t_k, diag_k, cnt, tgt_off; };                 // slot of a_ik in row i; diagonal of row k; |U(k)|; targets
// Block schedule of k_lu_factor: `nrows` consecutive rows sit in shared memory (row b at slot b * max_row) while the
// pivots k of the union of their L parts are applied in ascending order; one step = one pivot, whose U row is read
// ONCE (from global memory, or from the block's own shared rows when k is itself in the block) and applied to every
// row of the block that holds a_ik (its items).
struct LuBlock { int32_t row0, nrows, step_begin, step_end; };
struct LuStep { int32_t diag_k, cnt, src, item_begin, n_items, pad; };   // src < 0: U row k in global memory from diag_k + 1; else its first shared slot
struct LuItem { int32_t slot_ik, base, tgt_off, pad; };                  // shared slot of a_ik; first slot of the row; targets (tgt)
struct LuHost {
  bool enabled = false;
  int32_t n = 0, max_row = 0;
  int64_t nnz = 0, n_updates = 0;
  std::vector<int32_t> perm, pos_of;        // perm[p] = species eliminated p-th; pos_of[species] = p
  std::vector<int64_t> row_ptr;             // [n + 1]
  std::vector<int32_t> col, diag, src;      // [nnz] permuted column; [n] position of the diagonal; [nnz] Jacobian entry or -1 (fill)
  std::vector<LuRow> rows;                  // [n]
  std::vector<LuPair> pairs;                // sum_i |L(i)|, row by row, ascending k
  std::vector<uint16_t> tgt;                // for pair (i, k): slot in row i of every column of U(k)
  int32_t block_rows = 0;                   // rows per block (<= kLuMaxBlockRows, bounded by shared memory)
  int64_t n_block_loads = 0;                // sum over the steps of |U(k)|: U values read per column by k_lu_factor
  std::vector<LuBlock> blocks;
  std::vector<LuStep> steps;
  std::vector<LuItem> items;
};
struct LuDev {
  int32_t enabled, n, max_row;
  int64_t nnz;
  const int32_t *perm, *diag, *src, *col;
  const int64_t *row_ptr;
  const LuRow *rows;
  const LuPair *pairs;
  const uint16_t *tgt;
  int32_t block_rows, n_blocks;
  const LuBlock *blocks;
  const LuStep *steps;
  const LuItem *items;
};

// ---- tables of the pathway analyser (f4: xod_pathway; pack_path.cpp, pathway.cuh) ----------------
// Incoming-edge lists per destination species and a step schedule for a CTA of kFWarps warps: in every step a
// warp relaxes one part of one node's incoming edges (its four lane groups take every fourth edge); the parts of a
// node sit on consecutive warps of the same step and are combined in a fixed order by the first of them.
struct PathTask { int32_t node, begin, end, first_warp_parts; };   // first_warp_parts: first warp of the node | parts << 16; node < 0: idle
struct PathHost {
  bool enabled = false;
  int32_t n_steps = 0;
  int64_t n_edges = 0;
  std::vector<int64_t> in_ptr;          // [ns + 1]
  std::vector<uint16_t> in_u, in_rd;    // [n_edges]: source species; 2 * user reaction + direction
  std::vector<PathTask> sched;          // [n_steps][kFWarps]
};
struct PathDev {
  int32_t enabled, n_steps;
  int64_t n_edges;
  const uint16_t *in_u, *in_rd;
  const PathTask *sched;
};

// ---- tables of the equilibrium-composition kernel (f4: xod_equilibrium; equil.cuh) ----------------
constexpr int kEqThreads = 64;      // columns per CTA
constexpr int kEqMaxElem = 16;      // elements (including a charge column) the shared-memory layout is sized for
struct EquilDev {
  int32_t ns, ne;
  const int32_t *sp_ptr;    // [ns + 1] into sp_ea
  const int32_t *sp_ea;     // element + 256 * count (count signed: a charge column has both signs)
  const int32_t *el_neg;    // [ne] 1 if the element's composition column has a negative entry (abundance 0 allowed)
  const double *nasa, *tmid;
};

struct HostTables {
  int32_t ns = 0, ne = 0, nr = 0, n_photo = 0;
  std::vector<int32_t> eq_ptr, eq_ea, eq_neg;   // composition as (element, count) lists per species; signed columns
  int32_t uni_begin = 0, bi_begin = 0, fo_begin = 0, ph_begin = 0;
  std::vector<int32_t> packed_to_user, user_to_packed, photo_user;
  std::vector<double> c0, c1, c2, l0, l1, l2, fcl, cN;
  std::vector<int32_t> sp, flags, photo_row;
  std::vector<double> nasa, nasa_l2, tmid;
  // user-facing CSRs
  std::vector<int64_t> src_ptr;
  std::vector<int32_t> src_rxn_user, src_nu;
  std::vector<int64_t> jac_ptr;
  std::vector<int32_t> jac_col;
  // device-facing
  std::vector<int32_t> src_rxn_packed;
  std::vector<float> src_nu_f;
  std::vector<SrcSeg> src_seg;
  std::vector<int64_t> jac_term_ptr;
  std::vector<JacTerm> jac_terms;
  FusedHost f;
  JacTiledHost jt;
  LuHost lu;
  PathHost path;
};

// one row task of a chunk schedule: an accumulator row and its entries (q row | nu bits)
struct SchedSeg { int32_t row; const uint32_t *ent; int len; };
void build_chunk_schedule(std::vector<SchedSeg> segs, uint32_t zero_entry, std::vector<int32_t> &blob,
                          int64_t &n_tasks, int64_t &n_entries);

// pack.cpp
xod_status pack_network(const xod_network_desc *d, HostTables &h, std::string &err);
// pack_fused.cpp: tables of the fused path for a given chunk size (0 = does not fit: disabled)
void pack_fused(const xod_network_desc *d, HostTables &h, int chunk);
// host-only consistency check of the fused-path tables (pack_fused.cpp)
bool check_fused(const HostTables &h, std::string &err);
// shared-memory bytes k_fused needs for these tables
size_t fused_smem_bytes(int ns, int n_acc, int chunk, int meta_cap);
// pack_jac.cpp: tables of the tiled Jacobian kernel for a given chunk size and accumulator-row budget
void pack_jac_tiled(HostTables &h, int chunk, int acc_budget);
bool check_jac_tiled(const HostTables &h, std::string &err);
// pack_lu.cpp: minimum-degree ordering, filled pattern and update schedule of the implicit step
void pack_lu(HostTables &h);
bool check_lu(const HostTables &h, std::string &err);
// pack_path.cpp: incoming-edge lists and step schedule of the pathway analyser
void pack_path(const xod_network_desc *d, HostTables &h);
size_t path_smem_bytes(int ns);
size_t jac_tiled_smem_bytes(int ns, int acc_rows, int chunk, int meta_cap);

}  // namespace xod

// optional per-kernel timing (xod_network_tune(XOD_TUNE_TIMING)): CUDA event pairs recorded around
// every launch on the caller's stream, summed by xod_network_timing_read
namespace xod {
enum KernelId { KID_THERMO = 0, KID_PROLOGUE, KID_RATES, KID_RATES_FROM_K, KID_SOURCE, KID_JACOBIAN, KID_FUSED, KID_FUSED_COMBINE, KID_RATE_COEFFS, KID_JAC_TILED, KID_NEWTON_ASSEMBLE, KID_LU_FACTOR, KID_LU_SOLVE, KID_PHOTO_GEMM, KID_PHOTO_FLUX, KID_TRANSPORT, KID_PATH_WEIGHTS, KID_PATHWAY, KID_EQUILIBRIUM, KID_COUNT };
struct TimingState {
  bool on = false;
  std::vector<void *> pool;                       // cudaEvent_t, reused
  size_t used = 0;
  std::vector<int> kid;                           // kernel id of pair p = events 2p, 2p+1
};
}  // namespace xod

// f2: wavelength grid and cross-sections on the device (xod_photo_create)
struct xod_photo {
  const xod_network *net = nullptr;
  int device = -1;
  int32_t n_bins = 0, n_abs = 0, n_photo = 0;
  std::vector<double> h_dlambda, h_sigma_ext, h_sigma_ph;
  std::vector<int32_t> h_abs;
  double *dlambda = nullptr, *sigma_ext = nullptr, *sigma_ph = nullptr;
  int32_t *abs_species = nullptr;
};

constexpr int kHostSlots = 3;  // staging slots of xod_source_fused_host

struct xod_network {
  xod::HostTables h;
  xod::DevTables d{};
  xod::FusedDev fd{};
  xod::JacTiledDev jd{};
  xod::LuDev ld{};
  xod::PathDev pd{};
  xod::EquilDev ed{};
  int64_t force_split = 0;  // XOD_TUNE_SPLIT: 0 = automatic
  int64_t use_fused = 1;    // XOD_TUNE_FUSED_KERNEL: 0 = always the multi-kernel path
  int64_t use_jac_tiled = 1;  // XOD_TUNE_JAC_TILED: 0 = the one-warp-per-entry gather kernel
  int sm_count = 148;       // replaced by the device attribute at create
  int device = -1;
  std::vector<void *> dev_allocs;
  int64_t chunk_cols = 0;  // 0 = default
  // staging for the *_host call
  void *stage = nullptr;
  size_t stage_bytes = 0;
  void *host_streams[3] = {nullptr, nullptr, nullptr};  // cudaStream_t of the *_host pipeline slots
  mutable xod::TimingState timing;
};
