// psr_tables.h -- device-side mechanism table layout, shared by the host table builder
// (psr_api.cu) and the kernels (psr_kernels.cu).  Internal to the library.
//
// The mechanism is cut into chunks of at most `rc` reactions.  Every chunk is one contiguous,
// 16-byte aligned blob that a CTA pulls into shared memory with a single cp.async.bulk:
//
//   ChunkHdr | RxRec[n_rx] | AuxRec[n_aux] | EffEnt[n_eff] | u16 pool | u32 gptr[2K+1] | u32 gent[n_g]
//
// RxRec carries the log-linear rate forms that replace the paper's per-thread pow()/species sums
// (Eq. 6, 8, 9):
//   ln k_f = c0 + c1 ln T + c2/T
//   ln k_r = ln k_f - ln K_c = e0 + e1 ln T + e2/T + T (d0 + d1 T + d2 T^2 + d3 T^3)
// where ln K_c = sum_i nu_ik (s_i/R - h_i/RT) + (sum_i nu_ik) ln(P_atm/(R T)) with the NASA-7
// polynomials summed per reaction at load time (exact in real arithmetic for a single range).
#ifndef PSR_TABLES_H_
#define PSR_TABLES_H_
#include <stdint.h>

namespace psr {

constexpr int kTile = 32;       // reactors per tile = lanes of a warp
constexpr int kRowBytes = kTile * 8;  // one species / reaction row of a tile in shared memory
constexpr int kSlots = 3;       // inline concentration-factor slots per reaction side
constexpr int kMaxSide = 15;    // concentration factors per reaction side (long form)
constexpr int kMaxStages = 8;     // chunk blobs that can be resident in shared memory at once
constexpr int kMaxChunkRx = 1024; // reactions per chunk (rows of the q tile, +1 zero row)

// meta bits
constexpr uint32_t kMetaTypeMask = 0x3u;      // PSR_RX_*
constexpr uint32_t kMetaRev = 0x4u;           // reversible
constexpr uint32_t kMetaLong = 0x8u;          // factor list lives in the u16 pool at off[0]; counts in meta
constexpr int kMetaNrShift = 4;               // bits 4..7  reactant factor count (long form)
constexpr int kMetaNpShift = 8;               // bits 8..11 product factor count (long form)
constexpr int kMetaSgnShift = 12;              // bits 12..13 sign of A, bits 14..15 sign of A0: 0 positive, 1 negative, 2 zero
                                              // (non-zero only in long-form records: a reaction with A <= 0 or A0 <= 0
                                              // is stored in the long form, so the class loops of ordinary reactions
                                              // carry no sign handling; c[0], c0[0] then hold ln|A|, or 0 for A = 0)
constexpr int kMetaAuxShift = 16;             // bits 16..31 index into AuxRec[]

struct __attribute__((aligned(16))) RxRec {   // 112 bytes
  double c[3];            // ln A, b, -Ea/R_c
  double e[3];            // ln k_r coefficients over (1, ln T, 1/T)
  double d[4];            // ln k_r coefficients over (T, T^2, T^3, T^4)
  uint32_t meta;
  uint32_t off[2 * kSlots];  // byte offsets of the factor rows in the C tile: 3 reactant slots, 3 product
                             // slots, nu expanded by repetition, unused slots -> the unit row (index K)
  uint32_t korig;         // caller's reaction index (row of kf/kr/q outputs)
};
static_assert(sizeof(RxRec) == 112, "RxRec layout");

struct __attribute__((aligned(16))) AuxRec {  // 80 bytes; one per three-body / falloff reaction
  double c0[3];           // ln A0, b0, -Ea0/R_c (falloff only)
  double troe[4];         // alpha, -1/T***, -1/T*, -T**
  uint32_t eff_off, n_eff;
  uint32_t pad[2];
};
static_assert(sizeof(AuxRec) == 80, "AuxRec layout");

struct __attribute__((aligned(16))) EffEnt {  // 16 bytes
  double am1;             // alpha - 1
  uint32_t off;           // byte offset of the species row in the C tile
  uint32_t pad;
};

constexpr int kClsLong = 4;      // record classes: 0..3 = PSR_RX_* type in the 3+3 slot form, 4 = long factor lists (any type)
constexpr int kMaxWarps = 24;

struct __attribute__((aligned(16))) ChunkHdr {  // 336 bytes
  uint32_t n_rx, n_aux, n_eff, rec_base;   // rec_base: mechanism-wide index of the chunk's first record (rate table row)
  uint32_t off_aux, off_eff, off_pool, off_gptr, off_gent;
  uint32_t bytes;         // bytes to copy (multiple of 16)
  // warp w evaluates the records wb[w][c] .. wb[w][c+1]-1 of class c (cost-balanced over warps at load
  // time; a warp's records are contiguous and sorted by class)
  uint16_t wb[kMaxWarps][kClsLong + 2];
};
static_assert(sizeof(ChunkHdr) == 336, "ChunkHdr layout");

// Gather lists of nu^T (Eq. 4) per chunk: species s adds the q rows gent[gptr[2s] .. gptr[2s+1]) and
// subtracts gent[gptr[2s+1] .. gptr[2s+2]).  An entry is the byte offset of a row of the q tile;
// |nu| > 1 repeats the entry; every group is padded to a multiple of 4 entries with the offset of
// the all-zero row (index rc) so the inner loop is a branch-free 4-wide step.

// Kernel-side view of a loaded mechanism (passed by value as a kernel parameter).
struct MechView {
  const unsigned char* chunks;  // n_chunks blobs, chunk_stride bytes apart
  const double* invW;           // [K] 1/W
  const double* Wm;             // [K] W
  const double* nasa;           // [K][7] NASA-7 coefficients a0..a6 (energy row only)
  const int32_t* sp_of;         // [nw*spw] species owned by (warp, slot) in the gather, -1 = none (nnz-balanced)
  const double* exp_tab;        // [32] 2^(j/32), one entry per lane (psr_math.cuh)
  const int32_t* chunk_rec_base;  // [n_chunks + 1] mechanism-wide index of each chunk's first record
  int32_t K, I;
  int32_t n_chunks, rc;
  int32_t need_lnctot;          // some Troe reaction has no efficiency list (uses ln C_tot)
  int32_t resident;             // every chunk blob stays in shared memory (loaded once per CTA)
  int32_t jy_dense;             // Y-column launch packs the columns of consecutive reactors densely (K <= 64)
  int32_t ring_stages;          // otherwise: stages of the chunk ring (2, or 1 when only that fits)
  int32_t n_cbuf;               // C-tile buffers: 2 = the next tile's state is prefetched during this tile's chunks
  uint32_t chunk_stride;        // bytes, multiple of 16
  uint32_t smem_cs, smem_q, smem_mech, smem_tab, smem_misc, smem_total;  // byte offsets / sizes of the dynamic smem carve-up
};


// ---- warp-specialised kernel (psr_ws.cu): 12 reaction warps + 4 helper warps per CTA, the mechanism cut into
// n_parts resident blobs (same ChunkHdr layout, records dealt to the 12 reaction warps, gather lists per part)
constexpr int kWsRxWarps = 13, kWsHelpWarps = 7, kWsWarps = kWsRxWarps + kWsHelpWarps;
constexpr int kWsStRows = 8;      // per-tile state rows: T, ln T, 1/T, rho, C_tot, ln C_tot, 1/tau, 1/rho
constexpr int kWsMaxParts = 8;
// Gather lists of the warp-specialised kernel: one flat stream of 4-entry groups per (part, helper warp), groups
// wb[kWsRxWarps + hw][0] .. wb[kWsRxWarps + hw][1] - 1 of the part's gent array.  A group holds four byte offsets
// of q rows (multiples of kRowBytes, the zero row pads) that belong to ONE species and ONE sign; the low bits of
// its first entry say what to do with the group's sum.
constexpr uint32_t kGatherNeg = 1u;    // subtract the group's sum instead of adding it
constexpr uint32_t kGatherLast = 2u;   // last group of the species: its row of nu^T q is complete for this part

struct WsView {
  const unsigned char* chunks;  // n_parts blobs, chunk_stride bytes apart
  const double* invW;           // [K] 1/W
  const double* Wm;             // [K] W
  const int32_t* sp_of;         // [kWsHelpWarps][spw] species owned by a helper warp (owned ones first, then -1)
  const double* exp_tab;        // [32] 2^(j/32)
  int32_t K, I;
  int32_t n_parts, rc;          // rc: rows of a q buffer (+1 zero row)
  int32_t spw;                  // species slots per helper warp (<= 32)
  int32_t need_lnctot;
  uint32_t chunk_stride;
  uint32_t smem_cs, smem_ds, smem_q, smem_acc, smem_mech, smem_misc, smem_total;
  int32_t tm_cols;              // tensor-memory columns to allocate for the copies of the two C tiles (power of two), 0: none
  int32_t tm_buf;               // columns per tile: 2 per row, rows rounded up to four
};

// ---- warp-specialised kernel for LARGE mechanisms (psr_wsl.cu): the same roles as psr_ws.cu with what does not fit
// one CTA's shared memory given up -- a single C tile, no Y - Y_in tile (the epilogue reads Y, Y_in from global
// memory), the parts streamed through a two-stage ring instead of resident, and the running sums of nu^T q in a
// shared-memory tile when that fits, else in an L2-resident scratch [CTA][K][32] (acc_global).
// Gather streams per (part, helper warp) as for psr_ws.cu, except that species without a term in a part are left
// out (part 0 keeps every owned species: its flushes initialise the sums) and every flush takes its target -- the
// byte offset of the species' row in a [K][32] tile -- from a list in the blob (gptr area):
//   wb[kWslRxWarps + hw][0..2] = first group, one past the last group, first entry of the target list.
constexpr int kWslRxWarps = 12, kWslHelpWarps = 8, kWslWarps = kWslRxWarps + kWslHelpWarps;
constexpr int kWslMaxParts = 64;

struct WslView {
  const unsigned char* chunks;  // n_parts blobs, chunk_stride bytes apart
  const double* invW;
  const double* Wm;
  const int32_t* sp_of;         // [kWslHelpWarps][spw] species owned by a helper warp (owned ones first, then -1)
  const double* exp_tab;
  double* acc_g;                // acc_global: [CTAs][K][32] running sums; else unused
  int32_t K, I;
  int32_t n_parts, rc;
  int32_t spw;
  int32_t need_lnctot;
  int32_t acc_global;           // where the running sums of nu^T q live: 0 shared memory, 1 L2-resident scratch (acc_g), 2 tensor memory
  uint32_t chunk_stride;
  uint32_t smem_cs, smem_acc, smem_q, smem_mech, smem_misc, smem_total;
  int32_t tm_cols;              // tensor-memory columns to allocate (power of two), 0: none
  int32_t tm_acc_col;           // acc_global == 2: first column of the running sums (after the copy of the C tile);
                                // helper warp hw, owned species number jj: columns tm_acc_col + 2 ((hw / 4) spw + jj) of its quadrant
};

// ---- fused finite-difference Jacobian kernel (psr_jac.cu): lane <-> reactor, one CTA per tile of 32 reactors.
// Phase 1 evaluates the tile (at T + h_T, then at T) and sums the forward and reverse rates of every reaction
// into per-species sums BY CONCENTRATION ORDER; phase 2 builds the K species columns from them, warp <-> column.
constexpr int kJacWarps = 10;
constexpr int kJacMaxOrder = 6;   // highest concentration order of a rate term the kernel takes (else: the generic sweep)
constexpr int kJacAccLd = 33;     // row stride (doubles) of a warp's phase-2 tile: conflict-free by rows and by columns
constexpr int kJacStage = 8;       // incidence records per staging chunk of a warp (two chunks in flight)
constexpr int kJacStRows = 4;     // per-tile state rows (T, ln T, 1/T, rho, 1/rho, C_tot, ln C_tot, sum Y/W, 1/tau, h_T, ...)

// Species j takes part in reaction k ("incidence"): what column j needs to correct the rate of reaction k beyond
// the uniform scaling of all concentrations.
struct __attribute__((aligned(16))) JacInc {   // 96 bytes
  uint32_t off[6];   // the reaction's 3 + 3 factor slots: byte offsets of C-tile rows (unit row = unused, zero row =
                     // reverse side of an irreversible reaction)
  uint32_t row;      // scratch row of the reaction: k_f, k_r, E = [M] - C_tot of every reactor of the tile
  uint8_t tb;        // 1: three-body reaction (q = [M] (...)); 0: rate constants do not change under a Y perturbation
  uint8_t nf, nr;    // concentration orders of the forward / reverse rate (numbers of factors, >= 1)
  uint8_t af;        // how many of the forward slots are species j
  uint8_t ar;        // ... of the reverse slots
  uint8_t n_sc;      // scatter entries in use
  uint16_t pad;
  uint32_t pad2;
  double am1;        // three-body reaction with j in its efficiency list: alpha_kj - 1; else 0
  struct {           // reaction k changes species i (unused entries: the scratch row K of the tile, nu = 0)
    uint32_t row_off;  // byte offset of row i in a [K+1][kJacAccLd] tile
    float nu;          // net stoichiometric coefficient nu_ik
  } sc[6];
};
static_assert(sizeof(JacInc) == 96, "JacInc layout");

struct JacView {
  const unsigned char* chunks;   // n_parts blobs (records dealt to kJacWarps warps; gather streams by species and order)
  const JacInc* inc;             // incidence records, species after species
  const int32_t* inc_ptr;        // [K + 1]
  const uint32_t* inc_row;       // [records + 2] scratch row of every record (read two records ahead)
  const int32_t* col_order;      // [K] columns in descending order of their number of records
  const double* invW;
  const double* Wm;
  const double* exp_tab;
  double* scratch;               // [grid][I][3][32]: k_f, k_r, E of the tile a CTA works on
  int32_t K, I, n_parts, n_cls;  // n_cls: highest concentration order present
  int32_t rows_max;              // rows of the rate tile of a part (+1 zero row)
  int32_t need_lnctot;
  uint32_t chunk_stride;
  uint32_t smem_cs, smem_d, smem_ar, smem_mech, smem_misc, smem_stage, smem_total;
};

// what one launch produces
enum : uint32_t {
  kOutWdot = 1u, kOutQ = 2u, kOutKf = 4u, kOutKr = 8u, kOutF = 16u, kOutF0 = 64u,
  kModeJac = 32u,    // states are (reactor, column) pairs over all K+1 columns, every state a full evaluation
  kModeJacT = 128u,  // states are the T columns only (one per reactor), full evaluation
  kModeJacY = 256u,  // states are the Y columns, tiles aligned to reactors, T-only factors from the rate table
  kOutTab = 512u,    // also write the rate table (kRateVals doubles per reactor and reaction)
  kOutFT = 1024u     // also write the energy row F_T [N] (needs Tin)
};

// Rate table written by the base-residual launch of psr_fd_jacobian and read by the Y-column launch:
// the factors of a reaction that depend on T only, which a Y perturbation leaves unchanged.
//   plain, three-body: k_f, k_r            Lindemann: k_inf, 1/K_c, k_0/k_inf
//   Troe: ln k_0, 1/K_c, ln k_inf, ln F_cent
// Row of reactor r, record index j (chunk order): tab[(r * I + j) * kRateVals ...].
constexpr int kRateVals = 4;

struct EvalArgs {
  int64_t N, ld, ldk;
  const double *T, *P, *Y, *Yin, *tau;
  const double* Tin;      // kOutFT: inlet temperature [N]
  double* FT;             // kOutFT: energy row [N]
  double *wdot, *q, *kf, *kr, *F;
  double *J;              // Jacobian mode output
  double* tab_out;        // kOutTab: rate table [N][I][kRateVals]
  const double* tab;      // kModeJacY: the same table
  const double* F0;       // Jacobian mode: base residual [N][K+1]
  double* F0out;          // residual mode: also write [N][K+1] base residual (row 0 = 0)
  uint32_t flags;
  int64_t n_tiles;
  // psr_solve_hybrid only (null elsewhere): reactors whose skip_dt entry is NaN are finished -- a tile of finished
  // reactors is left out -- and *skip_count is the number of reactors still active (0: the launch does nothing)
  const double* skip_dt;
  const int32_t* skip_count;
};

// ---- psr_solve_hybrid: a sub-batch's state in the workspace (psr_solve.cu); row stride of Y, Yin: ldw
struct HybridState {
  double *T, *P, *tau, *Tin;   // [ldw]; Tin: null for the isothermal system
  double *Y, *Yin;             // [K][ldw]
  double *dt_cur, *dt_arg;     // [ldw]
  int32_t *mode, *it, *status, *nn, *np, *orig;   // [ldw]; orig: the reactor's index in the caller's sub-batch
  int64_t ldw;
};

}  // namespace psr
#endif
