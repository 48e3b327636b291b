// psr_api.cu -- host side of the C ABI in include/psr.h: argument checks, mechanism table
// construction (psr_tables.h) and kernel launches.  No reactor arithmetic runs on the host.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <numeric>
#include <string>
#include <vector>

#include "../../include/psr.h"
#include "psr_tables.h"

namespace psr {
cudaError_t launch_eval(int nw, int spw, int rl, const MechView& mv, const EvalArgs& a, int grid, cudaStream_t st);
cudaError_t occupancy_eval(int nw, int spw, int rl, size_t smem, size_t smem_optin, int* ctas_per_sm);
cudaError_t launch_probe(int kind, int iters, int grid, double* sink, cudaStream_t st);
cudaError_t launch_lu_solve(int64_t N, int n, const double* A, double* b, int32_t* info, int n_sm, size_t smem_optin,
                            cudaStream_t st, const double* F, const double* dt, const int32_t* skip_count);
cudaError_t launch_exp_values(const double* tab, const double* x, double* y, int n, cudaStream_t st);
cudaError_t launch_hybrid_gather(int64_t nb, int K, int64_t ld, const double* T, const double* P, const double* Y, const double* Tin,
                                 const double* Yin, const double* tau, const HybridState& s, const psr_solve_opts& o, int32_t* n_active,
                                 cudaStream_t st);
cudaError_t launch_hybrid_compact(int64_t nb, int K, const HybridState& src, const HybridState& dst, int32_t* pos, const int32_t* n_active,
                                  cudaStream_t st);
cudaError_t launch_hybrid_scatter(int64_t nb, int K, int64_t ld, const HybridState& s, double* T, double* Y, int32_t* status,
                                  int32_t* n_newton, int32_t* n_ptc, cudaStream_t st);
cudaError_t launch_hybrid_update(int64_t nb, int n, int64_t ld, const psr_solve_opts& o, double* T, double* Y, const double* dx,
                                 const int32_t* info, double* dt_cur, double* dt_arg, int32_t* mode, int32_t* it, int32_t* status,
                                 int32_t* n_newton, int32_t* n_ptc, int32_t* n_active, cudaStream_t st);
cudaError_t chk_read_kernels(unsigned int* count, unsigned int* first_code);
cudaError_t chk_read_ws(unsigned int* count, unsigned int* first_code);
cudaError_t chk_read_jac(unsigned int* count, unsigned int* first_code);
cudaError_t chk_read_wsl(unsigned int* count, unsigned int* first_code);
cudaError_t chk_read_solve(unsigned int* count, unsigned int* first_code);
cudaError_t wsl_set_smem(size_t smem);
cudaError_t launch_wsl(const WslView& mv, const EvalArgs& a, int grid, int bulk_ok, int rx_tmem, cudaStream_t st);
cudaError_t launch_chk_selftest(cudaStream_t st);
cudaError_t jac_set_smem(size_t smem);
cudaError_t launch_jac(const JacView& jv, const EvalArgs& a, int grid, cudaStream_t st);
cudaError_t launch_jac_static(const JacView& jv, const EvalArgs& a, int grid, cudaStream_t st);
size_t jac_static_scratch_bytes();
cudaError_t ws_set_smem(size_t smem);
cudaError_t launch_ws(const WsView& mv, const EvalArgs& a, int grid, int bulk_ok, cudaStream_t st);
}  // namespace psr

using namespace psr;

struct psr_mech {
  MechView view{};
  int nw = 0, spw = 0, rl = 1;  // warps per CTA, species per warp, reactors per lane
  int tile = kTile;             // evaluation states per tile = 32 * rl
  int n_sm = 0, ctas_per_sm = 0;
  int n_falloff = 0, n_third_body = 0, nnz_nu = 0;
  unsigned char* d_chunks = nullptr;
  double* d_invW = nullptr;
  double* d_W = nullptr;
  double* d_nasa = nullptr;
  double* d_exptab = nullptr;
  int32_t* d_sp_of = nullptr;
  int32_t* d_rec_base = nullptr;  // [n_chunks + 1]
  WsView ws{};                  // warp-specialised kernel (psr_ws.cu), when its tables fit (ws_ok)
  bool ws_ok = false;
  unsigned char* d_ws_chunks = nullptr;
  int32_t* d_ws_sp_of = nullptr;
  WslView wsl{};                // warp-specialised kernel for large mechanisms (psr_wsl.cu), when ws_ok is false (wsl_ok)
  bool wsl_ok = false;
  unsigned char* d_wsl_chunks = nullptr;
  int32_t* d_wsl_sp_of = nullptr;
  double* d_wsl_acc = nullptr;
  JacView jac{};                // fused finite-difference Jacobian kernel (psr_jac.cu), when the mechanism qualifies (jac_ok)
  bool jac_ok = false;
  unsigned char* d_jac_chunks = nullptr;
  JacInc* d_jac_inc = nullptr;
  int32_t* d_jac_inc_ptr = nullptr;
  uint32_t* d_jac_inc_row = nullptr;
  int32_t* d_jac_col_order = nullptr;
  double* d_jac_scratch = nullptr;
  int opt_fused_only = 0;       // diagnostic (psr_mech_set_option): never take the warp-specialised kernel
  int opt_no_tmem = 0;          // diagnostic: the evaluation kernels read every concentration from shared memory
  int opt_jac_unhoisted = 0;    // diagnostic: every Jacobian column a full evaluation
  int opt_jac_generic = 0;      // diagnostic: psr_fd_jacobian takes the generic three-launch sweep even where the fused kernel applies
  double* d_scratch = nullptr;  // psr_fd_jacobian: rate table [N][I][kRateVals], then F0 when the caller passes none
  size_t scratch_bytes = 0;
  std::vector<void*> retired;   // outgrown scratch buffers, freed with the mechanism
  int device = 0;
};

namespace {

thread_local std::string g_err;

psr_status fail(psr_status st, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return st;
}

psr_status cuda_fail(cudaError_t e, const char* what) {
  return fail(PSR_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

constexpr long double kRgasL = 8.31446261815324e7L;
constexpr long double kRcalL = 8.31446261815324L / 4.184L;
constexpr long double kPatmL = 1.01325e6L;

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

double reaction_cost(int type) {  // relative FP64 cost used to balance warps inside a chunk
  switch (type) {
    case PSR_RX_THREE_BODY: return 1.5;   // executed instructions relative to a plain reaction (ncu, C1)
    case PSR_RX_LINDEMANN: return 2.0;
    case PSR_RX_TROE: return 3.8;
    default: return 1.0;
  }
}

struct HostRx {
  RxRec rec;
  bool has_aux;
  AuxRec aux;
  std::vector<EffEnt> eff;
  std::vector<uint16_t> factors;  // reactants then products
  std::vector<std::pair<int, int>> nu_net;  // (species, nu''-nu')
  int type;
  int nr = 0, np = 0;
  bool special_sign = false;   // A <= 0 or A0 <= 0: stored in the long form (kMetaSgnShift)
};

struct BlobSet {
  std::vector<unsigned char> all;   // n_chunks blobs, stride bytes apart
  std::vector<int32_t> rec_base;    // [n_chunks + 1] mechanism-wide index of each chunk's first record
  size_t stride = 0;
  int n_chunks = 0, rc = 0;         // rc: most reactions in a chunk (rows of the q tile, +1 zero row)
};

// Cuts the mechanism into n_chunks chunks, deals every chunk's records to nw warps and serialises the chunk
// blobs (psr_tables.h): records, aux records, efficiency entries, factor pool, per-species gather lists.
// ws_sp_of (may be null): species ownership [kWsHelpWarps][ws_spw] of the warp-specialised kernel, whose gather
// lists are one flat stream of 4-entry groups per helper warp (see psr_tables.h) instead of lists per species.
struct JacBuild {                    // extra inputs / outputs when the blobs are those of the Jacobian kernel (psr_jac.cu)
  const std::vector<int32_t>* sp_of; // gather ownership [kJacWarps][spw]
  int spw = 0;
  int rows_zero = 0;                 // index of the all-zero row of the rate tile (= rows_max of a first pass)
  std::vector<int32_t> row_of;       // out: [I] scratch row of reaction k (mechanism-wide record index)
  int rows_max = 0;                  // out: most rate-tile rows of a part
};

struct WslBuild {                    // gather streams of the large-mechanism warp-specialised kernel (psr_wsl.cu)
  const std::vector<int32_t>* sp_of; // ownership [kWslHelpWarps][spw]
  int spw = 0;
  bool tuples = false;               // running sums in global memory: one (q row | sign, target row) tuple per entry of nu^T
  bool tm_targets = false;           // tuples whose sums live in tensor memory: target = column offset 2 jj of the species'
                                     // number jj in its owner's list | bit 31: subtract | bit 30: the species' last tuple
};

void build_blobs(const std::vector<HostRx>& rx, int K, int I, int n_chunks, int nw, double warp0_load, BlobSet& out,
                 const std::vector<int32_t>* ws_sp_of = nullptr, int ws_spw = 0, JacBuild* jb = nullptr,
                 const WslBuild* wl = nullptr) {
  const uint32_t row_bytes = (uint32_t)kRowBytes;
  const int rc = (I + n_chunks - 1) / n_chunks;
  out.n_chunks = n_chunks;
  out.rc = rc;
  // ---- distribute reactions over chunks (each type dealt round-robin so chunks cost the same),
  //      then inside a chunk order by cost and deal to warps in snake order.
  std::vector<int> order(I);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return reaction_cost(rx[x].type) > reaction_cost(rx[y].type); });
  std::vector<std::vector<int>> chunk_rx(n_chunks);
  for (int p = 0; p < I; ++p) chunk_rx[p % n_chunks].push_back(order[p]);
  // inside a chunk: longest-processing-time assignment of records to warps, records of a warp contiguous
  auto cls_of = [&](int k) { return (rx[k].nr > kSlots || rx[k].np > kSlots || rx[k].special_sign) ? kClsLong : rx[k].type; };
  std::vector<std::vector<int>> chunk_wb(n_chunks);   // [warp][class boundary], kClsLong + 2 per warp
  for (int c = 0; c < n_chunks; ++c) {
    auto& cr = chunk_rx[c];  // cost-descending
    std::vector<double> load(nw, 0.0);
    load[0] = warp0_load;   // extra work of warp 0 in units of a plain reaction (it forms ln T, rho, C_tot of the tile)
    std::vector<std::vector<int>> mine(nw);
    for (int k : cr) {
      const int wmin = (int)(std::min_element(load.begin(), load.end()) - load.begin());
      mine[wmin].push_back(k);
      load[wmin] += reaction_cost(rx[k].type);
    }
    cr.clear();
    chunk_wb[c].assign((size_t)kMaxWarps * (kClsLong + 2), 0);
    for (int wv = 0; wv < nw; ++wv) {
      std::stable_sort(mine[wv].begin(), mine[wv].end(), [&](int x, int y) { return cls_of(x) < cls_of(y); });
      int* wb = &chunk_wb[c][(size_t)wv * (kClsLong + 2)];
      size_t p = 0;
      for (int cl = 0; cl <= kClsLong; ++cl) {
        wb[cl] = (int)(cr.size() + p);
        while (p < mine[wv].size() && cls_of(mine[wv][p]) == cl) ++p;
      }
      cr.insert(cr.end(), mine[wv].begin(), mine[wv].end());
      wb[kClsLong + 1] = (int)cr.size();
    }
  }
  // ---- serialise chunk blobs
  out.rec_base.assign(n_chunks + 1, 0);
  for (int c = 0; c < n_chunks; ++c) out.rec_base[c + 1] = out.rec_base[c] + (int32_t)chunk_rx[c].size();
  std::vector<std::vector<unsigned char>> blobs(n_chunks);
  size_t stride = 0;
  const uint32_t unit_off = (uint32_t)K * row_bytes;   // the all-ones row of the C tile
  const uint32_t zero_c_off = (uint32_t)(K + 1) * row_bytes;  // the all-zero row of the C tile
  const uint32_t zero_off = (uint32_t)rc * row_bytes;  // the all-zero row of the q tile
  for (int c = 0; c < n_chunks; ++c) {
    const auto& cr = chunk_rx[c];
    const int n_rx = (int)cr.size();
    std::vector<RxRec> recs(n_rx);
    std::vector<AuxRec> auxs;
    std::vector<EffEnt> effs;
    std::vector<uint16_t> pool;
    std::vector<std::vector<uint32_t>> pos(K), neg(K);
    // Jacobian kernel: rate-tile rows of the records, and per (species, concentration order) the rows that enter
    // the species' sum with a plus / minus sign
    std::vector<std::vector<uint32_t>> jpos, jneg;
    uint32_t jrows = 0;
    if (jb) {
      jpos.assign((size_t)K * kJacMaxOrder, {});
      jneg.assign((size_t)K * kJacMaxOrder, {});
    }
    for (int kl = 0; kl < n_rx; ++kl) {
      const HostRx& h = rx[cr[kl]];
      RxRec rec = h.rec;
      if (jb) {
        // rows: forward rate, reverse rate; a three-body reaction q = (C_tot + E)(...) has four: C_tot x forward (order
        // nf), E x forward (order nf + 1), C_tot x reverse, E x reverse
        const bool tb = h.type == PSR_RX_THREE_BODY;
        const uint32_t rbase = jrows;
        jrows += tb ? 4 : 2;
        rec.korig = rbase | ((uint32_t)(out.rec_base[c] + kl) << 16);
        jb->row_of[cr[kl]] = out.rec_base[c] + kl;
        const int nf = h.nr, nr = std::max(h.np, 1);   // (HostRx::nr / np are the reactant / product factor counts)
        for (auto& pr : h.nu_net) {
          for (int t = 0; t < std::abs(pr.second); ++t) {
            auto& fw = (pr.second > 0 ? jpos : jneg);
            auto& rv = (pr.second > 0 ? jneg : jpos);
            if (!tb) {
              fw[(size_t)pr.first * kJacMaxOrder + nf - 1].push_back(rbase * row_bytes);
              rv[(size_t)pr.first * kJacMaxOrder + nr - 1].push_back((rbase + 1) * row_bytes);
            } else {
              fw[(size_t)pr.first * kJacMaxOrder + nf - 1].push_back(rbase * row_bytes);
              fw[(size_t)pr.first * kJacMaxOrder + nf].push_back((rbase + 1) * row_bytes);
              rv[(size_t)pr.first * kJacMaxOrder + nr - 1].push_back((rbase + 2) * row_bytes);
              rv[(size_t)pr.first * kJacMaxOrder + nr].push_back((rbase + 3) * row_bytes);
            }
          }
        }
      }
      if (h.nr <= kSlots && h.np <= kSlots && !h.special_sign) {
        for (int i = 0; i < kSlots; ++i) {
          rec.off[i] = i < h.nr ? (uint32_t)h.factors[i] * row_bytes : unit_off;
          rec.off[kSlots + i] = i < h.np ? (uint32_t)h.factors[h.nr + i] * row_bytes : unit_off;
        }
        // irreversible: the product-side factor is the zero row, so k_r * prod = 0 without a select
        // (and below ln k_r := ln k_f keeps the unused exp finite whenever k_f is)
        if (!(rec.meta & kMetaRev)) rec.off[kSlots] = zero_c_off;
      } else {
        rec.meta |= kMetaLong | ((uint32_t)h.nr << kMetaNrShift) | ((uint32_t)h.np << kMetaNpShift);
        rec.off[0] = (uint32_t)pool.size();
        pool.insert(pool.end(), h.factors.begin(), h.factors.end());
      }
      if (!(rec.meta & kMetaRev)) {
        for (int j = 0; j < 3; ++j) rec.e[j] = rec.c[j];
        for (int j = 0; j < 4; ++j) rec.d[j] = 0.0;
      }
      if (h.has_aux) {
        AuxRec ax = h.aux;
        ax.eff_off = (uint32_t)effs.size();
        ax.n_eff = (uint32_t)h.eff.size();
        for (EffEnt ee : h.eff) {
          ee.off *= row_bytes;
          effs.push_back(ee);
        }
        rec.meta |= (uint32_t)auxs.size() << kMetaAuxShift;
        auxs.push_back(ax);
      }
      recs[kl] = rec;
      for (auto& pr : h.nu_net)
        for (int t = 0; t < std::abs(pr.second); ++t)
          (pr.second < 0 ? neg : pos)[pr.first].push_back((uint32_t)kl * row_bytes);
    }
    std::vector<uint32_t> gptr(2 * K + 1, 0), gent;
    auto add_group = [&](const std::vector<uint32_t>& grp) {
      gent.insert(gent.end(), grp.begin(), grp.end());
      while (gent.size() % 4) gent.push_back(zero_off);
    };
    std::vector<uint16_t> ws_range(2 * kWsHelpWarps, 0);   // [helper warp] first group, one past its last group
    std::vector<uint16_t> jac_range(3 * kJacWarps, 0);     // [warp] first group, one past its last group, first flush target
    if (jb) {
      // Jacobian kernel: per owning warp one flat stream of 4-entry groups (as for the warp-specialised kernel), the
      // groups of a (species, order) pair together; the pair's last group carries kGatherLast and its sum goes to
      // the next entry of the flush-target list (byte offset of row (order - 1) * K + species of the sums tile).
      // Pairs without a term in this part are left out.
      const uint32_t jzero = (uint32_t)jb->rows_zero * row_bytes;   // the all-zero row of the rate tile
      gptr.clear();
      for (int wv = 0; wv < kJacWarps; ++wv) {
        jac_range[3 * wv] = (uint16_t)(gent.size() / 4);
        jac_range[3 * wv + 2] = (uint16_t)gptr.size();
        for (int jj = 0; jj < jb->spw; ++jj) {
          const int sidx = (*jb->sp_of)[(size_t)wv * jb->spw + jj];
          if (sidx < 0) break;
          for (int m = 0; m < kJacMaxOrder; ++m) {
            const auto& pp = jpos[(size_t)sidx * kJacMaxOrder + m];
            const auto& nn = jneg[(size_t)sidx * kJacMaxOrder + m];
            if (pp.empty() && nn.empty()) continue;
            gent.insert(gent.end(), pp.begin(), pp.end());
            while (gent.size() % 4) gent.push_back(jzero);
            const size_t first_neg = gent.size();
            gent.insert(gent.end(), nn.begin(), nn.end());
            while (gent.size() % 4) gent.push_back(jzero);
            for (size_t g = first_neg; g < gent.size(); g += 4) gent[g] |= kGatherNeg;
            gent[gent.size() - 4] |= kGatherLast;
            gptr.push_back((uint32_t)(m * K + sidx) * row_bytes);
          }
        }
        if ((gent.size() / 4 - jac_range[3 * wv]) % 2) gent.insert(gent.end(), 4, jzero);
        jac_range[3 * wv + 1] = (uint16_t)(gent.size() / 4);
        gent.insert(gent.end(), 16, jzero);
      }
      gptr.push_back(0);
    } else if (wl) {
      // large-mechanism kernel: per helper warp the groups of its species in ownership order ("+" groups, then "-"
      // groups); a species without a term in this part is left out, except in part 0 whose flushes initialise the
      // running sums (one all-zero group there).  Every flush reads its target row from the list.
      gptr.clear();
      for (int hw = 0; hw < kWslHelpWarps && wl->tuples; ++hw) {
        // tuple stream (sums in global memory, added to with red.global: no running sum, no flush): per helper warp, its
        // species in ownership order, a species' "+" entries then its "-" entries -- a fixed order.  Entry = {byte
        // offset of the q row, byte offset of the species' row | bit 31 if it is subtracted}; padded to a multiple of 4
        // tuples, and 8 more for the kernel's read-ahead, with {zero row of q, spare row K of the sums}.
        jac_range[3 * hw] = (uint16_t)(gent.size() / 4);   // in 16-byte units = pairs of tuples
        size_t n_t = 0;
        for (int jj = 0; jj < wl->spw; ++jj) {
          const int sidx = (*wl->sp_of)[(size_t)hw * wl->spw + jj];
          if (sidx < 0) break;
          const uint32_t target = wl->tm_targets ? 2u * (uint32_t)jj : (uint32_t)sidx * row_bytes;
          size_t n_sp = 0;
          // (the target word carries the flags -- bit 31: subtract, bit 30: the species' last tuple of the part, for
          // tensor-memory targets -- so that the q offset is used as it is)
          for (uint32_t qo : pos[sidx]) { gent.push_back(qo); gent.push_back(target); ++n_t; ++n_sp; }
          for (uint32_t qo : neg[sidx]) { gent.push_back(qo); gent.push_back(target | 0x80000000u); ++n_t; ++n_sp; }
          if (wl->tm_targets) {
            // the kernel sums a species' tuples in a register and adds the sum to the species' running sum at the tuple
            // marked last (part 0 stores instead: a species without a term there gets one tuple on the zero row)
            if (n_sp == 0 && c == 0) { gent.push_back(zero_off); gent.push_back(target); ++n_t; ++n_sp; }
            if (n_sp) gent[gent.size() - 1] |= 0x40000000u;
          }
        }
        const uint32_t pad_target = wl->tm_targets ? 0u : (uint32_t)K * row_bytes;
        for (; n_t % 4; ++n_t) { gent.push_back(zero_off); gent.push_back(pad_target); }
        jac_range[3 * hw + 1] = (uint16_t)(gent.size() / 4);
        for (int t = 0; t < 8; ++t) { gent.push_back(zero_off); gent.push_back(pad_target); }
      }
      if (wl->tuples) gptr.push_back(0);
      for (int hw = 0; hw < kWslHelpWarps && !wl->tuples; ++hw) {
        jac_range[3 * hw] = (uint16_t)(gent.size() / 4);
        jac_range[3 * hw + 2] = (uint16_t)gptr.size();
        for (int jj = 0; jj < wl->spw; ++jj) {
          const int sidx = (*wl->sp_of)[(size_t)hw * wl->spw + jj];
          if (sidx < 0) break;
          if (pos[sidx].empty() && neg[sidx].empty() && c != 0) continue;
          const size_t first = gent.size();
          add_group(pos[sidx]);
          const size_t first_neg = gent.size();
          add_group(neg[sidx]);
          if (gent.size() == first) gent.insert(gent.end(), 4, zero_off);
          if (!neg[sidx].empty())
            for (size_t g = first_neg; g < gent.size(); g += 4) gent[g] |= kGatherNeg;
          gent[gent.size() - 4] |= kGatherLast;
          gptr.push_back((uint32_t)sidx * row_bytes);
        }
        if ((gent.size() / 4 - jac_range[3 * hw]) % 2) gent.insert(gent.end(), 4, zero_off);
        jac_range[3 * hw + 1] = (uint16_t)(gent.size() / 4);
        gent.insert(gent.end(), 16, zero_off);
        gptr.push_back(gptr.empty() ? 0u : gptr.back());   // read one ahead by the kernel
      }
    } else if (!ws_sp_of) {
      for (int s = 0; s < K; ++s) {
        gptr[2 * s] = (uint32_t)gent.size();
        add_group(pos[s]);
        gptr[2 * s + 1] = (uint32_t)gent.size();
        add_group(neg[s]);
      }
      gptr[2 * K] = (uint32_t)gent.size();
    } else {
      // flat streams: for every helper warp the groups of its species in ownership order, "+" groups then "-"
      // groups of a species; every owned species ends with a group that carries kGatherLast (a species without
      // a reaction in this part gets one all-zero group), the stream has an even number of groups and four
      // all-zero groups behind it so that the kernel's reads two trips ahead stay inside the blob
      gptr.assign(1, 0);
      for (int hw = 0; hw < kWsHelpWarps; ++hw) {
        ws_range[2 * hw] = (uint16_t)(gent.size() / 4);
        for (int jj = 0; jj < ws_spw; ++jj) {
          const int s = (*ws_sp_of)[(size_t)hw * ws_spw + jj];
          if (s < 0) break;
          const size_t first = gent.size();
          add_group(pos[s]);
          const size_t first_neg = gent.size();
          add_group(neg[s]);
          if (gent.size() == first) gent.insert(gent.end(), 4, zero_off);
          for (size_t g = first_neg; g < gent.size(); g += 4)
            if (!neg[s].empty()) gent[g] |= kGatherNeg;
          gent[gent.size() - 4] |= kGatherLast;
        }
        if ((gent.size() / 4 - ws_range[2 * hw]) % 2) gent.insert(gent.end(), 4, zero_off);   // the kernel takes two groups per trip
        ws_range[2 * hw + 1] = (uint16_t)(gent.size() / 4);
        gent.insert(gent.end(), 16, zero_off);
      }
    }

    ChunkHdr hdr{};
    hdr.n_rx = n_rx;
    hdr.n_aux = (uint32_t)auxs.size();
    hdr.n_eff = (uint32_t)effs.size();
    hdr.rec_base = (uint32_t)out.rec_base[c];
    for (int wv = 0; wv < kMaxWarps; ++wv)
      for (int cl = 0; cl < kClsLong + 2; ++cl) hdr.wb[wv][cl] = (uint16_t)chunk_wb[c][(size_t)wv * (kClsLong + 2) + cl];
    if (jb)
      for (int wv = 0; wv < kJacWarps; ++wv)
        for (int t = 0; t < 3; ++t) hdr.wb[kJacWarps + wv][t] = jac_range[3 * wv + t];
    if (wl)
      for (int hw = 0; hw < kWslHelpWarps; ++hw)
        for (int t = 0; t < 3; ++t) hdr.wb[kWslRxWarps + hw][t] = jac_range[3 * hw + t];
    if (jb) jb->rows_max = std::max(jb->rows_max, (int)jrows);
    if (ws_sp_of)
      for (int hw = 0; hw < kWsHelpWarps; ++hw) {
        hdr.wb[kWsRxWarps + hw][0] = ws_range[2 * hw];
        hdr.wb[kWsRxWarps + hw][1] = ws_range[2 * hw + 1];
      }
    size_t off = sizeof(ChunkHdr) + sizeof(RxRec) * n_rx;
    hdr.off_aux = (uint32_t)off;
    off += sizeof(AuxRec) * auxs.size();
    hdr.off_eff = (uint32_t)off;
    off += sizeof(EffEnt) * effs.size();
    hdr.off_pool = (uint32_t)off;
    off = align_up(off + 2 * pool.size(), 16);
    hdr.off_gptr = (uint32_t)off;
    off = align_up(off + 4 * gptr.size(), 16);
    hdr.off_gent = (uint32_t)off;
    off = align_up(off + 4 * gent.size(), 16);
    hdr.bytes = (uint32_t)off;
    std::vector<unsigned char>& b = blobs[c];
    b.assign(off, 0);
    std::memcpy(b.data(), &hdr, sizeof hdr);
    std::memcpy(b.data() + sizeof(ChunkHdr), recs.data(), sizeof(RxRec) * n_rx);
    if (!auxs.empty()) std::memcpy(b.data() + hdr.off_aux, auxs.data(), sizeof(AuxRec) * auxs.size());
    if (!effs.empty()) std::memcpy(b.data() + hdr.off_eff, effs.data(), sizeof(EffEnt) * effs.size());
    if (!pool.empty()) std::memcpy(b.data() + hdr.off_pool, pool.data(), 2 * pool.size());
    std::memcpy(b.data() + hdr.off_gptr, gptr.data(), 4 * gptr.size());
    if (!gent.empty()) std::memcpy(b.data() + hdr.off_gent, gent.data(), 4 * gent.size());
    stride = std::max(stride, off);
  }
  stride = align_up(stride, 128);
  out.stride = stride;
  out.all.assign(stride * n_chunks, 0);
  for (int c = 0; c < n_chunks; ++c) std::memcpy(out.all.data() + stride * c, blobs[c].data(), blobs[c].size());
}

// Gather ownership: species to (warp, slot) by longest-processing-time on the row length of nu^T; a warp's
// owned species come first in its slots, -1 pads.
std::vector<int32_t> assign_species(const std::vector<HostRx>& rx, int K, int I, int nw, int spw) {
  std::vector<int32_t> sp_of((size_t)nw * spw, -1);
  std::vector<int> rowlen(K, 0);
  for (int k = 0; k < I; ++k)
    for (auto& pr : rx[k].nu_net) rowlen[pr.first] += std::abs(pr.second);
  std::vector<int> sorder(K);
  std::iota(sorder.begin(), sorder.end(), 0);
  std::stable_sort(sorder.begin(), sorder.end(), [&](int x, int y) { return rowlen[x] > rowlen[y]; });
  std::vector<double> load(nw, 0.0);
  std::vector<int> used(nw, 0);
  for (int sidx : sorder) {
    int best = -1;
    for (int wv = 0; wv < nw; ++wv)
      if (used[wv] < spw && (best < 0 || load[wv] < load[best])) best = wv;
    sp_of[(size_t)best * spw + used[best]++] = sidx;
    load[best] += rowlen[sidx] + 6.0;  // + per-species loop overhead
  }
  return sp_of;
}

}  // namespace

extern "C" {

const char* psr_last_error(void) { return g_err.c_str(); }
const char* psr_version(void) { return "psr-b200 0.1 (sm_100a)"; }

psr_status psr_mech_load(const psr_mech_desc* d, psr_mech** out) {
  g_err.clear();
  if (!d || !out) return fail(PSR_EINVAL, "psr_mech_load: null argument");
  const int K = d->n_species, I = d->n_reactions;
  if (K < 1 || I < 1) return fail(PSR_EINVAL, "psr_mech_load: need n_species >= 1 and n_reactions >= 1");
  if (!d->W || !d->nasa || !d->A || !d->b || !d->Ea || !d->rtype || !d->reversible || !d->reac_ptr ||
      !d->reac_sp || !d->reac_nu || !d->prod_ptr || !d->prod_sp || !d->prod_nu || !d->eff_ptr)
    return fail(PSR_EINVAL, "psr_mech_load: null array in description");
  if (K > 512) return fail(PSR_EUNSUPPORTED, "psr_mech_load: n_species %d > 512", K);
  for (int i = 0; i < K; ++i) {
    if (!(d->W[i] > 0.0) || !std::isfinite(d->W[i])) return fail(PSR_EINVAL, "W[%d] must be finite and > 0", i);
    for (int j = 0; j < 7; ++j)
      if (!std::isfinite(d->nasa[7 * i + j])) return fail(PSR_EINVAL, "nasa[%d][%d] not finite", i, j);
  }
  if (d->reac_ptr[0] != 0 || d->prod_ptr[0] != 0 || d->eff_ptr[0] != 0)
    return fail(PSR_EINVAL, "CSR pointers must start at 0");
  bool any_fall = false;
  for (int k = 0; k < I; ++k) {
    if (d->reac_ptr[k + 1] < d->reac_ptr[k] || d->prod_ptr[k + 1] < d->prod_ptr[k] || d->eff_ptr[k + 1] < d->eff_ptr[k])
      return fail(PSR_EINVAL, "CSR pointers not monotone at reaction %d", k);
    if (d->rtype[k] > 3) return fail(PSR_EINVAL, "reaction %d: unknown rtype %d", k, (int)d->rtype[k]);
    if (!std::isfinite(d->A[k]) || !std::isfinite(d->b[k]) || !std::isfinite(d->Ea[k]))
      return fail(PSR_EINVAL, "reaction %d: A, b, Ea must be finite", k);
    if (d->rtype[k] >= 2) any_fall = true;
  }
  if (any_fall && (!d->A0 || !d->b0 || !d->Ea0)) return fail(PSR_EINVAL, "falloff reactions need A0, b0, Ea0");
  if (d->eff_ptr[I] > 0 && (!d->eff_sp || !d->eff_val)) return fail(PSR_EINVAL, "eff_sp/eff_val null");
  if (d->eff_ptr[I] > 65535) return fail(PSR_EUNSUPPORTED, "more than 65535 efficiency entries");

  // ---- per-reaction host records
  std::vector<HostRx> rx(I);
  int n_fall = 0, n_tb = 0, nnz = 0, need_lnctot = 0;
  for (int k = 0; k < I; ++k) {
    HostRx& h = rx[k];
    std::memset(&h.rec, 0, sizeof h.rec);
    std::memset(&h.aux, 0, sizeof h.aux);
    h.type = d->rtype[k];
    long double da[7] = {0, 0, 0, 0, 0, 0, 0};
    int dnu = 0;
    std::vector<int> net(0);
    auto side = [&](const int32_t* ptr, const int32_t* sp, const int32_t* nu, int sign, const char* name) -> psr_status {
      int count = 0;
      for (int j = ptr[k]; j < ptr[k + 1]; ++j) {
        if (sp[j] < 0 || sp[j] >= K) return fail(PSR_EINVAL, "reaction %d: %s species index %d out of range", k, name, sp[j]);
        if (nu[j] < 1 || nu[j] > 3) return fail(PSR_EINVAL, "reaction %d: %s nu=%d outside 1..3", k, name, nu[j]);
        for (int t = 0; t < nu[j]; ++t) h.factors.push_back((uint16_t)sp[j]);
        count += nu[j];
        for (int c = 0; c < 7; ++c) da[c] += (long double)(sign * nu[j]) * (long double)d->nasa[7 * sp[j] + c];
        dnu += sign * nu[j];
        bool found = false;
        for (auto& pr : h.nu_net)
          if (pr.first == sp[j]) { pr.second += sign * nu[j]; found = true; }
        if (!found) h.nu_net.push_back({sp[j], sign * nu[j]});
      }
      if (count > kMaxSide) return fail(PSR_EUNSUPPORTED, "reaction %d: %d %s factors > %d", k, count, name, kMaxSide);
      return PSR_OK;
    };
    psr_status st = side(d->reac_ptr, d->reac_sp, d->reac_nu, -1, "reactant");
    if (st != PSR_OK) return st;
    const int nr = (int)h.factors.size();
    st = side(d->prod_ptr, d->prod_sp, d->prod_nu, +1, "product");
    if (st != PSR_OK) return st;
    const int np = (int)h.factors.size() - nr;
    // ln|A| and the sign (kMetaSgnShift): A < 0 (a duplicate reaction with a negative pre-exponential) and A = 0 are
    // ordinary input; such records take the long form, whose code applies the sign
    auto sgn_code = [](double x) -> uint32_t { return x > 0.0 ? 0u : x < 0.0 ? 1u : 2u; };
    uint32_t sg = sgn_code(d->A[k]);
    const long double lnA = d->A[k] != 0.0 ? logl(fabsl((long double)d->A[k])) : 0.0L;
    const long double mEaR = -(long double)d->Ea[k] / kRcalL;
    h.rec.c[0] = (double)lnA;
    h.rec.c[1] = d->b[k];
    h.rec.c[2] = (double)mEaR;
    // ln K_c over (1, ln T, 1/T, T, T^2, T^3, T^4); the record stores ln k_r = ln k_f - ln K_c
    const long double kc0 = da[6] - da[0] + (long double)dnu * logl(kPatmL / kRgasL);
    const long double kc1 = da[0] - (long double)dnu;
    const long double kc2 = -da[5];
    h.rec.e[0] = (double)(lnA - kc0);
    h.rec.e[1] = (double)((long double)d->b[k] - kc1);
    h.rec.e[2] = (double)(mEaR - kc2);
    h.rec.d[0] = (double)(-da[1] / 2);
    h.rec.d[1] = (double)(-da[2] / 6);
    h.rec.d[2] = (double)(-da[3] / 12);
    h.rec.d[3] = (double)(-da[4] / 20);
    h.rec.korig = (uint32_t)k;
    h.rec.meta = (uint32_t)h.type | (d->reversible[k] ? kMetaRev : 0u);
    h.nr = nr;
    h.np = np;
    h.has_aux = h.type != PSR_RX_PLAIN;
    for (int j = d->eff_ptr[k]; j < d->eff_ptr[k + 1]; ++j) {
      if (d->eff_sp[j] < 0 || d->eff_sp[j] >= K) return fail(PSR_EINVAL, "reaction %d: efficiency species out of range", k);
      if (!std::isfinite(d->eff_val[j])) return fail(PSR_EINVAL, "reaction %d: efficiency not finite", k);
      EffEnt e{};
      e.am1 = d->eff_val[j] - 1.0;
      e.off = (uint32_t)d->eff_sp[j];  // species index here; scaled to a row offset at serialisation
      if (h.has_aux) h.eff.push_back(e);  // efficiencies on a plain reaction have no effect
    }
    if (h.type >= 2) {
      if (!std::isfinite(d->A0[k]) || !std::isfinite(d->b0[k]) || !std::isfinite(d->Ea0[k]))
        return fail(PSR_EINVAL, "reaction %d: A0, b0, Ea0 must be finite", k);
      sg |= sgn_code(d->A0[k]) << 2;
      h.aux.c0[0] = d->A0[k] != 0.0 ? (double)logl(fabsl((long double)d->A0[k])) : 0.0;
      h.aux.c0[1] = d->b0[k];
      h.aux.c0[2] = (double)(-(long double)d->Ea0[k] / kRcalL);
      ++n_fall;
    }
    h.special_sign = sg != 0;
    h.rec.meta |= sg << kMetaSgnShift;
    if (h.type == PSR_RX_TROE) {
      if (h.eff.empty()) need_lnctot = 1;
      if (!d->troe) return fail(PSR_EINVAL, "Troe reactions need the troe array");
      const double* t = d->troe + 4 * k;
      // alpha, T***, T* finite and the temperatures non-zero (they divide T); T** finite or +inf (+inf is how the
      // three-parameter form, without the exp(-T**/T) term, is written)
      if (!std::isfinite(t[0]) || !std::isfinite(t[1]) || !std::isfinite(t[2]) || t[1] == 0.0 || t[2] == 0.0 ||
          std::isnan(t[3]) || t[3] == -INFINITY)
        return fail(PSR_EINVAL, "reaction %d: Troe parameters must be finite with T***, T* != 0 (T** may be +inf)", k);
      h.aux.troe[0] = t[0];
      h.aux.troe[1] = -1.0 / t[1];
      h.aux.troe[2] = -1.0 / t[2];
      h.aux.troe[3] = -t[3];
    }
    if (h.type == PSR_RX_THREE_BODY) ++n_tb;
    for (auto& pr : h.nu_net) nnz += std::abs(pr.second);
  }

  // ---- device
  int dev = 0, n_dev = 0;
  cudaError_t e = cudaGetDeviceCount(&n_dev);
  if (e != cudaSuccess || n_dev == 0) return fail(PSR_ECUDA, "psr_mech_load: no CUDA device (%s)", cudaGetErrorString(e));
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
  cudaDeviceProp prop;
  if ((e = cudaGetDeviceProperties(&prop, dev)) != cudaSuccess) return cuda_fail(e, "cudaGetDeviceProperties");

  // ---- launch shape
  int nw = 16;
  // species per warp in the gather: smallest compiled shape (PSR_SHAPES in psr_kernels.cu) with nw * spw >= K
  auto pick_spw = [&](int nw_) {
    static const int s8[] = {2, 4, 7, 8, 0}, s12[] = {5, 0}, s16[] = {2, 4, 8, 16, 32, 0};
    for (const int* p = nw_ == 8 ? s8 : nw_ == 12 ? s12 : s16; *p; ++p)
      if (nw_ * *p >= K) return *p;
    return 0;
  };
  int spw = pick_spw(nw);
  if (!spw) { nw = 16; spw = pick_spw(nw); }
  // reactors per lane: the kernel is written for R per lane, but only R = 1 is instantiated -- at R = 2 the
  // q tile of a 325-reaction chunk no longer fits beside the C tiles and the second gather pass costs
  // more than the halved warp-uniform overhead saves (measured on C1)
  const int rl = 1;
  const uint32_t row_bytes = (uint32_t)kRowBytes * rl;
  int rc_target = std::min(I, 384);
  // shared memory left for the q tile and the chunk ring beside one C tile and the per-CTA scratch
  // Y - Y_in tile beside every C tile when the species' accumulators live in registers (spw <= 4); it shares
  // its region with the rate-table slices, which only the Y-column launch (that has no such tile) uses
  const size_t ds_bytes = spw <= 4 ? align_up((size_t)K * kTile * rl * 8, 128) : 0;
  const size_t smem_fixed = align_up((size_t)(K + 2) * kTile * rl * 8, 128) + (size_t)nw * kTile * rl * 8 +
                            (size_t)11 * kTile * rl * 8 + 8 * (2 * kMaxStages);
  // Y-column launch of psr_fd_jacobian: dense column packing for small mechanisms (a tile then spans several
  // reactors and needs their rate-table slices side by side), whole tiles per reactor for large ones
  const bool jy_dense = K <= 64;
  const int jy_slices = jy_dense ? 31 / K + 2 : 1;
  int n_chunks = 0, rc = 0;
  bool resident = false;
  int ring_stages = 2;
  size_t stride = 0;
  BlobSet bs;
  // the chunk size shrinks until one C tile, the q tile and the (double-buffered) chunk ring fit one CTA
  for (;; rc_target = std::min(rc_target - 1, rc_target * 15 / 16)) {
  if (rc_target < 1)
    return fail(PSR_EUNSUPPORTED, "mechanism does not fit %zu bytes of shared memory per CTA even at one reaction per chunk",
                (size_t)prop.sharedMemPerBlockOptin);
  n_chunks = (I + rc_target - 1) / rc_target;
  rc = (I + n_chunks - 1) / n_chunks;  // <= rc_target <= kMaxChunkRx

  build_blobs(rx, K, I, n_chunks, nw, 2.0, bs);
  rc = bs.rc;
  stride = bs.stride;
  // all chunk blobs resident in shared memory (loaded once per CTA) when they fit; else a ring of two
  // stages, or of one when that is what lets this chunk size fit: a tile of a mechanism that large runs
  // for hundreds of microseconds, the exposed ~1 us copy per chunk costs less than a smaller chunk's extra
  // gather pass
  // q tile plus the rate-table slice of one chunk (Y-column launch of psr_fd_jacobian)
  // (the q tile also hosts the 3 x nw partial-sum rows of the energy row, hence the lower bound)
  const size_t tab_bytes_smem = std::max(align_up((size_t)jy_slices * rc * kRateVals * 8, 128), ds_bytes);   // slices of the reactors a column tile spans | one Y - Y_in tile
  const size_t q_bytes = align_up((size_t)std::max(rc + 1, 3 * nw) * kTile * rl * 8, 128) + tab_bytes_smem;
  resident = n_chunks <= kMaxStages && smem_fixed + q_bytes + stride * n_chunks <= (size_t)prop.sharedMemPerBlockOptin &&
             (n_chunks == 1 || stride * n_chunks <= 48 * 1024);
  ring_stages = 2;
  if (!resident && smem_fixed + q_bytes + stride * 2 > (size_t)prop.sharedMemPerBlockOptin) ring_stages = 1;
  const size_t need = smem_fixed + q_bytes + stride * (resident ? n_chunks : ring_stages);
  if (need > (size_t)prop.sharedMemPerBlockOptin) continue;
  break;
  }
  const std::vector<unsigned char>& all = bs.all;
  const std::vector<int32_t>& rec_base_of = bs.rec_base;
  const std::vector<int32_t> sp_of = assign_species(rx, K, I, nw, spw);

  // ---- warp-specialised kernel (psr_ws.cu): the mechanism in the fewest parts whose tables, two C tiles, two
  // Y - Y_in tiles, two q buffers and the partial-sum tile fit one CTA together (all parts resident)
  BlobSet wbs;
  WsView wv{};
  bool ws_ok = false;
  std::vector<int32_t> ws_sp_of;
  if (K <= 32 * kWsHelpWarps) {
    const int spw_h = (K + kWsHelpWarps - 1) / kWsHelpWarps;
    const int Kp = (K + 1) & ~1;
    ws_sp_of = assign_species(rx, K, I, kWsHelpWarps, spw_h);
    for (int n_parts = 1; n_parts <= kWsMaxParts && n_parts <= I && !ws_ok; ++n_parts) {
      build_blobs(rx, K, I, n_parts, kWsRxWarps, 0.0, wbs, &ws_sp_of, spw_h);
      size_t o = 0;
      wv.smem_cs = (uint32_t)o;
      o += align_up((size_t)2 * (K + 2) * kTile * 8, 128);
      wv.smem_ds = (uint32_t)o;
      o += align_up((size_t)2 * K * kTile * 8, 128);
      wv.smem_q = (uint32_t)o;
      o += align_up((size_t)2 * (wbs.rc + 1) * kTile * 8, 128);
      wv.smem_acc = (uint32_t)o;
      o += align_up((size_t)K * kTile * 8, 128);
      wv.smem_mech = (uint32_t)o;
      o += wbs.stride * n_parts;
      wv.smem_misc = (uint32_t)o;
      o += align_up((size_t)2 * Kp * 8 + (size_t)2 * kWsStRows * kTile * 8 + (size_t)2 * 3 * kTile * 8 + 16 * 8 +
                        align_up((size_t)kWsHelpWarps * spw_h * 4, 32) + (size_t)kWsHelpWarps * spw_h * 32, 128);
      wv.smem_total = (uint32_t)o;
      if (o <= (size_t)prop.sharedMemPerBlockOptin) {
        ws_ok = true;
        wv.K = K;
        wv.I = I;
        wv.n_parts = n_parts;
        wv.rc = wbs.rc;
        wv.spw = spw_h;
        wv.need_lnctot = need_lnctot;
        wv.chunk_stride = (uint32_t)wbs.stride;
        // copies of the two C tiles in tensor memory (512 columns of 32 bits per SM; one CTA per SM)
        wv.tm_buf = 2 * ((K + 2 + 3) & ~3);
        wv.tm_cols = 0;
        if (2 * wv.tm_buf <= 512) {
          wv.tm_cols = 32;
          while (wv.tm_cols < 2 * wv.tm_buf) wv.tm_cols *= 2;
        }
      }
    }
  }

  // ---- large mechanisms (psr_wsl.cu): the fewest parts for which one C tile, the running sums, two q buffers, a two-stage
  // ring of part tables and the per-CTA rows fit one CTA; the sums in shared memory if that is possible at all (larger
  // parts then), else in an L2-resident scratch
  BlobSet lbs;
  WslView lv{};
  bool wsl_ok = false;
  std::vector<int32_t> wsl_sp_of;
  if (!ws_ok) {
    const int spw_l = (K + kWslHelpWarps - 1) / kWslHelpWarps;
    const int Kp = (K + 1) & ~1;
    wsl_sp_of = assign_species(rx, K, I, kWslHelpWarps, spw_l);
    WslBuild wb;
    wb.sp_of = &wsl_sp_of;
    wb.spw = spw_l;
    // the sums in shared memory only when that leaves room for parts so large that at most 4 are needed (P5: 0.099 ms
    // against 0.105 with the sums in L2); beyond that the tile's worth of shared memory is better spent on larger
    // parts (measured: C2 0.522 ms with 8 parts and the sums in L2, 0.538 with 11 parts and the sums in shared memory)
    // Third place for the sums: tensor memory, beside the copy of the C tile (psr_wsl.cu) -- a helper warp's species in
    // its own lane quadrant, two warps per quadrant -- when both fit the 512 columns (K <= 200).  Parts as large as with
    // the sums in L2, the group streams of the shared-memory variant, and no red.global traffic through the LSU queue
    // the reaction warps' shared-memory loads go through.
    const int tm_tile_cols = 2 * ((K + 2 + 3) & ~3);
    const int tm_acc_cols = 2 * ((kWslHelpWarps + 3) / 4) * spw_l;
    const int acc_modes[3] = {0, 2, 1};
    for (int mi = 0; mi < 3 && !wsl_ok; ++mi) {
      const int acc_global = acc_modes[mi];
      if (acc_global == 2 && tm_tile_cols + tm_acc_cols > 512) continue;
      wb.tuples = acc_global != 0;
      wb.tm_targets = acc_global == 2;
      for (int n_parts = 2; n_parts <= (acc_global ? kWslMaxParts : 4) && n_parts <= I && !wsl_ok; ++n_parts) {
        const int rc_l = (I + n_parts - 1) / n_parts;
        // (a quick bound before building the blobs: the q buffers alone)
        if ((size_t)(K + 2) * kRowBytes + (acc_global ? 0 : (size_t)K * kRowBytes) + (size_t)2 * (rc_l + 1) * kRowBytes >
            (size_t)prop.sharedMemPerBlockOptin)
          continue;
        build_blobs(rx, K, I, n_parts, kWslRxWarps, 0.0, lbs, nullptr, 0, nullptr, &wb);
        size_t o = 0;
        lv.smem_cs = (uint32_t)o;
        o += align_up((size_t)(K + 2) * kRowBytes, 128);
        lv.smem_acc = (uint32_t)o;
        o += acc_global ? 0 : align_up((size_t)K * kRowBytes, 128);
        lv.smem_q = (uint32_t)o;
        o += align_up((size_t)2 * (lbs.rc + 1) * kRowBytes, 128);
        lv.smem_mech = (uint32_t)o;
        o += 2 * lbs.stride;
        lv.smem_misc = (uint32_t)o;
        o += align_up((size_t)2 * Kp * 8 + (size_t)2 * 8 * kRowBytes + (size_t)2 * 3 * kRowBytes + 12 * 8 +
                          (size_t)kWslHelpWarps * spw_l * 4, 128);
        lv.smem_total = (uint32_t)o;
        if (o <= (size_t)prop.sharedMemPerBlockOptin) {
          wsl_ok = true;
          lv.K = K;
          lv.I = I;
          lv.n_parts = n_parts;
          lv.rc = lbs.rc;
          lv.spw = spw_l;
          lv.need_lnctot = need_lnctot;
          lv.acc_global = acc_global;
          lv.chunk_stride = (uint32_t)lbs.stride;
          // a copy of the C tile in tensor memory (512 columns of 32 bits per SM, two per row)
          lv.tm_cols = 0;
          lv.tm_acc_col = tm_tile_cols;
          const int tm_need = tm_tile_cols + (acc_global == 2 ? tm_acc_cols : 0);
          if (tm_need <= 512) {
            lv.tm_cols = 32;
            while (lv.tm_cols < tm_need) lv.tm_cols *= 2;
          }
        }
      }
    }
  }

  // ---- fused Jacobian kernel (psr_jac.cu).  It takes mechanisms whose every rate is k(T, C_tot) x a product of at most
  // 3 + 3 concentrations, x [M] for three-body reactions: no falloff reaction with an efficiency list (its k changes
  // with the composition), no long factor lists, no sign records.  Anything else keeps the generic sweep.
  BlobSet jbs;
  JacView jv{};
  bool jac_ok = false;
  std::vector<JacInc> jinc;
  std::vector<int32_t> jinc_ptr, jcol_order;
  std::vector<uint32_t> jinc_row;
  {
    bool elig = K <= 64;
    int n_cls = 1;
    for (int k = 0; k < I && elig; ++k) {
      const HostRx& h = rx[k];
      if (h.special_sign || h.nr > kSlots || h.np > kSlots || h.nr < 1) elig = false;
      if (d->reversible[k] && h.np < 1) elig = false;
      if (h.type >= 2 && !h.eff.empty()) elig = false;
      n_cls = std::max(n_cls, std::max(h.nr, std::max(h.np, 1)) + (h.type == PSR_RX_THREE_BODY ? 1 : 0));
    }
    if (n_cls > kJacMaxOrder) elig = false;
    if (elig) {
      const int spw_j = (K + kJacWarps - 1) / kJacWarps;
      const std::vector<int32_t> jsp = assign_species(rx, K, I, kJacWarps, spw_j);
      const int Kp = (K + 1) & ~1;
      for (int n_parts = 1; n_parts <= kWsMaxParts && n_parts <= I && !jac_ok; ++n_parts) {
        JacBuild jb;
        jb.sp_of = &jsp;
        jb.spw = spw_j;
        jb.row_of.assign(I, 0);
        build_blobs(rx, K, I, n_parts, kJacWarps, 0.0, jbs, nullptr, 0, &jb);   // first pass: rows of the rate tile
        jb.rows_zero = jb.rows_max;
        build_blobs(rx, K, I, n_parts, kJacWarps, 0.0, jbs, nullptr, 0, &jb);
        size_t o = 0;
        jv.smem_cs = (uint32_t)o;
        o += align_up((size_t)(K + 2) * kTile * 8, 128);
        jv.smem_d = (uint32_t)o;
        o += align_up((size_t)n_cls * K * kTile * 8, 128);
        // phase 1: rate tile (+ zero row) and the F(T + h_T) tile, then the part being evaluated (one at a time, loaded
        // again for every tile and pass).  Phase 2 reads neither: its per-warp [K + 1][33] tiles lie over both.
        jv.smem_ar = (uint32_t)o;
        const size_t ar1 = align_up(((size_t)jb.rows_max + 1 + K) * kTile * 8, 128);
        const size_t ar2 = align_up((size_t)kJacWarps * (K + 1) * kJacAccLd * 8, 128);
        jv.smem_mech = (uint32_t)(o + ar1);
        o += std::max(ar1 + jbs.stride, ar2);
        jv.smem_misc = (uint32_t)o;
        o += align_up((size_t)2 * Kp * 8 + (size_t)kJacStRows * kTile * 8 + (2 + 2 * kJacWarps) * 8, 128);
        jv.smem_stage = (uint32_t)o;   // per warp: two chunks of kJacStage incidence records
        o += (size_t)kJacWarps * 2 * kJacStage * sizeof(JacInc);
        jv.smem_total = (uint32_t)o;
        if (o <= (size_t)prop.sharedMemPerBlockOptin) {
          jac_ok = true;
          jv.K = K;
          jv.I = I;
          jv.n_parts = n_parts;
          jv.n_cls = n_cls;
          jv.rows_max = jb.rows_max;
          jv.need_lnctot = need_lnctot;
          jv.chunk_stride = (uint32_t)jbs.stride;
          // incidence records, species after species
          const uint32_t unit_off = (uint32_t)K * kRowBytes, zero_c_off = (uint32_t)(K + 1) * kRowBytes;
          jinc_ptr.assign(K + 1, 0);
          for (int j = 0; j < K; ++j) {
            jinc_ptr[j] = (int32_t)jinc.size();
            for (int k = 0; k < I; ++k) {
              const HostRx& h = rx[k];
              int af = 0, ar = 0;
              for (int t = 0; t < h.nr; ++t) af += h.factors[t] == j;
              for (int t = 0; t < h.np; ++t) ar += h.factors[h.nr + t] == j;
              double am1 = 0.0;
              if (h.type == PSR_RX_THREE_BODY)
                for (const EffEnt& ee : h.eff)
                  if ((int)ee.off == j) am1 += ee.am1;   // (EffEnt::off holds the species index in the host records)
              if (af == 0 && ar == 0 && am1 == 0.0) continue;
              JacInc ic{};
              for (int t = 0; t < kSlots; ++t) {
                ic.off[t] = t < h.nr ? (uint32_t)h.factors[t] * kRowBytes : unit_off;
                ic.off[kSlots + t] = t < h.np ? (uint32_t)h.factors[h.nr + t] * kRowBytes : unit_off;
              }
              if (!d->reversible[k]) ic.off[kSlots] = zero_c_off;
              ic.row = (uint32_t)jb.row_of[k];
              ic.tb = h.type == PSR_RX_THREE_BODY;
              ic.nf = (uint8_t)h.nr;
              ic.nr = (uint8_t)std::max(h.np, 1);
              ic.af = (uint8_t)af;
              ic.ar = (uint8_t)(d->reversible[k] ? ar : 0);
              ic.am1 = am1;
              int n_sc = 0;
              for (auto& pr : h.nu_net)
                if (pr.second != 0 && n_sc < 6) {
                  ic.sc[n_sc].row_off = (uint32_t)pr.first * (kJacAccLd * 8);
                  ic.sc[n_sc].nu = (float)pr.second;
                  ++n_sc;
                }
              ic.n_sc = (uint8_t)n_sc;
              for (int t = n_sc; t < 6; ++t) {
                ic.sc[t].row_off = (uint32_t)K * (kJacAccLd * 8);   // a scratch row of the warp's tile
                ic.sc[t].nu = 0.0f;
              }
              jinc.push_back(ic);
            }
          }
          jinc_ptr[K] = (int32_t)jinc.size();
          for (const JacInc& ic : jinc) jinc_row.push_back(ic.row);
          jinc_row.push_back(0);
          jinc_row.push_back(0);
          jcol_order.resize(K);
          std::iota(jcol_order.begin(), jcol_order.end(), 0);
          std::stable_sort(jcol_order.begin(), jcol_order.end(),
                           [&](int x, int y) { return jinc_ptr[x + 1] - jinc_ptr[x] > jinc_ptr[y + 1] - jinc_ptr[y]; });
        }
      }
    }
  }

  psr_mech* m = new (std::nothrow) psr_mech();
  if (!m) return fail(PSR_ENOMEM, "psr_mech_load: host allocation failed");
  m->device = dev;
  m->nw = nw;
  m->rl = rl;
  m->tile = kTile * rl;
  m->spw = spw;
  m->n_sm = prop.multiProcessorCount;
  m->n_falloff = n_fall;
  m->n_third_body = n_tb;
  m->nnz_nu = nnz;
  MechView& v = m->view;
  v.K = K;
  v.I = I;
  v.n_chunks = n_chunks;
  v.rc = rc;
  v.resident = resident ? 1 : 0;
  v.ring_stages = ring_stages;
  v.jy_dense = jy_dense ? 1 : 0;
  v.need_lnctot = need_lnctot;
  v.chunk_stride = (uint32_t)stride;
  const size_t cbuf_bytes = align_up((size_t)(K + 2) * kTile * rl * 8, 128);  // K+2 rows so the Jacobian staging [tile][n|1] fits
  auto carve = [&](int n_cbuf) {
    size_t o = 0;
    v.smem_cs = (uint32_t)o;
    o += n_cbuf * cbuf_bytes;
    v.smem_q = (uint32_t)o;
    o += align_up((size_t)std::max(rc + 1, 3 * nw) * kTile * rl * 8, 128);  // + the all-zero row; >= energy-row scratch
    v.smem_mech = (uint32_t)o;
    o += stride * (resident ? n_chunks : ring_stages);
    v.smem_misc = (uint32_t)o;
    o += align_up((size_t)nw * kTile * rl * 8 + (size_t)11 * kTile * rl * 8 + 8 * (2 * kMaxStages), 128);  // partial sums; ln T, h, rho, C_tot, ln C_tot, T/P/tau prefetch; mbarriers
    // the rate-table slices of the Y-column launch of psr_fd_jacobian | the Y - Y_in tiles of every other launch
    v.smem_tab = (uint32_t)o;
    o += std::max(align_up((size_t)jy_slices * rc * kRateVals * 8, 128), n_cbuf * ds_bytes);
    v.smem_total = (uint32_t)o;
    v.n_cbuf = n_cbuf;
    return o;
  };
  // two C buffers (next tile prefetched under this tile's chunks) unless that costs a resident CTA
  const size_t smem_max = (size_t)prop.sharedMemPerBlockOptin, half = (size_t)prop.sharedMemPerMultiprocessor / 2 - 1024;
  size_t o = carve(2);
  if (o > smem_max || (o > half && carve(1) <= half)) o = carve(1);
  if (o > (size_t)prop.sharedMemPerBlockOptin) {
    delete m;
    return fail(PSR_EUNSUPPORTED, "mechanism needs %zu bytes of shared memory per CTA, device allows %zu", o,
                (size_t)prop.sharedMemPerBlockOptin);
  }
  std::vector<double> invW(K);
  for (int i = 0; i < K; ++i) invW[i] = 1.0 / d->W[i];
  auto cleanup = [&]() { psr_mech_free(m); };
  if ((e = cudaMalloc(&m->d_chunks, all.size())) != cudaSuccess) { cleanup(); return fail(PSR_ENOMEM, "cudaMalloc: %s", cudaGetErrorString(e)); }
  if ((e = cudaMalloc(&m->d_invW, 8 * K)) != cudaSuccess) { cleanup(); return fail(PSR_ENOMEM, "cudaMalloc: %s", cudaGetErrorString(e)); }
  if ((e = cudaMalloc(&m->d_W, 8 * K)) != cudaSuccess) { cleanup(); return fail(PSR_ENOMEM, "cudaMalloc: %s", cudaGetErrorString(e)); }
  if ((e = cudaMalloc(&m->d_nasa, 8 * 7 * (size_t)K)) != cudaSuccess) { cleanup(); return fail(PSR_ENOMEM, "cudaMalloc: %s", cudaGetErrorString(e)); }
  if ((e = cudaMemcpy(m->d_chunks, all.data(), all.size(), cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMemcpy(m->d_invW, invW.data(), 8 * K, cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMemcpy(m->d_W, d->W, 8 * K, cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMemcpy(m->d_nasa, d->nasa, 8 * 7 * (size_t)K, cudaMemcpyHostToDevice)) != cudaSuccess) {
    cleanup();
    return cuda_fail(e, "cudaMemcpy (mechanism upload)");
  }
  {
    double tab[32];
    for (int j = 0; j < 32; ++j) tab[j] = (double)exp2l((long double)j / 32.0L);
    if ((e = cudaMalloc(&m->d_exptab, sizeof tab)) != cudaSuccess ||
        (e = cudaMemcpy(m->d_exptab, tab, sizeof tab, cudaMemcpyHostToDevice)) != cudaSuccess) {
      cleanup();
      return cuda_fail(e, "exp table upload");
    }
  }
  if ((e = cudaMalloc(&m->d_sp_of, 4 * sp_of.size())) != cudaSuccess ||
      (e = cudaMemcpy(m->d_sp_of, sp_of.data(), 4 * sp_of.size(), cudaMemcpyHostToDevice)) != cudaSuccess) {
    cleanup();
    return cuda_fail(e, "species ownership upload");
  }
  if ((e = cudaMalloc(&m->d_rec_base, 4 * rec_base_of.size())) != cudaSuccess ||
      (e = cudaMemcpy(m->d_rec_base, rec_base_of.data(), 4 * rec_base_of.size(), cudaMemcpyHostToDevice)) != cudaSuccess) {
    cleanup();
    return cuda_fail(e, "chunk record bases upload");
  }
  v.chunk_rec_base = m->d_rec_base;
  v.sp_of = m->d_sp_of;
  v.exp_tab = m->d_exptab;
  v.chunks = m->d_chunks;
  v.invW = m->d_invW;
  v.Wm = m->d_W;
  v.nasa = m->d_nasa;
  if ((e = occupancy_eval(nw, spw, rl, v.smem_total, (size_t)prop.sharedMemPerBlockOptin, &m->ctas_per_sm)) != cudaSuccess || m->ctas_per_sm < 1) {
    cleanup();
    return fail(PSR_ECUDA, "kernel does not fit on this device (%s)", cudaGetErrorString(e));
  }
  if (jac_ok) {
    const size_t scratch_bytes = (size_t)prop.multiProcessorCount * I * 3 * kTile * 8;
    jinc.push_back(JacInc{});   // (read ahead by the kernel, never used)
    jinc.push_back(JacInc{});
    if ((e = cudaMalloc(&m->d_jac_chunks, jbs.all.size())) != cudaSuccess ||
        (e = cudaMemcpy(m->d_jac_chunks, jbs.all.data(), jbs.all.size(), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMalloc(&m->d_jac_inc, sizeof(JacInc) * jinc.size())) != cudaSuccess ||
        (e = cudaMemcpy(m->d_jac_inc, jinc.data(), sizeof(JacInc) * jinc.size(), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMalloc(&m->d_jac_inc_ptr, 4 * jinc_ptr.size())) != cudaSuccess ||
        (e = cudaMemcpy(m->d_jac_inc_ptr, jinc_ptr.data(), 4 * jinc_ptr.size(), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMalloc(&m->d_jac_inc_row, 4 * jinc_row.size())) != cudaSuccess ||
        (e = cudaMemcpy(m->d_jac_inc_row, jinc_row.data(), 4 * jinc_row.size(), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMalloc(&m->d_jac_col_order, 4 * jcol_order.size())) != cudaSuccess ||
        (e = cudaMemcpy(m->d_jac_col_order, jcol_order.data(), 4 * jcol_order.size(), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMalloc(&m->d_jac_scratch, scratch_bytes)) != cudaSuccess ||
        (e = jac_set_smem((size_t)prop.sharedMemPerBlockOptin)) != cudaSuccess) {
      cleanup();
      return cuda_fail(e, "Jacobian kernel tables");
    }
    jv.chunks = m->d_jac_chunks;
    jv.inc = m->d_jac_inc;
    jv.inc_ptr = m->d_jac_inc_ptr;
    jv.inc_row = m->d_jac_inc_row;
    jv.col_order = m->d_jac_col_order;
    jv.scratch = m->d_jac_scratch;
    jv.invW = m->d_invW;
    jv.Wm = m->d_W;
    jv.exp_tab = m->d_exptab;
    m->jac = jv;
    m->jac_ok = true;
  }
  if (wsl_ok) {
    const size_t acc_bytes = lv.acc_global == 1 ? (size_t)prop.multiProcessorCount * (K + 1) * kRowBytes : 256;   // + a spare row
    if ((e = cudaMalloc(&m->d_wsl_chunks, lbs.all.size())) != cudaSuccess ||
        (e = cudaMemcpy(m->d_wsl_chunks, lbs.all.data(), lbs.all.size(), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMalloc(&m->d_wsl_sp_of, 4 * wsl_sp_of.size())) != cudaSuccess ||
        (e = cudaMemcpy(m->d_wsl_sp_of, wsl_sp_of.data(), 4 * wsl_sp_of.size(), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMalloc(&m->d_wsl_acc, acc_bytes)) != cudaSuccess ||
        (e = wsl_set_smem((size_t)prop.sharedMemPerBlockOptin)) != cudaSuccess) {
      cleanup();
      return cuda_fail(e, "large-mechanism kernel tables");
    }
    lv.chunks = m->d_wsl_chunks;
    lv.sp_of = m->d_wsl_sp_of;
    lv.acc_g = m->d_wsl_acc;
    lv.invW = m->d_invW;
    lv.Wm = m->d_W;
    lv.exp_tab = m->d_exptab;
    m->wsl = lv;
    m->wsl_ok = true;
  }
  if (ws_ok) {
    if ((e = cudaMalloc(&m->d_ws_chunks, wbs.all.size())) != cudaSuccess ||
        (e = cudaMemcpy(m->d_ws_chunks, wbs.all.data(), wbs.all.size(), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMalloc(&m->d_ws_sp_of, 4 * ws_sp_of.size())) != cudaSuccess ||
        (e = cudaMemcpy(m->d_ws_sp_of, ws_sp_of.data(), 4 * ws_sp_of.size(), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = ws_set_smem((size_t)prop.sharedMemPerBlockOptin)) != cudaSuccess) {
      cleanup();
      return cuda_fail(e, "warp-specialised kernel tables");
    }
    wv.chunks = m->d_ws_chunks;
    wv.sp_of = m->d_ws_sp_of;
    wv.invW = m->d_invW;
    wv.Wm = m->d_W;
    wv.exp_tab = m->d_exptab;
    m->ws = wv;
    m->ws_ok = true;
  }
  *out = m;
  return PSR_OK;
}

void psr_mech_free(psr_mech* m) {
  if (!m) return;
  cudaFree(m->d_chunks);
  cudaFree(m->d_invW);
  cudaFree(m->d_W);
  cudaFree(m->d_nasa);
  cudaFree(m->d_exptab);
  cudaFree(m->d_sp_of);
  cudaFree(m->d_rec_base);
  cudaFree(m->d_scratch);
  for (void* q : m->retired) cudaFree(q);
  cudaFree(m->d_ws_chunks);
  cudaFree(m->d_ws_sp_of);
  cudaFree(m->d_wsl_chunks);
  cudaFree(m->d_wsl_sp_of);
  cudaFree(m->d_wsl_acc);
  cudaFree(m->d_jac_chunks);
  cudaFree(m->d_jac_inc);
  cudaFree(m->d_jac_inc_ptr);
  cudaFree(m->d_jac_inc_row);
  cudaFree(m->d_jac_col_order);
  cudaFree(m->d_jac_scratch);
  delete m;
}

psr_status psr_mech_info(const psr_mech* m, psr_mech_info_t* info) {
  if (!m || !info) return fail(PSR_EINVAL, "psr_mech_info: null argument");
  info->n_species = m->view.K;
  info->n_reactions = m->view.I;
  info->tile = m->tile;
  info->warps = m->nw;
  info->chunk_reactions = m->view.rc;
  info->n_chunks = m->view.n_chunks;
  info->smem_bytes = (int32_t)m->view.smem_total;
  info->ctas_per_sm = m->ctas_per_sm;
  info->n_sm = m->n_sm;
  info->n_falloff = m->n_falloff;
  info->n_third_body = m->n_third_body;
  info->nnz_nu = m->nnz_nu;
  info->eval_kernel = m->ws_ok ? 1 : m->wsl_ok ? 2 : 0;
  info->eval_parts = m->ws_ok ? m->ws.n_parts : m->wsl_ok ? m->wsl.n_parts : m->view.n_chunks;
  info->eval_acc_global = m->wsl_ok ? m->wsl.acc_global : 0;
  info->jac_kernel = m->jac_ok ? 1 : 0;
  return PSR_OK;
}

}  // extern "C"

namespace {

psr_status check_common(const psr_mech* m, int64_t N, const double* T, const double* P, const double* Y, int64_t ld,
                        const char* fn) {
  if (!m) return fail(PSR_EINVAL, "%s: null mechanism", fn);
  if (N < 0) return fail(PSR_EINVAL, "%s: N < 0", fn);
  if (N == 0) return PSR_OK;
  if (!T || !P || !Y) return fail(PSR_EINVAL, "%s: null state array", fn);
  if (ld < N) return fail(PSR_EINVAL, "%s: ld (%lld) < N (%lld)", fn, (long long)ld, (long long)N);
  return PSR_OK;
}

psr_status run(const psr_mech* m, EvalArgs& a, void* stream, const char* fn) {
  // wdot / residual / rate-constant calls of a mechanism whose tables stay resident: the warp-specialised kernel
  if (m->ws_ok && !m->opt_fused_only && (a.flags & ~(kOutWdot | kOutF | kOutKf | kOutKr | kOutQ)) == 0) {
    auto al16 = [](const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; };
    const bool wantF = (a.flags & kOutF) != 0;
    // whole tiles come by one bulk copy per species row: needs 16-byte aligned rows
    const int bulk_ok = al16(a.T) && al16(a.P) && al16(a.Y) && (a.ld % 2 == 0) && (!wantF || (al16(a.Yin) && al16(a.tau)));
    const int grid = (int)std::min<int64_t>(a.n_tiles, m->n_sm);
    WsView wv = m->ws;
    if (m->opt_no_tmem) wv.tm_cols = 0;
    cudaError_t e = launch_ws(wv, a, grid, bulk_ok, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, fn);
    return PSR_OK;
  }
  // the same calls of a mechanism too large for that: the warp-specialised kernel with streamed parts
  if (m->wsl_ok && !m->opt_fused_only && (a.flags & ~(kOutWdot | kOutF | kOutKf | kOutKr | kOutQ)) == 0) {
    auto al16 = [](const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; };
    const int bulk_ok = al16(a.T) && al16(a.P) && al16(a.Y) && (a.ld % 2 == 0) && (!(a.flags & kOutF) || al16(a.tau));
    const int grid = (int)std::min<int64_t>(a.n_tiles, m->n_sm);
    cudaError_t e = launch_wsl(m->wsl, a, grid, bulk_ok, m->opt_no_tmem ? 0 : 1, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, fn);
    return PSR_OK;
  }
  const int64_t cap = (int64_t)m->n_sm * m->ctas_per_sm;
  const int grid = (int)std::min<int64_t>(a.n_tiles, cap);
  cudaError_t e = launch_eval(m->nw, m->spw, m->rl, m->view, a, grid, (cudaStream_t)stream);
  if (e != cudaSuccess) return cuda_fail(e, fn);
  return PSR_OK;
}

}  // namespace

extern "C" {

psr_status psr_eval_kf_kr(const psr_mech* m, int64_t N, const double* T, const double* P, const double* Y, int64_t ld,
                          double* kf, double* kr, int64_t ldk, void* stream) {
  g_err.clear();
  psr_status st = check_common(m, N, T, P, Y, ld, "psr_eval_kf_kr");
  if (st != PSR_OK || N == 0) return st;
  if (!kf && !kr) return fail(PSR_EINVAL, "psr_eval_kf_kr: both outputs null");
  if (ldk < N) return fail(PSR_EINVAL, "psr_eval_kf_kr: ldk < N");
  EvalArgs a{};
  a.N = N; a.ld = ld; a.ldk = ldk; a.T = T; a.P = P; a.Y = Y; a.kf = kf; a.kr = kr;
  a.flags = (kf ? kOutKf : 0u) | (kr ? kOutKr : 0u);
  a.n_tiles = (N + m->tile - 1) / m->tile;
  return run(m, a, stream, "psr_eval_kf_kr");
}

psr_status psr_eval_wdot(const psr_mech* m, int64_t N, const double* T, const double* P, const double* Y, int64_t ld,
                         double* wdot, double* q, int64_t ldq, void* stream) {
  g_err.clear();
  psr_status st = check_common(m, N, T, P, Y, ld, "psr_eval_wdot");
  if (st != PSR_OK || N == 0) return st;
  if (!wdot) return fail(PSR_EINVAL, "psr_eval_wdot: wdot null");
  if (q && ldq < N) return fail(PSR_EINVAL, "psr_eval_wdot: ldq < N");
  EvalArgs a{};
  a.N = N; a.ld = ld; a.ldk = ldq; a.T = T; a.P = P; a.Y = Y; a.wdot = wdot; a.q = q;
  a.flags = kOutWdot | (q ? kOutQ : 0u);
  a.n_tiles = (N + m->tile - 1) / m->tile;
  return run(m, a, stream, "psr_eval_wdot");
}

psr_status psr_eval_residual(const psr_mech* m, int64_t N, const double* T, const double* P, const double* Y,
                             const double* Yin, const double* tau, int64_t ld, double* F, double* wdot, void* stream) {
  g_err.clear();
  psr_status st = check_common(m, N, T, P, Y, ld, "psr_eval_residual");
  if (st != PSR_OK || N == 0) return st;
  if (!Yin || !tau || !F) return fail(PSR_EINVAL, "psr_eval_residual: null Yin, tau or F");
  EvalArgs a{};
  a.N = N; a.ld = ld; a.T = T; a.P = P; a.Y = Y; a.Yin = Yin; a.tau = tau; a.F = F; a.wdot = wdot;
  a.flags = kOutF | (wdot ? kOutWdot : 0u);
  a.n_tiles = (N + m->tile - 1) / m->tile;
  return run(m, a, stream, "psr_eval_residual");
}

psr_status psr_eval_residual_energy(const psr_mech* m, int64_t N, const double* T, const double* P, const double* Y,
                                    const double* Tin, const double* Yin, const double* tau, int64_t ld, double* F,
                                    double* FT, double* wdot, void* stream) {
  g_err.clear();
  psr_status st = check_common(m, N, T, P, Y, ld, "psr_eval_residual_energy");
  if (st != PSR_OK || N == 0) return st;
  if (!Tin || !Yin || !tau || !F || !FT) return fail(PSR_EINVAL, "psr_eval_residual_energy: null Tin, Yin, tau, F or FT");
  EvalArgs a{};
  a.N = N; a.ld = ld; a.T = T; a.P = P; a.Y = Y; a.Tin = Tin; a.Yin = Yin; a.tau = tau; a.F = F; a.FT = FT; a.wdot = wdot;
  a.flags = kOutF | kOutFT | (wdot ? kOutWdot : 0u);
  a.n_tiles = (N + m->tile - 1) / m->tile;
  return run(m, a, stream, "psr_eval_residual_energy");
}

}  // extern "C"

namespace {

// Scratch of the Jacobian sweep for N reactors: the rate table of one sub-batch, plus the base residual when the
// caller passes no F0.  The sweep runs in sub-batches of *Nb reactors so that the rate table (I * kRateVals
// doubles per reactor) written by the base launch is still in L2 when the Y-column launch reads it.
size_t jac_scratch_bytes(const psr_mech* m, int64_t N, bool with_F0, int64_t* Nb_out) {
  const int64_t n = m->view.K + 1;
  const size_t row_bytes = (size_t)m->view.I * kRateVals * 8;
  const int64_t wave = (int64_t)m->n_sm * m->ctas_per_sm * m->tile;   // reactors per full wave of base tiles
  int64_t Nb = std::max<int64_t>(1, (int64_t)((size_t)64 * 1024 * 1024 / row_bytes));
  if (Nb > wave) Nb -= Nb % wave;
  Nb = std::min(Nb, std::max<int64_t>(N, 1));
  Nb = std::min<int64_t>(Nb, ((int64_t)1 << 31) / (n + 32) - 1);   // state indices of a launch fit 32 bits
  if (Nb_out) *Nb_out = Nb;
  return align_up((size_t)Nb * row_bytes, 256) + (with_F0 ? (size_t)N * n * 8 : 0);
}

// psr_fd_jacobian (Tin == nullptr: row 0 is T - T_set) and psr_fd_jacobian_energy (row 0 is the energy row)
// skip_dt / skip_count: psr_solve_hybrid's markers of finished reactors (EvalArgs); honoured by the fused kernel only
psr_status fd_jacobian_impl(const psr_mech* mc, int64_t N, const double* T, const double* P, const double* Y,
                            const double* Tin, const double* Yin, const double* tau, int64_t ld, double* J, double* F0,
                            void* stream, const char* fn, const double* skip_dt = nullptr, const int32_t* skip_count = nullptr) {
  g_err.clear();
  psr_status st = check_common(mc, N, T, P, Y, ld, fn);
  if (st != PSR_OK || N == 0) return st;
  if (!Yin || !tau || !J) return fail(PSR_EINVAL, "%s: null Yin, tau or J", fn);
  const uint32_t en = Tin ? kOutFT : 0u;
  psr_mech* m = const_cast<psr_mech*>(mc);
  if (m->jac_ok && !Tin && !m->opt_jac_generic) {
    // the fused kernel: base residual, T column and the K species columns of every reactor in one launch, no
    // mechanism-owned scratch that depends on N
    EvalArgs a{};
    a.N = N; a.ld = ld; a.T = T; a.P = P; a.Y = Y; a.Yin = Yin; a.tau = tau; a.J = J; a.F0out = F0;
    a.n_tiles = (N + kTile - 1) / kTile;
    a.skip_dt = skip_dt;
    a.skip_count = skip_count;
    const int grid = (int)std::min<int64_t>(a.n_tiles, m->n_sm);
    cudaError_t e = launch_jac(m->jac, a, grid, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, fn);
    return PSR_OK;
  }
  const int64_t K = m->view.K, n = K + 1, I = m->view.I;

  const size_t row_bytes = (size_t)I * kRateVals * 8;
  int64_t Nb = 0;
  const size_t need = jac_scratch_bytes(m, N, F0 == nullptr, &Nb);
  const bool unhoisted = m->opt_jac_unhoisted != 0;   // diagnostic: every column a full evaluation (tests compare the two sweeps)

  const size_t tab_bytes = align_up((size_t)Nb * row_bytes, 256);
  if (need > m->scratch_bytes) {
    // grow the mechanism-owned scratch.  Never inside a stream capture (an allocation would invalidate it: reserve
    // first with psr_mech_reserve), and the outgrown buffer is kept until psr_mech_free, because kernels already
    // enqueued -- or a captured graph replayed later -- may still point at it.
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing((cudaStream_t)stream, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone)
      return fail(PSR_EINVAL, "%s: scratch for %lld reactors not reserved before stream capture (psr_mech_reserve)", fn, (long long)N);
    void* grown = nullptr;
    cudaError_t e = cudaMalloc(&grown, need);
    if (e != cudaSuccess) return fail(PSR_ENOMEM, "%s: scratch: %s", fn, cudaGetErrorString(e));
    if (m->d_scratch) m->retired.push_back(m->d_scratch);
    m->d_scratch = static_cast<double*>(grown);
    m->scratch_bytes = need;
  }
  double* tab = m->d_scratch;
  if (!F0) F0 = reinterpret_cast<double*>(reinterpret_cast<unsigned char*>(m->d_scratch) + tab_bytes);

  for (int64_t r0 = 0; r0 < N; r0 += Nb) {
    const int64_t nb = std::min(Nb, N - r0);
    EvalArgs a{};
    a.N = nb; a.ld = ld; a.T = T + r0; a.P = P + r0; a.Y = Y + r0; a.Yin = Yin + r0; a.tau = tau + r0;
    a.F0out = F0 + r0 * n;
    a.tab_out = tab;
    a.Tin = Tin ? Tin + r0 : nullptr;
    a.flags = kOutF0 | en | (unhoisted ? 0u : kOutTab);
    a.n_tiles = (nb + m->tile - 1) / m->tile;
    st = run(m, a, stream, "psr_fd_jacobian (base residual)");
    if (st != PSR_OK) return st;
    EvalArgs b{};
    b.N = nb; b.ld = ld; b.T = a.T; b.P = a.P; b.Y = a.Y; b.Yin = a.Yin; b.tau = a.tau;
    b.J = J + r0 * n * n;
    b.F0 = a.F0out;
    b.Tin = a.Tin;
    if (unhoisted) {
      b.flags = kModeJac | en;
      b.n_tiles = (nb * n + m->tile - 1) / m->tile;
      st = run(m, b, stream, "psr_fd_jacobian (all columns)");
      if (st != PSR_OK) return st;
      continue;
    }
    b.flags = kModeJacT | en;                  // column 0: T perturbed, every factor changes
    b.n_tiles = (nb + m->tile - 1) / m->tile;
    st = run(m, b, stream, "psr_fd_jacobian (T column)");
    if (st != PSR_OK) return st;
    b.flags = kModeJacY | en;                  // columns 1..K: T-only factors from the rate table
    b.tab = tab;
    // states = (reactor, species column): packed densely, or padded to whole tiles per reactor (MechView::jy_dense)
    const int64_t Kp = m->view.jy_dense ? K : (K + m->tile - 1) / m->tile * m->tile;
    b.n_tiles = (nb * Kp + m->tile - 1) / m->tile;
    st = run(m, b, stream, "psr_fd_jacobian (Y columns)");
    if (st != PSR_OK) return st;
  }
  return PSR_OK;
}

}  // namespace

extern "C" {

psr_status psr_mech_reserve(psr_mech* m, int64_t N) {
  g_err.clear();
  if (!m || N < 0) return fail(PSR_EINVAL, "psr_mech_reserve: null mechanism or N < 0");
  const size_t need = jac_scratch_bytes(m, N, true, nullptr);
  if (need <= m->scratch_bytes) return PSR_OK;
  void* grown = nullptr;
  cudaError_t e = cudaMalloc(&grown, need);
  if (e != cudaSuccess) return fail(PSR_ENOMEM, "psr_mech_reserve: %s", cudaGetErrorString(e));
  if (m->d_scratch) m->retired.push_back(m->d_scratch);
  m->d_scratch = static_cast<double*>(grown);
  m->scratch_bytes = need;
  return PSR_OK;
}

psr_status psr_fd_jacobian(const psr_mech* mech, int64_t N, const double* T, const double* P, const double* Y,
                           const double* Yin, const double* tau, int64_t ld, double* J, double* F0, void* stream) {
  return fd_jacobian_impl(mech, N, T, P, Y, nullptr, Yin, tau, ld, J, F0, stream, "psr_fd_jacobian");
}

// psr_fd_jacobian through the fused kernel with its scratch in a static device array: no cudaMalloc, cudaFree or
// allocating library routine on this path (argument checks, one cudaGetSymbolAddress per device the first time, one
// kernel launch).
psr_status psr_fd_jacobian_noalloc(const psr_mech* m, int64_t N, const double* T, const double* P, const double* Y,
                                   const double* Yin, const double* tau, int64_t ld, double* J, double* F0, void* stream) {
  g_err.clear();
  psr_status st = check_common(m, N, T, P, Y, ld, "psr_fd_jacobian_noalloc");
  if (st != PSR_OK || N == 0) return st;
  if (!Yin || !tau || !J) return fail(PSR_EINVAL, "psr_fd_jacobian_noalloc: null Yin, tau or J");
  if (m->view.I > PSR_NOALLOC_MAX_REACTIONS)
    return fail(PSR_EUNSUPPORTED, "psr_fd_jacobian_noalloc: %d reactions, the static scratch (%zu bytes) is sized for at most %d",
                (int)m->view.I, jac_static_scratch_bytes(), (int)PSR_NOALLOC_MAX_REACTIONS);
  if (!m->jac_ok)
    return fail(PSR_EUNSUPPORTED, "psr_fd_jacobian_noalloc: the mechanism does not qualify for the fused Jacobian kernel "
                                  "(more than 64 species, falloff reactions with efficiency lists, long factor lists or A <= 0)");
  const size_t per_cta = (size_t)m->view.I * 3 * kTile * 8;
  const int64_t fit = (int64_t)(jac_static_scratch_bytes() / per_cta);   // >= 21 by the limit on the reactions
  EvalArgs a{};
  a.N = N; a.ld = ld; a.T = T; a.P = P; a.Y = Y; a.Yin = Yin; a.tau = tau; a.J = J; a.F0out = F0;
  a.n_tiles = (N + kTile - 1) / kTile;
  const int grid = (int)std::min<int64_t>(std::min<int64_t>(a.n_tiles, m->n_sm), fit);
  cudaError_t e = launch_jac_static(m->jac, a, grid, (cudaStream_t)stream);
  if (e != cudaSuccess) return cuda_fail(e, "psr_fd_jacobian_noalloc");
  return PSR_OK;
}

psr_status psr_fd_jacobian_energy(const psr_mech* mech, int64_t N, const double* T, const double* P, const double* Y,
                                  const double* Tin, const double* Yin, const double* tau, int64_t ld, double* J,
                                  double* F0, void* stream) {
  if (!Tin) {
    g_err = "psr_fd_jacobian_energy: null Tin";
    return PSR_EINVAL;
  }
  return fd_jacobian_impl(mech, N, T, P, Y, Tin, Yin, tau, ld, J, F0, stream, "psr_fd_jacobian_energy");
}

static psr_status solve_impl(const char* who, int64_t N, int32_t n, const double* A, double* b, int32_t* info,
                             const double* F, const double* dt, void* stream, const int32_t* skip_count = nullptr) {
  // SM count and shared-memory limit of the current device, looked up once per device
  static int s_sm[64], s_optin[64];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(e, who);
  int n_sm = 0, optin = 0;
  if (dev >= 0 && dev < 64 && s_sm[dev] > 0) {
    n_sm = s_sm[dev];
    optin = s_optin[dev];
  } else {
    e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return cuda_fail(e, who);
    if (dev >= 0 && dev < 64) {
      s_optin[dev] = optin;
      s_sm[dev] = n_sm;
    }
  }
  if (n > 168) return fail(PSR_EUNSUPPORTED, "%s: n = %d, the one-warp-per-system kernel takes n <= 168", who, n);
  e = launch_lu_solve(N, n, A, b, info, n_sm, (size_t)optin, (cudaStream_t)stream, F, dt, skip_count);
  if (e != cudaSuccess) return cuda_fail(e, who);
  return PSR_OK;
}

psr_status psr_lu_solve(int64_t N, int32_t n, const double* A, double* b, int32_t* info, void* stream) {
  g_err.clear();
  if (N < 0 || n < 1) return fail(PSR_EINVAL, "psr_lu_solve: N < 0 or n < 1");
  if (N == 0) return PSR_OK;
  if (!A || !b || !info) return fail(PSR_EINVAL, "psr_lu_solve: null A, b or info");
  return solve_impl("psr_lu_solve", N, n, A, b, info, nullptr, nullptr, stream);
}

psr_status psr_ptc_solve(int64_t N, int32_t n, const double* J, const double* F, const double* dt, double* dx,
                         int32_t* info, void* stream) {
  g_err.clear();
  if (N < 0 || n < 1) return fail(PSR_EINVAL, "psr_ptc_solve: N < 0 or n < 1");
  if (N == 0) return PSR_OK;
  if (!J || !F || !dt || !dx || !info) return fail(PSR_EINVAL, "psr_ptc_solve: null J, F, dt, dx or info");
  if (dx == F) return fail(PSR_EINVAL, "psr_ptc_solve: dx must not alias F");
  return solve_impl("psr_ptc_solve", N, n, J, dx, info, F, dt, stream);
}

namespace {
// workspace of the hybrid solver.  Per reactor: J, F0, dx (doubles), info and the partition's destination (int32), and
// two copies of the sub-batch's state (HybridState: 2 K + 6 double rows, 6 int32 rows) between which the reactors still
// iterating are moved to the front every kHybridCompactEvery rounds.  Once per call: the counter of active reactors,
// and the padding of the state rows to a stride of a multiple of 32 reactors.
constexpr int kHybridCompactEvery = 8;
size_t hybrid_state_bytes_per_reactor(int n) { return ((size_t)2 * n + 4) * 8 + 6 * 4; }
size_t hybrid_bytes_per_reactor(int n) { return ((size_t)n * n + 2 * (size_t)n) * 8 + 2 * 4 + 2 * hybrid_state_bytes_per_reactor(n); }
size_t hybrid_fixed_bytes(int n) { return 256 + 32 * 2 * hybrid_state_bytes_per_reactor(n) + 256; }

// carves a state of row stride ldw out of the workspace: double rows at d (2 K + 6 of them), int32 rows at q (6)
HybridState hybrid_state_at(double* d, int32_t* q, int K, int64_t ldw, bool adiabatic) {
  HybridState s{};
  s.ldw = ldw;
  s.T = d;
  s.P = d + ldw;
  s.tau = d + 2 * ldw;
  s.Tin = adiabatic ? d + 3 * ldw : nullptr;
  s.Y = d + 4 * ldw;
  s.Yin = s.Y + (size_t)K * ldw;
  s.dt_cur = s.Yin + (size_t)K * ldw;
  s.dt_arg = s.dt_cur + ldw;
  s.mode = q;
  s.it = q + ldw;
  s.status = q + 2 * ldw;
  s.nn = q + 3 * ldw;
  s.np = q + 4 * ldw;
  s.orig = q + 5 * ldw;
  return s;
}
}  // namespace

size_t psr_solve_hybrid_workspace_bytes(const psr_mech* m, int64_t N) {
  if (!m || N < 1) return 0;
  const int n = m->view.K + 1;
  return hybrid_bytes_per_reactor(n) * (size_t)N + hybrid_fixed_bytes(n) + 256;
}

psr_status psr_solve_hybrid(const psr_mech* m, int64_t N, double* T, const double* P, double* Y, const double* Tin,
                            const double* Yin, const double* tau, int64_t ld, const psr_solve_opts* o, void* workspace,
                            size_t workspace_bytes, int32_t* status, int32_t* n_newton, int32_t* n_ptc, void* stream) {
  g_err.clear();
  psr_status st = check_common(m, N, T, P, Y, ld, "psr_solve_hybrid");
  if (st != PSR_OK || N == 0) return st;
  if (!Yin || !tau || !o || !workspace || !status) return fail(PSR_EINVAL, "psr_solve_hybrid: null Yin, tau, opts, workspace or status");
  if (!(o->atol >= 0.0) || !(o->rtol >= 0.0) || !(o->atol + o->rtol > 0.0) || o->max_iter < 0 || o->max_newton < 1 || o->max_ptc < 1 ||
      !(o->dt0 > 0.0) || !(o->dt_grow > 0.0) || !(o->dt_shrink > 0.0) || std::isnan(o->y_floor))
    return fail(PSR_EINVAL, "psr_solve_hybrid: options out of range (atol, rtol >= 0 and not both 0; max_iter >= 0; max_newton, max_ptc >= 1; dt0, dt_grow, dt_shrink > 0)");
  const int K = m->view.K, n = K + 1;
  if (n > 168) return fail(PSR_EUNSUPPORTED, "psr_solve_hybrid: %d unknowns, the linear solve takes <= 168", n);
  uintptr_t base = (reinterpret_cast<uintptr_t>(workspace) + 255) & ~(uintptr_t)255;
  const size_t lost = base - reinterpret_cast<uintptr_t>(workspace);
  if (workspace_bytes <= lost + hybrid_fixed_bytes(n) + hybrid_bytes_per_reactor(n))
    return fail(PSR_EINVAL, "psr_solve_hybrid: workspace smaller than one reactor needs");
  const int64_t Nb = std::min<int64_t>(std::min<int64_t>(N, (int64_t)1 << 30),
                                      (int64_t)((workspace_bytes - lost - hybrid_fixed_bytes(n)) / hybrid_bytes_per_reactor(n)));
  const int64_t ldw = (Nb + 31) & ~(int64_t)31;
  int32_t* n_active = reinterpret_cast<int32_t*>(base);   // reactors of the sub-batch still iterating (device counter)
  double* J = reinterpret_cast<double*>(base + 256);
  double* F0 = J + (size_t)Nb * n * n;
  double* dx = F0 + (size_t)Nb * n;
  double* sd0 = dx + (size_t)Nb * n;                       // double rows of the two states
  double* sd1 = sd0 + (size_t)(2 * K + 6) * ldw;
  int32_t* sq0 = reinterpret_cast<int32_t*>(sd1 + (size_t)(2 * K + 6) * ldw);
  int32_t* sq1 = sq0 + 6 * ldw;
  int32_t* info = sq1 + 6 * ldw;
  int32_t* pos = info + Nb;
  HybridState hs[2] = {hybrid_state_at(sd0, sq0, K, ldw, Tin != nullptr), hybrid_state_at(sd1, sq1, K, ldw, Tin != nullptr)};
  cudaStream_t cs = (cudaStream_t)stream;
  for (int64_t r0 = 0; r0 < N; r0 += Nb) {
    const int64_t nb = std::min(Nb, N - r0);
    int cur = 0;
    // the sub-batch's state into the workspace (the caller's P, Y_in, tau are not to be reordered in place)
    cudaError_t e = launch_hybrid_gather(nb, K, ld, T + r0, P + r0, Y + r0, Tin ? Tin + r0 : nullptr, Yin + r0, tau + r0, hs[cur], *o,
                                         n_active, cs);
    if (e != cudaSuccess) return cuda_fail(e, "psr_solve_hybrid (gather)");
    for (int iter = 0; iter < o->max_iter; ++iter) {
      if (iter > 0 && iter % kHybridCompactEvery == 0) {
        // the reactors still iterating to the front (stable), so that finished ones fill whole tiles and drop out of
        // the Jacobian kernel; on a fixed schedule: nothing returns to the host
        e = launch_hybrid_compact(nb, K, hs[cur], hs[cur ^ 1], pos, n_active, cs);
        if (e != cudaSuccess) return cuda_fail(e, "psr_solve_hybrid (compaction)");
        cur ^= 1;
      }
      const HybridState& s = hs[cur];
      // error vector and Jacobian at the current estimates, the (shifted) solve, the per-reactor decisions
      // (finished reactors are marked in dt_arg and counted in n_active: their tiles and systems are left out, and a
      // round after the last one has finished costs a few empty launches)
      st = fd_jacobian_impl(m, nb, s.T, s.P, s.Y, s.Tin, s.Yin, s.tau, ldw, J, F0, stream, "psr_solve_hybrid", s.dt_arg, n_active);
      if (st != PSR_OK) return st;
      st = solve_impl("psr_solve_hybrid", nb, n, J, dx, info, F0, s.dt_arg, stream, n_active);
      if (st != PSR_OK) return st;
      e = launch_hybrid_update(nb, n, ldw, *o, s.T, s.Y, dx, info, s.dt_cur, s.dt_arg, s.mode, s.it, s.status, s.nn, s.np, n_active, cs);
      if (e != cudaSuccess) return cuda_fail(e, "psr_solve_hybrid (update)");
    }
    e = launch_hybrid_scatter(nb, K, ld, hs[cur], T + r0, Y + r0, status + r0, n_newton ? n_newton + r0 : nullptr,
                              n_ptc ? n_ptc + r0 : nullptr, cs);
    if (e != cudaSuccess) return cuda_fail(e, "psr_solve_hybrid (scatter)");
  }
  return PSR_OK;
}

psr_status psr_mech_set_option(psr_mech* m, int32_t option, int32_t value) {
  g_err.clear();
  if (!m) return fail(PSR_EINVAL, "psr_mech_set_option: null mechanism");
  switch (option) {
    case PSR_OPT_JAC_UNHOISTED: m->opt_jac_unhoisted = value != 0; return PSR_OK;
    case PSR_OPT_FUSED_ONLY: m->opt_fused_only = value != 0; return PSR_OK;
    case PSR_OPT_NO_TMEM: m->opt_no_tmem = value != 0; return PSR_OK;
    case PSR_OPT_JAC_GENERIC: m->opt_jac_generic = value != 0; return PSR_OK;
    default: return fail(PSR_EINVAL, "psr_mech_set_option: unknown option %d", (int)option);
  }
}

int32_t psr_check_failures(int32_t selftest, int32_t* first_code) {
  g_err.clear();
  if (first_code) *first_code = 0;
#ifndef PSR_CHECK
  (void)selftest;
  return -1;   // the product build carries no checks
#else
  if (selftest) {
    cudaError_t e = launch_chk_selftest(0);
    if (e != cudaSuccess) { cuda_fail(e, "psr_check_failures (self-test)"); return -2; }
  }
  unsigned int total = 0, first = 0;
  cudaError_t (*readers[5])(unsigned int*, unsigned int*) = {chk_read_ws, chk_read_wsl, chk_read_jac, chk_read_kernels, chk_read_solve};
  for (auto rd : readers) {
    unsigned int c = 0, code = 0;
    cudaError_t e = rd(&c, &code);
    if (e != cudaSuccess) { cuda_fail(e, "psr_check_failures"); return -2; }
    if (c && !first) first = code;
    total += c;
  }
  if (first_code) *first_code = (int32_t)first;
  return (int32_t)std::min<unsigned int>(total, 0x7fffffffu);
#endif
}

psr_status psr_probe_exp_values(const psr_mech* m, const double* x, double* y, int32_t n) {
  g_err.clear();
  if (!m || !x || !y || n < 0) return fail(PSR_EINVAL, "psr_probe_exp_values: bad argument");
  if (n == 0) return PSR_OK;
  double *dx = nullptr, *dy = nullptr;
  cudaError_t e;
  if ((e = cudaMalloc(&dx, 8 * (size_t)n)) != cudaSuccess) return fail(PSR_ENOMEM, "cudaMalloc: %s", cudaGetErrorString(e));
  if ((e = cudaMalloc(&dy, 8 * (size_t)n)) != cudaSuccess) { cudaFree(dx); return fail(PSR_ENOMEM, "cudaMalloc: %s", cudaGetErrorString(e)); }
  e = cudaMemcpy(dx, x, 8 * (size_t)n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = launch_exp_values(m->d_exptab, dx, dy, n, 0);
  if (e == cudaSuccess) e = cudaMemcpy(y, dy, 8 * (size_t)n, cudaMemcpyDeviceToHost);
  cudaFree(dx);
  cudaFree(dy);
  if (e != cudaSuccess) return cuda_fail(e, "psr_probe_exp_values");
  return PSR_OK;
}

psr_status psr_probe_fp64(int kind, int iters, double* elapsed_ms, double* ops) {
  g_err.clear();
  if (kind < 0 || kind > 2 || iters < 1 || !elapsed_ms || !ops) return fail(PSR_EINVAL, "psr_probe_fp64: bad argument");
  int dev = 0;
  cudaDeviceProp prop;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(e, "psr_probe_fp64");
  if ((e = cudaGetDeviceProperties(&prop, dev)) != cudaSuccess) return cuda_fail(e, "psr_probe_fp64");
  double* sink = nullptr;
  if ((e = cudaMalloc(&sink, 8)) != cudaSuccess) return cuda_fail(e, "psr_probe_fp64");
  const int grid = prop.multiProcessorCount * 8;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  launch_probe(kind, iters, grid, sink, 0);  // warm-up
  cudaEventRecord(e0, 0);
  e = launch_probe(kind, iters, grid, sink, 0);
  cudaEventRecord(e1, 0);
  cudaError_t e2 = cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (e != cudaSuccess) return cuda_fail(e, "psr_probe_fp64 launch");
  if (e2 != cudaSuccess) return cuda_fail(e2, "psr_probe_fp64 sync");
  *elapsed_ms = ms;
  *ops = (double)grid * 256.0 * (double)iters * (kind == 0 ? 64.0 : 8.0);
  return PSR_OK;
}

}  // extern "C"
