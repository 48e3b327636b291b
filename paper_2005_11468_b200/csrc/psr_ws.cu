// psr_ws.cu -- warp-specialised evaluation kernel for mechanisms whose tables stay resident in shared memory.
//
// The fused kernel of psr_kernels.cu runs its per-tile phases (state preparation, reactions, gather,
// epilogue) one after another behind CTA-wide barriers with ONE CTA per SM: whatever a phase leaves idle
// stays idle (measured on C1: reactions 0.11 ms of a 0.21 ms launch; the loads, the state preparation and
// the barriers 0.05 ms, the gather 0.035 ms, the epilogue 0.01 ms, none of it overlapped).  Here the phases
// are roles of different warps that meet only through mbarriers:
//
//   reaction warps (13)  a3..a7: k_f, K_c, k_r, [M], falloff, q of their share of the reactions, tile after
//                        tile without a CTA barrier; q goes to one of two q buffers (one "part" of the
//                        mechanism each), concentrations and per-reactor state come from one of two C tiles.
//   helper warps (7)     a1: TMA bulk loads of the tile after next, state preparation (Wbar, rho, C_i, ln T,
//                        ln C_tot) of the next tile;  a8: gather of the q buffer the reaction warps have just
//                        filled (nu^T q, fixed order, partial sums in shared memory between parts);
//                        a9: residual and stores.
//
//   full_in[b]   bulk loads of a tile landed (tx bytes)            helpers  -> helpers
//   full_C[b]    C tile + state rows of a tile ready               helpers  -> reaction warps
//   empty_C[b]   reaction warps are done with the C tile           reaction -> helpers (next loads into it)
//   full_q[qb]   every reaction warp has written its q rows        reaction -> helpers
//   empty_q[qb]  the part has been gathered                        helpers  -> reaction warps
//
// Tensor memory (K <= 126): four helper warps copy each finished C tile into the four lane quadrants of the SM's
// tensor memory, and the reaction warps take the six factors of a 3+3 record from there (tcgen05.ld) instead of
// shared memory, whose data pipe is the busiest unit of this kernel.
//
// Same tables (psr_tables.h), same per-reaction arithmetic and the same exp as psr_kernels.cu; the steps are
// SURVEY.md 8(a) a1..a9 (Eq. 2, 4-9).
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "psr_math.cuh"
#include "psr_ptx.cuh"
#include "psr_rx.cuh"
#include "psr_tables.h"

namespace psr {

namespace {

__device__ constexpr double kRgasW = 8.31446261815324e7;  // erg/mol/K

// mbarrier slots
constexpr int B_BLOB = 0, B_IN = 1, B_FULLC = 3, B_EMPTYC = 5, B_FULLQ = 7, B_EMPTYQ = 9, B_COUNT = 11;
// per-tile state rows St[b][row][lane]
constexpr int ST_T = 0, ST_LNT = 1, ST_INVT = 2, ST_RHO = 3, ST_CTOT = 4, ST_LNCTOT = 5, ST_INVTAU = 6, ST_INVRHO = 7;

// what the gather needs when a species' row of nu^T q is complete (one entry per helper warp and species slot)
struct __align__(16) SpEnt {
  uint32_t row_off;        // byte offset of the species' row in a [K][32] tile
  uint32_t next_row_off;   // the same of the warp's next owned species
  uint64_t pad_;
  int64_t goff;            // byte offset of the species' row in the [K][ld] outputs
  double W;                // molar mass
};
static_assert(sizeof(SpEnt) == 32, "SpEnt layout");

}  // namespace

// TM: a copy of each C tile in tensor memory (all four lane quadrants), from which the reaction warps take four of a
// record's six concentration factors (psr_rx.cuh, kRxTm); mv.tm_cols columns are allocated.
template <bool OUTK, bool TM>
__global__ void __launch_bounds__(kWsWarps * 32, 1) psr_ws_kernel(const WsView mv, const EvalArgs a, const int bulk_ok) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int K = mv.K;
  const int cs_elems = (K + 2) * kTile, ds_elems = K * kTile, q_elems = (mv.rc + 1) * kTile;
  double* Cs0 = reinterpret_cast<double*>(smem + mv.smem_cs);      // [2][K+2][32]; rows K, K+1: ones, zeros
  double* Ds0 = reinterpret_cast<double*>(smem + mv.smem_ds);      // [2][K][32]: Y_in, then Y - Y_in
  double* qh0 = reinterpret_cast<double*>(smem + mv.smem_q);       // [2][rc+1][32]; row rc stays zero
  double* acc_s = reinterpret_cast<double*>(smem + mv.smem_acc);   // [K][32]: nu^T q summed over the parts so far
  const unsigned char* mech = smem + mv.smem_mech;                 // n_parts blobs
  double* invW_s = reinterpret_cast<double*>(smem + mv.smem_misc); // [Kp]
  const int Kp = (K + 1) & ~1;
  double* W_s = invW_s + Kp;                                       // [Kp]
  double* St0 = W_s + Kp;                                          // [2][kWsStRows][32]
  double* tp0 = St0 + 2 * kWsStRows * kTile;                       // [2][3][32]: T, P, tau as loaded
  uint64_t* bars = reinterpret_cast<uint64_t*>(tp0 + 2 * 3 * kTile);
  uint32_t* tm_slot = reinterpret_cast<uint32_t*>(bars + B_COUNT); // tensor-memory base address (TM)
  int32_t* sp_s = reinterpret_cast<int32_t*>(bars + B_COUNT + 1);  // [helper warps][spw]
  SpEnt* sptab = reinterpret_cast<SpEnt*>(sp_s + ((kWsHelpWarps * mv.spw + 7) & ~7));   // [helper warps][spw]

  const int lane = threadIdx.x & 31;
  const int w = threadIdx.x >> 5;
  const bool wantF = (a.flags & kOutF) != 0;

  if (threadIdx.x == 0) {
    mbar_init(&bars[B_BLOB], 1);
    for (int b = 0; b < 2; ++b) {
      mbar_init(&bars[B_IN + b], kWsHelpWarps);
      mbar_init(&bars[B_FULLC + b], kWsHelpWarps);
      mbar_init(&bars[B_EMPTYC + b], kWsRxWarps);
      mbar_init(&bars[B_FULLQ + b], kWsRxWarps);
      mbar_init(&bars[B_EMPTYQ + b], kWsHelpWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
    const uint32_t bytes = mv.chunk_stride * (uint32_t)mv.n_parts;
    mbar_expect_tx(&bars[B_BLOB], bytes);
    bulk_g2s(smem + mv.smem_mech, mv.chunks, bytes, &bars[B_BLOB]);
  }
  if (w == 0) {
    if constexpr (TM) tm_alloc(tm_slot, (uint32_t)mv.tm_cols);
    for (int b = 0; b < 2; ++b) {
      Cs0[b * cs_elems + K * kTile + lane] = 1.0;         // unit row: unused factor slots
      Cs0[b * cs_elems + (K + 1) * kTile + lane] = 0.0;   // zero row: product side of an irreversible reaction
      qh0[b * q_elems + mv.rc * kTile + lane] = 0.0;      // zero row: padding of the gather lists
    }
  }
  for (int i = threadIdx.x; i < K; i += kWsWarps * 32) {
    invW_s[i] = mv.invW[i];
    W_s[i] = mv.Wm[i];
  }
  for (int i = threadIdx.x; i < kWsHelpWarps * mv.spw; i += kWsWarps * 32) {
    sp_s[i] = mv.sp_of[i];
    // the flush table of the gather: slots past a warp's last owned species repeat that species
    const int hw_ = i / mv.spw;
    int jj = i - hw_ * mv.spw, jn = jj + 1;
    while (jj > 0 && mv.sp_of[hw_ * mv.spw + jj] < 0) --jj;
    if (jn >= mv.spw || mv.sp_of[hw_ * mv.spw + jn] < 0) jn = jj;
    const int s_ = max(mv.sp_of[hw_ * mv.spw + jj], 0), sn_ = max(mv.sp_of[hw_ * mv.spw + jn], 0);
    sptab[i].row_off = (uint32_t)s_ * kRowBytes;
    sptab[i].next_row_off = (uint32_t)sn_ * kRowBytes;
    sptab[i].goff = (int64_t)s_ * a.ld * 8;
    sptab[i].W = mv.Wm[s_];
  }
  if constexpr (TM) tm_fence_before_sync();
  __syncthreads();
  uint32_t tm_quad = 0;   // this warp's quadrant of the allocation, buffer 0; buffer 1 is mv.tm_buf columns further
  if constexpr (TM) {
    tm_fence_after_sync();
    tm_quad = *tm_slot + ((uint32_t)((w & 3) * 32) << 16);
  }

  if (w < kWsRxWarps) {
    // ================================================================== reaction warps
    RxCtx cx;
    cx.etab = exp_tab_load(mv.exp_tab);
#ifdef PSR_CHECK
    cx.chk_c_bytes = (uint32_t)cs_elems * 8u;
#endif
    mbar_wait(&bars[B_BLOB], 0);
    int64_t tile = blockIdx.x;
    for (uint32_t lt = 0; tile < a.n_tiles; ++lt, tile += gridDim.x) {
      const int b = lt & 1;
      mbar_wait(&bars[B_FULLC + b], (lt >> 1) & 1);
      if constexpr (TM) {
        tm_fence_after_sync();
        cx.tm_c = tm_quad + (uint32_t)b * (uint32_t)mv.tm_buf;
      }
      const uint32_t st_lane = smem_u32(St0 + b * kWsStRows * kTile) + lane * 8;
      cx.c_lane = smem_u32(Cs0 + b * cs_elems) + lane * 8;
      cx.ctot_lane = st_lane + ST_CTOT * kRowBytes;
      cx.lnctot_lane = st_lane + ST_LNCTOT * kRowBytes;
      cx.T = lds64(st_lane + ST_T * kRowBytes);
      cx.lnT = lds64(st_lane + ST_LNT * kRowBytes);
      cx.invT = lds64(st_lane + ST_INVT * kRowBytes);
      const int64_t r = tile * kTile + lane;
      const bool valid = r < a.N;
      for (int p = 0; p < mv.n_parts; ++p) {
        const uint32_t g = lt * (uint32_t)mv.n_parts + (uint32_t)p, qb = g & 1, u = g >> 1;
        if (u > 0) mbar_wait(&bars[B_EMPTYQ + qb], (u - 1) & 1);   // the part that used this buffer before has been gathered
        const uint32_t q_lane = smem_u32(qh0 + qb * q_elems) + lane * 8;
        const unsigned char* blob = mech + (size_t)p * mv.chunk_stride;
        // Eq. 5: q = k_f prod C^nu' - k_r prod C^nu'' (x [M] for a three-body reaction).  An irreversible reaction has
        // its product side on the zero row (pr = 0): no per-lane selects here.
        auto sink = [&](int kl, uint32_t meta, uint32_t korig, int type, double kf, double kr, double pf, double pr, double M) {
          if (type == RX_THREE_BODY) {
            pf *= M;
            pr *= M;
          }
          const double q = fma(kf, pf, -(kr * pr));
          PSR_CHK(kl >= 0 && kl < mv.rc, 201);                               // a row of the q buffer (row rc is the zero row)
          PSR_CHK(!OUTK || !valid || (int64_t)korig < (int64_t)mv.I, 202);   // a row of the kf / kr / q outputs
          sts64(q_lane + (uint32_t)kl * (uint32_t)kRowBytes, q);
          if constexpr (OUTK) {
            if (valid) {
              const int64_t o = (int64_t)korig * a.ldk + r;
              if (a.flags & kOutKf) a.kf[o] = kf;
              if (a.flags & kOutKr) a.kr[o] = (meta & kMetaRev) ? kr : 0.0;
              if (a.flags & kOutQ) a.q[o] = q;
            }
          }
        };
        cx.amax = 0.0f;
        rx_run_chunk<kRxFast | (TM ? kRxTm : 0)>(cx, blob, w, sink);
        // an exp argument out of the table form's range (NaN, Inf, overflow, underflow: never for physical
        // states): this warp repeats its records with the library exp, which keeps IEEE results
        if (__any_sync(kFullMask, !exp_max_in_range(cx.amax))) rx_run_chunk<(TM ? kRxTm : 0)>(cx, blob, w, sink);
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars[B_FULLQ + qb]);
      }
      if constexpr (TM) tm_fence_before_sync();   // (every tensor-memory read of the tile has been waited for)
      if (lane == 0) mbar_arrive(&bars[B_EMPTYC + b]);
    }
  } else {
    // ================================================================== helper warps
    const int hw = w - kWsRxWarps;
    const int32_t* my_sp = sp_s + hw * mv.spw;
    int n_my = 0;
    while (n_my < mv.spw && my_sp[n_my] >= 0) ++n_my;   // owned species come first, -1 pads the list
    auto tile_bulk = [&](int64_t t) { return bulk_ok && (t + 1) * kTile <= a.N; };
    // a1, first half: bring a tile's Y (into the C tile), Y_in, T, P, tau into buffer b.  Whole tiles of aligned
    // arrays come by one bulk copy per species row (256 contiguous bytes); the ragged last tile and unaligned
    // arrays by plain loads of this warp's own rows (lanes past N read reactor N-1, a valid state, unused).
    auto issue_loads = [&](int64_t t, int b) {
      double* Cb = Cs0 + b * cs_elems;
      double* Db = Ds0 + b * ds_elems;
      double* tb = tp0 + b * 3 * kTile;
      if (tile_bulk(t)) {
        fence_proxy_async();
        if (lane == 0) {
          const uint32_t bytes = (uint32_t)n_my * kRowBytes * (wantF ? 2u : 1u) + (hw == 0 ? (wantF ? 3u : 2u) * kRowBytes : 0u);
          mbar_expect_tx(&bars[B_IN + b], bytes);
        }
        __syncwarp();
        const int64_t r0 = t * kTile;
        if (lane < n_my) {
          const int s = my_sp[lane];
          bulk_g2s(Cb + s * kTile, a.Y + (int64_t)s * a.ld + r0, kRowBytes, &bars[B_IN + b]);
          if (wantF) bulk_g2s(Db + s * kTile, a.Yin + (int64_t)s * a.ld + r0, kRowBytes, &bars[B_IN + b]);
        }
        if (hw == 0 && lane == 31) {
          bulk_g2s(tb, a.T + r0, kRowBytes, &bars[B_IN + b]);
          bulk_g2s(tb + kTile, a.P + r0, kRowBytes, &bars[B_IN + b]);
          if (wantF) bulk_g2s(tb + 2 * kTile, a.tau + r0, kRowBytes, &bars[B_IN + b]);
        }
      } else {
        int64_t r = t * kTile + lane;
        if (r >= a.N) r = a.N - 1;
        for (int jj = 0; jj < n_my; ++jj) {
          const int s = my_sp[jj];
          Cb[s * kTile + lane] = ldg_nc(a.Y + (int64_t)s * a.ld + r);
          if (wantF) Db[s * kTile + lane] = ldg_nc(a.Yin + (int64_t)s * a.ld + r);
        }
        if (hw == 0) {
          tb[lane] = ldg_nc(a.T + r);
          tb[kTile + lane] = ldg_nc(a.P + r);
          if (wantF) tb[2 * kTile + lane] = ldg_nc(a.tau + r);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars[B_IN + b]);
      }
    };
    // a1, second half: W_bar = 1/sum Y_i/W_i, rho = P W_bar/(R T), C_i = rho Y_i/W_i, C_tot = rho sum Y_i/W_i, and
    // the per-reactor state rows of tile number lt (of this CTA) in buffer b = lt & 1.  Every helper warp forms
    // the sum over all species itself (no exchange of partial sums), then converts its own rows.
    auto prologue = [&](uint32_t lt) {
      const int b = lt & 1;
      double* Cb = Cs0 + b * cs_elems;
      double* Db = Ds0 + b * ds_elems;
      const double* tb = tp0 + b * 3 * kTile;
      double* St = St0 + b * kWsStRows * kTile;
      mbar_wait(&bars[B_IN + b], (lt >> 1) & 1);
      const double T = tb[lane], P = tb[kTile + lane];
      double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
      int s = 0;
      for (; s + 4 <= K; s += 4) {
        s0 = fma(Cb[s * kTile + lane], invW_s[s], s0);
        s1 = fma(Cb[(s + 1) * kTile + lane], invW_s[s + 1], s1);
        s2 = fma(Cb[(s + 2) * kTile + lane], invW_s[s + 2], s2);
        s3 = fma(Cb[(s + 3) * kTile + lane], invW_s[s + 3], s3);
      }
      for (; s < K; ++s) s0 = fma(Cb[s * kTile + lane], invW_s[s], s0);
      const double sY = (s0 + s1) + (s2 + s3);
      const double Wbar = 1.0 / sY;
      const double rho = P * Wbar / (kRgasW * T);
      if (hw == 0) {
        St[ST_T * kTile + lane] = T;
        St[ST_LNT * kTile + lane] = log(T);
        St[ST_INVT * kTile + lane] = 1.0 / T;
      } else if (hw == 1) {
        // C_tot = sum_i C_i = rho sum_i Y_i/W_i, from the sum already at hand (differs from the species-by-species
        // sum by rounding only)
        const double ct = rho * sY;
        St[ST_RHO * kTile + lane] = rho;
        St[ST_CTOT * kTile + lane] = ct;
        if (mv.need_lnctot) St[ST_LNCTOT * kTile + lane] = log(ct);   // Troe reactions without efficiencies
      } else if (hw == 2 && wantF) {
        St[ST_INVTAU * kTile + lane] = 1.0 / tb[2 * kTile + lane];
        St[ST_INVRHO * kTile + lane] = 1.0 / rho;
      }
      named_bar_sync(1, kWsHelpWarps * 32);   // every helper warp has read the Y rows; the rows above are visible
      for (int jj = 0; jj < n_my; ++jj) {
        const int sp = my_sp[jj];
        const double y = Cb[sp * kTile + lane];
        if (wantF) Db[sp * kTile + lane] = y - Db[sp * kTile + lane];
        Cb[sp * kTile + lane] = rho * (y * invW_s[sp]);
      }
      if constexpr (TM) {
        // the finished tile (unit and zero rows included) into tensor memory, once per lane quadrant: four
        // consecutive warps reach the four quadrants.  Buffer b was released by the reaction warps through empty_C,
        // which this warp has waited for (issue_loads of this tile).
        static_assert(kWsHelpWarps >= 4, "four helper warps copy the C tile to the four TMEM quadrants");
        named_bar_sync(2, kWsHelpWarps * 32);   // every row of the tile is final
        if (hw < 4) {
          tm_fence_after_sync();
          const uint32_t tq = tm_quad + (uint32_t)b * (uint32_t)mv.tm_buf;
          const int last = K + 1;
          for (int s4 = 0; s4 <= last; s4 += 4)
            tm_st64x4(tq + 2u * (uint32_t)s4, Cb[s4 * kTile + lane], Cb[min(s4 + 1, last) * kTile + lane],
                      Cb[min(s4 + 2, last) * kTile + lane], Cb[min(s4 + 3, last) * kTile + lane]);
          tm_wait_st();
          tm_fence_before_sync();
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars[B_FULLC + b]);
    };

    // a8 (Eq. 4) and a9 (Eq. 2): this warp's stream of 4-entry groups of nu^T q of one part (psr_tables.h), in a fixed
    // order, two groups per trip.  Software-pipelined: the q rows of a pair are read one trip before they are
    // added and its offsets two trips before (the stream ends with padding groups), so a trip adds values that
    // have already arrived.  A group's sum enters the species' running sum with the group's sign; the group that
    // ends a species stores the sum -- to the partial-sum tile, or (last part) as wdot and F to global memory.
    auto gather_part = [&](auto first_tag, auto last_tag, const uint32_t gs, const int n_groups, const uint32_t q_lane,
                           const int b, const int64_t r, const bool valid) {
      constexpr bool FIRST = decltype(first_tag)::value, LAST = decltype(last_tag)::value;
      auto ld_group = [&](uint32_t addr, uint4& o) {
        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(o.x), "=r"(o.y), "=r"(o.z), "=r"(o.w) : "r"(addr));
      };
      const uint32_t acc_lane = smem_u32(acc_s) + lane * 8;
      const uint32_t d_lane = smem_u32(Ds0 + b * ds_elems) + lane * 8;
      const uint32_t tbl = smem_u32(sptab + hw * mv.spw);
      double invtau = 0.0, invrho = 0.0;
      if (LAST && wantF) {
        invtau = St0[(b * kWsStRows + ST_INVTAU) * kTile + lane];
        invrho = St0[(b * kWsStRows + ST_INVRHO) * kTile + lane];
      }
      const bool out_w = (a.flags & kOutWdot) != 0;
      const char* wdot_r = reinterpret_cast<const char*>(a.wdot + r);
      const char* F_r = reinterpret_cast<const char*>(a.F + r);
      uint32_t te = tbl;   // table entry of the species being summed
      double acc = 0.0;
      if (!FIRST && n_groups > 0) acc = lds64(acc_lane + reinterpret_cast<const SpEnt*>(sptab + hw * mv.spw)->row_off);
      auto flush = [&]() {
        uint32_t row_off, pad;
        double W;
        int64_t goff;
        PSR_CHK(te >= tbl && te < tbl + (uint32_t)mv.spw * (uint32_t)sizeof(SpEnt), 203);   // one flush per owned species
        asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(row_off), "=r"(pad) : "r"(te));
        PSR_CHK(row_off < (uint32_t)ds_elems * 8u && pad < (uint32_t)ds_elems * 8u, 204);
        if (LAST) {
          asm volatile("ld.shared.v2.b64 {%0, %1}, [%2+16];" : "=l"(goff), "=d"(W) : "r"(te));
          PSR_CHK(!valid || (goff >= 0 && goff % 8 == 0 && r < a.N && goff / 8 + r < (int64_t)K * a.ld), 205);   // element (species, r) of a [K][ld] output
          if (valid) {
            if (out_w) *reinterpret_cast<double*>(const_cast<char*>(wdot_r) + goff) = acc;
            if (wantF)
              *reinterpret_cast<double*>(const_cast<char*>(F_r) + goff) = fma(lds64(d_lane + row_off), invtau, -(acc * (W * invrho)));
          }
        } else {
          sts64(acc_lane + row_off, acc);
        }
        te += sizeof(SpEnt);
        // (the entry after the last owned species is a copy of the last one: harmless read)
        if (FIRST) acc = 0.0;
        else acc = lds64(acc_lane + pad);   // pad = row offset of the NEXT owned species
      };
      auto sgn = [](uint32_t ctl) { return __hiloint2double((int)(0x3ff00000u ^ (ctl << 31)), 0); };
      uint4 oa, ob;
      ld_group(gs, oa);
      ld_group(gs + 16, ob);
      double a0 = lds64(q_lane + (oa.x & ~3u)), a1 = lds64(q_lane + oa.y), a2 = lds64(q_lane + oa.z), a3 = lds64(q_lane + oa.w);
      double b0 = lds64(q_lane + (ob.x & ~3u)), b1 = lds64(q_lane + ob.y), b2 = lds64(q_lane + ob.z), b3 = lds64(q_lane + ob.w);
      uint32_t ca = oa.x, cb = ob.x;
      ld_group(gs + 32, oa);
      ld_group(gs + 48, ob);
#pragma unroll 1
      for (int i = 0; i < n_groups; i += 2) {
        const double ta = (a0 + a2) + (a1 + a3), tb = (b0 + b2) + (b1 + b3);
        const uint32_t c0 = ca, c1 = cb;
        ca = oa.x;
        cb = ob.x;
        {   // the groups read ahead (padding groups included) point at rows of the q buffer, zero row included
          const uint32_t qmax = (uint32_t)q_elems * 8u;
          PSR_CHK((oa.x & ~3u) < qmax && oa.y < qmax && oa.z < qmax && oa.w < qmax && (ob.x & ~3u) < qmax && ob.y < qmax &&
                      ob.z < qmax && ob.w < qmax, 206);
        }
        a0 = lds64(q_lane + (oa.x & ~3u)), a1 = lds64(q_lane + oa.y), a2 = lds64(q_lane + oa.z), a3 = lds64(q_lane + oa.w);
        b0 = lds64(q_lane + (ob.x & ~3u)), b1 = lds64(q_lane + ob.y), b2 = lds64(q_lane + ob.z), b3 = lds64(q_lane + ob.w);
        ld_group(gs + (uint32_t)(i + 4) * 16u, oa);
        ld_group(gs + (uint32_t)(i + 5) * 16u, ob);
        acc = fma(ta, sgn(c0), acc);
        if (c0 & kGatherLast) flush();
        acc = fma(tb, sgn(c1), acc);
        if (c1 & kGatherLast) flush();
      }
    };

    const int64_t stride = gridDim.x;
    int64_t tile = blockIdx.x;
    if (tile < a.n_tiles) issue_loads(tile, 0);
    if (tile + stride < a.n_tiles) issue_loads(tile + stride, 1);
    if (tile < a.n_tiles) prologue(0);   // (needs no mechanism table: runs while the blobs are still landing)
    mbar_wait(&bars[B_BLOB], 0);
    for (uint32_t lt = 0; tile < a.n_tiles; ++lt, tile += stride) {
      const int b = lt & 1;
      if (tile + stride < a.n_tiles) prologue(lt + 1);
      const int64_t r = tile * kTile + lane;
      const bool valid = r < a.N;
      for (int p = 0; p < mv.n_parts; ++p) {
        const uint32_t g = lt * (uint32_t)mv.n_parts + (uint32_t)p, qb = g & 1, u = g >> 1;
        const bool first = p == 0, last = p == mv.n_parts - 1;
        const unsigned char* blob = mech + (size_t)p * mv.chunk_stride;
        const ChunkHdr* hdr = reinterpret_cast<const ChunkHdr*>(blob);
        const uint32_t gs = smem_u32(blob + hdr->off_gent) + (uint32_t)hdr->wb[kWsRxWarps + hw][0] * 16u;
        const int n_groups = (int)hdr->wb[kWsRxWarps + hw][1] - (int)hdr->wb[kWsRxWarps + hw][0];   // even
        const uint32_t q_lane = smem_u32(qh0 + qb * q_elems) + lane * 8;
        mbar_wait(&bars[B_FULLQ + qb], u & 1);
        if (first && last) gather_part(std::true_type{}, std::true_type{}, gs, n_groups, q_lane, b, r, valid);
        else if (first) gather_part(std::true_type{}, std::false_type{}, gs, n_groups, q_lane, b, r, valid);
        else if (last) gather_part(std::false_type{}, std::true_type{}, gs, n_groups, q_lane, b, r, valid);
        else gather_part(std::false_type{}, std::false_type{}, gs, n_groups, q_lane, b, r, valid);
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars[B_EMPTYQ + qb]);
      }
      // buffer b is free once the reaction warps have left the tile: the tile after next goes there
      if (tile + 2 * stride < a.n_tiles) {
        mbar_wait(&bars[B_EMPTYC + b], (lt >> 1) & 1);
        issue_loads(tile + 2 * stride, b);
      }
    }
  }
  if constexpr (TM) {
    tm_fence_before_sync();
    __syncthreads();   // no warp touches tensor memory any more
    if (w == 0) tm_dealloc(*tm_slot, (uint32_t)mv.tm_cols);
  }
}

// once per process: the kernels' dynamic shared-memory limit raised to the device's (mechanisms of different sizes
// share the kernel instances)
PSR_CHK_TU_READER(chk_read_ws)

cudaError_t ws_set_smem(size_t smem) {
  cudaError_t e = cudaFuncSetAttribute(psr_ws_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(psr_ws_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(psr_ws_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(psr_ws_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  return e;
}

cudaError_t launch_ws(const WsView& mv, const EvalArgs& a, int grid, int bulk_ok, cudaStream_t st) {
  const bool outk = (a.flags & (kOutKf | kOutKr | kOutQ)) != 0;
  if (mv.tm_cols > 0) {
    if (outk) psr_ws_kernel<true, true><<<grid, kWsWarps * 32, mv.smem_total, st>>>(mv, a, bulk_ok);
    else psr_ws_kernel<false, true><<<grid, kWsWarps * 32, mv.smem_total, st>>>(mv, a, bulk_ok);
  } else {
    if (outk) psr_ws_kernel<true, false><<<grid, kWsWarps * 32, mv.smem_total, st>>>(mv, a, bulk_ok);
    else psr_ws_kernel<false, false><<<grid, kWsWarps * 32, mv.smem_total, st>>>(mv, a, bulk_ok);
  }
  return cudaGetLastError();
}

}  // namespace psr
