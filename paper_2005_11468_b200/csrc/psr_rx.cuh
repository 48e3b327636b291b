// psr_rx.cuh -- evaluation of a warp's share of the reaction records of one chunk blob (SURVEY.md 8(a) a3..a7:
// k_f, K_c, k_r, [M], falloff, concentration products; Eq. 5-9), shared by the kernels that keep
// lane <-> reactor and the mechanism tables in shared memory (psr_ws.cu, psr_jac.cu).  What a kernel does with a
// reaction's rates -- form q and store it, tabulate the factors -- is its own: the `sink` functor.
// Internal to the library.
#ifndef PSR_RX_CUH_
#define PSR_RX_CUH_
#include <cuda_runtime.h>
#include <stdint.h>

#include "psr_math.cuh"
#include "psr_ptx.cuh"
#include "psr_tables.h"

namespace psr {

__device__ constexpr double kRxLog10e = 0.43429448190325182765;
constexpr int RX_PLAIN = 0, RX_THREE_BODY = 1, RX_LINDEMANN = 2, RX_TROE = 3;  // = PSR_RX_* of psr.h

// per-lane state of the tile the records are evaluated on
struct RxCtx {
  double T, lnT, invT;
  uint32_t c_lane;      // this lane's column of row 0 of the C tile (shared-memory address); row K: ones, K+1: zeros
  uint32_t ctot_lane;   // this lane's C_tot, shared-memory address
  uint32_t lnctot_lane; // this lane's ln C_tot
  uint32_t tm_c;        // MODE & kRxTm: tensor-memory address of row 0 of a copy of the C tile (this warp's quadrant)
  ExpTab etab;
  float amax;           // NaN-propagating running max of |high word| of the exp arguments of this lane
#ifdef PSR_CHECK
  uint32_t chk_c_bytes; // size of the C tile in bytes, (K + 2) rows: bound of every factor / efficiency offset
#endif
};

// One record class of warp w's share of a chunk.  CLS: 0..3 = reaction type in the 3+3 slot form, kClsLong = long
// factor lists (any type, signs of A).  MODE & kRxFast: table exp, range noted in cx.amax; else the library exp.
// MODE & kRxTm: the six factors of a 3+3 record come from the copy of the C tile in tensor memory (cx.tm_c) instead
// of shared memory -- those row reads leave the shared-memory pipe; asked for at the top of a trip, waited for at
// its end; efficiency lists come four entries at a time, long factor lists one factor at a time: in this mode the
// reaction code does not read the shared-memory C tile at all (C_tot and ln C_tot are state rows, not tile rows).
// sink(kl, meta, korig, type, kf, kr, pf, pr, M): effective rate constants (falloff applied), the concentration
// products of the two sides WITHOUT [M], and [M] (1 for a plain reaction) of record kl.
constexpr int kRxFast = 1, kRxTm = 2;
template <int CLS, int MODE, class Sink>
__device__ __forceinline__ void rx_run_class(RxCtx& cx, const unsigned char* blob, const ChunkHdr* hdr, const RxRec* recs,
                                             const int kl_begin, const int kl_end, Sink&& sink) {
  constexpr bool FAST = (MODE & kRxFast) != 0, TMA = (MODE & kRxTm) != 0, TM = TMA && CLS < kClsLong;
  PSR_CHK(kl_begin >= 0 && kl_begin <= kl_end && kl_end <= (int)hdr->n_rx, 101);
  if (kl_begin >= kl_end) return;   // nothing of this class for this warp in this chunk (the rule in small parts)
  auto exps = [&](auto& ex, auto& ey) {
    constexpr int N = sizeof(ex) / sizeof(double);
    if constexpr (FAST) {
#pragma unroll
      for (int i = 0; i < N; ++i) cx.amax = exp_arg_max(cx.amax, ex[i]);
      exp_core_n<N>(ex, ey, cx.etab);
    } else {
#pragma unroll
      for (int i = 0; i < N; ++i) ey[i] = exp(ex[i]);
    }
  };
  // slot offsets (and meta, korig) of a record are read one trip ahead: they head the longest chain of a trip
  uint4 nxa, nxb;
  {
    const uint32_t ra = smem_u32(recs + kl_begin) + 80;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(nxa.x), "=r"(nxa.y), "=r"(nxa.z), "=r"(nxa.w) : "r"(ra));
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4+16];" : "=r"(nxb.x), "=r"(nxb.y), "=r"(nxb.z), "=r"(nxb.w) : "r"(ra));
  }
#pragma unroll 1
  for (int kl = kl_begin; kl < kl_end; ++kl) {
    const RxRec* rec = recs + kl;
    const uint4 ra_ = nxa, rb_ = nxb;   // {meta, off[0..2]}, {off[3..5], korig} of this record
    {
      const uint32_t ra = smem_u32(rec) + (112 + 80);
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(nxa.x), "=r"(nxa.y), "=r"(nxa.z), "=r"(nxa.w) : "r"(ra));
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4+16];" : "=r"(nxb.x), "=r"(nxb.y), "=r"(nxb.z), "=r"(nxb.w) : "r"(ra));
    }
    const uint32_t meta = ra_.x;
    const int type = CLS < kClsLong ? CLS : (int)(meta & kMetaTypeMask);
    const double T = cx.T, lnT = cx.lnT, invT = cx.invT;
    // Eq. 6 in log form, and ln k_r = ln k_f - ln K_c (Eq. 7-9 summed per reaction at load time)
    const double lnkf = fma(rec->c[1], lnT, fma(rec->c[2], invT, rec->c[0]));
    const double pn = fma(fma(fma(rec->d[3], T, rec->d[2]), T, rec->d[1]), T, rec->d[0]);
    const double lnkr = fma(pn, T, fma(rec->e[1], lnT, fma(rec->e[2], invT, rec->e[0])));
    double pf, pr, kf = 0.0, kr = 0.0, Mout = 1.0;
    TmF64 tf0, tf1, tf2, tp0, tp1, tp2;
    (void)tf0, (void)tf1, (void)tf2, (void)tp0, (void)tp1, (void)tp2;

    // concentration products (Eq. 5): integer powers by repetition, unused slots read the unit row
    if constexpr (CLS < kClsLong) {
      PSR_CHK(ra_.y < cx.chk_c_bytes && ra_.z < cx.chk_c_bytes && ra_.w < cx.chk_c_bytes && rb_.x < cx.chk_c_bytes &&
                  rb_.y < cx.chk_c_bytes && rb_.z < cx.chk_c_bytes && ((ra_.y | ra_.z | ra_.w | rb_.x | rb_.y | rb_.z) % kRowBytes) == 0, 102);
      if constexpr (TM) {
        // row offsets are multiples of kRowBytes = 256: row r <-> columns 2r, 2r + 1
        tm_ld64(cx.tm_c + (ra_.y >> 7), tf0);
        tm_ld64(cx.tm_c + (ra_.z >> 7), tf1);
        tm_ld64(cx.tm_c + (rb_.x >> 7), tp0);
        tm_ld64(cx.tm_c + (rb_.y >> 7), tp1);
        tm_ld64(cx.tm_c + (ra_.w >> 7), tf2);
        tm_ld64(cx.tm_c + (rb_.z >> 7), tp2);
      } else {
        const double f0 = lds64(cx.c_lane + ra_.y), f1 = lds64(cx.c_lane + ra_.z), f2 = lds64(cx.c_lane + ra_.w);
        const double p0 = lds64(cx.c_lane + rb_.x), p1 = lds64(cx.c_lane + rb_.y), p2 = lds64(cx.c_lane + rb_.z);
        pf = f0 * f1 * f2;
        pr = p0 * p1 * p2;
      }
    } else {
      const uint16_t* fsp = reinterpret_cast<const uint16_t*>(blob + hdr->off_pool) + ra_.y;
      const int nr = (int)((meta >> kMetaNrShift) & 0xF);
      const int np = (int)((meta >> kMetaNpShift) & 0xF);
      pf = 1.0;
      pr = 1.0;
#pragma unroll 1
      for (int j = 0; j < nr + np; ++j) {
        PSR_CHK((uint32_t)fsp[j] * (uint32_t)kRowBytes < cx.chk_c_bytes, 103);
        double cv;
        if constexpr (TMA) {   // (rare records: one factor at a time)
          TmF64 t;
          tm_ld64(cx.tm_c + 2u * (uint32_t)fsp[j], t);
          tm_wait_ld1(t);
          cv = t.get();
        } else {
          cv = lds64(cx.c_lane + (uint32_t)fsp[j] * (uint32_t)kRowBytes);
        }
        if (j < nr) pf *= cv;
        else pr *= cv;
      }
      if (!(meta & kMetaRev)) pr = 0.0;
    }

    // sign of A and of A0/A (any finite A is accepted: negative pre-exponentials of duplicate reactions, A = 0): only
    // long-form records carry them (psr_tables.h), so this folds away in the other class loops
    double sA = 1.0, sPr = 1.0;
    if constexpr (CLS == kClsLong) {
      const uint32_t sg = (meta >> kMetaSgnShift) & 0xFu;
      if (sg) {
        const double s0 = (sg >> 2) == 0 ? 1.0 : (sg >> 2) == 1 ? -1.0 : 0.0;
        sA = (sg & 3u) == 0 ? 1.0 : (sg & 3u) == 1 ? -1.0 : 0.0;
        sPr = sA == 0.0 ? __longlong_as_double(0x7ff8000000000000LL) : s0 * sA;   // k0 [M] / 0 is not a number
      }
    }
    if (type <= RX_THREE_BODY) {
      double ex[2], ey[2];
      ex[0] = lnkf;
      ex[1] = lnkr;
      exps(ex, ey);
      kf = ey[0];
      kr = ey[1];
      if constexpr (CLS == kClsLong) {
        kf *= sA;
        kr *= sA;
      }
    }
    if (type != RX_PLAIN) {
      const AuxRec* ax = reinterpret_cast<const AuxRec*>(blob + hdr->off_aux) + (meta >> kMetaAuxShift);
      const EffEnt* effs = reinterpret_cast<const EffEnt*>(blob + hdr->off_eff);
      double M = lds64(cx.ctot_lane);
      const uint32_t e1 = ax->eff_off + ax->n_eff;
      PSR_CHK((meta >> kMetaAuxShift) < hdr->n_aux && e1 <= hdr->n_eff, 104);
      if constexpr (TMA) {
        // the efficiency list four entries at a time from the tensor-memory copy; slots past the end re-read the last
        // entry and are not added
#pragma unroll 1
        for (uint32_t e = ax->eff_off; e < e1; e += 4) {
          TmF64 t0, t1, t2, t3;
          const uint32_t i1 = min(e + 1, e1 - 1), i2 = min(e + 2, e1 - 1), i3 = min(e + 3, e1 - 1);
          PSR_CHK(effs[e].off < cx.chk_c_bytes && effs[i3].off < cx.chk_c_bytes, 105);
          tm_ld64(cx.tm_c + (effs[e].off >> 7), t0);
          tm_ld64(cx.tm_c + (effs[i1].off >> 7), t1);
          tm_ld64(cx.tm_c + (effs[i2].off >> 7), t2);
          tm_ld64(cx.tm_c + (effs[i3].off >> 7), t3);
          const double a0 = effs[e].am1, a1 = effs[i1].am1, a2 = effs[i2].am1, a3 = effs[i3].am1;
          tm_wait_ld4(t0, t1, t2, t3);
          M = fma(a0, t0.get(), M);
          if (e + 1 < e1) M = fma(a1, t1.get(), M);
          if (e + 2 < e1) M = fma(a2, t2.get(), M);
          if (e + 3 < e1) M = fma(a3, t3.get(), M);
        }
      } else {
        // four entries per trip, their loads issued together (one at a time the list is a chain of shared-memory
        // latencies: 3 % of the C1 kernel's samples); slots past the end re-read the last entry and are not added
#pragma unroll 1
        for (uint32_t e = ax->eff_off; e < e1; e += 4) {
          const uint32_t i1 = min(e + 1, e1 - 1), i2 = min(e + 2, e1 - 1), i3 = min(e + 3, e1 - 1);
          PSR_CHK(effs[e].off < cx.chk_c_bytes && effs[i3].off < cx.chk_c_bytes, 105);
          const double a0 = effs[e].am1, a1 = effs[i1].am1, a2 = effs[i2].am1, a3 = effs[i3].am1;
          const double c0 = lds64(cx.c_lane + effs[e].off), c1 = lds64(cx.c_lane + effs[i1].off),
                       c2 = lds64(cx.c_lane + effs[i2].off), c3 = lds64(cx.c_lane + effs[i3].off);
          M = fma(a0, c0, M);
          if (e + 1 < e1) M = fma(a1, c1, M);
          if (e + 2 < e1) M = fma(a2, c2, M);
          if (e + 3 < e1) M = fma(a3, c3, M);
        }
      }
      if (type == RX_THREE_BODY) {
        Mout = M;
      } else if (type == RX_LINDEMANN) {
        // k_f = k_inf Pr/(1+Pr), Pr = k0 [M]/k_inf
        double ex[3], ey[3];
        const double lnk0 = fma(ax->c0[1], lnT, fma(ax->c0[2], invT, ax->c0[0]));
        ex[0] = lnk0 - lnkf;
        ex[1] = lnkf;
        ex[2] = lnkr - lnkf;
        exps(ex, ey);
        double Pr = ey[0] * M;
        if constexpr (CLS == kClsLong) Pr *= sPr;
        kf = ey[1] * (Pr / (1.0 + Pr));
        if constexpr (CLS == kClsLong) kf *= sA;
        kr = kf * ey[2];
      } else {
        // Troe.  With ln Pr = ln k0 - ln k_inf + ln[M]:  k_f = k_inf Pr/(1+Pr) F = exp(ln k0 + ln[M] + ln F)/(1+Pr)
        const double lnM = ax->n_eff == 0 ? lds64(cx.lnctot_lane) : log(M);
        const double lnk0 = fma(ax->c0[1], lnT, fma(ax->c0[2], invT, ax->c0[0]));
        const double lnk0M = lnk0 + lnM;
        const double lnPr = lnk0M - lnkf;
        double ex[5], ey[5];
        ex[0] = lnPr;
        ex[1] = T * ax->troe[1];
        ex[2] = T * ax->troe[2];
        ex[3] = ax->troe[3] * invT;
        ex[4] = lnkr - lnkf;        // ln(k_r/k_f) = -ln K_c
        exps(ex, ey);
        const double Pr = ey[0], invKc = ey[4];
        const double al = ax->troe[0];
        const double Fcent = fma(1.0 - al, ey[1], fma(al, ey[2], ey[3]));
        const double lnFc = log(Fcent);
        const double lF = lnFc * kRxLog10e;
        const double cc = fma(-0.67, lF, -0.4);
        const double nn = fma(-1.27, lF, 0.75);
        const double lp = fma(lnPr, kRxLog10e, cc);
        const double den = fma(-0.14, lp, nn);
        // ln F = ln Fcent / (1 + (lp/den)^2) = ln Fcent den^2 / (den^2 + lp^2); both quotients (this one and
        // k_f = .../(1+Pr)) share one reciprocal
        const double den2 = den * den;
        const double bq = fma(lp, lp, den2), dq = 1.0 + Pr;
        const double inv = 1.0 / (bq * dq);
        double e2[1], k2[1];
        e2[0] = fma(lnFc * den2, dq * inv, lnk0M);
        exps(e2, k2);
        kf = k2[0] * (bq * inv);
        // the log form above needs Pr > 0; otherwise log10(Pr) of the definition is not a number
        if constexpr (CLS == kClsLong) kf = sPr > 0.0 ? kf * sA : __longlong_as_double(0x7ff8000000000000LL);
        kr = kf * invKc;
      }
    }
    if constexpr (TM) {
      tm_wait_ld6(tf0, tf1, tf2, tp0, tp1, tp2);
      pf = tf0.get() * tf1.get() * tf2.get();
      pr = tp0.get() * tp1.get() * tp2.get();
    }
    sink(kl, meta, rb_.w, type, kf, kr, pf, pr, Mout);
  }
}

template <int MODE, class Sink>
__device__ __forceinline__ void rx_run_chunk(RxCtx& cx, const unsigned char* blob, int w, Sink&& sink) {
  const ChunkHdr* hdr = reinterpret_cast<const ChunkHdr*>(blob);
  const RxRec* recs = reinterpret_cast<const RxRec*>(blob + sizeof(ChunkHdr));
  // the six class boundaries of this warp are read together, ahead of the loops (read one by one in front of every
  // class loop they cost a shared-memory round trip each: a quarter of a reaction warp's time when a part holds ten
  // records per warp, as at 500 species).  The same in every lane: REDUX says so, which keeps loop counters and record
  // addresses in the uniform datapath.
  int kb[kClsLong + 2];
#pragma unroll
  for (int c = 0; c < kClsLong + 2; ++c) kb[c] = (int)hdr->wb[w][c];
#pragma unroll
  for (int c = 0; c < kClsLong + 2; ++c) kb[c] = __reduce_min_sync(kFullMask, kb[c]);
  rx_run_class<0, MODE>(cx, blob, hdr, recs, kb[0], kb[1], sink);
  rx_run_class<1, MODE>(cx, blob, hdr, recs, kb[1], kb[2], sink);
  rx_run_class<2, MODE>(cx, blob, hdr, recs, kb[2], kb[3], sink);
  rx_run_class<3, MODE>(cx, blob, hdr, recs, kb[3], kb[4], sink);
  rx_run_class<kClsLong, MODE>(cx, blob, hdr, recs, kb[4], kb[5], sink);
}

}  // namespace psr
#endif
