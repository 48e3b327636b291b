// psr_ws.cu -- warp-specialised evaluation kernel for mechanisms whose tables stay resident in shared memory.
//
// The fused kernel of psr_kernels.cu runs its per-tile phases (state preparation, reactions, gather,
// epilogue) one after another behind CTA-wide barriers with ONE CTA per SM: whatever a phase leaves idle
// stays idle (measured on C1: reactions 0.11 ms of a 0.21 ms launch; the loads, the state preparation and
// the barriers 0.05 ms, the gather 0.035 ms, the epilogue 0.01 ms, none of it overlapped).  Here the phases
// are roles of different warps that meet only through mbarriers:
//
//   reaction warps (11)  a3..a7: k_f, K_c, k_r, [M], falloff, q of their share of the reactions, tile after
//                        tile without a CTA barrier; q goes to one of two q buffers (one "part" of the
//                        mechanism each), concentrations and per-reactor state come from one of two C tiles.
//   helper warps (5)     a1: TMA bulk loads of the tile after next, state preparation (Wbar, rho, C_i, ln T,
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
// Same tables (psr_tables.h), same per-reaction arithmetic and the same exp as psr_kernels.cu; the steps are
// SURVEY.md 8(a) a1..a9 (Eq. 2, 4-9).
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "psr_math.cuh"
#include "psr_ptx.cuh"
#include "psr_tables.h"

namespace psr {

namespace {

__device__ constexpr double kRgasW = 8.31446261815324e7;  // erg/mol/K
__device__ constexpr double kLog10eW = 0.43429448190325182765;
constexpr int T_PLAIN = 0, T_THREE_BODY = 1, T_LINDEMANN = 2, T_TROE = 3;  // = PSR_RX_* of psr.h

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

struct RxCtx {
  double T, lnT, invT;
  uint32_t c_lane;    // this lane's column of row 0 of the C tile (shared-memory address)
  uint32_t q_lane;    // this lane's column of row 0 of the q buffer
  uint32_t st_lane;   // this lane's column of row 0 of the tile's state rows
  ExpTab etab;
  float amax;         // NaN-propagating running max of |high word| of the exp arguments of this lane
};

// One record class of one warp's share of a part (a3..a7).  CLS: 0..3 = reaction type in the 3+3 slot form,
// kClsLong = long factor lists.  FAST: table exp, range noted in cx.amax; else the library exp.  OUTK: k_f, k_r,
// q also go to global memory (psr_eval_kf_kr, q of psr_eval_wdot).
template <int CLS, bool FAST, bool OUTK>
__device__ __forceinline__ void ws_run_class(RxCtx& cx, const unsigned char* blob, const ChunkHdr* hdr, const RxRec* recs,
                                             int w, const EvalArgs& a, int64_t r, bool valid) {
  const int kl_begin = __reduce_min_sync(kFullMask, (int)hdr->wb[w][CLS]);
  const int kl_end = __reduce_min_sync(kFullMask, (int)hdr->wb[w][CLS + 1]);
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
    double pf, pr, kf = 0.0, kr = 0.0;

    // concentration products (Eq. 5): integer powers by repetition, unused slots read the unit row
    if constexpr (CLS < kClsLong) {
      const double f0 = lds64(cx.c_lane + ra_.y), f1 = lds64(cx.c_lane + ra_.z), f2 = lds64(cx.c_lane + ra_.w);
      const double p0 = lds64(cx.c_lane + rb_.x), p1 = lds64(cx.c_lane + rb_.y), p2 = lds64(cx.c_lane + rb_.z);
      pf = f0 * f1 * f2;
      pr = p0 * p1 * p2;
    } else {
      const uint16_t* fsp = reinterpret_cast<const uint16_t*>(blob + hdr->off_pool) + ra_.y;
      const int nr = (int)((meta >> kMetaNrShift) & 0xF);
      const int np = (int)((meta >> kMetaNpShift) & 0xF);
      pf = 1.0;
      pr = 1.0;
#pragma unroll 1
      for (int j = 0; j < nr + np; ++j) {
        const double cv = lds64(cx.c_lane + (uint32_t)fsp[j] * (uint32_t)kRowBytes);
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
    if (type <= T_THREE_BODY) {
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
    if (type != T_PLAIN) {
      const AuxRec* ax = reinterpret_cast<const AuxRec*>(blob + hdr->off_aux) + (meta >> kMetaAuxShift);
      const EffEnt* effs = reinterpret_cast<const EffEnt*>(blob + hdr->off_eff);
      double M = lds64(cx.st_lane + ST_CTOT * kRowBytes);
      const uint32_t e1 = ax->eff_off + ax->n_eff;
#pragma unroll 1
      for (uint32_t e = ax->eff_off; e < e1; ++e) M = fma(effs[e].am1, lds64(cx.c_lane + effs[e].off), M);
      if (type == T_THREE_BODY) {
        pf *= M;
        pr *= M;
      } else if (type == T_LINDEMANN) {
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
        const double lnM = ax->n_eff == 0 ? lds64(cx.st_lane + ST_LNCTOT * kRowBytes) : log(M);
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
        const double lF = lnFc * kLog10eW;
        const double cc = fma(-0.67, lF, -0.4);
        const double nn = fma(-1.27, lF, 0.75);
        const double lp = fma(lnPr, kLog10eW, cc);
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
    // an irreversible reaction has its product side on the zero row (pr = 0), a three-body reaction carries
    // [M] in both products: no per-lane selects here
    const double q = fma(kf, pf, -(kr * pr));
    sts64(cx.q_lane + (uint32_t)kl * (uint32_t)kRowBytes, q);
    if constexpr (OUTK) {
      if (valid) {
        const int64_t o = (int64_t)rb_.w * a.ldk + r;
        if (a.flags & kOutKf) a.kf[o] = kf;
        if (a.flags & kOutKr) a.kr[o] = (meta & kMetaRev) ? kr : 0.0;
        if (a.flags & kOutQ) a.q[o] = q;
      }
    }
  }
}

template <bool FAST, bool OUTK>
__device__ __forceinline__ void ws_run_part(RxCtx& cx, const unsigned char* blob, int w, const EvalArgs& a, int64_t r, bool valid) {
  const ChunkHdr* hdr = reinterpret_cast<const ChunkHdr*>(blob);
  const RxRec* recs = reinterpret_cast<const RxRec*>(blob + sizeof(ChunkHdr));
  ws_run_class<0, FAST, OUTK>(cx, blob, hdr, recs, w, a, r, valid);
  ws_run_class<1, FAST, OUTK>(cx, blob, hdr, recs, w, a, r, valid);
  ws_run_class<2, FAST, OUTK>(cx, blob, hdr, recs, w, a, r, valid);
  ws_run_class<3, FAST, OUTK>(cx, blob, hdr, recs, w, a, r, valid);
  ws_run_class<kClsLong, FAST, OUTK>(cx, blob, hdr, recs, w, a, r, valid);
}

}  // namespace

template <bool OUTK>
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
  __syncthreads();

  if (w < kWsRxWarps) {
    // ================================================================== reaction warps
    RxCtx cx;
    cx.etab = exp_tab_load(mv.exp_tab);
    mbar_wait(&bars[B_BLOB], 0);
    int64_t tile = blockIdx.x;
    for (uint32_t lt = 0; tile < a.n_tiles; ++lt, tile += gridDim.x) {
      const int b = lt & 1;
      mbar_wait(&bars[B_FULLC + b], (lt >> 1) & 1);
      cx.st_lane = smem_u32(St0 + b * kWsStRows * kTile) + lane * 8;
      cx.c_lane = smem_u32(Cs0 + b * cs_elems) + lane * 8;
      cx.T = lds64(cx.st_lane + ST_T * kRowBytes);
      cx.lnT = lds64(cx.st_lane + ST_LNT * kRowBytes);
      cx.invT = lds64(cx.st_lane + ST_INVT * kRowBytes);
      const int64_t r = tile * kTile + lane;
      const bool valid = r < a.N;
      for (int p = 0; p < mv.n_parts; ++p) {
        const uint32_t g = lt * (uint32_t)mv.n_parts + (uint32_t)p, qb = g & 1, u = g >> 1;
        if (u > 0) mbar_wait(&bars[B_EMPTYQ + qb], (u - 1) & 1);   // the part that used this buffer before has been gathered
        cx.q_lane = smem_u32(qh0 + qb * q_elems) + lane * 8;
        const unsigned char* blob = mech + (size_t)p * mv.chunk_stride;
        cx.amax = 0.0f;
        ws_run_part<true, OUTK>(cx, blob, w, a, r, valid);
        // an exp argument out of the table form's range (NaN, Inf, overflow, underflow: never for physical
        // states): this warp repeats its records with the library exp, which keeps IEEE results
        if (__any_sync(kFullMask, !exp_max_in_range(cx.amax))) ws_run_part<false, OUTK>(cx, blob, w, a, r, valid);
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars[B_FULLQ + qb]);
      }
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
        asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(row_off), "=r"(pad) : "r"(te));
        if (LAST) {
          asm volatile("ld.shared.v2.b64 {%0, %1}, [%2+16];" : "=l"(goff), "=d"(W) : "r"(te));
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
    mbar_wait(&bars[B_BLOB], 0);
    if (tile < a.n_tiles) prologue(0);
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
}

// once per process: the kernels' dynamic shared-memory limit raised to the device's (mechanisms of different sizes
// share the kernel instances)
cudaError_t ws_set_smem(size_t smem) {
  cudaError_t e = cudaFuncSetAttribute(psr_ws_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(psr_ws_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  return e;
}

cudaError_t launch_ws(const WsView& mv, const EvalArgs& a, int grid, int bulk_ok, cudaStream_t st) {
  if (a.flags & (kOutKf | kOutKr | kOutQ)) psr_ws_kernel<true><<<grid, kWsWarps * 32, mv.smem_total, st>>>(mv, a, bulk_ok);
  else psr_ws_kernel<false><<<grid, kWsWarps * 32, mv.smem_total, st>>>(mv, a, bulk_ok);
  return cudaGetLastError();
}

}  // namespace psr
