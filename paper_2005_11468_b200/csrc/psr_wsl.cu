// psr_wsl.cu -- warp-specialised evaluation kernel for LARGE mechanisms (BASELINE configs 2 and 3: 200 / 1500 and
// 500 / 2500; "hundreds of species and thousands of reactions").
//
// psr_ws.cu keeps two C tiles, two Y - Y_in tiles and every part's tables resident in shared memory; none of that
// fits beyond ~160 species.  The round-1 kernel (psr_kernels.cu) that served the large mechanisms alternates a
// reaction phase and a gather phase per chunk behind CTA barriers, and its gather visits every (chunk, species)
// pair -- 13 x 500 visits of ~1.5 reactions each at C3, the running sums bouncing through L2 in between: 55 % of
// its instructions (profiles/r1d_psr_eval_kernel_C3.md).  Here the roles are those of psr_ws.cu:
//
//   reaction warps (12)  a3..a7 of their share of a part's records, part after part, tile after tile; q goes to
//                        one of two q buffers; the part's tables come from a two-stage ring (bulk copies).
//   helper warps (8)     a8: gather of the q buffer just filled.  Where the running sums of nu^T q live decides its form
//                        (WslView::acc_global): 0 -- a shared-memory tile, when that still leaves room for at most four
//                        parts (P5): flat streams of 4-entry groups that SKIP the species without a term in the part,
//                        each flush taking its target row from a list in the blob; 2 -- tensor memory, the warp's own
//                        species in its own lane quadrant (K <= 200: C2): a flat stream of (q row, target | flags)
//                        tuples, a species' tuples summed in a register and added to its running sum at its last tuple;
//                        1 -- an L2-resident scratch (C3): the same tuples, each added with red.global (one thread owns
//                        an element: deterministic order);
//                        a1: loads and state preparation of the NEXT tile;
//                        a9: per-tile epilogue (wdot, F) streaming Y, Y_in and the sums, eight rows in flight.
//
// Tensor memory (TMODE 1; K <= 250): a copy of the finished C tile in all four lane quadrants, from which the reaction
// warps read every concentration (psr_rx.cuh, kRxTm) -- the shared-memory tile is then only a staging area, the next tile
// is loaded and converted there while the current one is evaluated, and between two tiles only the copy into tensor
// memory remains.  Without it the next tile is prepared ahead of the last part's gather, once the reaction warps have
// left the single tile.
//
//   ring[st]     a part's tables landed (tx bytes)                  helper 0   -> everyone
//   full_C       C tile + state rows of a tile ready                helpers    -> reaction warps
//   empty_C      reaction warps are done with the C tile            reaction   -> helpers
//   full_q[qb]   every reaction warp has written its q rows         reaction   -> helpers
//   empty_q[qb]  the part has been gathered (its ring stage is free) helpers    -> reaction warps
//
// Same tables, per-reaction code (psr_rx.cuh) and exp as the other kernels; SURVEY.md 8(a) a1..a9 (Eq. 2, 4-9).
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "psr_math.cuh"
#include "psr_ptx.cuh"
#include "psr_rx.cuh"
#include "psr_tables.h"

namespace psr {

namespace {
__device__ constexpr double kRgasL = 8.31446261815324e7;  // erg/mol/K
constexpr int L_RING = 0, L_FULLC = 2, L_EMPTYC = 3, L_FULLQ = 4, L_EMPTYQ = 6, L_IN = 8, L_COUNT = 10;
constexpr int L_SLOTS = L_COUNT + 2;   // + the tensor-memory base address (8 bytes used of 16)
constexpr int LS_T = 0, LS_LNT = 1, LS_INVT = 2, LS_CTOT = 3, LS_LNCTOT = 4, LS_INVTAU = 5, LS_INVRHO = 6, LS_ROWS = 8;
}  // namespace

// The helper warps' side of psr_wsl_kernel (every thread of warps kWslRxWarps.. calls it).  TM: a finished C tile is
// also copied to tensor memory, once per lane quadrant (tm_quad: this warp's quadrant of the allocation), as in psr_ws.cu.
template <int TMODE>
__device__ __forceinline__ void psr_wsl_helpers(const WslView& mv, const EvalArgs& a, double* Cs, double* acc_s, double* qh0,
                                                unsigned char* ring, const double* invW_s, const double* W_s, double* St0,
                                                double* tp0, uint64_t* bars, const int32_t* sp_s, uint32_t total_parts, const int bulk_ok,
                                                const uint32_t tm_quad) {
  constexpr bool TM = TMODE != 0;   // tensor memory allocated: the copy of the C tile is kept there
  // The reaction warps read only that copy (TMODE 1): the shared-memory tile is then a staging area, and the NEXT tile
  // is loaded and converted there (stage_tile) while they work on the current one; what is left between two tiles is
  // the copy into tensor memory (publish_tile).  Otherwise the two run back to back at the tile boundary.
  constexpr bool EARLY = TMODE == 1;
  const int lane = threadIdx.x & 31, hw = (threadIdx.x >> 5) - kWslRxWarps;
  const int K = mv.K, q_elems = (mv.rc + 1) * kTile;
  const bool wantF = (a.flags & kOutF) != 0, out_w = (a.flags & kOutWdot) != 0;
  const int32_t* my_sp = sp_s + hw * mv.spw;
  int n_my = 0;
  while (n_my < mv.spw && my_sp[n_my] >= 0) ++n_my;   // owned species come first, -1 pads the list
  const bool accg = mv.acc_global == 1;
  const bool acct = TM && mv.acc_global == 2;   // the running sums of this warp's species in tensor memory, its own quadrant
  const uint32_t tm_acc = tm_quad + (uint32_t)mv.tm_acc_col + 2u * (uint32_t)((hw >> 2) * mv.spw);
  char* accg_lane = reinterpret_cast<char*>(mv.acc_g + (size_t)blockIdx.x * (K + 1) * kTile + lane);   // row s at + s * kRowBytes; row K: spare
  const uint32_t acc_lane = smem_u32(acc_s) + lane * 8;

  // a1: a tile's Y rows (into the C tile), T, P, tau; then W_bar = 1/sum Y_i/W_i, rho = P W_bar/(R T), C_i = rho Y_i/W_i,
  // C_tot = rho sum Y_i/W_i and the state rows of the tile.  Every helper warp forms the sum over all species itself.
  auto stage_tile = [&](int64_t t, uint32_t lt) {
    if constexpr (EARLY) named_bar_sync(3, kWslHelpWarps * 32);   // the copy of the previous tile out of Cs is complete
    int64_t r = t * kTile + lane;
    if (r >= a.N) r = a.N - 1;   // lanes past N repeat the last reactor (a valid state, nothing stored)
    double* tb = tp0 + (lt & 1) * 3 * kTile;
    double* St = St0 + (lt & 1) * LS_ROWS * kTile;
    if (bulk_ok && (t + 1) * kTile <= a.N) {
      // whole tiles of 16-byte aligned arrays: one bulk copy per species row (256 contiguous bytes), lanes over rows
      fence_proxy_async();
      if (lane == 0) mbar_expect_tx(&bars[L_IN], (uint32_t)n_my * kRowBytes + (hw == 0 ? (wantF ? 3u : 2u) * kRowBytes : 0u));
      __syncwarp();
      const int64_t r0 = t * kTile;
      for (int jj = lane; jj < n_my; jj += 32) {
        const int s = my_sp[jj];
        bulk_g2s(Cs + s * kTile, a.Y + (int64_t)s * a.ld + r0, kRowBytes, &bars[L_IN]);
      }
      if (hw == 0 && lane == 31) {
        bulk_g2s(tb, a.T + r0, kRowBytes, &bars[L_IN]);
        bulk_g2s(tb + kTile, a.P + r0, kRowBytes, &bars[L_IN]);
        if (wantF) bulk_g2s(tb + 2 * kTile, a.tau + r0, kRowBytes, &bars[L_IN]);
      }
    } else {
#pragma unroll 8
      for (int jj = 0; jj < n_my; ++jj) {
        const int s = my_sp[jj];
        Cs[s * kTile + lane] = ldg_nc(a.Y + (int64_t)s * a.ld + r);
      }
      if (hw == 0) {
        tb[lane] = ldg_nc(a.T + r);
        tb[kTile + lane] = ldg_nc(a.P + r);
        if (wantF) tb[2 * kTile + lane] = ldg_nc(a.tau + r);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars[L_IN]);
    }
    mbar_wait(&bars[L_IN], lt & 1);   // every row of the tile is in (one phase per tile)
    const double T = tb[lane], P = tb[kTile + lane];
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    int s = 0;
    for (; s + 4 <= K; s += 4) {
      s0 = fma(Cs[s * kTile + lane], invW_s[s], s0);
      s1 = fma(Cs[(s + 1) * kTile + lane], invW_s[s + 1], s1);
      s2 = fma(Cs[(s + 2) * kTile + lane], invW_s[s + 2], s2);
      s3 = fma(Cs[(s + 3) * kTile + lane], invW_s[s + 3], s3);
    }
    for (; s < K; ++s) s0 = fma(Cs[s * kTile + lane], invW_s[s], s0);
    const double sY = (s0 + s1) + (s2 + s3);
    const double Wbar = 1.0 / sY;
    const double rho = P * Wbar / (kRgasL * T);
    if (hw == 0) {
      St[LS_T * kTile + lane] = T;
      St[LS_LNT * kTile + lane] = log(T);
      St[LS_INVT * kTile + lane] = 1.0 / T;
    } else if (hw == 1) {
      const double ct = rho * sY;   // C_tot = sum_i C_i = rho sum_i Y_i/W_i
      St[LS_CTOT * kTile + lane] = ct;
      if (mv.need_lnctot) St[LS_LNCTOT * kTile + lane] = log(ct);
    } else if (hw == 2 && wantF) {
      St[LS_INVTAU * kTile + lane] = 1.0 / tb[2 * kTile + lane];
      St[LS_INVRHO * kTile + lane] = 1.0 / rho;
    }
    named_bar_sync(1, kWslHelpWarps * 32);   // every helper warp has read the Y rows; the state rows are visible
    for (int jj = 0; jj < n_my; ++jj) {
      const int sp = my_sp[jj];
      Cs[sp * kTile + lane] = rho * (Cs[sp * kTile + lane] * invW_s[sp]);
    }
  };
  // (the reaction warps have released the previous tile through empty_C, which this warp has waited for)
  auto publish_tile = [&]() {
    if constexpr (TM) {
      static_assert(kWslHelpWarps >= 4, "four helper warps copy the C tile to the four TMEM quadrants");
      named_bar_sync(2, kWslHelpWarps * 32);   // every row of the staged tile is final
      if (hw < 4) {
        tm_fence_after_sync();
        const int last = K + 1;
        for (int s4 = 0; s4 <= last; s4 += 4)
          tm_st64x4(tm_quad + 2u * (uint32_t)s4, Cs[s4 * kTile + lane], Cs[min(s4 + 1, last) * kTile + lane],
                    Cs[min(s4 + 2, last) * kTile + lane], Cs[min(s4 + 3, last) * kTile + lane]);
        tm_wait_st();
        tm_fence_before_sync();
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&bars[L_FULLC]);
  };

  // a8 (Eq. 4): this warp's stream of 4-entry groups of one part, two groups per trip, software-pipelined as in
  // psr_ws.cu.  The group that ends a species adds the species' sum for this part to its running sum (part 0 stores).
  auto gather = [&](auto first_tag, const unsigned char* blob, const uint32_t q_lane) {
    constexpr bool FIRST = decltype(first_tag)::value;
    const ChunkHdr* hdr = reinterpret_cast<const ChunkHdr*>(blob);
    const uint32_t gs = smem_u32(blob + hdr->off_gent) + (uint32_t)hdr->wb[kWslRxWarps + hw][0] * 16u;
    const int n_groups = (int)hdr->wb[kWslRxWarps + hw][1] - (int)hdr->wb[kWslRxWarps + hw][0];   // even
    uint32_t dst = smem_u32(blob + hdr->off_gptr) + (uint32_t)hdr->wb[kWslRxWarps + hw][2] * 4u;
    auto ld_group = [&](uint32_t addr, uint4& o) {
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(o.x), "=r"(o.y), "=r"(o.z), "=r"(o.w) : "r"(addr));
    };
    auto sgn = [](uint32_t ctl) { return __hiloint2double((int)(0x3ff00000u ^ (ctl << 31)), 0); };
    auto flush = [&](double& acc) {
      uint32_t off;
      asm volatile("ld.shared.u32 %0, [%1];" : "=r"(off) : "r"(dst));
      dst += 4;
      PSR_CHK(off < (uint32_t)K * kRowBytes && off % kRowBytes == 0, 503);   // a row of the [K][32] running sums
      const uint32_t addr = acc_lane + off;   // (sums in shared memory; in global memory: gather_tuples)
      sts64(addr, FIRST ? acc : lds64(addr) + acc);
      acc = 0.0;
    };
    const uint32_t qmax = (uint32_t)q_elems * 8u;
    (void)qmax;
    uint4 oa, ob;
    ld_group(gs, oa);
    ld_group(gs + 16, ob);
    double a0 = lds64(q_lane + (oa.x & ~3u)), a1 = lds64(q_lane + oa.y), a2 = lds64(q_lane + oa.z), a3 = lds64(q_lane + oa.w);
    double b0 = lds64(q_lane + (ob.x & ~3u)), b1 = lds64(q_lane + ob.y), b2 = lds64(q_lane + ob.z), b3 = lds64(q_lane + ob.w);
    uint32_t ca = oa.x, cb = ob.x;
    ld_group(gs + 32, oa);
    ld_group(gs + 48, ob);
    double acc = 0.0;
#pragma unroll 1
    for (int i = 0; i < n_groups; i += 2) {
      const double ta = (a0 + a2) + (a1 + a3), tb = (b0 + b2) + (b1 + b3);
      const uint32_t c0 = ca, c1 = cb;
      ca = oa.x;
      cb = ob.x;
      PSR_CHK((oa.x & ~3u) < qmax && oa.y < qmax && oa.z < qmax && oa.w < qmax && (ob.x & ~3u) < qmax && ob.y < qmax &&
                  ob.z < qmax && ob.w < qmax, 504);
      a0 = lds64(q_lane + (oa.x & ~3u)), a1 = lds64(q_lane + oa.y), a2 = lds64(q_lane + oa.z), a3 = lds64(q_lane + oa.w);
      b0 = lds64(q_lane + (ob.x & ~3u)), b1 = lds64(q_lane + ob.y), b2 = lds64(q_lane + ob.z), b3 = lds64(q_lane + ob.w);
      ld_group(gs + (uint32_t)(i + 4) * 16u, oa);
      ld_group(gs + (uint32_t)(i + 5) * 16u, ob);
      acc = fma(ta, sgn(c0), acc);
      if (c0 & kGatherLast) flush(acc);
      acc = fma(tb, sgn(c1), acc);
      if (c1 & kGatherLast) flush(acc);
    }
  };

  // a8 with the sums in global memory: the tuple stream of this warp for one part (psr_api.cu build_blobs) -- per entry of
  // nu^T one q value read from the buffer and one red.global.add to the species' sum, its sign applied on the way; four
  // tuples per trip, read one trip ahead.  One thread owns an element of the sums and issues its adds in program order,
  // so the order of the summation is fixed.
  auto gather_tuples = [&](const unsigned char* blob, const uint32_t q_lane) {
    const ChunkHdr* hdr = reinterpret_cast<const ChunkHdr*>(blob);
    const uint32_t ts = smem_u32(blob + hdr->off_gent) + (uint32_t)hdr->wb[kWslRxWarps + hw][0] * 16u;
    const int n_pairs = (int)hdr->wb[kWslRxWarps + hw][1] - (int)hdr->wb[kWslRxWarps + hw][0];   // 16-byte units, even
    auto ld4 = [&](uint32_t addr, uint4& o) {
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(o.x), "=r"(o.y), "=r"(o.z), "=r"(o.w) : "r"(addr));
    };
    auto add = [&](uint32_t qo, uint32_t to) {
      PSR_CHK(qo < (uint32_t)q_elems * 8u && (to & 0x7fffffffu) <= (uint32_t)K * kRowBytes && to % kRowBytes == 0, 506);
      const double v = lds64(q_lane + qo);
      const double sv = __hiloint2double(__double2hiint(v) ^ (int)(to & 0x80000000u), __double2loint(v));   // -v if bit 31 is set
      asm volatile("red.global.add.f64 [%0], %1;" ::"l"(accg_lane + (to & 0x7fffffffu)), "d"(sv) : "memory");
    };
    uint4 ta, tb;
    ld4(ts, ta);
    ld4(ts + 16, tb);
#pragma unroll 1
    for (int i = 0; i < n_pairs; i += 2) {
      const uint4 ca = ta, cb = tb;
      ld4(ts + (uint32_t)(i + 2) * 16u, ta);
      ld4(ts + (uint32_t)(i + 3) * 16u, tb);
      add(ca.x, ca.y);
      add(ca.z, ca.w);
      add(cb.x, cb.y);
      add(cb.z, cb.w);
    }
  };

  // a8 with the sums in tensor memory (this warp's species at columns tm_acc + 2 jj of its own lane quadrant): the tuple
  // stream again -- no padding to groups, which at 4.3 entries per species and part would double the stream -- but a
  // species' tuples are summed in a register, in stream order, and the tuple marked last adds the sum to the species'
  // running sum (part 0 stores it).  Tuples are read two trips ahead, q values one trip ahead.
  auto gather_tuples_tm = [&](auto first_tag, const unsigned char* blob, const uint32_t q_lane) {
    constexpr bool FIRST = decltype(first_tag)::value;
    const ChunkHdr* hdr = reinterpret_cast<const ChunkHdr*>(blob);
    const uint32_t ts = smem_u32(blob + hdr->off_gent) + (uint32_t)hdr->wb[kWslRxWarps + hw][0] * 16u;
    const int n_pairs = (int)hdr->wb[kWslRxWarps + hw][1] - (int)hdr->wb[kWslRxWarps + hw][0];   // 16-byte units, even
    auto ld4 = [&](uint32_t addr, uint4& o) {
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(o.x), "=r"(o.y), "=r"(o.z), "=r"(o.w) : "r"(addr));
    };
    if (!FIRST) tm_wait_st();   // the sums the previous part stored have landed
    double acc = 0.0;
    auto step = [&](uint32_t qo, uint32_t to, double v) {
      PSR_CHK(qo < (uint32_t)q_elems * 8u && (to & 0xffffu) < 2u * (uint32_t)mv.spw, 507);
      acc += __hiloint2double(__double2hiint(v) ^ (int)(to & 0x80000000u), __double2loint(v));   // -v if bit 31 is set
      if (to & 0x40000000u) {   // the species' last tuple of this part (the same in every lane)
        const uint32_t col = tm_acc + (to & 0xffffu);
        if (FIRST) {
          tm_st64(col, acc);
        } else {
          TmF64 t;
          tm_ld64(col, t);
          tm_wait_ld1(t);
          tm_st64(col, t.get() + acc);
        }
        acc = 0.0;
      }
    };
    uint4 ca, cb, na, nb;
    ld4(ts, ca);
    ld4(ts + 16, cb);
    double v0 = lds64(q_lane + ca.x), v1 = lds64(q_lane + ca.z), v2 = lds64(q_lane + cb.x), v3 = lds64(q_lane + cb.z);
    ld4(ts + 32, na);
    ld4(ts + 48, nb);
#pragma unroll 1
    for (int i = 0; i < n_pairs; i += 2) {
      const uint4 a_ = ca, b_ = cb;
      const double w0 = v0, w1 = v1, w2 = v2, w3 = v3;
      ca = na;
      cb = nb;
      v0 = lds64(q_lane + ca.x), v1 = lds64(q_lane + ca.z), v2 = lds64(q_lane + cb.x), v3 = lds64(q_lane + cb.z);
      ld4(ts + (uint32_t)(i + 4) * 16u, na);
      ld4(ts + (uint32_t)(i + 5) * 16u, nb);
      step(a_.x, a_.y, w0);
      step(a_.z, a_.w, w1);
      step(b_.x, b_.y, w2);
      step(b_.z, b_.w, w3);
    }
  };

  // a9 (Eq. 2 at steady state) and the wdot store of a tile: F_i = (Y_i - Y_in,i)/tau - wdot_i W_i/rho, eight rows in flight.
  // (A running sum kept in global memory is read past L1: the adds of the later parts were done at L2.)
  auto epilogue = [&](int64_t t, uint32_t lt) {
    const int64_t r = t * kTile + lane;
    const bool valid = r < a.N;
    const int64_t rcl = valid ? r : a.N - 1;
    const double* St = St0 + (lt & 1) * LS_ROWS * kTile;
    const double invtau = wantF ? St[LS_INVTAU * kTile + lane] : 0.0, invrho = wantF ? St[LS_INVRHO * kTile + lane] : 0.0;
    constexpr int EU = 8;   // rows in flight
    if constexpr (TM) {
      if (acct) tm_wait_st();
    }
    for (int jj = 0; jj < n_my; jj += EU) {
      double tot[EU], y[EU], yin[EU];
      int sp[EU];
#pragma unroll
      for (int u = 0; u < EU; ++u) {
        sp[u] = my_sp[min(jj + u, n_my - 1)];
        if (TM && acct) {
          TmF64 t;
          tm_ld64(tm_acc + 2u * (uint32_t)min(jj + u, n_my - 1), t);
          tm_wait_ld1(t);
          tot[u] = t.get();
        } else {
          tot[u] = accg ? __ldcg(reinterpret_cast<const double*>(accg_lane + (size_t)sp[u] * kRowBytes)) : acc_s[sp[u] * kTile + lane];
        }
        y[u] = wantF ? ldg_nc(a.Y + (int64_t)sp[u] * a.ld + rcl) : 0.0;
        yin[u] = wantF ? ldg_nc(a.Yin + (int64_t)sp[u] * a.ld + rcl) : 0.0;
      }
#pragma unroll
      for (int u = 0; u < EU; ++u) {
        if (valid && jj + u < n_my) {
          PSR_CHK(sp[u] >= 0 && sp[u] < K, 505);
          const int64_t o = (int64_t)sp[u] * a.ld + r;
          if (out_w) a.wdot[o] = tot[u];
          if (wantF) a.F[o] = fma(y[u] - yin[u], invtau, -(tot[u] * (W_s[sp[u]] * invrho)));
        }
        // sums kept in global memory start the next tile at zero (this thread's own later adds come after this store)
        if (accg && jj + u < n_my) __stcg(reinterpret_cast<double*>(accg_lane + (size_t)sp[u] * kRowBytes), 0.0);
      }
    }
  };

  if (accg) {   // this warp's rows of the sums (and the spare row) start at zero
    for (int jj = 0; jj < n_my; ++jj) __stcg(reinterpret_cast<double*>(accg_lane + (size_t)my_sp[jj] * kRowBytes), 0.0);
    if (hw == 0) __stcg(reinterpret_cast<double*>(accg_lane + (size_t)K * kRowBytes), 0.0);
  }
  const int64_t stride = gridDim.x;
  int64_t tile = blockIdx.x;
  if (tile < a.n_tiles) {
    stage_tile(tile, 0);
    publish_tile();
  }
  for (uint32_t lt = 0; tile < a.n_tiles; ++lt, tile += stride) {
    for (int p = 0; p < mv.n_parts; ++p) {
      const uint32_t g = lt * (uint32_t)mv.n_parts + (uint32_t)p, qb = g & 1, u = g >> 1;
      mbar_wait(&bars[L_FULLQ + qb], u & 1);
      mbar_wait(&bars[L_RING + qb], u & 1);   // (complete long ago: makes the bulk copy's bytes visible to this warp)
      if (p == mv.n_parts - 1 && tile + stride < a.n_tiles) {
        // the reaction warps leave the tile now: the next tile's C first, the last part's gather after it
        mbar_wait(&bars[L_EMPTYC], lt & 1);
        if constexpr (!EARLY) stage_tile(tile + stride, lt + 1);
        publish_tile();
      }
      const unsigned char* blob = ring + (size_t)qb * mv.chunk_stride;
      const uint32_t q_lane = smem_u32(qh0 + qb * q_elems) + lane * 8;
      if (accg) gather_tuples(blob, q_lane);
      else if (TM && acct) {
        if (p == 0) gather_tuples_tm(std::true_type{}, blob, q_lane);
        else gather_tuples_tm(std::false_type{}, blob, q_lane);
      } else if (p == 0) gather(std::true_type{}, blob, q_lane);
      else gather(std::false_type{}, blob, q_lane);
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars[L_EMPTYQ + qb]);
      if (hw == 0 && g + 2 < total_parts) {
        // once every helper warp is done with the part its ring stage is free: the part after next goes there
        // (only this warp waits for the others; the reaction warps wait for the same phase, then for the ring)
        mbar_wait(&bars[L_EMPTYQ + qb], u & 1);
        if (lane == 0) {
          fence_proxy_async();
          mbar_expect_tx(&bars[L_RING + qb], mv.chunk_stride);
          bulk_g2s(ring + (size_t)qb * mv.chunk_stride, mv.chunks + (size_t)((g + 2) % (uint32_t)mv.n_parts) * mv.chunk_stride,
                   mv.chunk_stride, &bars[L_RING + qb]);
        }
        __syncwarp();
      }
      if constexpr (EARLY) {
        if (p == 0 && tile + stride < a.n_tiles) stage_tile(tile + stride, lt + 1);
      }
    }
    epilogue(tile, lt);
  }
}

// TMODE: 0 no tensor memory; 1 the copy of the C tile there, read by the reaction warps (and the running sums, if
// mv.acc_global == 2); 2 the same allocation but the reaction warps read shared memory (PSR_OPT_NO_TMEM on a
// mechanism whose sums live in tensor memory).
template <bool OUTK, int TMODE>
__global__ void __launch_bounds__(kWslWarps * 32, 1) psr_wsl_kernel(const WslView mv, const EvalArgs a, const int bulk_ok) {
  extern __shared__ __align__(128) unsigned char smem[];
  constexpr bool TM = TMODE != 0, RXTM = TMODE == 1;
  const int K = mv.K;
  const int q_elems = (mv.rc + 1) * kTile;
  double* Cs = reinterpret_cast<double*>(smem + mv.smem_cs);        // [K+2][32]; rows K, K+1: ones, zeros
  double* acc_s = reinterpret_cast<double*>(smem + mv.smem_acc);    // [K][32] running sums (unless acc_global)
  double* qh0 = reinterpret_cast<double*>(smem + mv.smem_q);        // [2][rc+1][32]; row rc stays zero
  unsigned char* ring = smem + mv.smem_mech;                        // [2][chunk_stride]
  double* invW_s = reinterpret_cast<double*>(smem + mv.smem_misc);  // [Kp]
  const int Kp = (K + 1) & ~1;
  double* W_s = invW_s + Kp;                                        // [Kp]
  double* St0 = W_s + Kp;                                           // [2][LS_ROWS][32]: state rows, by tile parity
  double* tp0 = St0 + 2 * LS_ROWS * kTile;                          // [2][3][32]: T, P, tau as loaded
  uint64_t* bars = reinterpret_cast<uint64_t*>(tp0 + 2 * 3 * kTile);
  uint32_t* tm_slot = reinterpret_cast<uint32_t*>(bars + L_COUNT);  // tensor-memory base address (TM)
  int32_t* sp_s = reinterpret_cast<int32_t*>(bars + L_SLOTS);       // [helper warps][spw]

  const int lane = threadIdx.x & 31;
  const int w = threadIdx.x >> 5;
  const bool wantF = (a.flags & kOutF) != 0;
  const int64_t my_tiles = (a.n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x;
  const uint32_t total_parts = (uint32_t)my_tiles * (uint32_t)mv.n_parts;   // parts this CTA evaluates, in order

  if (threadIdx.x == 0) {
    mbar_init(&bars[L_RING], 1);
    mbar_init(&bars[L_RING + 1], 1);
    mbar_init(&bars[L_FULLC], kWslHelpWarps);
    mbar_init(&bars[L_EMPTYC], kWslRxWarps);
    mbar_init(&bars[L_IN], kWslHelpWarps);
    for (int b = 0; b < 2; ++b) {
      mbar_init(&bars[L_FULLQ + b], kWslRxWarps);
      mbar_init(&bars[L_EMPTYQ + b], kWslHelpWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
    for (uint32_t g = 0; g < 2 && g < total_parts; ++g) {
      mbar_expect_tx(&bars[L_RING + g], mv.chunk_stride);
      bulk_g2s(ring + (size_t)g * mv.chunk_stride, mv.chunks + (size_t)(g % mv.n_parts) * mv.chunk_stride, mv.chunk_stride,
               &bars[L_RING + g]);
    }
  }
  if (w == 0) {
    if constexpr (TM) tm_alloc(tm_slot, (uint32_t)mv.tm_cols);
    Cs[K * kTile + lane] = 1.0;         // unit row: unused factor slots
    Cs[(K + 1) * kTile + lane] = 0.0;   // zero row: product side of an irreversible reaction
    for (int b = 0; b < 2; ++b) qh0[b * q_elems + mv.rc * kTile + lane] = 0.0;   // zero row: padding of the gather streams
  }
  for (int i = threadIdx.x; i < K; i += kWslWarps * 32) {
    invW_s[i] = mv.invW[i];
    W_s[i] = mv.Wm[i];
  }
  for (int i = threadIdx.x; i < kWslHelpWarps * mv.spw; i += kWslWarps * 32) sp_s[i] = mv.sp_of[i];
  if constexpr (TM) tm_fence_before_sync();
  __syncthreads();
  uint32_t tm_quad = 0;   // this warp's quadrant of the copy of the C tile in tensor memory
  if constexpr (TM) {
    tm_fence_after_sync();
    tm_quad = *tm_slot + ((uint32_t)((w & 3) * 32) << 16);
  }

  if (w < kWslRxWarps) {
    // ================================================================== reaction warps
    RxCtx cx;
    cx.etab = exp_tab_load(mv.exp_tab);
    cx.c_lane = smem_u32(Cs) + lane * 8;
    cx.tm_c = tm_quad;
#ifdef PSR_CHECK
    cx.chk_c_bytes = (uint32_t)(K + 2) * kRowBytes;
#endif
    int64_t tile = blockIdx.x;
    for (uint32_t lt = 0; tile < a.n_tiles; ++lt, tile += gridDim.x) {
      mbar_wait(&bars[L_FULLC], lt & 1);
      if constexpr (TM) tm_fence_after_sync();
      const uint32_t st_lane = smem_u32(St0 + (lt & 1) * LS_ROWS * kTile) + lane * 8;
      cx.ctot_lane = st_lane + LS_CTOT * kRowBytes;
      cx.lnctot_lane = st_lane + LS_LNCTOT * kRowBytes;
      cx.T = lds64(st_lane + LS_T * kRowBytes);
      cx.lnT = lds64(st_lane + LS_LNT * kRowBytes);
      cx.invT = lds64(st_lane + LS_INVT * kRowBytes);
      const int64_t r = tile * kTile + lane;
      const bool valid = r < a.N;
      for (int p = 0; p < mv.n_parts; ++p) {
        const uint32_t g = lt * (uint32_t)mv.n_parts + (uint32_t)p, qb = g & 1, u = g >> 1;
        // the part two before this one used the same q buffer and ring stage: gathered, and its stage refilled
        if (u > 0) mbar_wait(&bars[L_EMPTYQ + qb], (u - 1) & 1);
        mbar_wait(&bars[L_RING + qb], u & 1);
        const uint32_t q_lane = smem_u32(qh0 + qb * q_elems) + lane * 8;
        const unsigned char* blob = ring + (size_t)qb * mv.chunk_stride;
        // Eq. 5: q = k_f prod C^nu' - k_r prod C^nu'' (x [M] for a three-body reaction); an irreversible reaction has
        // its product side on the zero row
        auto sink = [&](int kl, uint32_t meta, uint32_t korig, int type, double kf, double kr, double pf, double pr, double M) {
          if (type == RX_THREE_BODY) {
            pf *= M;
            pr *= M;
          }
          const double q = fma(kf, pf, -(kr * pr));
          PSR_CHK(kl >= 0 && kl < mv.rc, 501);
          PSR_CHK(!OUTK || !valid || (int64_t)korig < (int64_t)mv.I, 502);
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
        rx_run_chunk<kRxFast | (RXTM ? kRxTm : 0)>(cx, blob, w, sink);
        // an exp argument out of the table form's range: this warp repeats its records with the library exp
        if (__any_sync(kFullMask, !exp_max_in_range(cx.amax))) rx_run_chunk<(RXTM ? kRxTm : 0)>(cx, blob, w, sink);
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars[L_FULLQ + qb]);
      }
      if constexpr (TM) tm_fence_before_sync();   // (every tensor-memory read of the tile has been waited for)
      if (lane == 0) mbar_arrive(&bars[L_EMPTYC]);
    }
  } else {
    // ================================================================== helper warps: see above
    psr_wsl_helpers<TMODE>(mv, a, Cs, acc_s, qh0, ring, invW_s, W_s, St0, tp0, bars, sp_s, total_parts, bulk_ok, tm_quad);
  }
  if constexpr (TM) {
    tm_fence_before_sync();
    __syncthreads();   // no warp touches tensor memory any more
    if (w == 0) tm_dealloc(*tm_slot, (uint32_t)mv.tm_cols);
  }
}

PSR_CHK_TU_READER(chk_read_wsl)

cudaError_t wsl_set_smem(size_t smem) {
  const void* fns[] = {(const void*)psr_wsl_kernel<false, 0>, (const void*)psr_wsl_kernel<true, 0>, (const void*)psr_wsl_kernel<false, 1>,
                       (const void*)psr_wsl_kernel<true, 1>,  (const void*)psr_wsl_kernel<false, 2>, (const void*)psr_wsl_kernel<true, 2>};
  for (const void* f : fns) {
    cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

// rx_tmem: the reaction warps read the tensor-memory copy of the C tile (0: PSR_OPT_NO_TMEM)
cudaError_t launch_wsl(const WslView& mv, const EvalArgs& a, int grid, int bulk_ok, int rx_tmem, cudaStream_t st) {
  const bool outk = (a.flags & (kOutKf | kOutKr | kOutQ)) != 0;
  const int tmode = mv.tm_cols <= 0 ? 0 : rx_tmem ? 1 : mv.acc_global == 2 ? 2 : 0;
  const int nt = kWslWarps * 32;
  if (tmode == 1) {
    if (outk) psr_wsl_kernel<true, 1><<<grid, nt, mv.smem_total, st>>>(mv, a, bulk_ok);
    else psr_wsl_kernel<false, 1><<<grid, nt, mv.smem_total, st>>>(mv, a, bulk_ok);
  } else if (tmode == 2) {
    if (outk) psr_wsl_kernel<true, 2><<<grid, nt, mv.smem_total, st>>>(mv, a, bulk_ok);
    else psr_wsl_kernel<false, 2><<<grid, nt, mv.smem_total, st>>>(mv, a, bulk_ok);
  } else {
    if (outk) psr_wsl_kernel<true, 0><<<grid, nt, mv.smem_total, st>>>(mv, a, bulk_ok);
    else psr_wsl_kernel<false, 0><<<grid, nt, mv.smem_total, st>>>(mv, a, bulk_ok);
  }
  return cudaGetLastError();
}

}  // namespace psr
