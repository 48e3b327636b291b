// psr_kernels.cu -- sm_100a kernels of the batched PSR chemistry hot path.
//
// One fused kernel evaluates SURVEY.md 8(a) steps a1..a10 for a tile of 32 R evaluation states:
//   lane  <-> R reactors (or, in Jacobian mode, R perturbed copies of a reactor),
//   warp  <-> a share of the chunk's reactions (reaction phase) / a share of the species (gather).
// Every per-reaction quantity is therefore warp-uniform: mechanism constants are shared-memory
// broadcasts, reaction-type branches never diverge, and C[species][lane] reads are conflict-free.
//
// Per tile:   prologue  a1  Wbar, rho, C_i -> smem Cs[K][32 R]           (Eq. 5's X_i)
//             per chunk a3-a7  k_f, K_c, k_r, [M], falloff, q -> qs[rc][32 R]   (Eq. 5-9)
//                       a8     wdot += nu^T q : CSR gather, accumulators in registers (Eq. 4)
//             epilogue  a9/a10 residual (Eq. 2) / difference quotient, coalesced stores.
// The mechanism chunk blobs (psr_tables.h) stream global -> shared through cp.async.bulk with an
// mbarrier per stage; a mechanism that fits one chunk is staged once per CTA.
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "psr_math.cuh"
#include "psr_ptx.cuh"
#include "psr_tables.h"

namespace psr {

__device__ constexpr double kRgas = 8.31446261815324e7;  // erg/mol/K
__device__ constexpr double kLog10e = 0.43429448190325182765;
constexpr int PSR_T_PLAIN = 0, PSR_T_THREE_BODY = 1, PSR_T_LINDEMANN = 2, PSR_T_TROE = 3;  // = PSR_RX_* of psr.h

template <int R>
struct RowIO;
template <>
struct RowIO<1> {
  static __device__ __forceinline__ void ld(uint32_t addr, double (&v)[1]) { v[0] = lds64(addr); }
  static __device__ __forceinline__ void st(uint32_t addr, const double (&v)[1]) { sts64(addr, v[0]); }
};
template <>
struct RowIO<2> {
  static __device__ __forceinline__ void ld(uint32_t addr, double (&v)[2]) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v[0]), "=d"(v[1]) : "r"(addr));
  }
  static __device__ __forceinline__ void st(uint32_t addr, const double (&v)[2]) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v[0]), "d"(v[1]));
  }
};

#ifndef PSR_MINB
#define PSR_MINB(NW) ((NW) == 8 ? 2 : 1)   // CTAs per SM the register allocation is held to (128 regs/thread)
#endif
// ------------------------------------------------------------------ the fused kernel
// R reactors per lane: every warp-uniform instruction (mechanism loads, address arithmetic, branches)
// is amortised over R evaluations and the R exp chains interleave in the FP64 pipe.
// JY: the Y-column launch of psr_fd_jacobian (kModeJacY) -- tiles are aligned to reactors (the 32 lanes of
// a tile are 32 Y columns of ONE reactor) and the T-only factors of every reaction come from the rate
// table that the base-residual launch wrote, as warp-uniform broadcasts, instead of being recomputed.
// EN: psr_eval_residual_energy -- the epilogue also forms the energy row (kOutFT).  Its own instantiation so
// that the extra registers and code stay out of the other calls (measured: 2.7 % on C1 when shared).
constexpr int kVarPlain = 0, kVarJacY = 1, kVarEnergy = 2;   // bit flags: 3 = Y-column launch of the adiabatic Jacobian
template <int NW, int SPW, int R, int VAR>
__global__ void __launch_bounds__(NW * 32, PSR_MINB(NW)) psr_eval_kernel(const MechView mv, const EvalArgs a) {
  constexpr bool JY = (VAR & kVarJacY) != 0;
  constexpr bool EN = (VAR & kVarEnergy) != 0;
  // DS: the epilogue's operands Y - Y_in and tau come with the tile's prefetch (shared memory) instead of
  // being loaded into registers before the last gather, where they were spilled at once (measured: the
  // spill stores waited for the loads, 5 % of the kernel)
  constexpr bool DS = SPW <= 4 && !JY;   // (the Y-column launch has registers to spare and keeps the loads)
  static_assert(!JY || R == 1, "the Y-column mode maps one column to a lane");
  constexpr int TR = 32 * R;  // evaluation states per tile
  extern __shared__ __align__(128) unsigned char smem[];
  double* Cs0 = reinterpret_cast<double*>(smem + mv.smem_cs);         // [2][K+2][TR]; row K is the unit row
  double* qs = reinterpret_cast<double*>(smem + mv.smem_q);           // [rc+1][TR]; row rc stays zero
  unsigned char* mring = smem + mv.smem_mech;                         // stages * chunk_stride
  double* part = reinterpret_cast<double*>(smem + mv.smem_misc);      // [NW][TR] partial sums
  double* lane_s = part + NW * TR;                                    // [TR]: ln T per state
  double* hs = lane_s + TR;                                           // [TR]: finite-difference step per state
  double* rho_s = hs + TR;                                            // [TR]: density per state
  double* ctot_s = rho_s + TR;                                        // [TR]: C_tot per state
  double* lnctot_s = ctot_s + TR;                                     // [TR]: ln C_tot (formed on first use)
  double* tp = lnctot_s + TR;                                         // [2][3][TR]: prefetched T, P, tau
  uint64_t* bars = reinterpret_cast<uint64_t*>(tp + 6 * TR);          // [kMaxStages] chunk stages, [kMaxStages] rate table
  double* tab_s = reinterpret_cast<double*>(smem + mv.smem_tab);      // [kslices][rc][kRateVals]: rate table slices of the tile's reactors (JY)
  double* Ds0 = reinterpret_cast<double*>(smem + mv.smem_tab);        // [2][K][TR]: Y_in, then Y - Y_in, of the tile (DS; shares the region of the JY table slices)
  double* en_s = qs;   // [3][NW][TR]: partial sums of the energy row (the q tile is free after the last gather)

  const int lane = threadIdx.x & 31;
  const int w = threadIdx.x >> 5;
  const int K = mv.K;
  const int n = K + 1;
  const bool jac = (a.flags & (kModeJac | kModeJacT | kModeJacY)) != 0;
  const bool jacT = (a.flags & kModeJacT) != 0;
  // JY: state v = reactor * Kp + species column; a tile is 32 consecutive states.  Small mechanisms pack the
  // columns densely (Kp = K: a tile spans up to 31/K + 2 reactors, whose rate-table slices sit side by side
  // in tab_s); large ones (K > 64, where padding wastes little and shared memory is short) pad every
  // reactor to whole tiles (Kp = 32 ceil(K/32): one reactor, one slice per tile).
  const int Kp = mv.jy_dense ? K : ((K + 31) / 32) * 32;
  const int64_t n_states = a.N * Kp;
  const bool resident = mv.resident != 0;   // every chunk blob has its own stage and is loaded once per CTA
  const int nstage = resident ? mv.n_chunks : mv.ring_stages;
  const int cs_elems = (K + 2) * TR;
  const int ds_elems = K * TR;
  const bool wantF = jac || (a.flags & (kOutF | kOutF0)) != 0;
  const uint32_t q_lane = smem_u32(qs) + lane * (8 * R);

  const int64_t my_tiles = (a.n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x;
  const int64_t total_loads = resident ? mv.n_chunks : my_tiles * mv.n_chunks;

  if (threadIdx.x == 0) {
    for (int g = 0; g <= kMaxStages; ++g) mbar_init(&bars[g], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    for (int g = 0; g < nstage && g < total_loads; ++g) {
      mbar_expect_tx(&bars[g], mv.chunk_stride);
      bulk_g2s(mring + (size_t)g * mv.chunk_stride, mv.chunks + (size_t)(g % mv.n_chunks) * mv.chunk_stride,
               mv.chunk_stride, &bars[g]);
    }
  }
  const ExpTab etab = exp_tab_load(mv.exp_tab);
  // Species this warp owns in the prologue, gather and epilogue.  Up to 4 per warp they and their
  // accumulators live in registers across the chunks.  Beyond that (GA, K > 64) registers would spill:
  // the slot loops are not unrolled, the species index is re-read, and the running sum of a species goes
  // through the output array between chunks (L2-resident for the tile) instead of a register.
  constexpr bool GA = SPW > 4;
  constexpr int SPR = GA ? 1 : SPW;
  int sp[SPR];
  if constexpr (!GA) {
#pragma unroll
    for (int jj = 0; jj < SPW; ++jj) sp[jj] = mv.sp_of[w * SPW + jj];
  }
  auto for_species = [&](auto&& f) {
    if constexpr (GA) {
#pragma unroll 1
      for (int jj = 0; jj < SPW; ++jj) {
        const int s = __ldg(mv.sp_of + w * SPW + jj);
        if (s >= 0) f(0, s);
      }
    } else {
#pragma unroll
      for (int jj = 0; jj < SPW; ++jj) {
        const int s = sp[jj];
        if (s >= 0) f(jj, s);
      }
    }
  };
  if (w == 0) {
#pragma unroll
    for (int i = 0; i < R; ++i) qs[mv.rc * TR + lane * R + i] = 0.0;
  }

  // state i of this lane in tile t is evaluation v = t*TR + i*32 + lane (coalesced global access); in
  // shared memory it lives at column lane*R + i of every row.  Jacobian mode: v = reactor*n + column.
  auto state_of = [&](int64_t t, int i, int64_t& r_, int& jsp_, bool& valid_) {
    const int64_t v = t * TR + i * 32 + lane;
    if constexpr (JY) {
      valid_ = v < n_states;
      const uint32_t vv = (uint32_t)(valid_ ? v : n_states - 1);   // states of a sub-batch fit 32 bits (psr_fd_jacobian)
      const uint32_t rr = vv / (uint32_t)Kp;
      const int j = (int)(vv - rr * (uint32_t)Kp);
      r_ = rr;
      valid_ = valid_ && j < K;
      jsp_ = valid_ ? j : -2;   // padding lanes evaluate an unperturbed state, unused
    } else if (jacT) {
      valid_ = v < a.N;
      r_ = valid_ ? v : a.N - 1;
      jsp_ = -1;
    } else if (jac) {
      valid_ = v < a.N * n;
      const int64_t vv = valid_ ? v : a.N * n - 1;
      r_ = vv / n;
      jsp_ = (int)(vv - r_ * n) - 1;   // perturbed species; -1: the T column
    } else {
      valid_ = v < a.N;
      r_ = valid_ ? v : a.N - 1;
      jsp_ = -2;                      // nothing perturbed
    }
  };
  // asynchronous prefetch of a tile's T, P (warp 0) and of this thread's Y entries into C buffer `buf`
  auto prefetch = [&](int64_t t, int buf) {
    if (t < a.n_tiles) {
#pragma unroll
      for (int i = 0; i < R; ++i) {
        int64_t r_;
        int jsp_;
        bool valid_;
        state_of(t, i, r_, jsp_, valid_);
        const int col = lane * R + i;
        if (w == 0) {
          cp_async8(tp + (buf * 3 + 0) * TR + col, a.T + r_);
          cp_async8(tp + (buf * 3 + 1) * TR + col, a.P + r_);
          if (DS && wantF) cp_async8(tp + (buf * 3 + 2) * TR + col, a.tau + r_);
        }
        for_species([&](int, int s) {
          cp_async8(Cs0 + buf * cs_elems + s * TR + col, a.Y + (int64_t)s * a.ld + r_);
          if (DS && wantF) cp_async8(Ds0 + buf * ds_elems + s * TR + col, a.Yin + (int64_t)s * a.ld + r_);
        });
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  prefetch(blockIdx.x, 0);
  // JY: bulk copies of the rate-table slices of tile t's reactors for chunk c into tab_s (thread 0 only)
  auto tile_reactors = [&](int64_t t, uint32_t& r_first, uint32_t& r_last) {
    const int64_t v0 = t * TR, v1 = min(v0 + TR, n_states) - 1;
    r_first = (uint32_t)v0 / (uint32_t)Kp;
    r_last = (uint32_t)v1 / (uint32_t)Kp;
  };
  auto load_tab = [&](int64_t t, int c) {
    const int b0 = mv.chunk_rec_base[c], b1 = mv.chunk_rec_base[c + 1];
    const uint32_t bytes = (uint32_t)(b1 - b0) * (kRateVals * 8);
    uint32_t r0, r1;
    tile_reactors(t, r0, r1);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(&bars[kMaxStages], bytes * (r1 - r0 + 1));
    for (uint32_t rr = r0; rr <= r1; ++rr)
      bulk_g2s(tab_s + (size_t)(rr - r0) * mv.rc * kRateVals, a.tab + ((size_t)rr * mv.I + b0) * kRateVals, bytes,
               &bars[kMaxStages]);
  };
  int64_t gt = 0;  // rate-table slices consumed so far by this CTA
  if constexpr (JY) {
    if (threadIdx.x == 0 && blockIdx.x < a.n_tiles) load_tab(blockIdx.x, 0);
  }
  __syncthreads();

  int64_t g = 0;  // chunk loads consumed so far by this CTA
  int buf = 0;
  for (int64_t tile = blockIdx.x; tile < a.n_tiles; tile += gridDim.x, buf ^= (mv.n_cbuf - 1)) {
    // ---------------------------------------------------------------- prologue (a1)
    double* Cs = Cs0 + buf * cs_elems;
    double* Ds = Ds0 + buf * ds_elems;
    const uint32_t c_lane = smem_u32(Cs) + lane * (8 * R);   // this lane's R slots of row 0 of the C tile
    asm volatile("cp.async.wait_group 0;" ::: "memory");   // this thread's prefetched entries have landed

    double T[R];
    // Energy row (steady Eq. 3): this thread's share of  sum Yin_i (h_i(Tin) - h_i(T)),
    // sum h_i wdot_i W_i  and  sum Y_i cp_i  over the species it owns; h [erg/g] = (h/RT) R T / W (NASA-7).
    // The first and the last sum do not need wdot: with the Y - Y_in tile (DS) they are formed in the
    // prologue, where Y and Y_in are at hand, and the epilogue adds the middle one (same h, same order).
    double en[3][R];
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int i = 0; i < R; ++i) en[k][i] = 0.0;
    auto h_of = [&](int s, double t) {
      const double* c = mv.nasa + 7 * s;
      const double hRT = fma(fma(fma(fma(c[4] * 0.2, t, c[3] * 0.25), t, c[2] * (1.0 / 3.0)), t, c[1] * 0.5), t, c[0]) + c[5] / t;
      return hRT * (kRgas * mv.invW[s]) * t;
    };
    auto energy_pre = [&](int s, int i, double Tin_, double y, double yin) {
      if constexpr (!EN) return;
      const double* c = mv.nasa + 7 * s;
      const double cp = fma(fma(fma(fma(c[4], T[i], c[3]), T[i], c[2]), T[i], c[1]), T[i], c[0]) * (kRgas * mv.invW[s]);
      en[0][i] = fma(yin, h_of(s, Tin_) - h_of(s, T[i]), en[0][i]);
      en[2][i] = fma(y, cp, en[2][i]);
    };
    auto energy_post = [&](int s, int i, double wd) {
      if constexpr (!EN) return;
      en[1][i] = fma(h_of(s, T[i]) * wd, mv.Wm[s], en[1][i]);
    };
    auto energy_terms = [&](int s, int i, double Tin_, double y, double yin, double wd) {
      energy_pre(s, i, Tin_, y, yin);
      energy_post(s, i, wd);
    };
    {
      int jsp[R];
      double rho[R], tin[R];
#pragma unroll
      for (int i = 0; i < R; ++i) {
        int64_t r_;
        bool valid_;
        state_of(tile, i, r_, jsp[i], valid_);
        tin[i] = (EN && DS && wantF) ? ldg_nc(a.Tin + r_) : 0.0;
      }
      // x' = fl(x + delta), h = fl(x' - x) for the perturbed unknown of a Jacobian state (O11, g15)
      // pass 1: Y_i/W_i summed; a perturbed entry is replaced in the tile.  pass 2 (below) re-reads it.
      double sumYW[R];
#pragma unroll
      for (int i = 0; i < R; ++i) sumYW[i] = 0.0;
      for_species([&](int, int s) {
        const double iw = mv.invW[s];
#pragma unroll
        for (int i = 0; i < R; ++i) {
          double y = Cs[s * TR + lane * R + i];
          if (s == jsp[i]) {
            const double yp = y + 1e-8 * fmax(fabs(y), 1e-10);
            hs[lane * R + i] = yp - y;
            Cs[s * TR + lane * R + i] = yp;
            y = yp;
          }
          sumYW[i] += y * iw;
        }
      });
#pragma unroll
      for (int i = 0; i < R; ++i) part[w * TR + lane * R + i] = sumYW[i];
      if (w == 0) {
#pragma unroll
        for (int i = 0; i < R; ++i) {
          Cs[K * TR + lane * R + i] = 1.0;         // unit row: unused factor slots
          Cs[(K + 1) * TR + lane * R + i] = 0.0;   // zero row: product side of an irreversible reaction
        }
      }
      __syncthreads();   // partial sums and warp 0's T, P visible; every warp has left the previous tile
      if (mv.n_cbuf == 2) prefetch(tile + gridDim.x, buf ^ 1);
#pragma unroll
      for (int i = 0; i < R; ++i) {
        T[i] = tp[(buf * 3 + 0) * TR + lane * R + i];
        const double P = tp[(buf * 3 + 1) * TR + lane * R + i];
        if (jsp[i] == -1) {
          const double Tp = T[i] + 1e-8 * fmax(fabs(T[i]), 1e-10);
          if (w == 0) hs[lane * R + i] = Tp - T[i];
          T[i] = Tp;
        }
        double sY = 0.0;
#pragma unroll
        for (int ww = 0; ww < NW; ++ww) sY += part[ww * TR + lane * R + i];
        const double Wbar = 1.0 / sY;
        rho[i] = P * Wbar / (kRgas * T[i]);
        if (w == 0) {
          // C_tot = sum_i C_i = rho * sum_i Y_i/W_i: formed from the sum already at hand (differs from
          // the species-by-species sum by rounding only)
          const double ct = rho[i] * sY;
          lane_s[lane * R + i] = log(T[i]);
          rho_s[lane * R + i] = rho[i];
          ctot_s[lane * R + i] = ct;
          if (mv.need_lnctot) lnctot_s[lane * R + i] = log(ct);   // Troe reactions without efficiencies
        }
      }
      for_species([&](int, int s) {
        const double iw = mv.invW[s];
#pragma unroll
        for (int i = 0; i < R; ++i) {
          const double y = Cs[s * TR + lane * R + i];   // the perturbed value where this state perturbs s
          if (DS && wantF) {
            const double yin = Ds[s * TR + lane * R + i];
            Ds[s * TR + lane * R + i] = y - yin;
            energy_pre(s, i, tin[i], y, yin);
          }
          Cs[s * TR + lane * R + i] = rho[i] * (y * iw);
        }
      });
    }
    __syncthreads();
    double lnT[R], invT[R];
#pragma unroll
    for (int i = 0; i < R; ++i) {
      lnT[i] = lane_s[lane * R + i];
      invT[i] = 1.0 / T[i];
    }

    double acc[SPR][R];
#pragma unroll
    for (int jj = 0; jj < SPR; ++jj)
#pragma unroll
      for (int i = 0; i < R; ++i) acc[jj][i] = 0.0;

    // ---------------------------------------------------------------- chunks
    int stage = 0;
    const unsigned char* blob = nullptr;
    const ChunkHdr* hdr = nullptr;
    // gather (a8, Eq. 4) of the chunk in `stage`: every warp sums the rows of nu^T it owns in a fixed
    // order; afterwards the stage is handed back to the bulk-copy ring
    // adds the chunk's rows of nu^T q for species s to a0, in the fixed order of the gather lists
    auto sum_rows = [&](const uint32_t* gptr, const uint4* gent, int s, double (&a0)[R]) {
      const uint32_t g0 = gptr[2 * s] >> 2, g1 = gptr[2 * s + 1] >> 2, g2 = gptr[2 * s + 2] >> 2;
      double a1[R];
#pragma unroll
      for (int i = 0; i < R; ++i) a1[i] = 0.0;
#pragma unroll 1
      PSR_CHK(s >= 0 && s < K && g0 <= g1 && g1 <= g2, 407);
      for (uint32_t e = g0; e < g1; ++e) {
        const uint4 o = gent[e];
        {
          const uint32_t qmax = (uint32_t)(mv.rc + 1) * (uint32_t)(TR * 8);   // rows of the q tile, zero row included
          PSR_CHK(o.x < qmax && o.y < qmax && o.z < qmax && o.w < qmax, 408);
        }
        double v0[R], v1[R], v2[R], v3[R];
        RowIO<R>::ld(q_lane + o.x, v0);
        RowIO<R>::ld(q_lane + o.y, v1);
        RowIO<R>::ld(q_lane + o.z, v2);
        RowIO<R>::ld(q_lane + o.w, v3);
#pragma unroll
        for (int i = 0; i < R; ++i) {
          a0[i] += v0[i];
          a1[i] += v1[i];
          a0[i] += v2[i];
          a1[i] += v3[i];
        }
      }
#pragma unroll 1
      for (uint32_t e = g1; e < g2; ++e) {
        const uint4 o = gent[e];
        {
          const uint32_t qmax = (uint32_t)(mv.rc + 1) * (uint32_t)(TR * 8);
          PSR_CHK(o.x < qmax && o.y < qmax && o.z < qmax && o.w < qmax, 409);
        }
        double v0[R], v1[R], v2[R], v3[R];
        RowIO<R>::ld(q_lane + o.x, v0);
        RowIO<R>::ld(q_lane + o.y, v1);
        RowIO<R>::ld(q_lane + o.z, v2);
        RowIO<R>::ld(q_lane + o.w, v3);
#pragma unroll
        for (int i = 0; i < R; ++i) {
          a0[i] -= v0[i];
          a1[i] -= v1[i];
          a0[i] -= v2[i];
          a1[i] -= v3[i];
        }
      }
#pragma unroll
      for (int i = 0; i < R; ++i) a0[i] += a1[i];
    };
    // GA: where the running sum of (species s, state i of this lane) rests between chunks, and the
    // outputs of that entry once the last chunk is in (same arithmetic as the epilogue below)
    auto ga_slot = [&](int s, int64_t r_, int jsp_) -> double* {
      if (jac) return a.J + ((int64_t)r_ * n + (jsp_ + 1)) * n + 1 + s;
      if (a.flags & kOutWdot) return a.wdot + (int64_t)s * a.ld + r_;
      if (a.flags & kOutF) return a.F + (int64_t)s * a.ld + r_;
      return a.F0out + r_ * n + 1 + s;
    };
    auto ga_finish = [&](int s, int i, int64_t r_, int jsp_, double accv) {
      PSR_CHK(s >= 0 && s < K && r_ >= 0 && r_ < a.N, 410);   // element (species, r) of the [K][ld] arrays
      const int64_t o = (int64_t)s * a.ld + r_;
      if (!jac) {
        if (a.flags & kOutWdot) a.wdot[o] = accv;
        if (wantF) {
          const double invtau = 1.0 / ldg_nc(a.tau + r_);
          const double invrho = 1.0 / rho_s[lane * R + i];
          const double Fv = fma(ldg_nc(a.Y + o) - ldg_nc(a.Yin + o), invtau, -(accv * (mv.Wm[s] * invrho)));
          if (a.flags & kOutF) a.F[o] = Fv;
          if (a.flags & kOutF0) a.F0out[r_ * n + 1 + s] = Fv;
          if constexpr (EN) energy_terms(s, i, ldg_nc(a.Tin + r_), ldg_nc(a.Y + o), ldg_nc(a.Yin + o), accv);
        }
      } else {
        const double invtau = 1.0 / ldg_nc(a.tau + r_);
        const double invrho = 1.0 / rho_s[lane * R + i];
        const double invh = 1.0 / hs[lane * R + i];
        double y = ldg_nc(a.Y + o);
        if (s == jsp_) y = y + 1e-8 * fmax(fabs(y), 1e-10);   // the same x' as in the prologue
        const double yin = ldg_nc(a.Yin + o);
        const double Fv = fma(y - yin, invtau, -(accv * (mv.Wm[s] * invrho)));
        *ga_slot(s, r_, jsp_) = (Fv - ldg_nc(a.F0 + r_ * n + 1 + s)) * invh;
        if constexpr (EN) energy_terms(s, i, ldg_nc(a.Tin + r_), y, yin, accv);
      }
    };
    auto gather_and_release = [&](bool first, bool last) {
      if (jac || (a.flags & (kOutWdot | kOutF | kOutF0))) {
        const uint32_t* gptr = reinterpret_cast<const uint32_t*>(blob + hdr->off_gptr);
        const uint4* gent = reinterpret_cast<const uint4*>(blob + hdr->off_gent);
        if constexpr (GA) {
          int64_t r_[R];
          int jsp_[R];
          bool valid_[R];
#pragma unroll
          for (int i = 0; i < R; ++i) state_of(tile, i, r_[i], jsp_[i], valid_[i]);
          // the running sum of the NEXT species is requested before this species' rows are added, so that its
          // trip to L2 runs beside the summation instead of in front of it
          auto fetch = [&](int s, double (&v)[R]) {
#pragma unroll
            for (int i = 0; i < R; ++i) v[i] = (first || !valid_[i] || s < 0) ? 0.0 : *ga_slot(s, r_[i], jsp_[i]);
          };
          int s_nxt = __ldg(mv.sp_of + w * SPW);
          double nxt[R];
          fetch(s_nxt, nxt);
#pragma unroll 1
          for (int jj = 0; jj < SPW; ++jj) {
            const int s = s_nxt;
            double a0[R];
#pragma unroll
            for (int i = 0; i < R; ++i) a0[i] = nxt[i];
            if (jj + 1 < SPW) {
              s_nxt = __ldg(mv.sp_of + w * SPW + jj + 1);
              fetch(s_nxt, nxt);
            }
            if (s < 0) continue;
            sum_rows(gptr, gent, s, a0);
#pragma unroll
            for (int i = 0; i < R; ++i) {
              if (valid_[i]) {
                if (last) ga_finish(s, i, r_[i], jsp_[i], a0[i]);
                else *ga_slot(s, r_[i], jsp_[i]) = a0[i];
              }
            }
          }
        } else {
          for_species([&](int jj, int s) { sum_rows(gptr, gent, s, acc[jj]); });
        }
      }
      __syncthreads();
      if (!resident) {
        if (threadIdx.x == 0 && g + nstage < total_loads) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          mbar_expect_tx(&bars[stage], mv.chunk_stride);
          bulk_g2s(mring + (size_t)stage * mv.chunk_stride,
                   mv.chunks + (size_t)((g + nstage) % mv.n_chunks) * mv.chunk_stride, mv.chunk_stride, &bars[stage]);
        }
      }
      ++g;
    };
    for (int c = 0; c < mv.n_chunks; ++c) {
      stage = (int)(g % nstage);
      if (!resident || g < nstage) mbar_wait(&bars[stage], (uint32_t)((g / nstage) & 1));
      blob = mring + (size_t)stage * mv.chunk_stride;
      hdr = reinterpret_cast<const ChunkHdr*>(blob);
      const RxRec* recs = reinterpret_cast<const RxRec*>(blob + sizeof(ChunkHdr));

      // ---- reaction phase (a3..a7): warp w takes its cost-balanced share of the chunk's records, sorted
      // by class (plain, three-body, Lindemann, Troe in the 3+3 slot form; then the long-list form), one
      // loop per class so that no reaction-type test is left inside a loop.  FAST: every exp takes the
      // table form and a lane only notes an out-of-range argument; the CTA then repeats the phase with
      // the library exp (IEEE results for NaN, Inf, overflow, gradual underflow).  That never happens for
      // physical states, so the range test costs two compares per reaction and no vote or branch.
      const double* tvb = tab_s;   // JY: the table slice of this lane's reactor
      if constexpr (JY) {
        int64_t r_;
        int jsp_;
        bool valid_;
        uint32_t r0, r1;
        state_of(tile, 0, r_, jsp_, valid_);
        tile_reactors(tile, r0, r1);
        tvb = tab_s + (size_t)((uint32_t)r_ - r0) * mv.rc * kRateVals;
      }
      float amax = 0.0f;   // NaN-propagating running max of |high word| of every exp argument of this lane
      auto run_class = [&](auto cls_tag, auto fast_tag, auto out_tag) {
        constexpr int CLS = decltype(cls_tag)::value;
        constexpr bool FAST = decltype(fast_tag)::value;
        // 0: nothing leaves the loop but q; 1: k_f, k_r, q go to global memory (psr_eval_kf_kr, q of
        // psr_eval_wdot); 2: the T-only factors go to the rate table (base launch of psr_fd_jacobian);
        // 3: decided by the flags at run time (the rare library-exp repeat, to keep the code small)
        constexpr int OUTT = decltype(out_tag)::value;
        const bool out_k = OUTT == 1 || (OUTT == 3 && (a.flags & (kOutKf | kOutKr | kOutQ)) != 0);
        const bool out_tab = OUTT == 2 || (OUTT == 3 && (a.flags & kOutTab) != 0);
        // the record range is the same in every lane: say so (REDUX writes a uniform register), which
        // keeps the loop counter and the record addresses in the uniform datapath
        const int kl_begin = __reduce_min_sync(kFullMask, (int)hdr->wb[w][CLS]);
        const int kl_end = __reduce_min_sync(kFullMask, (int)hdr->wb[w][CLS + 1]);
        PSR_CHK(kl_begin >= 0 && kl_begin <= kl_end && kl_end <= (int)hdr->n_rx && kl_end <= mv.rc, 401);
        auto exps = [&](auto& ex, auto& ey) {
          constexpr int N = sizeof(ex) / sizeof(double);
          if constexpr (FAST) {
#pragma unroll
            for (int i = 0; i < N; ++i) amax = exp_arg_max(amax, ex[i]);
            exp_core_n<N>(ex, ey, etab);
          } else {
#pragma unroll
            for (int i = 0; i < N; ++i) ey[i] = exp(ex[i]);
          }
        };
        // rate table row of this lane's reactor (OUT == 2 only)
        auto tab_row = [&](int kl, int i, bool& valid_) -> double* {
          int64_t r_;
          int jsp_;
          state_of(tile, i, r_, jsp_, valid_);
          return a.tab_out + ((size_t)r_ * mv.I + hdr->rec_base + kl) * kRateVals;
        };
        // The slot offsets (and meta, korig) of a record are read one trip ahead: they head the longest
        // chain of the trip (offsets -> C tile loads -> products), and read at the top of their own trip
        // they cost a shared-memory round trip before anything else can start.  Reading one record past
        // the warp's range stays inside the chunk blob.
        // (Not in the energy-row instantiation, whose epilogue operands leave no registers for it.)
        constexpr int PF = EN ? 0 : 1;
        uint4 nxa, nxb;
        if constexpr (PF) {
          const uint32_t ra = smem_u32(recs + kl_begin) + 80;
          asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(nxa.x), "=r"(nxa.y), "=r"(nxa.z), "=r"(nxa.w) : "r"(ra));
          asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4+16];" : "=r"(nxb.x), "=r"(nxb.y), "=r"(nxb.z), "=r"(nxb.w) : "r"(ra));
        }
#pragma unroll 1
        for (int kl = kl_begin; kl < kl_end; ++kl) {
          const RxRec* rec = recs + kl;
          if constexpr (!PF) {
            const uint32_t ra = smem_u32(rec) + 80;
            asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(nxa.x), "=r"(nxa.y), "=r"(nxa.z), "=r"(nxa.w) : "r"(ra));
            asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4+16];" : "=r"(nxb.x), "=r"(nxb.y), "=r"(nxb.z), "=r"(nxb.w) : "r"(ra));
          }
          const uint4 ra_ = nxa, rb_ = nxb;   // {meta, off[0..2]}, {off[3..5], korig} of this record
          if constexpr (PF) {
            const uint32_t ra = smem_u32(rec) + (112 + 80);
            asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(nxa.x), "=r"(nxa.y), "=r"(nxa.z), "=r"(nxa.w) : "r"(ra));
            asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4+16];" : "=r"(nxb.x), "=r"(nxb.y), "=r"(nxb.z), "=r"(nxb.w) : "r"(ra));
          }
          const uint32_t meta = ra_.x;
          const int type = CLS < kClsLong ? CLS : (int)(meta & kMetaTypeMask);
          const double* tv = tvb + kl * kRateVals;     // JY: the T-only factors of this reaction for the lane's reactor
          double lnkf[R], lnkr[R], pf[R], pr[R], kf[R], kr[R], M[R];
          // Eq. 6 in log form, and ln k_r = ln k_f - ln K_c (Eq. 7-9 summed per reaction at load time)
          if constexpr (!JY) {
#pragma unroll
            for (int i = 0; i < R; ++i) {
              lnkf[i] = fma(rec->c[1], lnT[i], fma(rec->c[2], invT[i], rec->c[0]));
              const double pn = fma(fma(fma(rec->d[3], T[i], rec->d[2]), T[i], rec->d[1]), T[i], rec->d[0]);
              lnkr[i] = fma(pn, T[i], fma(rec->e[1], lnT[i], fma(rec->e[2], invT[i], rec->e[0])));
            }
          }
#pragma unroll
          for (int i = 0; i < R; ++i) M[i] = 1.0;

          // concentration products (Eq. 5): integer powers by repetition, unused slots read the unit row
          if constexpr (CLS < kClsLong) {
            double f0[R], f1[R], f2[R], p0[R], p1[R], p2[R];
            {
              const uint32_t cmax = (uint32_t)cs_elems * 8u;   // factor rows of the C tile, unit and zero rows included
              PSR_CHK(ra_.y < cmax && ra_.z < cmax && ra_.w < cmax && rb_.x < cmax && rb_.y < cmax && rb_.z < cmax, 402);
            }
            RowIO<R>::ld(c_lane + ra_.y, f0);
            RowIO<R>::ld(c_lane + ra_.z, f1);
            RowIO<R>::ld(c_lane + ra_.w, f2);
            RowIO<R>::ld(c_lane + rb_.x, p0);
            RowIO<R>::ld(c_lane + rb_.y, p1);
            RowIO<R>::ld(c_lane + rb_.z, p2);
#pragma unroll
            for (int i = 0; i < R; ++i) {
              pf[i] = f0[i] * f1[i] * f2[i];
              pr[i] = p0[i] * p1[i] * p2[i];
            }
          } else {
            const uint16_t* fsp = reinterpret_cast<const uint16_t*>(blob + hdr->off_pool) + ra_.y;
            const int nr = (int)((meta >> kMetaNrShift) & 0xF);
            const int np = (int)((meta >> kMetaNpShift) & 0xF);
#pragma unroll
            for (int i = 0; i < R; ++i) {
              pf[i] = 1.0;
              pr[i] = 1.0;
            }
#pragma unroll 1
            for (int j = 0; j < nr + np; ++j) {
              double cv[R];
              PSR_CHK((uint32_t)fsp[j] < (uint32_t)(K + 2), 403);
              RowIO<R>::ld(c_lane + (uint32_t)fsp[j] * (uint32_t)(TR * 8), cv);
#pragma unroll
              for (int i = 0; i < R; ++i) {
                if (j < nr) pf[i] *= cv[i];
                else pr[i] *= cv[i];
              }
            }
            if (!(meta & kMetaRev)) {
#pragma unroll
              for (int i = 0; i < R; ++i) pr[i] = 0.0;
            }
          }

          // sign of A and of A0/A (psr.h accepts any finite A: negative pre-exponentials of duplicate reactions, A = 0):
          // only long-form records carry them (psr_tables.h), so this folds away in the other class loops
          double sA = 1.0, sPr = 1.0;
          if constexpr (CLS == kClsLong) {
            const uint32_t sg = (meta >> kMetaSgnShift) & 0xFu;
            if (sg) {
              const double s0 = (sg >> 2) == 0 ? 1.0 : (sg >> 2) == 1 ? -1.0 : 0.0;
              sA = (sg & 3u) == 0 ? 1.0 : (sg & 3u) == 1 ? -1.0 : 0.0;
              sPr = sA == 0.0 ? __longlong_as_double(0x7ff8000000000000LL) : s0 * sA;   // k0 [M] / 0 is not a number
            }
          }
          if (type <= PSR_T_THREE_BODY) {
            if constexpr (JY) {
#pragma unroll
              for (int i = 0; i < R; ++i) {
                kf[i] = tv[0];
                kr[i] = tv[1];
              }
            } else {
              double ex[2 * R], ey[2 * R];
#pragma unroll
              for (int i = 0; i < R; ++i) {
                ex[2 * i] = lnkf[i];
                ex[2 * i + 1] = lnkr[i];
              }
              exps(ex, ey);
#pragma unroll
              for (int i = 0; i < R; ++i) {
                kf[i] = ey[2 * i];
                kr[i] = ey[2 * i + 1];
              }
              if (out_tab) {
#pragma unroll
                for (int i = 0; i < R; ++i) {
                  bool valid_;
                  double* row = tab_row(kl, i, valid_);
                  if (valid_) {
                    row[0] = kf[i];
                    row[1] = kr[i];
                  }
                }
              }
            }
          }
          if constexpr (CLS == kClsLong) {
            if (type <= PSR_T_THREE_BODY) {
#pragma unroll
              for (int i = 0; i < R; ++i) {
                kf[i] *= sA;
                kr[i] *= sA;
              }
            }
          }
          if (type != PSR_T_PLAIN) {
            const AuxRec* ax = reinterpret_cast<const AuxRec*>(blob + hdr->off_aux) + (meta >> kMetaAuxShift);
            const EffEnt* effs = reinterpret_cast<const EffEnt*>(blob + hdr->off_eff);
#pragma unroll
            for (int i = 0; i < R; ++i) M[i] = ctot_s[lane * R + i];
            const uint32_t e1 = ax->eff_off + ax->n_eff;
            PSR_CHK((meta >> kMetaAuxShift) < hdr->n_aux && e1 <= hdr->n_eff, 404);
#pragma unroll 1
            for (uint32_t e = ax->eff_off; e < e1; ++e) {
              PSR_CHK(effs[e].off < (uint32_t)cs_elems * 8u, 405);
              double cv[R];
              RowIO<R>::ld(c_lane + effs[e].off, cv);
#pragma unroll
              for (int i = 0; i < R; ++i) M[i] = fma(effs[e].am1, cv[i], M[i]);
            }
            if (type == PSR_T_THREE_BODY) {
#pragma unroll
              for (int i = 0; i < R; ++i) {
                pf[i] *= M[i];
                pr[i] *= M[i];
              }
            } else if (type == PSR_T_LINDEMANN) {
              // k_f = k_inf Pr/(1+Pr), Pr = k0 [M]/k_inf
              double ey[3 * R];
              if constexpr (JY) {
#pragma unroll
                for (int i = 0; i < R; ++i) {
                  ey[3 * i] = tv[2];
                  ey[3 * i + 1] = tv[0];
                  ey[3 * i + 2] = tv[1];
                }
              } else {
                double ex[3 * R];
#pragma unroll
                for (int i = 0; i < R; ++i) {
                  const double lnk0 = fma(ax->c0[1], lnT[i], fma(ax->c0[2], invT[i], ax->c0[0]));
                  ex[3 * i] = lnk0 - lnkf[i];
                  ex[3 * i + 1] = lnkf[i];
                  ex[3 * i + 2] = lnkr[i] - lnkf[i];
                }
                exps(ex, ey);
                if (out_tab) {
#pragma unroll
                  for (int i = 0; i < R; ++i) {
                    bool valid_;
                    double* row = tab_row(kl, i, valid_);
                    if (valid_) {
                      row[0] = ey[3 * i + 1];
                      row[1] = ey[3 * i + 2];
                      row[2] = ey[3 * i];
                    }
                  }
                }
              }
#pragma unroll
              for (int i = 0; i < R; ++i) {
                double Pr = ey[3 * i] * M[i];
                if constexpr (CLS == kClsLong) Pr *= sPr;
                kf[i] = ey[3 * i + 1] * (Pr / (1.0 + Pr));
                if constexpr (CLS == kClsLong) kf[i] *= sA;
                kr[i] = kf[i] * ey[3 * i + 2];
              }
            } else {
              // Troe.  With ln Pr = ln k0 - ln k_inf + ln[M]:
              //   k_f = k_inf Pr/(1+Pr) F = exp(ln k0 + ln[M] + ln F)/(1+Pr)
              // one reactor at a time: five exps in lock step are enough to fill the FP64 pipe.  The JY
              // form repeats the same operations on the tabulated ln k0, ln k_inf, ln F_cent, 1/K_c, so the
              // T-only part of a perturbed state is bit-identical to that of the base state.
#pragma unroll
              for (int i = 0; i < R; ++i) {
                const double lnM = ax->n_eff == 0 ? lnctot_s[lane * R + i] : log(M[i]);
                double lnk0, lnkinf, lnFc, invKc, Pr;
                if constexpr (JY) {
                  lnk0 = tv[0];
                  invKc = tv[1];
                  lnkinf = tv[2];
                  lnFc = tv[3];
                } else {
                  lnk0 = fma(ax->c0[1], lnT[i], fma(ax->c0[2], invT[i], ax->c0[0]));
                  lnkinf = lnkf[i];
                }
                const double lnk0M = lnk0 + lnM;
                const double lnPr = lnk0M - lnkinf;
                if constexpr (JY) {
                  double ex[1], ey[1];
                  ex[0] = lnPr;
                  exps(ex, ey);
                  Pr = ey[0];
                } else {
                  double ex[5], ey[5];
                  ex[0] = lnPr;
                  ex[1] = T[i] * ax->troe[1];
                  ex[2] = T[i] * ax->troe[2];
                  ex[3] = ax->troe[3] * invT[i];
                  ex[4] = lnkr[i] - lnkf[i];        // ln(k_r/k_f) = -ln K_c
                  exps(ex, ey);
                  Pr = ey[0];
                  invKc = ey[4];
                  const double al = ax->troe[0];
                  const double Fcent = fma(1.0 - al, ey[1], fma(al, ey[2], ey[3]));
                  lnFc = log(Fcent);
                  if (out_tab) {
                    bool valid_;
                    double* row = tab_row(kl, i, valid_);
                    if (valid_) {
                      row[0] = lnk0;
                      row[1] = invKc;
                      row[2] = lnkinf;
                      row[3] = lnFc;
                    }
                  }
                }
                const double lF = lnFc * kLog10e;
                const double cc = fma(-0.67, lF, -0.4);
                const double nn = fma(-1.27, lF, 0.75);
                const double lp = fma(lnPr, kLog10e, cc);
                const double den = fma(-0.14, lp, nn);
                // ln F = ln Fcent / (1 + (lp/den)^2) = ln Fcent den^2 / (den^2 + lp^2); den = 0 with lp != 0 gives F = 1 (g17);
                // den = lp = 0 (0/0) and Pr = inf (inf/inf) are not numbers here as in the definition
                // both quotients (this one and k_f = .../(1+Pr)) share one reciprocal
                const double den2 = den * den;
                const double bq = fma(lp, lp, den2), dq = 1.0 + Pr;
                const double inv = 1.0 / (bq * dq);
                double e2[1], k2[1];
                e2[0] = fma(lnFc * den2, dq * inv, lnk0M);
                exps(e2, k2);
                kf[i] = k2[0] * (bq * inv);
                // the log form above needs Pr > 0; otherwise log10(Pr) of the definition is not a number (or -inf,
                // which makes F not a number): same result here
                if constexpr (CLS == kClsLong) kf[i] = sPr > 0.0 ? kf[i] * sA : __longlong_as_double(0x7ff8000000000000LL);
                kr[i] = kf[i] * invKc;
              }
            }
          }
          // an irreversible reaction has its product side on the zero row (pr = 0), a three-body reaction
          // carries [M] in both products: no per-lane selects here
          double q[R];
#pragma unroll
          for (int i = 0; i < R; ++i) q[i] = fma(kf[i], pf[i], -(kr[i] * pr[i]));
          RowIO<R>::st(q_lane + (uint32_t)kl * (uint32_t)(TR * 8), q);

          if (out_k) {
#pragma unroll
            for (int i = 0; i < R; ++i) {
              int64_t r_;
              int jsp_;
              bool valid_;
              state_of(tile, i, r_, jsp_, valid_);
              if (valid_) {
                PSR_CHK((int64_t)rb_.w < (int64_t)mv.I && r_ < a.N, 406);   // element (reaction, r) of the [I][ldk] outputs
                const int64_t o = (int64_t)rb_.w * a.ldk + r_;
                if (a.flags & kOutKf) a.kf[o] = kf[i];
                if (a.flags & kOutKr) a.kr[o] = (meta & kMetaRev) ? kr[i] : 0.0;
                if (a.flags & kOutQ) a.q[o] = q[i];
              }
            }
          }
        }
      };
      auto run_out = [&](auto fast_tag, auto out_tag) {
        run_class(std::integral_constant<int, 0>{}, fast_tag, out_tag);
        run_class(std::integral_constant<int, 1>{}, fast_tag, out_tag);
        run_class(std::integral_constant<int, 2>{}, fast_tag, out_tag);
        run_class(std::integral_constant<int, 3>{}, fast_tag, out_tag);
        run_class(std::integral_constant<int, kClsLong>{}, fast_tag, out_tag);
      };
      auto run_all = [&](auto fast_tag) {
        if constexpr (JY) {
          run_out(fast_tag, std::integral_constant<int, 0>{});
        } else if constexpr (!decltype(fast_tag)::value) {
          run_out(fast_tag, std::integral_constant<int, 3>{});
        } else {
          if (a.flags & (kOutKf | kOutKr | kOutQ)) run_out(fast_tag, std::integral_constant<int, 1>{});
          else if (a.flags & kOutTab) run_out(fast_tag, std::integral_constant<int, 2>{});
          else run_out(fast_tag, std::integral_constant<int, 0>{});
        }
      };
      if constexpr (JY) mbar_wait(&bars[kMaxStages], (uint32_t)(gt & 1));   // the rate table slices of this tile
      run_all(std::true_type{});
      if (__syncthreads_or(!exp_max_in_range(amax))) {   // also the barrier that publishes the q tile
        run_all(std::false_type{});
        __syncthreads();
      }
      if constexpr (JY) {
        // the table buffer is free: request the slice of the next (tile, chunk) of this CTA
        ++gt;
        const bool more_chunks = c + 1 < mv.n_chunks;
        const int64_t nt = more_chunks ? tile : tile + gridDim.x;
        if (threadIdx.x == 0 && nt < a.n_tiles) load_tab(nt, more_chunks ? c + 1 : 0);
      }

      if (c + 1 < mv.n_chunks) gather_and_release(c == 0, false);
    }

    // operands of the epilogue are requested now so that they arrive during the last gather
    double e_tau[R], e_y[SPR][R], e_yin[SPR][R], e_f0[SPR][R];
    int64_t r[R];
    int jsp[R];
    bool valid[R];
#pragma unroll
    for (int i = 0; i < R; ++i) state_of(tile, i, r[i], jsp[i], valid[i]);
      if (wantF) {
#pragma unroll
        for (int i = 0; i < R; ++i) {
          e_tau[i] = DS ? tp[(buf * 3 + 2) * TR + lane * R + i] : ldg_nc(a.tau + r[i]);
          if constexpr (!GA) {
            for_species([&](int jj, int s) {
              const int64_t o = (int64_t)s * a.ld + r[i];
              if constexpr (!DS) {
                e_y[jj][i] = ldg_nc(a.Y + o);
                e_yin[jj][i] = ldg_nc(a.Yin + o);
              }
              if (jac) e_f0[jj][i] = ldg_nc(a.F0 + r[i] * n + 1 + s);
            });
          }
        }
      }

    gather_and_release(mv.n_chunks == 1, true);

    // Energy row: the three sums over all species -- per-warp shares through shared memory (the q tile is
    // free by now), added in warp order by warp 0, whose lanes get F_T = -dT/dt of their states.  Every
    // thread of the CTA calls this.
    auto energy_reduce = [&](double (&ft)[R]) {
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int i = 0; i < R; ++i) en_s[(k * NW + w) * TR + lane * R + i] = en[k][i];
      __syncthreads();
#pragma unroll
      for (int i = 0; i < R; ++i) {
        ft[i] = 0.0;
        if (w == 0) {
          double e[3];
#pragma unroll
          for (int k = 0; k < 3; ++k) {
            e[k] = 0.0;
#pragma unroll
            for (int ww = 0; ww < NW; ++ww) e[k] += en_s[(k * NW + ww) * TR + lane * R + i];
          }
          ft[i] = -((e[0] / ldg_nc(a.tau + r[i]) - e[1] / rho_s[lane * R + i]) / e[2]);
        }
      }
      __syncthreads();
      if (w == 0) {   // the partial sums may have covered the q tile's zero row
#pragma unroll
        for (int i = 0; i < R; ++i) qs[mv.rc * TR + lane * R + i] = 0.0;
      }
    };

    // ---------------------------------------------------------------- epilogue (a8 store, a9, a10)
    if constexpr (GA) {
      // every (species, state) entry left with the last gather; what remains is row 0 of the unknowns
      if (w == 0) {
#pragma unroll
        for (int i = 0; i < R; ++i) {
          if (valid[i]) {
            if (EN) continue;
            if (jac) a.J[((int64_t)r[i] * n + (jsp[i] + 1)) * n] = (jsp[i] == -1) ? 1.0 : 0.0;   // F_T = T - T_set
            else if (a.flags & kOutF0) a.F0out[r[i] * n] = 0.0;
          }
        }
      }
      if constexpr (EN) {
        double ft[R];
        energy_reduce(ft);
        if (w == 0) {
#pragma unroll
          for (int i = 0; i < R; ++i) {
            if (!valid[i]) continue;
            if (jac) a.J[((int64_t)r[i] * n + (jsp[i] + 1)) * n] = (ft[i] - ldg_nc(a.F0 + r[i] * n)) / hs[lane * R + i];
            else {
              if (a.FT) a.FT[r[i]] = ft[i];
              if (a.flags & kOutF0) a.F0out[r[i] * n] = ft[i];
            }
          }
        }
        __syncthreads();   // warp 0 has read the steps hs[] before the next tile's prologue writes them
      }
    } else if (!jac) {
#pragma unroll
      for (int i = 0; i < R; ++i) {
        if (valid[i]) {
          const double invtau = 1.0 / e_tau[i];
          const double invrho = 1.0 / rho_s[lane * R + i];
#pragma unroll
          for (int jj = 0; jj < SPW; ++jj) {
            const int s = sp[jj];
            if (s >= 0) {
              PSR_CHK(s < K && r[i] >= 0 && r[i] < a.N, 411);
              const int64_t o = (int64_t)s * a.ld + r[i];
              if (a.flags & kOutWdot) a.wdot[o] = acc[jj][i];
              if (wantF) {
                const double dy = DS ? Ds[s * TR + lane * R + i] : e_y[jj][i] - e_yin[jj][i];
                const double Fv = fma(dy, invtau, -(acc[jj][i] * (mv.Wm[s] * invrho)));
                if (a.flags & kOutF) a.F[o] = Fv;
                if (a.flags & kOutF0) a.F0out[r[i] * n + 1 + s] = Fv;
                if constexpr (EN && DS) energy_post(s, i, acc[jj][i]);
                else if constexpr (EN) energy_terms(s, i, ldg_nc(a.Tin + r[i]), e_y[jj][i], e_yin[jj][i], acc[jj][i]);
              }
            }
          }
          if (!EN && (a.flags & kOutF0) && w == 0) a.F0out[r[i] * n] = 0.0;
        }
      }
      if constexpr (EN) {
        double ft[R];
        energy_reduce(ft);
        if (w == 0) {
#pragma unroll
          for (int i = 0; i < R; ++i) {
            if (!valid[i]) continue;
            if (a.FT) a.FT[r[i]] = ft[i];
            if (a.flags & kOutF0) a.F0out[r[i] * n] = ft[i];
          }
        }
      }
    } else {
      // difference quotient, staged [state][npad] in this tile's C buffer, then one linear coalesced store
      const int npad = n | 1;
      double* stg = Cs;  // needs TR*npad doubles <= (K+2)*TR (host sizes smem_cs accordingly)
#pragma unroll
      for (int i = 0; i < R; ++i) {
        const double invtau = 1.0 / e_tau[i];
        const double invrho = 1.0 / rho_s[lane * R + i];
        const double invh = 1.0 / hs[lane * R + i];
        const int st = i * 32 + lane;  // position of this state inside the tile, in evaluation order
#pragma unroll
        for (int jj = 0; jj < SPW; ++jj) {
          const int s = sp[jj];
          if (s >= 0) {
            double y = 0.0, dy;
            if constexpr (DS) {
              dy = Ds[s * TR + lane * R + i];   // formed in the prologue from the perturbed y
            } else {
              y = e_y[jj][i];
              if (s == jsp[i]) y = y + 1e-8 * fmax(fabs(y), 1e-10);   // the same x' as in the prologue
              dy = y - e_yin[jj][i];
            }
            const double Fv = fma(dy, invtau, -(acc[jj][i] * (mv.Wm[s] * invrho)));
            stg[st * npad + 1 + s] = (Fv - e_f0[jj][i]) * invh;
            if constexpr (EN && DS) energy_post(s, i, acc[jj][i]);
            else if constexpr (EN) energy_terms(s, i, ldg_nc(a.Tin + r[i]), y, e_yin[jj][i], acc[jj][i]);
          }
        }
        if (!EN && w == 0) stg[st * npad] = (jsp[i] == -1) ? 1.0 : 0.0;  // row 0: F_T = T - T_set
      }
      if constexpr (EN) {   // row 0: the energy row's difference quotient
        double ft[R];
        energy_reduce(ft);
        if (w == 0) {
#pragma unroll
          for (int i = 0; i < R; ++i)
            stg[(i * 32 + lane) * npad] = (ft[i] - ldg_nc(a.F0 + r[i] * n)) / hs[lane * R + i];
        }
      }
      __syncthreads();
      if constexpr (JY) {
        // state l of the tile is column 1 + j of reactor r: n contiguous doubles in J; consecutive states are
        // consecutive columns except across a reactor boundary (the T column lies between)
        for (int idx = threadIdx.x; idx < TR * n; idx += NW * 32) {
          const int l = idx / n, i = idx - l * n;
          const int64_t v = tile * TR + l;
          if (v < n_states) {
            const uint32_t rr = (uint32_t)v / (uint32_t)Kp;
            const uint32_t j = (uint32_t)v - rr * (uint32_t)Kp;
            PSR_CHK(j >= (uint32_t)K || ((int64_t)rr * n + 1 + j) * n + i < a.N * (int64_t)n * n, 412);
            if (j < (uint32_t)K) a.J[((int64_t)rr * n + 1 + j) * n + i] = stg[l * npad + i];
          }
        }
      } else if (jacT) {
        // column 0 of reactors tile*TR ..: n contiguous doubles each, n*n apart
        for (int idx = threadIdx.x; idx < TR * n; idx += NW * 32) {
          const int l = idx / n, i = idx - l * n;
          const int64_t r_ = tile * TR + l;
          if (r_ < a.N) a.J[r_ * n * n + i] = stg[l * npad + i];
        }
      } else {
        const int64_t base = tile * TR * (int64_t)n;
        const int64_t lim = a.N * (int64_t)n * n;
        for (int idx = threadIdx.x; idx < TR * n; idx += NW * 32) {
          const int l = idx / n, i = idx - l * n;
          if (base + idx < lim) a.J[base + idx] = stg[l * npad + i];
        }
      }
      __syncthreads();
    }
    if (mv.n_cbuf == 1) prefetch(tile + gridDim.x, 0);   // single C buffer: it is free only now
  }
}

// ------------------------------------------------------------------ launch wrapper
#ifdef PSR_EXP_SHAPES   // development builds: fewer shapes compile in a fraction of the time
#define PSR_SHAPES(X) X(16, 4)
#else
#define PSR_SHAPES(X) X(16, 2) X(16, 4) X(16, 8) X(16, 16) X(16, 32)
#endif

template <int NW, int SPW, int R, int VAR>
static cudaError_t launch_t(const MechView& mv, const EvalArgs& a, int grid, cudaStream_t st) {
  auto kern = psr_eval_kernel<NW, SPW, R, VAR>;   // its dynamic shared-memory limit was raised once, at load (occupancy_eval)
  const uint32_t smem = mv.smem_total;
  kern<<<grid, NW * 32, smem, st>>>(mv, a);
  return cudaGetLastError();
}

cudaError_t launch_eval(int nw, int spw, int rl, const MechView& mv, const EvalArgs& a, int grid, cudaStream_t st) {
  const int var = ((a.flags & kModeJacY) ? kVarJacY : 0) | ((a.flags & kOutFT) ? kVarEnergy : 0);
#define PSR_L(NW_, SPW_)                                                                        \
  if (nw == NW_ && spw == SPW_ && rl == 1) {                                                    \
    if (var == 3) return launch_t<NW_, SPW_, 1, 3>(mv, a, grid, st);                            \
    if (var == kVarJacY) return launch_t<NW_, SPW_, 1, kVarJacY>(mv, a, grid, st);              \
    if (var == kVarEnergy) return launch_t<NW_, SPW_, 1, kVarEnergy>(mv, a, grid, st);          \
    return launch_t<NW_, SPW_, 1, kVarPlain>(mv, a, grid, st);                                  \
  }
  PSR_SHAPES(PSR_L)
#undef PSR_L
  return cudaErrorInvalidConfiguration;
}

template <int NW, int SPW, int R>
static cudaError_t occ_t(size_t smem, size_t smem_optin, int* ctas_per_sm) {
  // every variant is launched with the same grid: size it for the one with the lowest occupancy
  const void* kerns[4] = {(const void*)psr_eval_kernel<NW, SPW, R, 0>, (const void*)psr_eval_kernel<NW, SPW, R, 1>,
                          (const void*)psr_eval_kernel<NW, SPW, R, 2>, (const void*)psr_eval_kernel<NW, SPW, R, 3>};
  int least = 1 << 30;
  for (const void* k : kerns) {
    int nb = 0;
    // raised to the device's limit once per kernel instance: mechanisms of different sizes share the instance,
    // so the attribute must not follow the mechanism loaded last
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_optin);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k, NW * 32, smem);
    if (e != cudaSuccess) return e;
    least = nb < least ? nb : least;
  }
  *ctas_per_sm = least;
  return cudaSuccess;
}

cudaError_t occupancy_eval(int nw, int spw, int rl, size_t smem, size_t smem_optin, int* ctas_per_sm) {
#define PSR_O(NW_, SPW_) \
  if (nw == NW_ && spw == SPW_ && rl == 1) return occ_t<NW_, SPW_, 1>(smem, smem_optin, ctas_per_sm);
  PSR_SHAPES(PSR_O)
#undef PSR_O
  return cudaErrorInvalidConfiguration;
}

// ------------------------------------------------------------------ PSR_CHECK plumbing
PSR_CHK_TU_READER(chk_read_kernels)

// trips one check on purpose (code 999): "0 failures" must not be able to mean "the checks are compiled out"
__global__ void chk_selftest_kernel(int one) { PSR_CHK(one != 1, 999); }
cudaError_t launch_chk_selftest(cudaStream_t st) {
  chk_selftest_kernel<<<1, 1, 0, st>>>(1);
  return cudaGetLastError();
}

// ------------------------------------------------------------------ FP64 pipe probes
template <int KIND>
__global__ void __launch_bounds__(256) probe_kernel(int iters, double* sink) {
  double x0 = 1.0 + 1e-9 * threadIdx.x, x1 = 0.5 + 1e-9 * threadIdx.x, x2 = 0.25, x3 = 0.125;
  double x4 = 0.3, x5 = 0.7, x6 = 0.9, x7 = 1.1;
  const double a = 0.999999, b = 1e-7;
  for (int i = 0; i < iters; ++i) {
    if (KIND == 0) {
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
      }
    } else if (KIND == 1) {
      x0 = exp(x0 * -0.5); x1 = exp(x1 * -0.5); x2 = exp(x2 * -0.5); x3 = exp(x3 * -0.5);
      x4 = exp(x4 * -0.5); x5 = exp(x5 * -0.5); x6 = exp(x6 * -0.5); x7 = exp(x7 * -0.5);
    } else {
      x0 = log(x0 + 1.5); x1 = log(x1 + 1.5); x2 = log(x2 + 1.5); x3 = log(x3 + 1.5);
      x4 = log(x4 + 1.5); x5 = log(x5 + 1.5); x6 = log(x6 + 1.5); x7 = log(x7 + 1.5);
    }
  }
  const double s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
  if (s == 123.456) sink[0] = s;
}

// exp_fast on an array (diagnostic behind psr_probe_exp_values)
__global__ void exp_values_kernel(const double* __restrict__ tab, const double* __restrict__ x, double* __restrict__ y, int n) {
  const ExpTab etab = exp_tab_load(tab);
  const int stride = gridDim.x * blockDim.x;
  for (int i0 = blockIdx.x * blockDim.x; i0 < n; i0 += stride) {   // warp-uniform trip count
    const int i = i0 + threadIdx.x;
    const double v = exp_fast(x[i < n ? i : n - 1], etab);
    if (i < n) y[i] = v;
  }
}

cudaError_t launch_exp_values(const double* tab, const double* x, double* y, int n, cudaStream_t st) {
  exp_values_kernel<<<148, 256, 0, st>>>(tab, x, y, n);
  return cudaGetLastError();
}

cudaError_t launch_probe(int kind, int iters, int grid, double* sink, cudaStream_t st) {
  if (kind == 0) probe_kernel<0><<<grid, 256, 0, st>>>(iters, sink);
  else if (kind == 1) probe_kernel<1><<<grid, 256, 0, st>>>(iters, sink);
  else probe_kernel<2><<<grid, 256, 0, st>>>(iters, sink);
  return cudaGetLastError();
}

}  // namespace psr
