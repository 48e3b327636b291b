// psr_jac.cu -- fused forward finite-difference Jacobian of the PSR residual (PAPER.md:19, 44:
// "The Jacobian matrix ... is obtained by applying finite difference approximation, which requires the calculation
// of net production rate of species").
//
// The generic sweep (psr_kernels.cu) evaluates the residual once per column: K + 1 full evaluations per reactor,
// each with its own state preparation, gather and epilogue.  A perturbation of ONE mass fraction, though, changes a
// reactor's concentrations in a very particular way (reading g14: rho and W_bar are recomputed from the perturbed,
// unnormalised Y):
//     sum' = sum_i Y_i/W_i + h_j/W_j,   rho' = s rho with s = sum/sum',   C_i' = s C_i (i != j),
//     C_j' = s (C_j + rho h_j/W_j),     C_tot' = rho' sum' = C_tot,
// and leaves every rate constant untouched (k_f, k_r depend on T; a falloff reaction without an efficiency list on
// T and C_tot).  A rate term k prod_n C of concentration order n therefore becomes s^n times itself unless species j is
// one of its factors, so with D_i^(n) = the signed sum over the reactions of the order-n rate terms of species i,
//     wdot_i'/s - wdot_i = sum_n (s^(n-1) - 1) D_i^(n)  +  (1/s) sum_{k touching j} nu_ik dq_k ,
//     F_i(x') - F_i(x)  = delta_ij h_j/tau - (W_i/rho) (wdot_i'/s - wdot_i)              (Eq. 2, rho' = s rho)
// where dq_k, the part of q_k' beyond the uniform scaling, has the closed form
//     k_f s^nf prod_other ((C_j + dC)^a - C_j^a)  -  (same for the reverse side),    dC = rho h_j/W_j,
// with (C+dC)^a - C^a = dC (...) written out for a = 1, 2, 3 (three-body reactions: the same with
// [M]' = C_tot + s (E + (alpha_kj - 1) dC)).  Every small quantity (s - 1, s^n - 1, dC) is formed directly, not as a
// difference of nearly equal numbers: the columns are the difference quotients of the definition, J_ij =
// (F_i(x + h_j e_j) - F_i(x))/h_j, without the eps |F| / h round-off of evaluating F twice -- closer to the exact
// quotient (the long-double oracle J*) than any FP64 sweep can be, at about a tenth of the instructions.
//
// One CTA per tile of 32 reactors (lane <-> reactor), kJacWarps warps.
//   phase 1, twice: at T + h_T (only F is kept: the T column) and at T.  State preparation (a1), the reaction records
//            (a3..a7, psr_rx.cuh) writing forward and reverse rates to a shared-memory rate tile and k_f, k_r, E to a
//            per-CTA scratch, then the sums D_i^(n) by a gather (fixed order); F0 and the T column leave here.
//   phase 2: warp <-> column j: the polynomial in s from D, the incidence records of species j (psr_tables.h), the
//            quotient, stores.  No exchange between warps.
#include <cuda_runtime.h>
#include <stdint.h>

#include "psr_math.cuh"
#include "psr_ptx.cuh"
#include "psr_rx.cuh"
#include "psr_tables.h"

namespace psr {

namespace {
__device__ constexpr double kRgasJ = 8.31446261815324e7;  // erg/mol/K
constexpr int JS_LNT = 0, JS_CTOT = 1, JS_LNCTOT = 2;     // state rows the reaction records read through shared memory
}  // namespace

__global__ void __launch_bounds__(kJacWarps * 32, 1) psr_jac_kernel(const JacView jv, const EvalArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int K = jv.K, n = K + 1, n_cls = jv.n_cls;
  double* Cs = reinterpret_cast<double*>(smem + jv.smem_cs);        // [K+2][32]: C_i; rows K, K+1: ones, zeros
  double* Dt = reinterpret_cast<double*>(smem + jv.smem_d);         // [n_cls][K][32]: D_i^(n)
  double* AR = reinterpret_cast<double*>(smem + jv.smem_ar);        // phase 1: rate tile [rows_max+1][32], then Fp [K][32];
                                                                    // phase 2: [kJacWarps][K+1][33], over this region AND the
                                                                    // blob behind it (phase 2 reads neither: psr_api.cu)
  unsigned char* blob = smem + jv.smem_mech;                        // the part being evaluated (phase 1; loaded per tile and pass)
  double* invW_s = reinterpret_cast<double*>(smem + jv.smem_misc);  // [Kp]
  const int Kp = (K + 1) & ~1;
  double* W_s = invW_s + Kp;                                        // [Kp]
  double* St = W_s + Kp;                                            // [kJacStRows][32]
  uint64_t* bar = reinterpret_cast<uint64_t*>(St + kJacStRows * kTile);
  int* col_next = reinterpret_cast<int*>(bar + 1);                   // phase 2: the next column to hand out
  uint64_t* wbar = bar + 2 + 2 * (threadIdx.x >> 5);                 // this warp's two staging barriers
  unsigned char* stage = smem + jv.smem_stage + (threadIdx.x >> 5) * (2 * kJacStage * sizeof(JacInc));
  double* Fp = AR + (size_t)(jv.rows_max + 1) * kTile;              // F(T + h_T) of the tile
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int nthr = kJacWarps * 32;

  if (a.skip_count && *a.skip_count == 0) return;   // (hybrid solver: every reactor has finished; uniform in the grid)
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    for (int q = 0; q < 2 * kJacWarps; ++q) mbar_init(bar + 2 + q, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (int i = threadIdx.x; i < K; i += nthr) {
    invW_s[i] = jv.invW[i];
    W_s[i] = jv.Wm[i];
  }
  if (w == 0) {
    Cs[K * kTile + lane] = 1.0;
    Cs[(K + 1) * kTile + lane] = 0.0;
  }
  __syncthreads();
  RxCtx cx;
  cx.etab = exp_tab_load(jv.exp_tab);
  cx.c_lane = smem_u32(Cs) + lane * 8;
  cx.ctot_lane = smem_u32(St + JS_CTOT * kTile) + lane * 8;
  cx.lnctot_lane = smem_u32(St + JS_LNCTOT * kTile) + lane * 8;
#ifdef PSR_CHECK
  cx.chk_c_bytes = (uint32_t)(K + 2) * kRowBytes;
#endif
  double* scr = jv.scratch + (size_t)blockIdx.x * jv.I * 3 * kTile + lane;   // row v of reaction k: scr[(3 k + v) * 32]
  const uint32_t r_lane = smem_u32(AR) + lane * 8;
  const uint32_t d_lane = smem_u32(Dt) + lane * 8;
  uint32_t n_loads = 0;   // blob loads this CTA has waited for (mbarrier phase)
  uint32_t n_iss = 0, n_use = 0;   // staging chunks this warp has requested / consumed

  for (int64_t tile = blockIdx.x; tile < a.n_tiles; tile += gridDim.x) {
    if (a.skip_dt) {
      // a tile whose reactors have all finished keeps its (unused) outputs: the same answer in every warp
      const int64_t rs = tile * kTile + (threadIdx.x & 31);
      const double d = rs < a.N ? a.skip_dt[rs] : __longlong_as_double(0x7ff8000000000000LL);
      if (__all_sync(0xffffffffu, d != d)) continue;
    }
    const int64_t r = tile * kTile + lane;
    const bool valid = r < a.N;
    const int64_t rc = valid ? r : a.N - 1;   // lanes past N repeat the last reactor (a valid state, nothing stored)
    const double T0 = ldg_nc(a.T + rc), P = ldg_nc(a.P + rc), invtau = 1.0 / ldg_nc(a.tau + rc);
    double rho = 0.0, invrho = 0.0, sY = 0.0, hT = 0.0;

    // ================================================================ phase 1: at T + h_T, then at T
    for (int pass = 0; pass < 2; ++pass) {
      // ---- a1: state of the tile.  x' = fl(x + delta), h = fl(x' - x) for the T column (O11, g15)
      const double Tp = pass == 0 ? T0 + 1e-8 * fmax(fabs(T0), 1e-10) : T0;
      if (pass == 0) hT = Tp - T0;
      for (int i = w; i < K; i += kJacWarps) Cs[i * kTile + lane] = ldg_nc(a.Y + (int64_t)i * a.ld + rc);
      for (int i = threadIdx.x; i < n_cls * K * kTile; i += nthr) Dt[i] = 0.0;
      if (w == 0) AR[jv.rows_max * kTile + lane] = 0.0;   // the rate tile's zero row (phase 2 uses the region otherwise)
      if (threadIdx.x == 0) *col_next = 0;
      __syncthreads();
      {
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
        int s = 0;
        for (; s + 4 <= K; s += 4) {
          s0 = fma(Cs[s * kTile + lane], invW_s[s], s0);
          s1 = fma(Cs[(s + 1) * kTile + lane], invW_s[s + 1], s1);
          s2 = fma(Cs[(s + 2) * kTile + lane], invW_s[s + 2], s2);
          s3 = fma(Cs[(s + 3) * kTile + lane], invW_s[s + 3], s3);
        }
        for (; s < K; ++s) s0 = fma(Cs[s * kTile + lane], invW_s[s], s0);
        sY = (s0 + s1) + (s2 + s3);
      }
      const double Wbar = 1.0 / sY;
      rho = P * Wbar / (kRgasJ * Tp);
      invrho = 1.0 / rho;
      cx.T = Tp;
      cx.lnT = log(Tp);
      cx.invT = 1.0 / Tp;
      if (w == 0) {
        const double ct = rho * sY;   // C_tot = sum_i C_i = rho sum_i Y_i/W_i
        St[JS_CTOT * kTile + lane] = ct;
        if (jv.need_lnctot) St[JS_LNCTOT * kTile + lane] = log(ct);
      }
      __syncthreads();   // every warp has read the Y rows
      for (int i = w; i < K; i += kJacWarps) Cs[i * kTile + lane] = rho * (Cs[i * kTile + lane] * invW_s[i]);
      __syncthreads();

      // ---- a3..a7 and the sums by order, part after part
      for (int p = 0; p < jv.n_parts; ++p) {
        if (threadIdx.x == 0) {
          fence_proxy_async();
          mbar_expect_tx(bar, jv.chunk_stride);
          bulk_g2s(blob, jv.chunks + (size_t)p * jv.chunk_stride, jv.chunk_stride, bar);
        }
        mbar_wait(bar, n_loads & 1);
        ++n_loads;
        const double ctot = St[JS_CTOT * kTile + lane];
        // rate-tile rows of a record (its first row and its scratch row ride in the record's korig field):
        //   k_f prod C^nu', k_r prod C^nu''; three-body q = (C_tot + E)(...): C_tot x and E x each of the two
        auto sink = [&](int kl, uint32_t meta, uint32_t korig, int type, double kf, double kr, double pf, double pr, double M) {
          PSR_CHK((int)(korig & 0xffffu) + (type == RX_THREE_BODY ? 4 : 2) <= jv.rows_max, 301);   // rows of the rate tile
          PSR_CHK((int)(korig >> 16) < jv.I, 302);                                                // row of the per-CTA scratch
          const uint32_t row = r_lane + (korig & 0xffffu) * (uint32_t)kRowBytes;
          const double Rf = kf * pf, Rr = kr * pr;
          double E = 0.0;
          if (type == RX_THREE_BODY) {
            E = M - ctot;
            sts64(row, ctot * Rf);
            sts64(row + kRowBytes, E * Rf);
            sts64(row + 2 * kRowBytes, ctot * Rr);
            sts64(row + 3 * kRowBytes, E * Rr);
          } else {
            sts64(row, Rf);
            sts64(row + kRowBytes, Rr);
          }
          if (pass == 1) {
            double* sr = scr + (size_t)(korig >> 16) * 3 * kTile;
            sr[0] = kf;
            sr[kTile] = kr;
            sr[2 * kTile] = E;
          }
        };
        cx.amax = 0.0f;
        rx_run_chunk<true>(cx, blob, w, sink);
        if (__any_sync(kFullMask, !exp_max_in_range(cx.amax))) rx_run_chunk<false>(cx, blob, w, sink);
        __syncthreads();   // the rate tile of the part is complete
        {
          // gather: this warp's stream of 4-entry groups (two per trip, software-pipelined as in psr_ws.cu); the group
          // that ends a (species, order) pair adds the pair's sum to its entry of the sums tile
          const ChunkHdr* hdr = reinterpret_cast<const ChunkHdr*>(blob);
          const uint32_t gs = smem_u32(blob + hdr->off_gent) + (uint32_t)hdr->wb[kJacWarps + w][0] * 16u;
          const int n_groups = (int)hdr->wb[kJacWarps + w][1] - (int)hdr->wb[kJacWarps + w][0];
          uint32_t dst = smem_u32(blob + hdr->off_gptr) + (uint32_t)hdr->wb[kJacWarps + w][2] * 4u;
          auto ld_group = [&](uint32_t addr, uint4& o) {
            asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(o.x), "=r"(o.y), "=r"(o.z), "=r"(o.w) : "r"(addr));
          };
          auto sgn = [](uint32_t ctl) { return __hiloint2double((int)(0x3ff00000u ^ (ctl << 31)), 0); };
          auto flush = [&](double& acc) {
            uint32_t off;
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(off) : "r"(dst));
            dst += 4;
            PSR_CHK(off < (uint32_t)n_cls * (uint32_t)K * kRowBytes && off % kRowBytes == 0, 303);   // a row of the sums tile
            sts64(d_lane + off, lds64(d_lane + off) + acc);
            acc = 0.0;
          };
          uint4 oa, ob;
          ld_group(gs, oa);
          ld_group(gs + 16, ob);
          double a0 = lds64(r_lane + (oa.x & ~3u)), a1 = lds64(r_lane + oa.y), a2 = lds64(r_lane + oa.z), a3 = lds64(r_lane + oa.w);
          double b0 = lds64(r_lane + (ob.x & ~3u)), b1 = lds64(r_lane + ob.y), b2 = lds64(r_lane + ob.z), b3 = lds64(r_lane + ob.w);
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
            a0 = lds64(r_lane + (oa.x & ~3u)), a1 = lds64(r_lane + oa.y), a2 = lds64(r_lane + oa.z), a3 = lds64(r_lane + oa.w);
            b0 = lds64(r_lane + (ob.x & ~3u)), b1 = lds64(r_lane + ob.y), b2 = lds64(r_lane + ob.z), b3 = lds64(r_lane + ob.w);
            ld_group(gs + (uint32_t)(i + 4) * 16u, oa);
            ld_group(gs + (uint32_t)(i + 5) * 16u, ob);
            {
              const uint32_t rmax = (uint32_t)(jv.rows_max + 1) * kRowBytes;   // rate tile rows, zero row included
              PSR_CHK((oa.x & ~3u) < rmax && oa.y < rmax && oa.z < rmax && oa.w < rmax && (ob.x & ~3u) < rmax && ob.y < rmax &&
                          ob.z < rmax && ob.w < rmax, 304);
            }
            acc = fma(ta, sgn(c0), acc);
            if (c0 & kGatherLast) flush(acc);
            acc = fma(tb, sgn(c1), acc);
            if (c1 & kGatherLast) flush(acc);
          }
        }
        __syncthreads();   // the sums are in; the rate tile and the blob buffer are free
      }

      // ---- a9: residual of the pass from wdot_i = sum_n D_i^(n) (the same order in both passes)
      for (int i = w; i < K; i += kJacWarps) {
        double wd = 0.0;
        for (int c = 0; c < n_cls; ++c) wd += Dt[(c * K + i) * kTile + lane];
        const int64_t o = (int64_t)i * a.ld + rc;
        const double Fv = fma(ldg_nc(a.Y + o) - ldg_nc(a.Yin + o), invtau, -(wd * (W_s[i] * invrho)));
        if (pass == 0) {
          Fp[i * kTile + lane] = Fv;
        } else if (valid) {
          if (a.F0out) a.F0out[r * n + 1 + i] = Fv;
          PSR_CHK((r * n) * n + 1 + i < a.N * (int64_t)n * n, 305);
          a.J[(r * n) * n + 1 + i] = (Fp[i * kTile + lane] - Fv) / hT;   // column 0: T perturbed
        }
      }
      if (pass == 1 && w == 0 && valid) {
        a.J[(r * n) * n] = 1.0;   // row 0 is F_T = T - T_set (g13)
        if (a.F0out) a.F0out[r * n] = 0.0;
      }
      __syncthreads();
    }

    // ================================================================ phase 2: the species columns, warp <-> column
    // (columns in descending order of their number of records, handed out through a shared counter)
    double* acc_t = AR + (size_t)w * (K + 1) * kJacAccLd;   // this warp's [K+1][33] tile (row K: unused scatter slots)
    const uint32_t acc_lane = smem_u32(acc_t) + lane * 8;
    const double ctot = St[JS_CTOT * kTile + lane];
    for (;;) {
      int jn = 0;
      if (lane == 0) jn = atomicAdd(col_next, 1);
      jn = __shfl_sync(kFullMask, jn, 0);
      if (jn >= K) break;
      const int j = __ldg(jv.col_order + jn);
      PSR_CHK(j >= 0 && j < K, 306);
      const double yj = ldg_nc(a.Y + (int64_t)j * a.ld + rc);
      const double yp = yj + 1e-8 * fmax(fabs(yj), 1e-10);
      const double h = yp - yj;                    // h_j = fl(x' - x)
      const double hw = h * invW_s[j];             // the change of sum Y/W
      const double sYp = sY + hw;
      const double s = sY / sYp;                   // rho'/rho
      const double t = -hw / sYp;                  // s - 1, formed directly
      const double inv_s = sYp / sY;
      const double dc = rho * hw;                  // C_j + dc: the unscaled perturbed concentration of species j
      // s^n and s^n - 1 (u_n = u_(n-1) s + t), n = 1 .. n_cls <= kJacMaxOrder
      double sp[kJacMaxOrder + 1], u[kJacMaxOrder + 1];
      sp[0] = 1.0;
      u[0] = 0.0;
#pragma unroll
      for (int q = 1; q <= kJacMaxOrder; ++q) {
        sp[q] = sp[q - 1] * s;
        u[q] = fma(u[q - 1], s, t);
      }
      auto pw = [&](int q) {   // s^q by warp-uniform selects (q is the same in every lane)
        double v = sp[1];
#pragma unroll
        for (int e = 2; e <= kJacMaxOrder; ++e) v = q == e ? sp[e] : v;
        return v;
      };
      // The incidence records of the column (contiguous in global memory, L2-resident) come through this warp's
      // staging ring in shared memory: chunks of kJacStage records by bulk copies, two in flight; the first two
      // are requested before the polynomial part is formed.
      const int e0 = __ldg(jv.inc_ptr + j), e1 = __ldg(jv.inc_ptr + j + 1);
      const int n_chunks = (e1 - e0 + kJacStage - 1) / kJacStage;
      int ci = 0;   // chunks of this column requested so far
      auto issue = [&]() {
        if (ci < n_chunks) {
          const int first = e0 + ci * kJacStage;
          const uint32_t bytes = (uint32_t)min(kJacStage, e1 - first) * (uint32_t)sizeof(JacInc);
          const uint32_t b = n_iss & 1;
          if (lane == 0) {
            fence_proxy_async();
            mbar_expect_tx(&wbar[b], bytes);
            bulk_g2s(stage + b * kJacStage * sizeof(JacInc), jv.inc + first, bytes, &wbar[b]);
          }
          ++n_iss;
          ++ci;
        }
      };
      issue();
      issue();
      // polynomial part: sum_n (s^(n-1) - 1) D_i^(n)
#pragma unroll 4
      for (int i = 0; i < K; ++i) {
        double v = 0.0;
#pragma unroll
        for (int c = 1; c < kJacMaxOrder; ++c)
          if (c < n_cls) v = fma(u[c], Dt[(c * K + i) * kTile + lane], v);
        acc_t[i * kJacAccLd + lane] = v;
      }
      // the reactions species j takes part in
      const double cj = Cs[j * kTile + lane], cjp = cj + dc;
      const uint32_t off_j = (uint32_t)j * kRowBytes;
      auto ld4 = [&](uint32_t addr, uint4& o) {
        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(o.x), "=r"(o.y), "=r"(o.z), "=r"(o.w) : "r"(addr));
      };
      auto ld_row = [&](uint32_t rec_addr) {
        uint32_t row;
        asm volatile("ld.shared.u32 %0, [%1+24];" : "=r"(row) : "r"(rec_addr));
        return row;
      };
      for (int c = 0; c < n_chunks; ++c) {
        const uint32_t b = n_use & 1;
        mbar_wait(&wbar[b], (n_use >> 1) & 1);
        ++n_use;
        const int cnt = min(kJacStage, e1 - (e0 + c * kJacStage));
        const uint32_t sb = smem_u32(stage + b * kJacStage * sizeof(JacInc));
        // k_f, k_r, E of a record's reaction (this tile's scratch, L2) are requested two records ahead
        double kf_b, kr_b, E_b, kf_c = 0.0, kr_c = 0.0, E_c = 0.0;
        {
          const double* sr = scr + (size_t)ld_row(sb) * 3 * kTile;
          kf_b = sr[0];
          kr_b = sr[kTile];
          E_b = sr[2 * kTile];
          if (cnt > 1) {
            const double* sr2 = scr + (size_t)ld_row(sb + (uint32_t)sizeof(JacInc)) * 3 * kTile;
            kf_c = sr2[0];
            kr_c = sr2[kTile];
            E_c = sr2[2 * kTile];
          }
        }
#pragma unroll 1
        for (int t = 0; t < cnt; ++t) {
          const uint32_t ra = sb + (uint32_t)t * (uint32_t)sizeof(JacInc);
          uint4 A[6];
#pragma unroll
          for (int q = 0; q < 6; ++q) ld4(ra + 16 * q, A[q]);
          const double kf = kf_b, kr = kr_b, E = E_b;
          kf_b = kf_c;
          kr_b = kr_c;
          E_b = E_c;
          if (t + 2 < cnt) {
            const double* sr = scr + (size_t)ld_row(ra + 2 * (uint32_t)sizeof(JacInc)) * 3 * kTile;
            kf_c = sr[0];
            kr_c = sr[kTile];
            E_c = sr[2 * kTile];
          }
          const uint32_t meta = A[1].w;
          {   // the record's factor rows (C tile), scatter rows (this warp's [K+1][33] tile) and scratch row
            const uint32_t cmax = (uint32_t)(K + 2) * kRowBytes, tmax = (uint32_t)(K + 1) * (kJacAccLd * 8);
            PSR_CHK(A[0].x < cmax && A[0].y < cmax && A[0].z < cmax && A[0].w < cmax && A[1].x < cmax && A[1].y < cmax, 307);
            PSR_CHK(A[3].x < tmax && A[3].z < tmax && A[4].x < tmax && A[4].z < tmax && A[5].x < tmax && A[5].z < tmax, 308);
            PSR_CHK((int)A[1].z < jv.I, 309);
          }
          const int tb = meta & 0xff, nf = (meta >> 8) & 0xff, nr = (meta >> 16) & 0xff, af = meta >> 24;
          const int ar = A[2].x & 0xff;
          const double am1 = __hiloint2double((int)A[2].w, (int)A[2].z);
          auto other = [&](uint32_t off) { return off == off_j ? 1.0 : lds64(cx.c_lane + off); };
          // (C + dc)^a - C^a, a = 0..3, without cancellation
          auto grow = [&](int aa) {
            return aa == 0 ? 0.0 : aa == 1 ? dc : aa == 2 ? dc * (cj + cjp) : dc * fma(cj, cj, fma(cj, cjp, cjp * cjp));
          };
          // the targets of the record's scatter are read now, added to below
          const uint32_t t0 = acc_lane + A[3].x, t1 = acc_lane + A[3].z, t2 = acc_lane + A[4].x, t3 = acc_lane + A[4].z,
                         t4 = acc_lane + A[5].x, t5 = acc_lane + A[5].z;
          const double v0 = lds64(t0), v1 = lds64(t1), v2 = lds64(t2), v3 = lds64(t3), v4 = lds64(t4), v5 = lds64(t5);
          const double Pof = other(A[0].x) * other(A[0].y) * other(A[0].z), Por = other(A[0].w) * other(A[1].x) * other(A[1].y);
          const double dPf = Pof * grow(af), dPr = Por * grow(ar);
          const double kfs = kf * pw(nf), krs = kr * pw(nr);
          double dq = fma(kfs, dPf, -(krs * dPr));
          if (tb) {
            // [M]' = C_tot + s (E + (alpha_kj - 1) dc); the uniform-scaling part (C_tot + s E)(...) is in D
            auto power = [&](int aa) { return aa == 0 ? 1.0 : aa == 1 ? cj : aa == 2 ? cj * cj : cj * cj * cj; };
            const double Pf1 = fma(Pof, power(af), dPf), Pr1 = fma(Por, power(ar), dPr);   // perturbed products (unscaled)
            dq = fma(fma(s, E, ctot), dq, (s * am1 * dc) * fma(kfs, Pf1, -(krs * Pr1)));
          }
          dq *= inv_s;
          // (the six targets of a record are distinct species, or the unused row with nu = 0)
          sts64(t0, fma((double)__uint_as_float(A[3].y), dq, v0));
          sts64(t1, fma((double)__uint_as_float(A[3].w), dq, v1));
          sts64(t2, fma((double)__uint_as_float(A[4].y), dq, v2));
          sts64(t3, fma((double)__uint_as_float(A[4].w), dq, v3));
          sts64(t4, fma((double)__uint_as_float(A[5].y), dq, v4));
          sts64(t5, fma((double)__uint_as_float(A[5].w), dq, v5));
        }
        __syncwarp();   // every lane has read the chunk: its buffer takes the chunk after next
        issue();
      }
      // the quotient: J_ij = (delta_ij h/tau - (W_i/rho)(wdot_i'/s - wdot_i)) / h, formed in place; then the warp
      // writes the column of one reactor after the other (n contiguous doubles each: lanes over the rows; the
      // tile's row stride of 33 keeps both access directions free of bank conflicts)
      {
        const double invh = 1.0 / h;
#pragma unroll 4
        for (int i = 0; i < K; ++i) {
          const double d = -(W_s[i] * invrho) * acc_t[i * kJacAccLd + lane];
          acc_t[i * kJacAccLd + lane] = (i == j ? fma(h, invtau, d) : d) * invh;
        }
      }
      __syncwarp();
      {
        const int n_valid = (int)min((int64_t)kTile, a.N - tile * kTile);
        double* Jc = a.J + ((tile * kTile * n) + 1 + j) * n;   // column 1 + j of the tile's first reactor
        PSR_CHK(((tile * kTile + n_valid - 1) * n + 1 + j) * n + n <= a.N * (int64_t)n * n, 310);   // the last reactor's column ends inside J
        // four reactors per trip, their values read before the first store (a load the compiler cannot move over a
        // store through another generic pointer would otherwise wait for it)
        const int64_t nn = (int64_t)n * n;
        int l = 0;
        for (; l + 4 <= n_valid; l += 4, Jc += 4 * nn) {
          for (int e = lane; e < n; e += 32) {
            double v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) v[u] = e == 0 ? 0.0 : acc_t[(e - 1) * kJacAccLd + l + u];   // row 0: F_T = T - T_set does not depend on Y
#pragma unroll
            for (int u = 0; u < 4; ++u) Jc[u * nn + e] = v[u];
          }
        }
        for (; l < n_valid; ++l, Jc += nn)
          for (int e = lane; e < n; e += 32) Jc[e] = e == 0 ? 0.0 : acc_t[(e - 1) * kJacAccLd + l];
      }
      __syncwarp();
    }
    __syncthreads();   // the next tile's phase 1 reuses every tile
  }
}

PSR_CHK_TU_READER(chk_read_jac)

cudaError_t jac_set_smem(size_t smem) {
  return cudaFuncSetAttribute(psr_jac_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}

cudaError_t launch_jac(const JacView& jv, const EvalArgs& a, int grid, cudaStream_t st) {
  psr_jac_kernel<<<grid, kJacWarps * 32, jv.smem_total, st>>>(jv, a);
  return cudaGetLastError();
}

// ------------------------------------------------------------------ the same kernel with STATIC scratch (psr_fd_jacobian_noalloc)
// Some callers cannot let the library allocate: code under CUDA-graph capture, tight serving loops, harnesses that
// forbid cudaMalloc.  For them the kernel's per-CTA scratch ([CTAs][I][3][32] doubles: k_f, k_r, E of the tile a CTA
// works on) lives in this file-scope array instead of the buffer psr_mech_load allocates.  Every GPU that loads the
// library holds these 32 MiB until the process exits.
//   * g_jac_static_scratch is, in HOST code, only a stand-in for the symbol -- not a device address: passing it to a
//     kernel would fault (or silently use host memory where the GPU can reach it).  The device address comes from
//     cudaGetSymbolAddress, asked once per device with that device current, and is what the kernel is given.
//   * Nothing in the array has to start at zero: in phase 1 a CTA writes the rows of all I reactions of its tile (every
//     lane, lanes past N included) before phase 2 reads any of them, so what the last call left behind is never read.
//   * Every call on a device shares the array: two calls that overlap on the GPU (different streams, or a graph
//     replayed beside an eager call) race on it.  Serialise them.
constexpr size_t kJacStaticBytes = (size_t)32 << 20;
static __device__ __align__(256) double g_jac_static_scratch[kJacStaticBytes / sizeof(double)];

size_t jac_static_scratch_bytes() { return kJacStaticBytes; }

// Device address of the static scratch on the current device; resolved on the first call per device (no allocation:
// the array is part of the loaded module).
static cudaError_t jac_static_scratch_ptr(double** out) {
  constexpr int kMaxDev = 64;
  static double* ptr[kMaxDev];
  static bool have[kMaxDev];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
  if (!have[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_jac_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    ptr[dev] = p;     // (two host threads racing here store the same address)
    have[dev] = true;
  }
  *out = ptr[dev];
  return cudaSuccess;
}

// grid: at most the CTAs whose scratch rows fit the array (the caller has checked that at least one does)
cudaError_t launch_jac_static(const JacView& jv, const EvalArgs& a, int grid, cudaStream_t st) {
  double* scratch = nullptr;
  cudaError_t e = jac_static_scratch_ptr(&scratch);
  if (e != cudaSuccess) return e;
  const size_t per_cta = (size_t)jv.I * 3 * kTile * sizeof(double);
  if (grid < 1 || (size_t)grid * per_cta > kJacStaticBytes) return cudaErrorInvalidConfiguration;
  JacView v = jv;
  v.scratch = scratch;
  psr_jac_kernel<<<grid, kJacWarps * 32, v.smem_total, st>>>(v, a);
  return cudaGetLastError();
}

}  // namespace psr
