// psr_lu.cu -- batched dense solve of the Newton step.
//
// "The Jacobian matrix is decomposed into lower and upper triangular matrices, and then a back-solving
// operation is carried out to obtain the final solution".  One warp per system: the n x n
// matrix (column-major per reactor, the layout psr_fd_jacobian writes) lives in shared memory with an odd
// column stride, lane l owns rows l, l+32, ...  Gaussian elimination with partial pivoting (largest
// |a_ik|, the first one on ties -- the same choice as the oracle), rank-1 updates with the multipliers of a
// lane's rows in registers and the pivot row as shared-memory broadcasts, then a column-oriented back
// substitution.  Row accesses along a column are contiguous and row exchanges run along the odd stride:
// no bank conflicts.  Several systems (warps) per CTA so that one warp's global loads overlap another's
// elimination.
#include <cuda_runtime.h>
#include <stdint.h>

namespace psr {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kNB = 8;   // pivots per pass over the trailing matrix

// RPL: rows per lane (n <= 32 * RPL).  The column stride ld = n | 1 is a run-time value, so the update walks
// the columns with two running pointers (pivot-row entry, this lane's rows) instead of forming j*ld + i for
// every access (that index arithmetic cost more instructions than the elimination itself: 51 k
// instructions per 54 x 54 system, 4 k of them FMA, in the first version).
// PTC: the pseudo-transient variant (psr_ptc_solve): matrix J + I/dt, right-hand side -F.
template <int RPL, bool PTC>
__global__ void __launch_bounds__(128) lu_solve_kernel(int64_t N, int n, const double* __restrict__ A,
                                                       double* __restrict__ b, int32_t* __restrict__ info,
                                                       int sys_doubles, const double* __restrict__ F,
                                                       const double* __restrict__ dt, const int32_t* __restrict__ skip_count) {
  extern __shared__ __align__(16) double sm[];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, wpc = blockDim.x >> 5;
  const int ld = n | 1;
  double* As = sm + (size_t)w * sys_doubles;   // entry (i, j) at As[j*ld + i]
  double* bs = As + (size_t)n * ld;            // [n]
  double* dinv = bs + n;                       // [n] reciprocals of the pivots

  // psr_solve_hybrid (skip_count non-null): nothing to do once every reactor has finished, and a finished reactor's
  // system -- its dt is NaN -- is left out (dx, info unchanged and unused)
  if (PTC && skip_count && *skip_count == 0) return;
  for (int64_t r = (int64_t)blockIdx.x * wpc + w; r < N; r += (int64_t)gridDim.x * wpc) {
    if (PTC && skip_count && dt[r] != dt[r]) continue;
    const double* Ar = A + (size_t)r * n * n;
    // pseudo-transient step (psr_ptc_solve): the matrix is J + I/dt, the right-hand side -F
    const double shift = PTC ? 1.0 / dt[r] : 0.0;
    {
      // column-major stream, 32 consecutive entries per trip, kStageU trips in flight (with one warp per system and
      // nine warps per SM nothing else hides the latency of these loads: at 4 in flight they were 18 % of the samples);
      // (i, j) tracked without a divide.  The warp's NEXT system is asked into L2 meanwhile.
      constexpr int kStageU = 24;
      {
        const int64_t rn = r + (int64_t)gridDim.x * wpc;
        if (rn < N) {
          const char* pn = reinterpret_cast<const char*>(A + (size_t)rn * n * n);
          for (int o = lane * 128; o < n * n * 8; o += 32 * 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(pn + o));
        }
      }
      int i = lane, j = 0;
      while (i >= n) { i -= n; ++j; }
      for (int t = lane; t < n * n; t += 32 * kStageU) {
        double v[kStageU];
        int off[kStageU];
#pragma unroll
        for (int u = 0; u < kStageU; ++u) {
          off[u] = j * ld + i;
          v[u] = (t + 32 * u < n * n) ? Ar[t + 32 * u] : 0.0;
          if (PTC && i == j) v[u] += shift;
          i += 32;
          while (i >= n) { i -= n; ++j; }
        }
#pragma unroll
        for (int u = 0; u < kStageU; ++u)
          if (t + 32 * u < n * n) As[off[u]] = v[u];
      }
    }
    for (int i = lane; i < n; i += 32) bs[i] = PTC ? -F[r * n + i] : b[r * n + i];
    __syncwarp();

    // Blocked right-looking elimination, kNB pivots per pass over the trailing matrix: every trailing entry
    // is read and written once per kNB pivots instead of once per pivot (shared-memory traffic is what bounds
    // this kernel), with the kNB multipliers of a lane's rows held in registers.
    int fail = 0;
    for (int k0 = 0; k0 < n && !fail; k0 += kNB) {
      const int nb = min(kNB, n - k0);
      // ---- panel: columns k0 .. k0+nb-1, one pivot at a time; row exchanges span the whole row
      double* colk = As + (size_t)k0 * ld;
      for (int k = k0; k < k0 + nb; ++k, colk += ld) {
        // pivot: largest |a_ik| over rows i >= k, the smallest i on ties.  |a| as an integer is ordered like
        // the double, so the warp arg-max is three REDUX steps (high word, low word among the ties, row
        // index among those) instead of five shuffle rounds.
        double best = -1.0;
        int p = n;
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr) {
          const int i = lane + 32 * rr;
          if (i >= k && i < n) {
            const double v = fabs(colk[i]);
            if (v > best) { best = v; p = i; }
          }
        }
        const unsigned bhi = best >= 0.0 ? (unsigned)__double2hiint(best) : 0u;
        const unsigned blo = best >= 0.0 ? (unsigned)__double2loint(best) : 0u;
        const unsigned mhi = __reduce_max_sync(kFull, bhi);
        const unsigned mlo = __reduce_max_sync(kFull, (best >= 0.0 && bhi == mhi) ? blo : 0u);
        p = (int)__reduce_min_sync(kFull, (best >= 0.0 && bhi == mhi && blo == mlo) ? (unsigned)p : 0xffffffffu);
        best = __hiloint2double((int)mhi, (int)mlo);
        if (!(best > 0.0) || p >= n) {   // zero (or NaN) pivot column
          fail = k + 1;
          break;
        }
        if (p != k) {
          double* pj = As + lane * ld;
          for (int j = lane; j < n; j += 32, pj += 32 * ld) {
            const double u = pj[k];
            pj[k] = pj[p];
            pj[p] = u;
          }
          if (lane == 0) {
            const double u = bs[k];
            bs[k] = bs[p];
            bs[p] = u;
          }
        }
        __syncwarp();
        const double rinv = 1.0 / colk[k];   // one division per pivot: multipliers and the back substitution use it
        const double bk = bs[k];
        if (lane == 0) dinv[k] = rinv;
        double l[RPL];
        bool mine[RPL];
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr) {
          const int i = lane + 32 * rr;
          mine[rr] = i > k && i < n;
          l[rr] = 0.0;
          if (mine[rr]) {
            l[rr] = colk[i] * rinv;
            colk[i] = l[rr];
            bs[i] = fma(-l[rr], bk, bs[i]);
          }
        }
        // the remaining columns of the panel (at most kNB - 1)
        const double* pk = colk + ld + k;
        double* pl = colk + ld + lane;
        for (int j = k + 1; j < k0 + nb; ++j, pk += ld, pl += ld) {
          const double akj = *pk;
#pragma unroll
          for (int rr = 0; rr < RPL; ++rr)
            if (mine[rr]) pl[32 * rr] = fma(-l[rr], akj, pl[32 * rr]);
        }
        __syncwarp();
      }
      if (fail) break;
      const int jt = k0 + nb;   // first trailing column
      if (jt >= n) break;
      // ---- U12: the pivot rows of the trailing columns, forward substitution with the unit-lower panel
      // block; lanes over columns (a column's nb entries are contiguous, columns an odd stride apart)
      for (int j = jt + lane; j < n; j += 32) {
        double* cj = As + (size_t)j * ld + k0;
        double u[kNB];
#pragma unroll
        for (int t = 0; t < kNB; ++t) u[t] = t < nb ? cj[t] : 0.0;
#pragma unroll
        for (int t = 1; t < kNB; ++t) {
          if (t < nb) {
#pragma unroll
            for (int s2 = 0; s2 < t; ++s2) u[t] = fma(-As[(size_t)(k0 + s2) * ld + k0 + t], u[s2], u[t]);
            cj[t] = u[t];
          }
        }
      }
      __syncwarp();
      // ---- A22 -= L21 U12: lanes over rows, the nb multipliers of each row in registers, two columns per trip
      double lm[RPL][kNB];
      bool below[RPL];
#pragma unroll
      for (int rr = 0; rr < RPL; ++rr) {
        const int i = lane + 32 * rr;
        below[rr] = i >= jt && i < n;
#pragma unroll
        for (int t = 0; t < kNB; ++t) lm[rr][t] = (below[rr] && t < nb) ? As[(size_t)(k0 + t) * ld + i] : 0.0;
      }
      double* cu = As + (size_t)jt * ld + k0;     // U12 entries of the current column
      double* cl = As + (size_t)jt * ld + lane;   // this lane's rows of the current column
      int j = jt;
      for (; j + 2 <= n; j += 2, cu += 2 * ld, cl += 2 * ld) {
        double u0[kNB], u1[kNB], a0[RPL], a1[RPL];
#pragma unroll
        for (int t = 0; t < kNB; ++t) {
          u0[t] = cu[t];          // entries beyond nb belong to other rows; their multipliers are 0
          u1[t] = cu[ld + t];
        }
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr) {
          a0[rr] = below[rr] ? cl[32 * rr] : 0.0;
          a1[rr] = below[rr] ? cl[ld + 32 * rr] : 0.0;
        }
#pragma unroll
        for (int t = 0; t < kNB; ++t)
#pragma unroll
          for (int rr = 0; rr < RPL; ++rr) {
            a0[rr] = fma(-lm[rr][t], u0[t], a0[rr]);
            a1[rr] = fma(-lm[rr][t], u1[t], a1[rr]);
          }
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr) {
          if (below[rr]) {
            cl[32 * rr] = a0[rr];
            cl[ld + 32 * rr] = a1[rr];
          }
        }
      }
      if (j < n) {
        double a0[RPL];
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr) a0[rr] = below[rr] ? cl[32 * rr] : 0.0;
#pragma unroll
        for (int t = 0; t < kNB; ++t) {
          const double ut = cu[t];
#pragma unroll
          for (int rr = 0; rr < RPL; ++rr) a0[rr] = fma(-lm[rr][t], ut, a0[rr]);
        }
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr)
          if (below[rr]) cl[32 * rr] = a0[rr];
      }
      __syncwarp();
    }
    if (!fail) {
      // back substitution, column oriented: x_i = b_i / u_ii, then b_r -= u_ri x_i for r < i
      const double* coli = As + (size_t)(n - 1) * ld;
      for (int i = n - 1; i >= 0; --i, coli -= ld) {
        const double xi = bs[i] * dinv[i];
        __syncwarp();
        if (lane == 0) bs[i] = xi;
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr) {
          const int rw = lane + 32 * rr;
          if (rw < i) bs[rw] = fma(-coli[rw], xi, bs[rw]);
        }
        __syncwarp();
      }
      for (int i = lane; i < n; i += 32) b[r * n + i] = bs[i];
    }
    if (lane == 0) info[r] = fail;
    __syncwarp();
  }
}

cudaError_t launch_lu_solve(int64_t N, int n, const double* A, double* b, int32_t* info, int n_sm, size_t smem_optin,
                            cudaStream_t st, const double* F, const double* dt, const int32_t* skip_count) {
  const int ld = n | 1;
  const int sys_doubles = n * ld + 2 * n + (n & 1);   // matrix, right-hand side, pivot reciprocals; even
  const size_t per_sys = (size_t)sys_doubles * 8;
  if (per_sys > smem_optin) return cudaErrorInvalidConfiguration;
  // systems (warps) per CTA: the count, up to 4, that packs the most systems into one SM's shared memory
  const size_t sm_total = smem_optin + 1024;
  int wpc = 1, best_sys = 0;
  for (int c = 1; c <= 4; ++c) {
    if (c * per_sys > smem_optin) break;
    const int sys = (int)(sm_total / (c * per_sys + 1024)) * c;
    if (sys >= best_sys) { best_sys = sys; wpc = c; }
  }
  const size_t smem = per_sys * wpc;
  const int rpl = (n + 31) / 32;
  int64_t ctas = (N + wpc - 1) / wpc;
  const int64_t cap = (int64_t)n_sm * (best_sys / wpc);   // persistent: every CTA strides over the systems
  if (ctas > cap) ctas = cap;
#define PSR_LU(RPL_)                                                                                         \
  if (rpl <= RPL_) {                                                                                         \
    auto kern = dt ? lu_solve_kernel<RPL_, true> : lu_solve_kernel<RPL_, false>;                             \
    static bool raised[2] = {false, false};   /* dynamic shared-memory limit: once per kernel instance */    \
    if (!raised[dt ? 1 : 0]) {                                                                               \
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_optin); \
      if (e != cudaSuccess) return e;                                                                        \
      raised[dt ? 1 : 0] = true;                                                                             \
    }                                                                                                        \
    kern<<<(int)ctas, wpc * 32, smem, st>>>(N, n, A, b, info, sys_doubles, F, dt, skip_count);               \
    return cudaGetLastError();                                                                               \
  }
  PSR_LU(1) PSR_LU(2) PSR_LU(4) PSR_LU(6)
#undef PSR_LU
  return cudaErrorInvalidConfiguration;
}

}  // namespace psr
