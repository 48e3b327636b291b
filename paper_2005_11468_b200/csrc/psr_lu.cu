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

// RPL: rows per lane (n <= 32 * RPL).  The column stride ld = n | 1 is a run-time value, so the update walks
// the columns with two running pointers (pivot-row entry, this lane's rows) instead of forming j*ld + i for
// every access (that index arithmetic cost more instructions than the elimination itself: 51 k
// instructions per 54 x 54 system, 4 k of them FMA, in the first version).
template <int RPL>
__global__ void __launch_bounds__(128) lu_solve_kernel(int64_t N, int n, const double* __restrict__ A,
                                                       double* __restrict__ b, int32_t* __restrict__ info,
                                                       int sys_doubles) {
  extern __shared__ __align__(16) double sm[];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, wpc = blockDim.x >> 5;
  const int ld = n | 1;
  double* As = sm + (size_t)w * sys_doubles;   // entry (i, j) at As[j*ld + i]
  double* bs = As + (size_t)n * ld;            // [n]

  for (int64_t r = (int64_t)blockIdx.x * wpc + w; r < N; r += (int64_t)gridDim.x * wpc) {
    const double* Ar = A + (size_t)r * n * n;
    {
      // column-major stream, 32 consecutive entries per trip, 4 trips in flight; (i, j) tracked without a divide
      int i = lane, j = 0;
      while (i >= n) { i -= n; ++j; }
      for (int t = lane; t < n * n; t += 128) {
        double v[4];
        int off[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          off[u] = j * ld + i;
          v[u] = (t + 32 * u < n * n) ? Ar[t + 32 * u] : 0.0;
          i += 32;
          while (i >= n) { i -= n; ++j; }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)
          if (t + 32 * u < n * n) As[off[u]] = v[u];
      }
    }
    for (int i = lane; i < n; i += 32) bs[i] = b[r * n + i];
    __syncwarp();

    int fail = 0;
    double* colk = As;   // column k
    for (int k = 0; k < n; ++k, colk += ld) {
      // pivot: largest |a_ik| over rows i >= k, the smallest i on ties
      double best = -1.0;
      int p = k;
#pragma unroll
      for (int rr = 0; rr < RPL; ++rr) {
        const int i = lane + 32 * rr;
        if (i >= k && i < n) {
          const double v = fabs(colk[i]);
          if (v > best) { best = v; p = i; }
        }
      }
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) {
        const double ob = __shfl_xor_sync(kFull, best, off);
        const int op = __shfl_xor_sync(kFull, p, off);
        if (ob > best || (ob == best && op < p)) { best = ob; p = op; }
      }
      if (!(best > 0.0)) {   // zero (or NaN) pivot column
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
      const double piv = colk[k];
      const double bk = bs[k];
      double l[RPL];
      bool mine[RPL];
#pragma unroll
      for (int rr = 0; rr < RPL; ++rr) {
        const int i = lane + 32 * rr;
        mine[rr] = i > k && i < n;
        l[rr] = 0.0;
        if (mine[rr]) {
          l[rr] = colk[i] / piv;
          colk[i] = l[rr];
          bs[i] = fma(-l[rr], bk, bs[i]);
        }
      }
      // rank-1 update of the trailing columns, kCB columns per trip: all loads of a trip are issued before
      // its first store (stores to As would otherwise order every later load behind them)
      constexpr int kCB = RPL <= 2 ? 8 : 4;
      const double* pk = colk + ld + k;      // pivot-row entry of the current column
      double* pl = colk + ld + lane;         // this lane's first row of the current column
      int j0 = k + 1;
      for (; j0 + kCB <= n; j0 += kCB) {
        double akj[kCB], av[kCB][RPL];
        const double* qk = pk;
        const double* ql = pl;
#pragma unroll
        for (int u = 0; u < kCB; ++u, qk += ld, ql += ld) {
          akj[u] = *qk;   // broadcast
#pragma unroll
          for (int rr = 0; rr < RPL; ++rr) av[u][rr] = mine[rr] ? ql[32 * rr] : 0.0;
        }
#pragma unroll
        for (int u = 0; u < kCB; ++u, pk += ld, pl += ld)
#pragma unroll
          for (int rr = 0; rr < RPL; ++rr)
            if (mine[rr]) pl[32 * rr] = fma(-l[rr], akj[u], av[u][rr]);
      }
      for (; j0 < n; ++j0, pk += ld, pl += ld) {
        const double akj = *pk;
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr)
          if (mine[rr]) pl[32 * rr] = fma(-l[rr], akj, pl[32 * rr]);
      }
      __syncwarp();
    }
    if (!fail) {
      // back substitution, column oriented: x_i = b_i / u_ii, then b_r -= u_ri x_i for r < i
      const double* coli = As + (size_t)(n - 1) * ld;
      for (int i = n - 1; i >= 0; --i, coli -= ld) {
        const double xi = bs[i] / coli[i];
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
                            cudaStream_t st) {
  const int ld = n | 1;
  const int sys_doubles = n * ld + ((n + 1) & ~1);
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
    cudaError_t e = cudaFuncSetAttribute(lu_solve_kernel<RPL_>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                         (int)smem);                                                         \
    if (e != cudaSuccess) return e;                                                                          \
    lu_solve_kernel<RPL_><<<(int)ctas, wpc * 32, smem, st>>>(N, n, A, b, info, sys_doubles);                 \
    return cudaGetLastError();                                                                               \
  }
  PSR_LU(1) PSR_LU(2) PSR_LU(4) PSR_LU(6)
#undef PSR_LU
  return cudaErrorInvalidConfiguration;
}

}  // namespace psr
