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

// RPL: rows per lane (n <= 32 * RPL)
template <int RPL>
__global__ void __launch_bounds__(128) lu_solve_kernel(int64_t N, int n, const double* __restrict__ A,
                                                       double* __restrict__ b, int32_t* __restrict__ info,
                                                       int sys_doubles) {
  extern __shared__ __align__(16) double sm[];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, wpc = blockDim.x >> 5;
  const int ld = n | 1;
  double* As = sm + (size_t)w * sys_doubles;   // [n][ld], entry (i, j) at As[j*ld + i]
  double* bs = As + (size_t)n * ld;            // [n]

  for (int64_t r = (int64_t)blockIdx.x * wpc + w; r < N; r += (int64_t)gridDim.x * wpc) {
    const double* Ar = A + (size_t)r * n * n;
    for (int t = lane; t < n * n; t += 32) {
      const int j = t / n, i = t - j * n;
      As[j * ld + i] = Ar[t];
    }
    for (int i = lane; i < n; i += 32) bs[i] = b[r * n + i];
    __syncwarp();

    int fail = 0;
    for (int k = 0; k < n; ++k) {
      // pivot: largest |a_ik| over rows i >= k, the smallest i on ties
      double best = -1.0;
      int p = k;
#pragma unroll
      for (int rr = 0; rr < RPL; ++rr) {
        const int i = lane + 32 * rr;
        if (i >= k && i < n) {
          const double v = fabs(As[k * ld + i]);
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
        for (int j = lane; j < n; j += 32) {
          const double u = As[j * ld + k];
          As[j * ld + k] = As[j * ld + p];
          As[j * ld + p] = u;
        }
        if (lane == 0) {
          const double u = bs[k];
          bs[k] = bs[p];
          bs[p] = u;
        }
      }
      __syncwarp();
      const double piv = As[k * ld + k];
      const double bk = bs[k];
      double l[RPL];
#pragma unroll
      for (int rr = 0; rr < RPL; ++rr) {
        const int i = lane + 32 * rr;
        l[rr] = 0.0;
        if (i > k && i < n) {
          l[rr] = As[k * ld + i] / piv;
          As[k * ld + i] = l[rr];
          bs[i] = fma(-l[rr], bk, bs[i]);
        }
      }
      for (int j = k + 1; j < n; ++j) {
        const double akj = As[j * ld + k];   // broadcast
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr) {
          const int i = lane + 32 * rr;
          if (i > k && i < n) As[j * ld + i] = fma(-l[rr], akj, As[j * ld + i]);
        }
      }
      __syncwarp();
    }
    if (!fail) {
      // back substitution, column oriented: x_i = b_i / u_ii, then b_r -= u_ri x_i for r < i
      for (int i = n - 1; i >= 0; --i) {
        const double xi = bs[i] / As[i * ld + i];
        __syncwarp();
        if (lane == 0) bs[i] = xi;
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr) {
          const int rw = lane + 32 * rr;
          if (rw < i) bs[rw] = fma(-As[i * ld + rw], xi, bs[rw]);
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
  int wpc = (int)(smem_optin / per_sys);
  if (wpc < 1) return cudaErrorInvalidConfiguration;
  if (wpc > 4) wpc = 4;
  const size_t smem = per_sys * wpc;
  const int rpl = (n + 31) / 32;
  int64_t ctas = (N + wpc - 1) / wpc;
  const int64_t cap = (int64_t)n_sm * 8;   // persistent: every CTA strides over the systems
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
