// psr_math.cuh -- FP64 elementary functions sized for the rate kernels (internal to the library).
//
// Eq. 6 and Eq. 9 of the paper put one exp per rate constant on the hot path ("time consuming,
// specifically due to the exponential term").  CUDA's exp(double) costs ~20 FP64
// issue slots plus a guarded slow path per call.  exp_fast is the table-driven form:
//     x = (64 m + j) ln2/64 + r,  |r| <= ln2/128,   exp(x) = 2^m * 2^(j/64) * (1 + r + ... + r^5/120)
// with 2^(j/64) read from a 64-entry table in shared memory: 10 FP64 instructions, no branch.
// Truncation error r^6/720 <= 3.5e-17; measured max error < 1 ulp-ish (tests pin it at 4e-16 rel).
// Valid while the result is a normal number; callers guard with exp_in_range (|x| < 700, which also
// routes NaN and Inf to the library exp so IEEE propagation is kept).
#ifndef PSR_MATH_CUH_
#define PSR_MATH_CUH_
#include <cuda_runtime.h>
#include <stdint.h>

namespace psr {

constexpr int kExpTabN = 64;

__device__ __forceinline__ double exp_core(double x, const double* __restrict__ tab) {
  constexpr double kMagic = 6755399441055744.0;            // 1.5 * 2^52: round-to-nearest-integer shifter
  constexpr double k64InvLn2 = 92.33248261689366;          // 64 / ln 2
  constexpr double kLn2o64Hi = 0x1.62e42ff000000p-7;       // ln2/64, 32 significant bits (n * hi exact)
  constexpr double kLn2o64Lo = -6.563929801064195e-13;     // ln2/64 - hi
  const double t = fma(x, k64InvLn2, kMagic);
  const int n = __double2loint(t);
  const double nd = t - kMagic;
  double r = fma(nd, -kLn2o64Hi, x);
  r = fma(nd, -kLn2o64Lo, r);
  const double tj = tab[n & (kExpTabN - 1)];
  double s = fma(r, 1.0 / 120.0, 1.0 / 24.0);
  s = fma(s, r, 1.0 / 6.0);
  s = fma(s, r, 0.5);
  s = fma(s, r, 1.0);
  const double y = fma(tj, s * r, tj);
  return __hiloint2double(__double2hiint(y) + ((n >> 6) << 20), __double2loint(y));
}

// true iff |a| < 512 and |b| < 512 at least, and never true when either is >= 700, NaN or Inf
__device__ __forceinline__ bool exp_in_range(double a, double b) {
  return (uint32_t)((__double2hiint(a) | __double2hiint(b)) & 0x7fffffff) < 0x4085e000u;
}
__device__ __forceinline__ bool exp_in_range(double a) {
  return (uint32_t)(__double2hiint(a) & 0x7fffffff) < 0x4085e000u;
}

__device__ __forceinline__ double exp_fast(double x, const double* __restrict__ tab) {
  return exp_in_range(x) ? exp_core(x, tab) : exp(x);
}

}  // namespace psr
#endif
