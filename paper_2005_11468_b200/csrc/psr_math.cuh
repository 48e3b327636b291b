// psr_math.cuh -- FP64 elementary functions sized for the rate kernels (internal to the library).
//
// Eq. 6 and Eq. 9 of the paper put one exp per rate constant on the hot path ("time consuming,
// specifically due to the exponential term").  CUDA's exp(double) costs ~21 FP64
// issue slots per call (measured).  exp_core is the table-driven form
//     x = (32 m + j) ln2/32 + r,  |r| <= ln2/64,   exp(x) = 2^m * 2^(j/32) * (1 + r + ... + r^6/720)
// with the 32-entry table 2^(j/32) held one entry per lane and read with two warp shuffles: a
// shared-memory table costs ~7 crossbar cycles per lookup from bank conflicts (measured), a shuffle
// costs one each.  11 FP64 instructions, no branch.  Truncation error r^7/5040 <= 3.5e-18; the tests
// pin the result at <= 4e-16 relative against 50-digit arithmetic.
// Valid while the result is a normal number: callers guard with exp_in_range (|x| < 700, which also
// routes NaN and Inf to the library exp so IEEE propagation is kept), decided per WARP because the
// shuffles need all 32 lanes.
#ifndef PSR_MATH_CUH_
#define PSR_MATH_CUH_
#include <cuda_runtime.h>
#include <stdint.h>

namespace psr {

constexpr int kExpTabN = 32;
constexpr unsigned kFullMask = 0xffffffffu;

struct ExpTab {  // this lane's entry 2^(lane/32)
  int hi, lo;
};

__device__ __forceinline__ ExpTab exp_tab_load(const double* __restrict__ tab_global) {
  const double v = tab_global[threadIdx.x & 31];
  return ExpTab{__double2hiint(v), __double2loint(v)};
}

// all 32 lanes of the warp must call this together
__device__ __forceinline__ double exp_core(double x, const ExpTab& tab) {
  constexpr double kMagic = 6755399441055744.0;            // 1.5 * 2^52: round-to-nearest-integer shifter
  constexpr double k32InvLn2 = 46.16624130844683;          // 32 / ln 2
  constexpr double kLn2o32Hi = 0x1.62e42ff000000p-6;       // ln2/32, 32 significant bits (n * hi exact)
  constexpr double kLn2o32Lo = -1.312785960212839e-12;     // ln2/32 - hi
  const double t = fma(x, k32InvLn2, kMagic);
  const int n = __double2loint(t);
  const double nd = t - kMagic;
  const int thi = __shfl_sync(kFullMask, tab.hi, n);       // source lane = n mod 32
  const int tlo = __shfl_sync(kFullMask, tab.lo, n);
  double r = fma(nd, -kLn2o32Hi, x);
  r = fma(nd, -kLn2o32Lo, r);
  double s = fma(r, 1.0 / 720.0, 1.0 / 120.0);
  s = fma(s, r, 1.0 / 24.0);
  s = fma(s, r, 1.0 / 6.0);
  s = fma(s, r, 0.5);
  s = fma(s, r, 1.0);
  const double tj = __hiloint2double(thi + ((n >> 5) << 20), tlo);   // 2^m * 2^(j/32)
  return fma(tj, s * r, tj);
}

// |x| < 700 decided on the high word read as a float (one FSETP with |.|): false for NaN and Inf too
__device__ __forceinline__ bool exp_in_range(double a) {
  return fabsf(__int_as_float(__double2hiint(a))) < __int_as_float(0x4085e000);
}

// all 32 lanes of the warp must call this together
__device__ __forceinline__ double exp_fast(double x, const ExpTab& tab) {
  return __all_sync(kFullMask, exp_in_range(x)) ? exp_core(x, tab) : exp(x);
}

}  // namespace psr
#endif
