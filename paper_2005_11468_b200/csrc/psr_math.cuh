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

// Constants.  A DFMA immediate supplies only the high 32 bits of a double, so every constant whose low
// word can be zero without hurting the result is chosen that way and costs no instruction:
//   kMagic = 1.5 * 2^52 (exact); k32InvLn2 only picks the integer n, so 21 bits do (|r| grows by < 3 %);
//   kLn2o32Hi has 21 significant bits (n * hi exact for |n| < 2^32), kLn2o32Lo carries the rest in full;
//   1/720 and 1/120 truncated to 21 bits move the result by < 1e-19 relative.
// 1/24, 1/6 and kLn2o32Lo need all 64 bits (two moves each, shared by the N exps of a lock-step batch).
constexpr double kMagic = 6755399441055744.0;
constexpr double k32InvLn2 = 0x1.7154700000000p+5;
constexpr double kLn2o32Hi = 0x1.62e4300000000p-6;
constexpr double kLn2o32Lo = -5.952044687368025e-11;   // ln2/32 - kLn2o32Hi
constexpr double kC6 = 0x1.6c16c00000000p-10;           // ~1/720
constexpr double kC5 = 0x1.1111100000000p-7;            // ~1/120
constexpr double kC4 = 1.0 / 24.0, kC3 = 1.0 / 6.0;

struct ExpTab {  // this lane's entry 2^(lane/32)
  int hi, lo;
};

__device__ __forceinline__ ExpTab exp_tab_load(const double* __restrict__ tab_global) {
  const double v = tab_global[threadIdx.x & 31];
  return ExpTab{__double2hiint(v), __double2loint(v)};
}

// all 32 lanes of the warp must call this together
__device__ __forceinline__ double exp_core(double x, const ExpTab& tab) {
  const double t = fma(x, k32InvLn2, kMagic);
  const int n = __double2loint(t);
  const double nd = t - kMagic;
  const int thi = __shfl_sync(kFullMask, tab.hi, n);       // source lane = n mod 32
  const int tlo = __shfl_sync(kFullMask, tab.lo, n);
  double r = fma(nd, -kLn2o32Hi, x);
  r = fma(nd, -kLn2o32Lo, r);
  double s = fma(r, kC6, kC5);
  s = fma(s, r, kC4);
  s = fma(s, r, kC3);
  s = fma(s, r, 0.5);
  s = fma(s, r, 1.0);
  const double tj = __hiloint2double(thi + ((n >> 5) << 20), tlo);   // 2^m * 2^(j/32)
  return fma(tj, s * r, tj);
}

// N independent exps advanced in lock step, so that the FP64 pipe always has N dependency chains to
// pick from (the one-at-a-time form leaves the scheduler a single 11-deep chain per call).
template <int N>
__device__ __forceinline__ void exp_core_n(const double (&x)[N], double (&y)[N], const ExpTab& tab) {
  double t[N], r[N], s[N], tj[N];
  int n[N];
#pragma unroll
  for (int i = 0; i < N; ++i) t[i] = fma(x[i], k32InvLn2, kMagic);
#pragma unroll
  for (int i = 0; i < N; ++i) {
    n[i] = __double2loint(t[i]);
    t[i] = t[i] - kMagic;
  }
  // the table entries are requested now and first touched after the polynomial: a shuffle takes about as
  // long as three dependent DFMAs, and a consumer placed right behind it stalls the warp for that time
  int thi[N], tlo[N];
#pragma unroll
  for (int i = 0; i < N; ++i) {
    thi[i] = __shfl_sync(kFullMask, tab.hi, n[i]);
    tlo[i] = __shfl_sync(kFullMask, tab.lo, n[i]);
  }
#pragma unroll
  for (int i = 0; i < N; ++i) r[i] = fma(t[i], -kLn2o32Hi, x[i]);
#pragma unroll
  for (int i = 0; i < N; ++i) r[i] = fma(t[i], -kLn2o32Lo, r[i]);
#pragma unroll
  for (int i = 0; i < N; ++i) s[i] = fma(r[i], kC6, kC5);
#pragma unroll
  for (int i = 0; i < N; ++i) s[i] = fma(s[i], r[i], kC4);
#pragma unroll
  for (int i = 0; i < N; ++i) s[i] = fma(s[i], r[i], kC3);
#pragma unroll
  for (int i = 0; i < N; ++i) s[i] = fma(s[i], r[i], 0.5);
#pragma unroll
  for (int i = 0; i < N; ++i) s[i] = fma(s[i], r[i], 1.0);
#pragma unroll
  for (int i = 0; i < N; ++i) s[i] = s[i] * r[i];
#pragma unroll
  for (int i = 0; i < N; ++i) {
    // 2^m * 2^(j/32): m = n >> 5 added to the exponent field.  The asm keeps the assembler from moving the
    // integer work back up to the shuffles.
    int hi;
    asm volatile("mad.lo.s32 %0, %1, 32768, %2;" : "=r"(hi) : "r"(n[i] & ~31), "r"(thi[i]));
    tj[i] = __hiloint2double(hi, tlo[i]);
  }
#pragma unroll
  for (int i = 0; i < N; ++i) y[i] = fma(tj[i], s[i], tj[i]);
}

// |x| < 700 decided on the high word read as a float (one FSETP with |.|): false for NaN and Inf too
__device__ __forceinline__ bool exp_in_range(double a) {
  return fabsf(__int_as_float(__double2hiint(a))) < __int_as_float(0x4085e000);
}

// Deferred form of the same test: m = max(m, |high word of a| read as a float), NaN-propagating (the high
// word of a double NaN or Inf reads as a float NaN), then one compare per lane at the end of a phase.
__device__ __forceinline__ float exp_arg_max(float m, double a) {
  float r;
  asm("max.NaN.f32 %0, %1, %2;" : "=f"(r) : "f"(fabsf(__int_as_float(__double2hiint(a)))), "f"(m));
  return r;
}
__device__ __forceinline__ bool exp_max_in_range(float m) { return m < __int_as_float(0x4085e000); }

// all 32 lanes of the warp must call this together
__device__ __forceinline__ double exp_fast(double x, const ExpTab& tab) {
  return __all_sync(kFullMask, exp_in_range(x)) ? exp_core(x, tab) : exp(x);
}

// N exps behind ONE warp vote: the table form if every argument of every lane is in range, else the
// library exp (NaN, Inf, overflow, gradual underflow keep their IEEE results).  All 32 lanes call together.
template <int N>
__device__ __forceinline__ void exp_fast_n(const double (&x)[N], double (&y)[N], const ExpTab& tab) {
  bool ok = true;
#pragma unroll
  for (int i = 0; i < N; ++i) ok = ok && exp_in_range(x[i]);
  if (__all_sync(kFullMask, ok)) {
    exp_core_n<N>(x, y, tab);
  } else {
#pragma unroll
    for (int i = 0; i < N; ++i) y[i] = exp(x[i]);
  }
}

}  // namespace psr
#endif
