// psr_solve.cu -- per-reactor bookkeeping of the hybrid Newton / pseudo-transient solver (psr_solve_hybrid,
// SURVEY.md 8(f) NEXT-4).  The residual, the finite-difference Jacobian and the linear solves are the
// library's own calls; what is here is the part between them: take or refuse the trial estimate x + dx, test the
// Newton correction against the tolerances, switch a reactor between the Newton iteration and the pseudo-transient
// conditioning, adapt its pseudo-time step -- one warp per reactor, nothing returns to the host.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "../../include/psr.h"
#include "psr_ptx.cuh"
#include "psr_tables.h"

namespace psr {

constexpr unsigned kAll = 0xffffffffu;
enum : int32_t { kModeNewton = 0, kModePtc = 1, kModeDone = 2 };

// One step of every reactor's state machine (readings g22-g25), after the solve of
// (I/dt_arg + J) dx = -F at the current estimate x = (T, Y).
__global__ void __launch_bounds__(256) hybrid_update_kernel(int64_t nb, int n, int64_t ld, psr_solve_opts o, double* __restrict__ T,
                                                            double* __restrict__ Y, const double* __restrict__ dx,
                                                            const int32_t* __restrict__ info, double* __restrict__ dt_cur,
                                                            double* __restrict__ dt_arg, int32_t* __restrict__ mode,
                                                            int32_t* __restrict__ it, int32_t* __restrict__ status,
                                                            int32_t* __restrict__ n_newton, int32_t* __restrict__ n_ptc,
                                                            int32_t* __restrict__ n_active) {
  const int lane = threadIdx.x & 31;
  const int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (r >= nb) return;
  if (*reinterpret_cast<volatile int32_t*>(n_active) == 0) return;   // every reactor finished in an earlier round
  const int32_t md = mode[r];
  if (md == kModeDone) return;
  // trial x' = x + dx; admissible when the system solved to a finite dx and every mass fraction stays >= -y_floor
  bool ok = info[r] == 0;
  bool adm = true;
  double err = 0.0;
  for (int i = lane; i < n; i += 32) {
    const double d = dx[r * n + i];
    const double x = i == 0 ? T[r] : Y[(int64_t)(i - 1) * ld + r];
    ok = ok && isfinite(d);
    // |dx_i| / (atol + rtol |x_i|), operation by operation (no contraction: the test decides an integer)
    err = fmax(err, __ddiv_rn(fabs(d), __dadd_rn(o.atol, __dmul_rn(o.rtol, fabs(x)))));
    if (i > 0) adm = adm && (__dadd_rn(x, d) >= -o.y_floor);
  }
  ok = __all_sync(kAll, ok);
  adm = __all_sync(kAll, adm) && ok;
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) err = fmax(err, __shfl_xor_sync(kAll, err, s));
  int32_t k = it[r];
  double dtc = dt_cur[r];
  int32_t new_mode = md;
  bool take = false;
  if (md == kModeNewton) {
    if (lane == 0 && n_newton) n_newton[r] += 1;
    if (adm && err <= 1.0) {
      take = true;
      new_mode = kModeDone;
      if (lane == 0) status[r] = 0;
    } else if (adm) {
      take = true;
      if (++k >= o.max_newton) {   // the stage is over without convergence: condition the estimate
        new_mode = kModePtc;
        k = 0;
      }
    } else {
      new_mode = kModePtc;
      k = 0;
    }
  } else {
    if (lane == 0 && n_ptc) n_ptc[r] += 1;
    if (adm) {
      take = true;
      dtc = __dmul_rn(dtc, o.dt_grow);
    } else {
      dtc = __dmul_rn(dtc, o.dt_shrink);
    }
    if (++k >= o.max_ptc) {   // back to the Newton iteration from the conditioned estimate
      new_mode = kModeNewton;
      k = 0;
    }
  }
  if (take) {
    for (int i = lane; i < n; i += 32) {
      const double d = dx[r * n + i];
      if (i == 0) T[r] = __dadd_rn(T[r], d);
      else Y[(int64_t)(i - 1) * ld + r] = __dadd_rn(Y[(int64_t)(i - 1) * ld + r], d);
    }
  }
  if (lane == 0) {
    mode[r] = new_mode;
    it[r] = k;
    dt_cur[r] = dtc;
    // a finished reactor is marked with dt = NaN: the Jacobian and solve launches of the remaining rounds leave it
    // out (psr_jac.cu: tiles whose reactors have all finished; psr_lu.cu: its system), and n_active counts the rest
    dt_arg[r] = new_mode == kModeDone ? __longlong_as_double(0x7ff8000000000000LL) : new_mode == kModePtc ? dtc : INFINITY;
    if (new_mode == kModeDone) atomicSub(n_active, 1);
  }
}

cudaError_t launch_hybrid_update(int64_t nb, int n, int64_t ld, const psr_solve_opts& o, double* T, double* Y, const double* dx,
                                 const int32_t* info, double* dt_cur, double* dt_arg, int32_t* mode, int32_t* it, int32_t* status,
                                 int32_t* n_newton, int32_t* n_ptc, int32_t* n_active, cudaStream_t st) {
  hybrid_update_kernel<<<(unsigned)((nb * 32 + 255) / 256), 256, 0, st>>>(nb, n, ld, o, T, Y, dx, info, dt_cur, dt_arg, mode, it,
                                                                          status, n_newton, n_ptc, n_active);
  return cudaGetLastError();
}

// ------------------------------------------------------------------ compaction of the reactors still iterating
// psr_solve_hybrid works on a copy of the sub-batch's state in its workspace (HybridState, two of them).  Every few
// rounds the reactors are partitioned -- the ones still iterating first, in their order, the finished ones behind
// them -- into the other copy: finished reactors then fill whole tiles of 32, which the Jacobian kernel leaves out
// (psr_jac.cu), so that a round costs what the active reactors cost.  A reactor's arithmetic does not depend on its
// position, so its path is the same with or without the moves.

// rows of a state: T, P, tau, Tin, Y[0..K), Yin[0..K) (doubles, row stride ldw), then dt_cur, dt_arg, then the integers
__device__ __forceinline__ double* hs_row(const HybridState& s, int row, int K) {
  if (row == 0) return s.T;
  if (row == 1) return s.P;
  if (row == 2) return s.tau;
  if (row == 3) return s.Tin;
  if (row < 4 + K) return s.Y + (int64_t)(row - 4) * s.ldw;
  if (row < 4 + 2 * K) return s.Yin + (int64_t)(row - 4 - K) * s.ldw;
  return row == 4 + 2 * K ? s.dt_cur : s.dt_arg;
}

// the caller's arrays of the sub-batch into a state; bookkeeping initialised (grid.y: rows; the last row: integers)
__global__ void hybrid_gather_kernel(int64_t nb, int K, int64_t ld, const double* T, const double* P, const double* Y, const double* Tin,
                                     const double* Yin, const double* tau, HybridState s, psr_solve_opts o, int32_t* n_active) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int row = blockIdx.y;
  if (row == 0 && r == 0) *n_active = (int32_t)nb;
  if (r >= nb) return;
  if (row == 0) s.T[r] = T[r];
  else if (row == 1) s.P[r] = P[r];
  else if (row == 2) s.tau[r] = tau[r];
  else if (row == 3) { if (Tin) s.Tin[r] = Tin[r]; }
  else if (row < 4 + K) s.Y[(int64_t)(row - 4) * s.ldw + r] = Y[(int64_t)(row - 4) * ld + r];
  else if (row < 4 + 2 * K) s.Yin[(int64_t)(row - 4 - K) * s.ldw + r] = Yin[(int64_t)(row - 4 - K) * ld + r];
  else if (row == 4 + 2 * K) {
    s.dt_cur[r] = o.dt0;
    s.dt_arg[r] = INFINITY;   // Newton iteration: the pseudo-transient system without its shift
  } else {
    s.mode[r] = kModeNewton;
    s.it[r] = 0;
    s.status[r] = 1;
    s.nn[r] = 0;
    s.np[r] = 0;
    s.orig[r] = (int32_t)r;
  }
}

// destination of every reactor under the stable partition (active first); one CTA walks the sub-batch
__global__ void __launch_bounds__(1024) hybrid_scan_kernel(int64_t nb, const int32_t* __restrict__ mode, const int32_t* __restrict__ n_active,
                                                            int32_t* __restrict__ pos) {
  __shared__ int32_t wsum[32];
  __shared__ int32_t base_s;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int32_t n_act = *n_active;
  if (n_act == 0) return;   // nothing iterates any more: the order no longer matters
  if (threadIdx.x == 0) base_s = 0;
  __syncthreads();
  for (int64_t c0 = 0; c0 < nb; c0 += 1024) {
    const int64_t r = c0 + threadIdx.x;
    const int f = (r < nb && mode[r] != kModeDone) ? 1 : 0;
    int v = f;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int u = __shfl_up_sync(kAll, v, d);
      if (lane >= d) v += u;
    }
    if (lane == 31) wsum[w] = v;
    __syncthreads();
    if (w == 0) {
      int t = wsum[lane];
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int u = __shfl_up_sync(kAll, t, d);
        if (lane >= d) t += u;
      }
      wsum[lane] = t;   // inclusive sums of the warps' totals
    }
    __syncthreads();
    const int32_t base = base_s;
    const int32_t before = base + (w ? wsum[w - 1] : 0) + v - f;   // active reactors in front of r
    if (r < nb) pos[r] = f ? before : n_act + (int32_t)(r - before);
    __syncthreads();
    if (threadIdx.x == 0) base_s = base + wsum[31];
    __syncthreads();
  }
}

__global__ void hybrid_permute_kernel(int64_t nb, int K, HybridState src, HybridState dst, const int32_t* __restrict__ pos,
                                      const int32_t* __restrict__ n_active) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int row = blockIdx.y;
  if (r >= nb) return;
  // (nothing iterates any more: no partition was formed; the copy is still made, in place order, because the host side
  // swaps the two states on a fixed schedule)
  const int64_t d = *n_active == 0 ? r : (int64_t)pos[r];
  PSR_CHK(d >= 0 && d < nb, 601);   // the partition's destination is a reactor of the sub-batch
  if (row < 6 + 2 * K) {
    if (row == 3 && !src.Tin) return;
    hs_row(dst, row, K)[d] = hs_row(src, row, K)[r];
  } else {
    dst.mode[d] = src.mode[r];
    dst.it[d] = src.it[r];
    dst.status[d] = src.status[r];
    dst.nn[d] = src.nn[r];
    dst.np[d] = src.np[r];
    dst.orig[d] = src.orig[r];
  }
}

// the state back into the caller's arrays, every reactor at the index it came from
__global__ void hybrid_scatter_kernel(int64_t nb, int K, int64_t ld, HybridState s, double* T, double* Y, int32_t* status, int32_t* n_newton,
                                      int32_t* n_ptc) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int row = blockIdx.y;
  if (r >= nb) return;
  const int64_t o = s.orig[r];
  PSR_CHK(o >= 0 && o < nb, 602);   // the index a reactor came from
  if (row == 0) {
    T[o] = s.T[r];
    status[o] = s.status[r];
    if (n_newton) n_newton[o] = s.nn[r];
    if (n_ptc) n_ptc[o] = s.np[r];
  } else {
    Y[(int64_t)(row - 1) * ld + o] = s.Y[(int64_t)(row - 1) * s.ldw + r];
  }
}

PSR_CHK_TU_READER(chk_read_solve)

cudaError_t launch_hybrid_gather(int64_t nb, int K, int64_t ld, const double* T, const double* P, const double* Y, const double* Tin,
                                 const double* Yin, const double* tau, const HybridState& s, const psr_solve_opts& o, int32_t* n_active,
                                 cudaStream_t st) {
  const dim3 grid((unsigned)((nb + 255) / 256), (unsigned)(2 * K + 6));
  hybrid_gather_kernel<<<grid, 256, 0, st>>>(nb, K, ld, T, P, Y, Tin, Yin, tau, s, o, n_active);
  return cudaGetLastError();
}

cudaError_t launch_hybrid_compact(int64_t nb, int K, const HybridState& src, const HybridState& dst, int32_t* pos, const int32_t* n_active,
                                  cudaStream_t st) {
  hybrid_scan_kernel<<<1, 1024, 0, st>>>(nb, src.mode, n_active, pos);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const dim3 grid((unsigned)((nb + 255) / 256), (unsigned)(2 * K + 7));
  hybrid_permute_kernel<<<grid, 256, 0, st>>>(nb, K, src, dst, pos, n_active);
  return cudaGetLastError();
}

cudaError_t launch_hybrid_scatter(int64_t nb, int K, int64_t ld, const HybridState& s, double* T, double* Y, int32_t* status,
                                  int32_t* n_newton, int32_t* n_ptc, cudaStream_t st) {
  const dim3 grid((unsigned)((nb + 255) / 256), (unsigned)(K + 1));
  hybrid_scatter_kernel<<<grid, 256, 0, st>>>(nb, K, ld, s, T, Y, status, n_newton, n_ptc);
  return cudaGetLastError();
}

}  // namespace psr
