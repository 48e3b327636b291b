// psr_solve.cu -- per-reactor bookkeeping of the hybrid Newton / pseudo-transient solver (psr_solve_hybrid,
// SURVEY.md 8(f) NEXT-4).  The residual, the finite-difference Jacobian and the linear solves are the
// library's own calls; what is here is the part between them: take or refuse the trial estimate x + dx, test the
// Newton correction against the tolerances, switch a reactor between the Newton iteration and the pseudo-transient
// conditioning, adapt its pseudo-time step -- one warp per reactor, nothing returns to the host.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "../../include/psr.h"

namespace psr {

constexpr unsigned kAll = 0xffffffffu;
enum : int32_t { kModeNewton = 0, kModePtc = 1, kModeDone = 2 };

__global__ void hybrid_init_kernel(int64_t nb, psr_solve_opts o, double* dt_cur, double* dt_arg, int32_t* mode, int32_t* it,
                                   int32_t* status, int32_t* n_newton, int32_t* n_ptc, int32_t* n_active) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r == 0) *n_active = (int32_t)nb;   // reactors still iterating (the block is at most 2^31 - 1 reactors: checked by the caller)
  if (r >= nb) return;
  dt_cur[r] = o.dt0;
  dt_arg[r] = INFINITY;   // Newton iteration: the pseudo-transient system without its shift
  mode[r] = kModeNewton;
  it[r] = 0;
  status[r] = 1;
  if (n_newton) n_newton[r] = 0;
  if (n_ptc) n_ptc[r] = 0;
}

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

cudaError_t launch_hybrid_init(int64_t nb, const psr_solve_opts& o, double* dt_cur, double* dt_arg, int32_t* mode, int32_t* it,
                               int32_t* status, int32_t* n_newton, int32_t* n_ptc, int32_t* n_active, cudaStream_t st) {
  hybrid_init_kernel<<<(unsigned)((nb + 255) / 256), 256, 0, st>>>(nb, o, dt_cur, dt_arg, mode, it, status, n_newton, n_ptc, n_active);
  return cudaGetLastError();
}

cudaError_t launch_hybrid_update(int64_t nb, int n, int64_t ld, const psr_solve_opts& o, double* T, double* Y, const double* dx,
                                 const int32_t* info, double* dt_cur, double* dt_arg, int32_t* mode, int32_t* it, int32_t* status,
                                 int32_t* n_newton, int32_t* n_ptc, int32_t* n_active, cudaStream_t st) {
  hybrid_update_kernel<<<(unsigned)((nb * 32 + 255) / 256), 256, 0, st>>>(nb, n, ld, o, T, Y, dx, info, dt_cur, dt_arg, mode, it,
                                                                          status, n_newton, n_ptc, n_active);
  return cudaGetLastError();
}

}  // namespace psr
