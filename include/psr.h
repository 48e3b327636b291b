/* psr.h -- C ABI of the B200 (sm_100a) batched perfectly-stirred-reactor chemistry library.
 *
 * The hot path of arxiv 2005.11468 ("Towards using GPGPU units for accelerating the batched PSR
 * calculations"): for N independent reactors that share one reaction mechanism, evaluate in FP64
 *   k_f (Eq. 6), K_p/K_c/k_r (Eq. 7-9), the rate of progress q
 *   (Eq. 5), the net production rate wdot (Eq. 4), the steady
 *   species residual of PAPER.md:33-35 Eq. 2, and the forward finite-difference Jacobian the Newton
 *   solver builds from it,
 * with NASA-7 thermo, third-body concentrations and Lindemann/Troe falloff in their CHEMKIN-II form
 * (BASELINE.json: north_star; DESIGN.md lists every reading of the paper).
 * Unlike the paper's three kernels + host loop, every step runs on the device and
 * nothing returns to the host between them.
 *
 * Units (CHEMKIN cgs): T [K], P [dyn/cm^2], Y mass fraction, tau [s], W [g/mol], Ea [cal/mol],
 * A in (mol/cm^3)^(1-order)/s, C [mol/cm^3], wdot and q [mol/cm^3/s], F [1/s].
 * Constants: R = 8.31446261815324e7 erg/mol/K, R_c = R/4.184e7 cal/mol/K, P_atm = 1.01325e6.
 *
 * Memory: mechanism descriptions are HOST pointers, borrowed for the call.  Reactor state and
 * outputs are DEVICE pointers owned by the caller, species-major struct-of-arrays: element
 * (species or reaction k, reactor r) is at base[k*ld + r] with ld >= N, 8-byte aligned.  The
 * library never frees or keeps caller arrays; inputs and outputs must not alias.
 *
 * Execution: every psr_eval_* / psr_fd_jacobian call enqueues kernels on `stream` (a cudaStream_t
 * cast to void*, NULL = legacy default stream) of the current device and returns without
 * synchronising.  Calls on one psr_mech from several host threads must be serialised by the caller.
 * Overlap on the GPU: a mechanism handle owns device scratch that some kernels use (the per-CTA rate
 * constants of the fused Jacobian kernel; the running sums of nu^T q of the large-mechanism evaluation
 * kernel, psr_mech_info: eval_acc_global = 1; the rate table of the generic Jacobian sweep).  Calls on ONE
 * handle that may run at the same time on the device -- different streams without an ordering between
 * them -- therefore race, except psr_eval_wdot / _residual / _kf_kr on a mechanism with eval_kernel = 1
 * (no scratch).  Order them (one stream, or events), or load the mechanism once per stream.
 *
 * Errors: every call returns a psr_status; on failure nothing was launched and psr_last_error()
 * describes why.  N == 0 is PSR_OK.  Non-finite or negative T/Y are not checked and propagate by
 * IEEE rules.  There is no CPU fallback: without a CUDA device the calls return PSR_ECUDA.
 */
#ifndef PSR_H_
#define PSR_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct psr_mech psr_mech; /* opaque; owns the device-side mechanism tables */

typedef enum {
  PSR_OK = 0,
  PSR_EINVAL = 1,       /* bad argument or malformed mechanism */
  PSR_EUNSUPPORTED = 2, /* valid but outside what the kernels handle (see psr_mech_load) */
  PSR_ENOMEM = 3,
  PSR_ECUDA = 4,        /* CUDA runtime error or no device */
  PSR_EIO = 5
} psr_status;

/* Reaction types (rtype) */
enum { PSR_RX_PLAIN = 0, PSR_RX_THREE_BODY = 1, PSR_RX_LINDEMANN = 2, PSR_RX_TROE = 3 };

/* Mechanism description: K species, I reactions.  All HOST pointers. */
typedef struct {
  int32_t n_species, n_reactions;
  const double* W;           /* [K]   molar mass, > 0 */
  const double* nasa;        /* [K][7] NASA-7 a0..a6, one temperature range:
                                cp/R = a0+a1 T+a2 T^2+a3 T^3+a4 T^4
                                h/RT = a0+a1 T/2+a2 T^2/3+a3 T^3/4+a4 T^4/5+a5/T
                                s/R  = a0 ln T+a1 T+a2 T^2/2+a3 T^3/3+a4 T^4/4+a6 */
  const double *A, *b, *Ea;  /* [I]   k = A T^b exp(-Ea/(R_c T)) (Eq. 6); the high-pressure limit for falloff.
                                Any finite A: negative (duplicate reactions) and zero are evaluated as defined */
  const uint8_t* rtype;      /* [I]   PSR_RX_* */
  const uint8_t* reversible; /* [I]   1: k_r = k_f/K_c (Eq. 7); 0: k_r = 0 */
  const int32_t *reac_ptr, *reac_sp, *reac_nu; /* CSR over reactions: reactant species and nu' in {1,2,3} */
  const int32_t *prod_ptr, *prod_sp, *prod_nu; /* products and nu'' in {1,2,3} */
  const int32_t *eff_ptr, *eff_sp;             /* CSR over reactions: third-body efficiencies (default 1) */
  const double* eff_val;
  const double *A0, *b0, *Ea0; /* [I]   low-pressure limit, read when rtype >= 2 */
  const double* troe;          /* [I][4] alpha, T***, T*, T**, read when rtype == 3; T***, T* != 0; the
                                  three-parameter form (no exp(-T** / T) term) is written T** = +inf */
} psr_mech_desc;

/* psr_mech_load: validate the description, build the device tables (per-reaction log-linear rate and
 * equilibrium coefficients, factor lists, per-chunk CSR of nu^T) and upload them once.
 * PSR_EINVAL: null pointers, K or I < 1, species index out of range, nu outside 1..3, W <= 0,
 *   non-monotone CSR pointers, unknown rtype, non-finite coefficients (A, b, Ea, A0, b0, Ea0, NASA, efficiencies;
 *   T** of a Troe reaction may be +inf), T*** or T* = 0.
 * PSR_EUNSUPPORTED: K > 512, more than 15 concentration factors on one side of a reaction, more
 *   than 65535 efficiency entries.  *out is set only on PSR_OK.  Synchronous. */
psr_status psr_mech_load(const psr_mech_desc* desc, psr_mech** out);
void psr_mech_free(psr_mech* mech);

/* Effective forward and reverse rate constants (reading g18): kf has falloff
 * applied but no [M] factor; kr = kf/K_c, 0 if irreversible.  kf, kr: [I][ldk], either may be NULL. */
psr_status psr_eval_kf_kr(const psr_mech* mech, int64_t N, const double* T, const double* P,
                          const double* Y, int64_t ld, double* kf, double* kr, int64_t ldk, void* stream);

/* Net production rates wdot [K][ld] (Eq. 4) and, if q != NULL, rates of progress q [I][ldq] (Eq. 5). */
psr_status psr_eval_wdot(const psr_mech* mech, int64_t N, const double* T, const double* P,
                         const double* Y, int64_t ld, double* wdot, double* q, int64_t ldq, void* stream);

/* PSR species residual F_i = (Y_i - Yin_i)/tau - wdot_i W_i/rho (steady Eq. 2 with tau = rho V/mdot),
 * F [K][ld]; wdot [K][ld] may be NULL. */
psr_status psr_eval_residual(const psr_mech* mech, int64_t N, const double* T, const double* P,
                             const double* Y, const double* Yin, const double* tau, int64_t ld,
                             double* F, double* wdot, void* stream);

/* Adiabatic PSR residual: the species rows F [K][ld] exactly as psr_eval_residual,
 * plus the energy row FT [N], the steady form of the paper's Eq. 3 with Qdot = 0 and
 * dP/dt = 0 written as a residual,
 *   F_T = -[ (1/tau) sum_i Yin_i (h_i(Tin) - h_i(T)) - (sum_i h_i(T) wdot_i W_i)/rho ] / cp_mix,
 * h_i [erg/g] = (h/RT)_i R T / W_i and cp_mix = sum_i Y_i (cp/R)_i R / W_i from the NASA-7 fits of the
 * mechanism.  Tin [N]: inlet temperature [K].  wdot [K][ld] may be NULL.  F_T is in K/s. */
psr_status psr_eval_residual_energy(const psr_mech* mech, int64_t N, const double* T, const double* P,
                                    const double* Y, const double* Tin, const double* Yin, const double* tau,
                                    int64_t ld, double* F, double* FT, double* wdot, void* stream);

/* Forward finite-difference Jacobian of the residual in x = (T, Y_1..Y_K) (
 * BASELINE.json configs[4]): delta_j = 1e-8 max(|x_j|, 1e-10), x'_j = fl(x_j + delta_j),
 * h_j = fl(x'_j - x_j), J_ij = (F_i(x') - F_i(x))/h_j.  Row 0 is the fixed-temperature equation
 * F_T = T - T_set with T_set the input T, so row 0 of J is e_0.
 * J: [N][(K+1)*(K+1)], column-major per reactor (entry (i,j) of reactor r at J[r*n*n + j*n + i],
 * n = K+1), directly usable by a batched LU.  F0: [N][K+1] residual at x (row 0 = 0), may be NULL.
 * Enqueues, per sub-batch of reactors, three launches on `stream`: the base residual (which also
 * tabulates the reaction factors that depend on T only), the T column, and the K species columns
 * (which reuse those factors: a Y perturbation leaves them unchanged; the result is bit-identical to
 * evaluating every column in full).  The rate table (and F0 when NULL is passed) live in a scratch
 * buffer owned by `mech`: calls of psr_fd_jacobian on ONE mechanism handle must therefore not run
 * concurrently on different streams.  The buffer grows (cudaMalloc, PSR_ENOMEM on failure) the first time a
 * larger N is seen, or ahead of time through psr_mech_reserve; an outgrown buffer stays allocated until
 * psr_mech_free, so work already enqueued and captured graphs that point at it stay valid.
 * Stream capture: the call allocates nothing when the scratch is large enough, and returns PSR_EINVAL
 * instead of allocating inside a capture -- call psr_mech_reserve(mech, N) before capturing. */
psr_status psr_fd_jacobian(const psr_mech* mech, int64_t N, const double* T, const double* P,
                           const double* Y, const double* Yin, const double* tau, int64_t ld,
                           double* J, double* F0, void* stream);

/* psr_fd_jacobian for callers that cannot let the library allocate (code under CUDA-graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same arguments, same result (the fused Jacobian kernel), but
 * the kernel's scratch is a static device array of 32 MiB inside the library -- held by every GPU that loads the
 * library until the process exits -- and the call performs no cudaMalloc, cudaFree or allocating library routine.
 * Limits: PSR_EUNSUPPORTED if the mechanism has more than PSR_NOALLOC_MAX_REACTIONS reactions (the array is sized for
 * that), or does not qualify for the fused kernel (more than 64 species, a falloff reaction with an efficiency list,
 * more than 3 concentration factors on a side, A <= 0): use psr_fd_jacobian then.  Any N: the launch uses as many CTAs,
 * up to one per SM, as have room for their scratch rows (n_reactions * 768 bytes each).
 * The array is shared by every call on the device and keeps the previous call's contents (none of which is read
 * before it is rewritten): calls that OVERLAP on the GPU -- different streams, or a graph replayed beside an eager
 * call -- race on it and must be serialised by the caller.  Asynchronous on `stream`. */
#define PSR_NOALLOC_MAX_REACTIONS 2048
psr_status psr_fd_jacobian_noalloc(const psr_mech* mech, int64_t N, const double* T, const double* P,
                                   const double* Y, const double* Yin, const double* tau, int64_t ld,
                                   double* J, double* F0, void* stream);

/* Sizes the scratch of psr_fd_jacobian / psr_fd_jacobian_energy for batches of up to N reactors (including the
 * internal F0 used when the caller passes none).  Synchronous (cudaMalloc); never shrinks. */
psr_status psr_mech_reserve(psr_mech* mech, int64_t N);

/* The same sweep for the adiabatic system (NEXT-1): row 0 of the residual is the energy row F_T of
 * psr_eval_residual_energy instead of T - T_set, so row 0 of J is dF_T/dx_j by the same forward
 * differences and F0[r][0] = F_T.  Tin [N]: inlet temperature.  Rows 1..K are bit-identical to
 * psr_fd_jacobian's. */
psr_status psr_fd_jacobian_energy(const psr_mech* mech, int64_t N, const double* T, const double* P,
                                  const double* Y, const double* Tin, const double* Yin, const double* tau,
                                  int64_t ld, double* J, double* F0, void* stream);

/* Newton step's linear solve ("The Jacobian matrix is decomposed into
 * lower and upper triangular matrices, and then a back-solving operation is carried out"): N independent
 * dense systems A x = b by Gaussian elimination with partial pivoting, one warp per system.
 * A: DEVICE [N][n*n], column-major per system (the layout psr_fd_jacobian writes), not modified.
 * b: DEVICE [N][n], right-hand side in, solution out (unchanged for a system that fails).
 * info: DEVICE [N], 0 on success, k+1 if the pivot column of step k (0-based) is exactly zero.
 * n <= 168 on a 227 KB shared-memory device (PSR_EUNSUPPORTED beyond).  The Newton update is the solve of
 * J dx = -F: pass b = -F0.  Asynchronous on `stream`. */
psr_status psr_lu_solve(int64_t N, int32_t n, const double* A, double* b, int32_t* info, void* stream);

/* One pseudo-transient (implicit Euler) step ("If the Newton algorithm
 * fails to converge, then the solution estimate is conditioned by a pseudo-transient time integration of the
 * governing equations"): the transient system dx/dt = -F(x) stepped by implicit Euler and linearised about x,
 *     (I/dt + J) dx = -F,
 * solved for N independent reactors by the elimination of psr_lu_solve (one warp per system; the shift and the
 * sign are applied while J is staged into shared memory, so J and F are read once and not modified).
 * J: DEVICE [N][n*n] column-major per system (psr_fd_jacobian's layout); F: DEVICE [N][n] residual at x (the F0 of
 * psr_fd_jacobian); dt: DEVICE [N] pseudo-time step per reactor, > 0 (+inf gives the Newton step exactly);
 * dx: DEVICE [N][n] out, must not alias F (unchanged for a system that fails); info: DEVICE [N] as in psr_lu_solve.
 * The paper gives neither the step-size control nor the Newton/pseudo-transient switching constants ("See
 * [5]"): choosing dt and accepting steps is the caller's.  Asynchronous on `stream`. */
psr_status psr_ptc_solve(int64_t N, int32_t n, const double* J, const double* F, const double* dt, double* dx,
                         int32_t* info, void* stream);

/* Hybrid Newton / pseudo-transient solve of the PSR equations for N reactors (PAPER.md:44:
 * "The hybrid approach consists of two steps: a steady state Newton iteration and a pseudo-transient time
 * integration.  If convergence is not achieved using the Newton iteration, the solution estimate is conditioned
 * using the time integration.  The process of switching ... continues until convergence is achieved, which is based
 * on ... absolute and relative tolerances").  The paper leaves the constants and the step-size rule to its ref. [5]:
 * they are the caller's, in psr_solve_opts, and the rules below are DESIGN.md readings g21-g25.
 *   Unknowns x = (T, Y_1..Y_K); equations: the residual of psr_fd_jacobian (row 0: T stays at its input value),
 *   or with Tin != NULL that of psr_fd_jacobian_energy (row 0: the energy row; T is solved for).
 *   Every iteration: F and the forward-difference Jacobian at x, the solve of (I/dt + J) dx = -F (no shift in a
 *   Newton iteration), the trial x' = x + dx.  A trial is admissible when the system solved without a zero pivot,
 *   dx is finite and every mass fraction of x' is >= -y_floor (+inf switches the bound off).
 *   Newton iteration: converged when max_i |dx_i| / (atol + rtol |x_i|) <= 1 (the correction is applied); an
 *   inadmissible trial, or max_newton admissible iterations without convergence, end the Newton stage and max_ptc
 *   pseudo-transient steps follow, after which Newton resumes.  Pseudo-transient step: dt starts at dt0 and
 *   persists; an admissible step is taken and dt *= dt_grow, otherwise x stays and dt *= dt_shrink.
 *   Every solve counts; after max_iter of them a reactor is left as it is with status 1.
 * T [N], Y [K][ld]: DEVICE, initial estimate in, solution estimate out.  P, Tin (or NULL), Yin [K][ld], tau: DEVICE
 * inputs.  status [N]: 0 converged, 1 not converged within max_iter; n_newton, n_ptc [N] (may be NULL): iterations
 * of each kind performed.  workspace: DEVICE scratch of workspace_bytes >= psr_solve_hybrid_workspace_bytes(mech, 1)
 * bytes; with less than psr_solve_hybrid_workspace_bytes(mech, N) the batch is solved in sub-batches one after the
 * other.  Runs entirely on the device: max_iter rounds of (psr_fd_jacobian, psr_ptc_solve, one bookkeeping kernel)
 * are enqueued on `stream` for every sub-batch, with no host synchronisation.  Converged reactors are left
 * untouched by the later rounds and are marked on the device: their linear systems, and the tiles of 32 reactors of
 * the fused Jacobian kernel that hold only finished reactors, are left out, and once a sub-batch has none left a round
 * is three empty launches -- max_iter is a budget, not a cost.  Capturable in a CUDA graph after
 * psr_mech_reserve(mech, N). */
typedef struct {
  double atol, rtol;
  int32_t max_iter, max_newton, max_ptc, reserved;
  double dt0, dt_grow, dt_shrink, y_floor;
} psr_solve_opts;
size_t psr_solve_hybrid_workspace_bytes(const psr_mech* mech, int64_t N);
psr_status psr_solve_hybrid(const psr_mech* mech, int64_t N, double* T, const double* P, double* Y, const double* Tin,
                            const double* Yin, const double* tau, int64_t ld, const psr_solve_opts* opts,
                            void* workspace, size_t workspace_bytes, int32_t* status, int32_t* n_newton,
                            int32_t* n_ptc, void* stream);

/* Thread-local description of the last failure on this thread; valid until its next psr_* call. */
const char* psr_last_error(void);

/* Introspection: n_species, n_reactions, reactors per tile, warps per CTA, reactions per chunk,
 * number of chunks, dynamic shared memory bytes, CTAs per SM the launch is sized for (those six: of the general fused
 * kernel), then which kernel the evaluation calls and psr_fd_jacobian take for this mechanism. */
typedef struct {
  int32_t n_species, n_reactions, tile, warps, chunk_reactions, n_chunks, smem_bytes, ctas_per_sm;
  int32_t n_sm, n_falloff, n_third_body, nnz_nu;
  int32_t eval_kernel;   /* kernel of psr_eval_wdot / _residual / _kf_kr: 0 general fused, 1 warp-specialised (resident
                            tables), 2 warp-specialised for large mechanisms (streamed parts) */
  int32_t eval_parts;    /* parts the mechanism is cut into for that kernel */
  int32_t eval_acc_global; /* kernel 2: where the running sums of nu^T q live: 0 shared memory, 1 an L2-resident scratch
                              of the handle, 2 tensor memory */
  int32_t jac_kernel;    /* psr_fd_jacobian: 1 fused Jacobian kernel, 0 generic sweep */
} psr_mech_info_t;
psr_status psr_mech_info(const psr_mech* mech, psr_mech_info_t* info);

/* Diagnostic switches of a loaded mechanism, used by the tests and by profiling to compare code paths that
 * must agree (they are not tuning knobs; default 0).  PSR_OPT_JAC_UNHOISTED: psr_fd_jacobian evaluates every
 * column in full instead of reusing the T-only factors of the base state (the two sweeps are bit-identical).
 * PSR_OPT_FUSED_ONLY: psr_eval_wdot / psr_eval_residual / psr_eval_kf_kr take the single fused kernel even
 * where the warp-specialised one applies.  PSR_OPT_JAC_GENERIC: psr_fd_jacobian takes the generic
 * three-launch sweep even where the fused Jacobian kernel applies.  PSR_OPT_NO_TMEM: the warp-specialised evaluation
 * kernels (eval_kernel = 1, 2) read every concentration from shared memory instead of taking the factors of the rate
 * products from their copy of the tile in tensor memory (bit-identical results).  Not thread-safe against concurrent calls on `mech`. */
enum { PSR_OPT_JAC_UNHOISTED = 1, PSR_OPT_FUSED_ONLY = 2, PSR_OPT_JAC_GENERIC = 3, PSR_OPT_NO_TMEM = 4 };
psr_status psr_mech_set_option(psr_mech* mech, int32_t option, int32_t value);

/* Diagnostic of the bounds-checked build (libpsr_b200_check.so: the same sources with -DPSR_CHECK; DESIGN.md 6.7 --
 * compute-sanitizer is refused on the GPU pool this library is developed on).  In that build the kernels assert, on
 * the device, every shared-memory offset they take from the mechanism tables and every global output index against
 * its bound.  Returns the number of failed assertions since the last call and resets it (*first_code, if not NULL:
 * the code of the first one, see the PSR_CHK sites in csrc/); selftest != 0 first trips one assertion on purpose
 * (code 999) so that a caller can tell "no failure" from "no checks".  Returns -1 in the product build, which carries
 * no checks, and -2 on a CUDA error.  Synchronises the device. */
int32_t psr_check_failures(int32_t selftest, int32_t* first_code);

/* FP64 pipe probes used for the roofline denominator: run `iters` dependent-
 * chain iterations of (kind 0) DFMA, (kind 1) exp, (kind 2) log on every SM and return the device
 * time in milliseconds and the number of operations executed per thread-lane in total.
 * Synchronous; returns PSR_ECUDA without a device. */
psr_status psr_probe_fp64(int kind, int iters, double* elapsed_ms, double* ops);

/* Diagnostic: evaluate the kernels' table-driven exp (csrc/psr_math.cuh) on n HOST values x -> y
 * (HOST).  Synchronous, default stream.  Used by the tests to pin its accuracy. */
psr_status psr_probe_exp_values(const psr_mech* mech, const double* x, double* y, int32_t n);

const char* psr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PSR_H_ */
