// psr_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, scalar CPU implementation of the per-reactor chemical source term of
// arxiv 2005.11468 (section 3, Eq. 4-9; section 2, Eq. 2) with the CHEMKIN-II
// third-body / falloff forms and NASA-7 thermo that BASELINE.json: north_star adds.
// One reactor at a time, every step written as the paper / SURVEY.md section 8(c) O1..O11
// states it: no blocking, no fusion, no hoisting, pow() for T^b, species sums for Eq. 9.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may build, load or call this file.  It shares no code, header, table or constant with
// paper_2005_11468_b200/csrc (the CUDA path); its struct below is declared here on purpose.
//
// Templated on the real type: `double` is the oracle proper; `long double` (x87 80-bit) is
// the low-noise reference J* for the finite-difference Jacobian criterion.
//
// Pins (tests/test_oracle_pins.py, none of which call this file to get the expected value):
//   O1..O11 on the toy mechanism T3 against 17-digit values (tests/golden/t3_pins.json, values
//   printed in SURVEY.md 8(c), re-derived in the test with mpmath at 50 digits through an
//   independent dense-matrix formulation); Arrhenius hand values; NASA closed forms;
//   sum_i C_i = P/RT; K_c(R)*K_c(reverse R)=1; q sign flip under reactant/product swap;
//   k_f/k_r = K_c; sum_k W_k wdot_k = 0 on element-balanced mechanisms; Lindemann limits
//   k->k0[M], k->k_inf; Troe F=F_cent at log10 Pr=-c; sum_i F_i = (sum Y - sum Y_in)/tau;
//   Jacobian species rows of a Y column sum to 1/tau; J row 0 = e_0; the round-off scale S (roundoff_acc)
//   against its definition typed independently at 50 digits (tests/mp_dense.py roundoff_scale).
//   Energy row (NEXT-1): T3 values of h_i, C_p,mix and F_T from SURVEY.md 8(c), re-derived with mpmath;
//   F_T = 0 for an inert mechanism at T_in = T; linearity in 1/tau; enthalpy-balance identity.
//   Linear solve (NEXT-2): exact rational solutions of small integer systems, a system that needs a row
//   exchange, a singular system, LAPACK (numpy.linalg.solve) on random systems, backward error bound.
//   Pseudo-transient step (NEXT-4): exact rational solutions, the Newton limit dt -> inf, the explicit-Euler
//   limit dt -> 0 (dx -> -dt F), the scalar closed form dx = -F/(1/dt + J), LAPACK on the shifted matrix.
//   Hybrid solver (NEXT-4): an inert mechanism reaches Y = Y_in in one Newton step (to the forward-difference
//   accuracy) and stops after the confirming one; the closed-form steady state of A <=> B (a linear residual);
//   the root of 2A <=> B found with mpmath from the dense restatement, reached by Newton alone from a near guess
//   and through pseudo-transient stages from a guess whose Newton trial is inadmissible; exhausted budgets;
//   pseudo-transient steps with dt = 1e300 retrace the Newton iterates; the adiabatic inert reactor settles at
//   (T_in, Y_in).
//
// Units (paper silent; CHEMKIN cgs, reading g4): T [K], P [dyn/cm^2], C [mol/cm^3],
// rho [g/cm^3], W [g/mol], wdot [mol/cm^3/s], Ea [cal/mol].
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {
struct oracle_mech {  // all host pointers, borrowed
  int32_t n_species, n_reactions;
  const double* W;        // [K]
  const double* nasa;     // [K][7]
  const double *A, *b, *Ea;  // [I], Ea cal/mol
  const uint8_t* rtype;   // 0 plain, 1 three-body, 2 Lindemann, 3 Troe
  const uint8_t* reversible;
  const int32_t *reac_ptr, *reac_sp, *reac_nu;
  const int32_t *prod_ptr, *prod_sp, *prod_nu;
  const int32_t *eff_ptr, *eff_sp;
  const double* eff_val;
  const double *A0, *b0, *Ea0;
  const double* troe;     // [I][4] alpha, T3 (T***), T1 (T*), T2 (T**)
};
}

namespace {

// math in the template's precision
inline double m_exp(double x) { return std::exp(x); }
inline long double m_exp(long double x) { return expl(x); }
inline double m_log(double x) { return std::log(x); }
inline long double m_log(long double x) { return logl(x); }
inline double m_log10(double x) { return std::log10(x); }
inline long double m_log10(long double x) { return log10l(x); }
inline double m_pow(double x, double y) { return std::pow(x, y); }
inline long double m_pow(long double x, long double y) { return powl(x, y); }

template <class R> struct Consts {
  static constexpr R Rgas = (R)8.31446261815324e7L;                 // erg/mol/K
  static constexpr R Rcal = (R)8.31446261815324L / (R)4.184L;       // cal/mol/K
  static constexpr R Patm = (R)1.01325e6L;                          // dyn/cm^2
};

// per-reaction intermediates of one reactor (for the pins)
template <class R> struct RxnDetail {
  R kinf, k0, Pr, Fcent, F, M, Kp, Kc, kf, kr, q;
};

// O3: Eq. 6
template <class R> R arrhenius(R A, R b, R Ea, R T) {
  return A * m_pow(T, b) * m_exp(-Ea / (Consts<R>::Rcal * T));
}

// O2: NASA-7, single range
template <class R> void nasa7(const double* a, R T, R& cp_R, R& h_RT, R& s_R) {
  R a0 = a[0], a1 = a[1], a2 = a[2], a3 = a[3], a4 = a[4], a5 = a[5], a6 = a[6];
  R T2 = T * T, T3 = T2 * T, T4 = T3 * T;
  cp_R = a0 + a1 * T + a2 * T2 + a3 * T3 + a4 * T4;
  h_RT = a0 + a1 * T / 2 + a2 * T2 / 3 + a3 * T3 / 4 + a4 * T4 / 5 + a5 / T;
  s_R = a0 * m_log(T) + a1 * T + a2 * T2 / 2 + a3 * T3 / 3 + a4 * T4 / 4 + a6;
}

template <class R> R ipow(R x, int n) {  // nu in {1,2,3}: repeated multiply
  R r = x;
  for (int i = 1; i < n; ++i) r *= x;
  return r;
}

// One full evaluation O1..O10 for one reactor.  Y, Yin: K values (contiguous here).
// Outputs may be null.  Returns rho through *rho_out.
template <class R>
void eval_one(const oracle_mech& m, R T, R P, const R* Y, const R* Yin, R tau, R Tset,
              R* kf_out, R* kr_out, R* q_out, R* wdot_out, R* F_out /*K+1: F_T, F_1..F_K*/,
              RxnDetail<R>* det, R* C_out, R* rho_out) {
  const int K = m.n_species, I = m.n_reactions;
  const R Rg = Consts<R>::Rgas;
  // O1
  R sumYW = 0;
  for (int i = 0; i < K; ++i) sumYW += Y[i] / (R)m.W[i];
  R Wbar = (R)1 / sumYW;
  R rho = P * Wbar / (Rg * T);
  std::vector<R> C(K), h_RT(K), s_R(K), wdot(K, (R)0);
  R Ctot = 0;
  for (int i = 0; i < K; ++i) {
    C[i] = rho * Y[i] / (R)m.W[i];
    Ctot += C[i];
  }
  // O2
  for (int i = 0; i < K; ++i) {
    R cp;
    nasa7<R>(m.nasa + 7 * i, T, cp, h_RT[i], s_R[i]);
  }
  for (int k = 0; k < I; ++k) {
    // O3
    R kinf = arrhenius<R>((R)m.A[k], (R)m.b[k], (R)m.Ea[k], T);
    // O4: Eq. 9 then Eq. 8
    R dS = 0, dH = 0;
    int dnu = 0;
    for (int j = m.prod_ptr[k]; j < m.prod_ptr[k + 1]; ++j) {
      dS += (R)m.prod_nu[j] * s_R[m.prod_sp[j]];
      dH += (R)m.prod_nu[j] * h_RT[m.prod_sp[j]];
      dnu += m.prod_nu[j];
    }
    for (int j = m.reac_ptr[k]; j < m.reac_ptr[k + 1]; ++j) {
      dS -= (R)m.reac_nu[j] * s_R[m.reac_sp[j]];
      dH -= (R)m.reac_nu[j] * h_RT[m.reac_sp[j]];
      dnu -= m.reac_nu[j];
    }
    R Kp = m_exp(dS - dH);
    R Kc = Kp * m_pow(Consts<R>::Patm / (Rg * T), (R)dnu);
    // O5
    R M = Ctot;
    for (int j = m.eff_ptr[k]; j < m.eff_ptr[k + 1]; ++j) M += ((R)m.eff_val[j] - (R)1) * C[m.eff_sp[j]];
    // O6
    R kf = kinf, k0 = 0, Pr = 0, Fcent = 1, F = 1;
    const int rt = m.rtype[k];
    if (rt >= 2) {
      k0 = arrhenius<R>((R)m.A0[k], (R)m.b0[k], (R)m.Ea0[k], T);
      Pr = k0 * M / kinf;
      if (rt == 3) {
        const R al = m.troe[4 * k + 0], T3 = m.troe[4 * k + 1], T1 = m.troe[4 * k + 2], T2 = m.troe[4 * k + 3];
        Fcent = ((R)1 - al) * m_exp(-T / T3) + al * m_exp(-T / T1) + m_exp(-T2 / T);
        R lF = m_log10(Fcent);
        R c = (R)-0.4L - (R)0.67L * lF;
        R n = (R)0.75L - (R)1.27L * lF;
        R d = (R)0.14L;
        R lp = m_log10(Pr) + c;
        R f1 = lp / (n - d * lp);
        F = m_pow((R)10, lF / ((R)1 + f1 * f1));
      }
      kf = kinf * (Pr / ((R)1 + Pr)) * F;
    }
    // O7: Eq. 7
    R kr = m.reversible[k] ? kf / Kc : (R)0;
    // O8: Eq. 5
    R pf = 1, pr = 1;
    for (int j = m.reac_ptr[k]; j < m.reac_ptr[k + 1]; ++j) pf *= ipow<R>(C[m.reac_sp[j]], m.reac_nu[j]);
    for (int j = m.prod_ptr[k]; j < m.prod_ptr[k + 1]; ++j) pr *= ipow<R>(C[m.prod_sp[j]], m.prod_nu[j]);
    R q = kf * pf - kr * pr;
    if (rt == 1) q *= M;
    // O9: Eq. 4, k ascending
    for (int j = m.reac_ptr[k]; j < m.reac_ptr[k + 1]; ++j) wdot[m.reac_sp[j]] -= (R)m.reac_nu[j] * q;
    for (int j = m.prod_ptr[k]; j < m.prod_ptr[k + 1]; ++j) wdot[m.prod_sp[j]] += (R)m.prod_nu[j] * q;
    if (kf_out) kf_out[k] = kf;
    if (kr_out) kr_out[k] = kr;
    if (q_out) q_out[k] = q;
    if (det) det[k] = RxnDetail<R>{kinf, k0, Pr, Fcent, F, M, Kp, Kc, kf, kr, q};
  }
  if (wdot_out)
    for (int i = 0; i < K; ++i) wdot_out[i] = wdot[i];
  // O10
  if (F_out) {
    F_out[0] = T - Tset;
    for (int i = 0; i < K; ++i) F_out[1 + i] = (Y[i] - Yin[i]) / tau - wdot[i] * (R)m.W[i] / rho;
  }
  if (C_out)
    for (int i = 0; i < K; ++i) C_out[i] = C[i];
  if (rho_out) *rho_out = rho;
}

// Energy row: the steady form of Eq. 3 with Qdot = 0 and dP/dt = 0,
//   C_p,mix dT/dt = (mdot / rho V) sum_i Y_i,in (h_i,in - h_i) - (sum_i h_i wdot_i W_i) / rho,
// written as the residual F_T = -dT/dt with mdot/(rho V) = 1/tau.  h_i [erg/g] =
// (h/RT)_i R T / W_i at the reactor temperature, h_i,in the same at the inlet temperature T_in,
// C_p,mix = sum_i Y_i (cp/R)_i R / W_i  [erg/g/K]; NASA-7 fits as in O2.
template <class R>
R energy_row(const oracle_mech& m, R T, R Tin, const R* Y, const R* Yin, R tau, const R* wdot, R rho) {
  const int K = m.n_species;
  const R Rg = Consts<R>::Rgas;
  R inflow = 0, reaction = 0, cp_mix = 0;
  for (int i = 0; i < K; ++i) {
    R cp_R, h_RT, s_R, cpin_R, hin_RT, sin_R;
    nasa7<R>(m.nasa + 7 * i, T, cp_R, h_RT, s_R);
    nasa7<R>(m.nasa + 7 * i, Tin, cpin_R, hin_RT, sin_R);
    const R W = (R)m.W[i];
    const R h = h_RT * Rg * T / W;
    const R hin = hin_RT * Rg * Tin / W;
    inflow += Yin[i] * (hin - h);
    reaction += h * wdot[i] * W;
    cp_mix += Y[i] * cp_R * Rg / W;
  }
  const R dTdt = (inflow / tau - reaction / rho) / cp_mix;
  return -dTdt;
}

// Batch form of the adiabatic residual: species rows F [K][ld] as O10 and F_T [N] from energy_row.
template <class R>
int energy_batch(const oracle_mech& m, int64_t N, const double* T, const double* P, const double* Y,
                 const double* Tin, const double* Yin, const double* tau, int64_t ld, double* F, double* FT,
                 double* wdot, int nthreads) {
  const int K = m.n_species;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
#endif
  {
    std::vector<R> y(K), yin(K), ow(K), oF(K + 1);
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
    for (int64_t r = 0; r < N; ++r) {
      for (int i = 0; i < K; ++i) {
        y[i] = Y[(int64_t)i * ld + r];
        yin[i] = Yin[(int64_t)i * ld + r];
      }
      R rho;
      eval_one<R>(m, (R)T[r], (R)P[r], y.data(), yin.data(), (R)tau[r], (R)T[r], nullptr, nullptr, nullptr,
                  ow.data(), oF.data(), nullptr, nullptr, &rho);
      const R ft = energy_row<R>(m, (R)T[r], (R)Tin[r], y.data(), yin.data(), (R)tau[r], ow.data(), rho);
      if (F) for (int i = 0; i < K; ++i) F[(int64_t)i * ld + r] = (double)oF[1 + i];
      if (FT) FT[r] = (double)ft;
      if (wdot) for (int i = 0; i < K; ++i) wdot[(int64_t)i * ld + r] = (double)ow[i];
    }
  }
  return 0;
}

template <class R>
int eval_batch(const oracle_mech& m, int64_t N, const double* T, const double* P, const double* Y,
               const double* Yin, const double* tau, int64_t ld, double* kf, double* kr, double* q,
               int64_t ldk, double* wdot, double* F, int nthreads) {
  const int K = m.n_species, I = m.n_reactions;
  const bool want_F = F != nullptr;
  if (want_F && (!Yin || !tau)) return 1;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
#endif
  {
    std::vector<R> y(K), yin(K, (R)0), okf(I), okr(I), oq(I), ow(K), oF(K + 1);
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
    for (int64_t r = 0; r < N; ++r) {
      for (int i = 0; i < K; ++i) y[i] = Y[(int64_t)i * ld + r];
      if (want_F)
        for (int i = 0; i < K; ++i) yin[i] = Yin[(int64_t)i * ld + r];
      eval_one<R>(m, (R)T[r], (R)P[r], y.data(), yin.data(), want_F ? (R)tau[r] : (R)1, (R)T[r],
                  okf.data(), okr.data(), oq.data(), ow.data(), want_F ? oF.data() : nullptr, nullptr,
                  nullptr, nullptr);
      if (kf) for (int k = 0; k < I; ++k) kf[(int64_t)k * ldk + r] = (double)okf[k];
      if (kr) for (int k = 0; k < I; ++k) kr[(int64_t)k * ldk + r] = (double)okr[k];
      if (q) for (int k = 0; k < I; ++k) q[(int64_t)k * ldk + r] = (double)oq[k];
      if (wdot) for (int i = 0; i < K; ++i) wdot[(int64_t)i * ld + r] = (double)ow[i];
      if (F) for (int i = 0; i < K; ++i) F[(int64_t)i * ld + r] = (double)oF[1 + i];
    }
  }
  return 0;
}

// Round-off scale of the net production rates: acc_i = sum_k (nu'_ik + nu''_ik)
// (|k_f prod C^nu'| + |k_r prod C^nu''|), times |[M]_k| for a three-body reaction -- the magnitude of the
// terms whose signed sum is wdot_i (Eq. 4, 5), i.e. what one unit of relative rounding error in them moves
// wdot_i by.  C, kf, kr: the reactor's concentrations and effective rate constants (outputs of eval_one).
template <class R>
void roundoff_acc(const oracle_mech& m, const R* C, const R* kf, const R* kr, R* acc /*[K], zeroed*/) {
  const int K = m.n_species, I = m.n_reactions;
  for (int k = 0; k < I; ++k) {
    R pf = 1, pr = 1;
    for (int j = m.reac_ptr[k]; j < m.reac_ptr[k + 1]; ++j) pf *= ipow<R>(C[m.reac_sp[j]], m.reac_nu[j]);
    for (int j = m.prod_ptr[k]; j < m.prod_ptr[k + 1]; ++j) pr *= ipow<R>(C[m.prod_sp[j]], m.prod_nu[j]);
    R mag = std::fabs((double)(kf[k] * pf)) + std::fabs((double)(kr[k] * pr));
    if (m.rtype[k] == 1) {
      R M = 0;
      for (int i = 0; i < K; ++i) M += C[i];
      for (int j = m.eff_ptr[k]; j < m.eff_ptr[k + 1]; ++j) M += ((R)m.eff_val[j] - (R)1) * C[m.eff_sp[j]];
      mag *= std::fabs((double)M);
    }
    for (int j = m.reac_ptr[k]; j < m.reac_ptr[k + 1]; ++j) acc[m.reac_sp[j]] += (R)m.reac_nu[j] * mag;
    for (int j = m.prod_ptr[k]; j < m.prod_ptr[k + 1]; ++j) acc[m.prod_sp[j]] += (R)m.prod_nu[j] * mag;
  }
}

// O11: forward finite-difference Jacobian. x=(T,Y_1..Y_K); delta_j=1e-8*max(|x_j|,1e-10);
// x'_j = fl(x_j+delta_j) and h_j = fl(x'_j - x_j) are formed in DOUBLE for both precisions
// (the state is a double array; reading g15); each perturbed residual is a full independent
// O1..O10 evaluation.  J column-major per reactor, (K+1)x(K+1); S (optional) is the
// round-off scale S_i = |Y_i-Yin_i|/tau + (W_i/rho) sum_k |nu_ik| (|kf prod C'| + |kr prod C''|)
// of 8(c)-J, row 0 = |T|... row 0 is exact (S_0 = 0).
template <class R>
int jac_batch(const oracle_mech& m, int64_t N, const double* T, const double* P, const double* Y,
              const double* Tin /* null: row 0 is T - T_set; else the energy row */, const double* Yin,
              const double* tau, int64_t ld, double* J, double* F0, double* S, double* H, int nthreads) {
  const int K = m.n_species, I = m.n_reactions, n = K + 1;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
#endif
  {
    std::vector<double> x(n), xp(n);
    std::vector<R> y(K), yin(K), f0(n), f1(n), okf(I), okr(I), C(K), ow(K);
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
    for (int64_t r = 0; r < N; ++r) {
      x[0] = T[r];
      for (int i = 0; i < K; ++i) {
        x[1 + i] = Y[(int64_t)i * ld + r];
        yin[i] = Yin[(int64_t)i * ld + r];
        y[i] = x[1 + i];
      }
      const R Tset = (R)T[r];
      R rho;
      eval_one<R>(m, (R)x[0], (R)P[r], y.data(), yin.data(), (R)tau[r], Tset, okf.data(), okr.data(),
                  nullptr, ow.data(), f0.data(), nullptr, C.data(), &rho);
      if (Tin) f0[0] = energy_row<R>(m, (R)x[0], (R)Tin[r], y.data(), yin.data(), (R)tau[r], ow.data(), rho);
      double* Jr = J + (int64_t)r * n * n;
      if (F0) for (int i = 0; i < n; ++i) F0[(int64_t)r * n + i] = (double)f0[i];
      if (S) {
        double* Sr = S + (int64_t)r * n;
        Sr[0] = 0.0;
        std::vector<R> acc(K, (R)0);
        roundoff_acc<R>(m, C.data(), okf.data(), okr.data(), acc.data());
        for (int i = 0; i < K; ++i)
          Sr[1 + i] = (double)(std::fabs((double)((y[i] - yin[i]) / (R)tau[r])) + (R)m.W[i] / rho * acc[i]);
        if (Tin) {
          // round-off scale of the energy row: its terms in absolute value, the reaction part through the
          // same |nu| (|kf prod| + |kr prod|) sums as the species rows
          R st = 0, cp_mix = 0;
          for (int i = 0; i < K; ++i) {
            R cp_R, h_RT, s_R, cpin_R, hin_RT, sin_R;
            nasa7<R>(m.nasa + 7 * i, (R)x[0], cp_R, h_RT, s_R);
            nasa7<R>(m.nasa + 7 * i, (R)Tin[r], cpin_R, hin_RT, sin_R);
            const R W = (R)m.W[i];
            const R h = h_RT * Consts<R>::Rgas * (R)x[0] / W, hin = hin_RT * Consts<R>::Rgas * (R)Tin[r] / W;
            st += std::fabs((double)(yin[i] * (hin - h))) / (R)tau[r] + std::fabs((double)h) * W / rho * acc[i];
            cp_mix += y[i] * cp_R * Consts<R>::Rgas / W;
          }
          Sr[0] = (double)(st / cp_mix);
        }
      }
      for (int j = 0; j < n; ++j) {
        double ax = std::fabs(x[j]);
        double delta = 1e-8 * (ax > 1e-10 ? ax : 1e-10);
        volatile double xpj = x[j] + delta;   // fl(x_j + delta_j)
        volatile double hj = xpj - x[j];      // fl(x'_j - x_j)
        xp = x;
        xp[j] = xpj;
        if (H) H[(int64_t)r * n + j] = hj;
        for (int i = 0; i < K; ++i) y[i] = (R)xp[1 + i];
        R rho1;
        eval_one<R>(m, (R)xp[0], (R)P[r], y.data(), yin.data(), (R)tau[r], Tset, nullptr, nullptr, nullptr,
                    ow.data(), f1.data(), nullptr, nullptr, &rho1);
        if (Tin) f1[0] = energy_row<R>(m, (R)xp[0], (R)Tin[r], y.data(), yin.data(), (R)tau[r], ow.data(), rho1);
        for (int i = 0; i < n; ++i) Jr[(int64_t)j * n + i] = (double)((f1[i] - f0[i]) / (R)hj);
      }
      for (int i = 0; i < K; ++i) y[i] = (R)x[1 + i];
    }
  }
  return 0;
}

// NEXT-2: the Newton step's linear solve ("The Jacobian matrix is decomposed into lower and upper
// triangular matrices, and then a back-solving operation is carried out"): Gaussian
// elimination with partial pivoting (row of largest |a_ik|, the first one on ties), then forward and back
// substitution.  A: n x n column-major (entry (i,j) at A[j*n+i]), not modified; b -> x.  Returns 0, or
// k+1 if the pivot of step k is exactly zero (x is then left unset).
template <class R>
int lu_solve_one(int n, const double* A, const double* b, double* x) {
  std::vector<R> a((size_t)n * n), y(n);
  for (size_t t = 0; t < (size_t)n * n; ++t) a[t] = (R)A[t];
  for (int i = 0; i < n; ++i) y[i] = (R)b[i];
  for (int k = 0; k < n; ++k) {
    int p = k;
    R best = a[(size_t)k * n + k] < 0 ? -a[(size_t)k * n + k] : a[(size_t)k * n + k];
    for (int i = k + 1; i < n; ++i) {
      const R v = a[(size_t)k * n + i] < 0 ? -a[(size_t)k * n + i] : a[(size_t)k * n + i];
      if (v > best) { best = v; p = i; }
    }
    if (best == (R)0) return k + 1;
    if (p != k) {
      for (int j = 0; j < n; ++j) std::swap(a[(size_t)j * n + k], a[(size_t)j * n + p]);
      std::swap(y[k], y[p]);
    }
    for (int i = k + 1; i < n; ++i) {
      const R l = a[(size_t)k * n + i] / a[(size_t)k * n + k];
      a[(size_t)k * n + i] = l;
      for (int j = k + 1; j < n; ++j) a[(size_t)j * n + i] -= l * a[(size_t)j * n + k];
      y[i] -= l * y[k];
    }
  }
  for (int i = n - 1; i >= 0; --i) {
    R sum = y[i];
    for (int j = i + 1; j < n; ++j) sum -= a[(size_t)j * n + i] * y[j];
    y[i] = sum / a[(size_t)i * n + i];
  }
  for (int i = 0; i < n; ++i) x[i] = (double)y[i];
  return 0;
}

}  // namespace

extern "C" {

// Batched A x = b: A [N][n*n] column-major per system, b, x [N][n], info [N] (0 or k+1, see lu_solve_one).
int oracle_lu_solve(int64_t N, int n, const double* A, const double* b, double* x, int32_t* info,
                    int use_long_double) {
  for (int64_t r = 0; r < N; ++r) {
    const double* Ar = A + (size_t)r * n * n;
    info[r] = use_long_double ? lu_solve_one<long double>(n, Ar, b + r * n, x + r * n)
                              : lu_solve_one<double>(n, Ar, b + r * n, x + r * n);
  }
  return 0;
}

// NEXT-4: one pseudo-transient (implicit Euler) step.  "If the Newton algorithm fails to converge, then the
// solution estimate is conditioned by a pseudo-transient time integration of the governing equations"
// (PAPER.md:44).  The transient equations are dx/dt = -F(x) (Eq. 2 with this build's sign of F); implicit
// Euler over dt, linearised about x:  (x' - x)/dt = -F(x') ~ -F(x) - J (x' - x)   =>   (I/dt + J) dx = -F.
// Written out as that: form A = J + I/dt entry by entry, b = -F, then the elimination above.
// J: [N][n*n] column-major per system, F: [N][n], dt: [N] (> 0; +inf gives the Newton step), dx: [N][n].
int oracle_ptc_step(int64_t N, int n, const double* J, const double* F, const double* dt, double* dx, int32_t* info,
                    int use_long_double) {
  std::vector<double> A((size_t)n * n), b(n);
  for (int64_t r = 0; r < N; ++r) {
    const double shift = 1.0 / dt[r];
    for (int j = 0; j < n; ++j)
      for (int i = 0; i < n; ++i) A[(size_t)j * n + i] = J[(size_t)r * n * n + (size_t)j * n + i] + (i == j ? shift : 0.0);
    for (int i = 0; i < n; ++i) b[i] = -F[r * n + i];
    info[r] = use_long_double ? lu_solve_one<long double>(n, A.data(), b.data(), dx + r * n)
                              : lu_solve_one<double>(n, A.data(), b.data(), dx + r * n);
  }
  return 0;
}

// Batch evaluation, species-major SoA (element (k, r) at [k*ld + r]).  Any output may be null.
// use_long_double: 0 -> double (the oracle), 1 -> long double reference.
int oracle_eval(const oracle_mech* m, int64_t N, const double* T, const double* P, const double* Y,
                const double* Yin, const double* tau, int64_t ld, double* kf, double* kr, double* q,
                int64_t ldk, double* wdot, double* F, int use_long_double, int nthreads) {
  if (use_long_double)
    return eval_batch<long double>(*m, N, T, P, Y, Yin, tau, ld, kf, kr, q, ldk, wdot, F, nthreads);
  return eval_batch<double>(*m, N, T, P, Y, Yin, tau, ld, kf, kr, q, ldk, wdot, F, nthreads);
}

// Adiabatic PSR residual: F [K][ld] (species rows, O10), FT [N] (energy row), wdot [K][ld]; any may be null.
int oracle_eval_energy(const oracle_mech* m, int64_t N, const double* T, const double* P, const double* Y,
                       const double* Tin, const double* Yin, const double* tau, int64_t ld, double* F, double* FT,
                       double* wdot, int use_long_double, int nthreads) {
  if (use_long_double) return energy_batch<long double>(*m, N, T, P, Y, Tin, Yin, tau, ld, F, FT, wdot, nthreads);
  return energy_batch<double>(*m, N, T, P, Y, Tin, Yin, tau, ld, F, FT, wdot, nthreads);
}

// J: [N][(K+1)*(K+1)] column-major per reactor; F0, S, H: [N][K+1] (may be null).
int oracle_jacobian(const oracle_mech* m, int64_t N, const double* T, const double* P, const double* Y,
                    const double* Yin, const double* tau, int64_t ld, double* J, double* F0, double* S,
                    double* H, int use_long_double, int nthreads) {
  if (use_long_double) return jac_batch<long double>(*m, N, T, P, Y, nullptr, Yin, tau, ld, J, F0, S, H, nthreads);
  return jac_batch<double>(*m, N, T, P, Y, nullptr, Yin, tau, ld, J, F0, S, H, nthreads);
}

// The same with the energy row (NEXT-1) as row 0 of the residual: the adiabatic PSR system.
int oracle_jacobian_energy(const oracle_mech* m, int64_t N, const double* T, const double* P, const double* Y,
                           const double* Tin, const double* Yin, const double* tau, int64_t ld, double* J, double* F0,
                           double* S, double* H, int use_long_double, int nthreads) {
  if (use_long_double) return jac_batch<long double>(*m, N, T, P, Y, Tin, Yin, tau, ld, J, F0, S, H, nthreads);
  return jac_batch<double>(*m, N, T, P, Y, Tin, Yin, tau, ld, J, F0, S, H, nthreads);
}

// Round-off scales of a batch (the floor terms of the parity criteria): Sw [K][ld] =
// roundoff_acc (scale of wdot_i), SF [K][ld] = |Y_i - Yin_i|/tau + (W_i/rho) Sw_i (scale of F_i, the S of
// oracle_jacobian rows 1..K).  Either may be null; SF needs Yin and tau.
int oracle_roundoff_scale(const oracle_mech* m, int64_t N, const double* T, const double* P, const double* Y,
                          const double* Yin, const double* tau, int64_t ld, double* Sw, double* SF, int nthreads) {
  const int K = m->n_species, I = m->n_reactions;
  if (SF && (!Yin || !tau)) return 1;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
#endif
  {
    std::vector<double> y(K), yin(K, 0.0), okf(I), okr(I), C(K), acc(K);
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
    for (int64_t r = 0; r < N; ++r) {
      for (int i = 0; i < K; ++i) y[i] = Y[(int64_t)i * ld + r];
      double rho;
      eval_one<double>(*m, T[r], P[r], y.data(), yin.data(), 1.0, T[r], okf.data(), okr.data(), nullptr, nullptr,
                       nullptr, nullptr, C.data(), &rho);
      std::fill(acc.begin(), acc.end(), 0.0);
      roundoff_acc<double>(*m, C.data(), okf.data(), okr.data(), acc.data());
      for (int i = 0; i < K; ++i) {
        if (Sw) Sw[(int64_t)i * ld + r] = acc[i];
        if (SF) SF[(int64_t)i * ld + r] = std::fabs((y[i] - Yin[(int64_t)i * ld + r]) / tau[r]) + m->W[i] / rho * acc[i];
      }
    }
  }
  return 0;
}

// Single-reactor detail for the pins: per reaction 11 doubles
// (kinf,k0,Pr,Fcent,F,M,Kp,Kc,kf,kr,q); per species C; scalars out[0]=Wbar... rho only.
int oracle_detail(const oracle_mech* m, double T, double P, const double* Y, double* rxn /*[I][11]*/,
                  double* C /*[K]*/, double* rho) {
  const int K = m->n_species, I = m->n_reactions;
  std::vector<RxnDetail<double>> det(I);
  std::vector<double> yin(K, 0.0);
  double r;
  eval_one<double>(*m, T, P, Y, yin.data(), 1.0, T, nullptr, nullptr, nullptr, nullptr, nullptr, det.data(), C, &r);
  for (int k = 0; k < I; ++k) {
    const RxnDetail<double>& d = det[k];
    double v[11] = {d.kinf, d.k0, d.Pr, d.Fcent, d.F, d.M, d.Kp, d.Kc, d.kf, d.kr, d.q};
    std::memcpy(rxn + 11 * k, v, sizeof v);
  }
  if (rho) *rho = r;
  return 0;
}

double oracle_arrhenius(double A, double b, double Ea, double T) { return arrhenius<double>(A, b, Ea, T); }

void oracle_nasa7(const double* a, double T, double* cp_R, double* h_RT, double* s_R) {
  nasa7<double>(a, T, *cp_R, *h_RT, *s_R);
}

int oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
}

// NEXT-4, second half: the hybrid Newton / pseudo-transient solver of PAPER.md:44 --
//   "one of the first steps involves constructing an error vector by substituting the initial guesses into the
//    nonlinear-algebraic equations.  The next step is to construct a Jacobian matrix.  The Jacobian matrix is
//    decomposed into lower and upper triangular matrices, and then a back-solving operation is carried out ...
//    The hybrid approach consists of two steps: a steady state Newton iteration and a pseudo-transient time
//    integration.  If convergence is not achieved using the Newton iteration, the solution estimate is conditioned
//    using the time integration.  The process of switching between the Newton iteration and time integration
//    approaches continues until convergence is achieved, which is based on very specific criteria related to
//    absolute and relative tolerances."
// The paper leaves every constant and the step-size rule to its ref. [5]; they are the caller's (opts), and the
// points the paper does not fix are read as follows (readings g21-g25):
//   g21  unknowns x = (T, Y_1..Y_K); residual F of O10 (row 0 = T - T_set), or with Tin the adiabatic system
//        whose row 0 is the energy row; Jacobian by O11 (forward differences) at every iteration.
//   g22  Newton iteration: solve J dx = -F, trial x' = x + dx (full step).  Converged when
//        max_i |dx_i| / (atol + rtol |x_i|) <= 1 with x the estimate the correction was computed at; the
//        correction is applied before stopping.  A trial is admissible when dx is finite (the system solved
//        without a zero pivot) and every mass fraction of x' is >= -y_floor (the solver this one descends from,
//        PAPER.md:158 ref. [3], bounds its unknowns the same way; y_floor = +inf switches the bound off).
//   g23  "convergence is not achieved": the trial of a Newton iteration is not admissible (x then stays), or
//        max_newton admissible iterations of a Newton stage have passed without convergence.  The estimate is
//        then conditioned by max_ptc pseudo-transient steps ((I/dt + J) dx = -F, oracle_ptc_step's system)
//        before Newton resumes.
//   g24  step size: dt starts at dt0 and persists across stages; an admissible step is taken and
//        dt <- dt * dt_grow, otherwise x stays and dt <- dt * dt_shrink (either way it counts as one step).
//   g25  budget: every linear solve (Newton or pseudo-transient) counts; after max_iter of them a reactor that has
//        not converged is reported as such (status 1).  status 0 = converged.
// One reactor at a time, every step a call of the plain routines above (jac_batch on one reactor, lu_solve_one).
extern "C" {
struct oracle_solve_opts {
  double atol, rtol;
  int32_t max_iter, max_newton, max_ptc, reserved;
  double dt0, dt_grow, dt_shrink, y_floor;
};

int oracle_solve_hybrid(const oracle_mech* m, int64_t N, double* T, const double* P, double* Y, const double* Tin,
                        const double* Yin, const double* tau, int64_t ld, const oracle_solve_opts* o, int32_t* status,
                        int32_t* n_newton, int32_t* n_ptc, int nthreads) {
  const int K = m->n_species, n = K + 1;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
#endif
  {
    std::vector<double> x(n), xt(n), y(K), yin(K), J((size_t)n * n), F(n), A((size_t)n * n), b(n), dx(n);
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 1)
#endif
    for (int64_t r = 0; r < N; ++r) {
      x[0] = T[r];
      for (int i = 0; i < K; ++i) {
        x[1 + i] = Y[(int64_t)i * ld + r];
        yin[i] = Yin[(int64_t)i * ld + r];
      }
      const double Tset = T[r];   // the fixed-temperature equation holds T at its initial value
      const double Pr = P[r], taur = tau[r], Tinr = Tin ? Tin[r] : 0.0;
      bool newton = true, converged = false;
      int it = 0, nn = 0, np = 0;
      double dt = o->dt0;
      for (int iter = 0; iter < o->max_iter && !converged; ++iter) {
        // error vector and Jacobian at the current estimate (O10 / energy row, O11)
        for (int i = 0; i < K; ++i) y[i] = x[1 + i];
        const double Tr = x[0];
        jac_batch<double>(*m, 1, &Tr, &Pr, y.data(), Tin ? &Tinr : nullptr, yin.data(), &taur, 1, J.data(), F.data(),
                          nullptr, nullptr, 1);
        if (!Tin) F[0] = x[0] - Tset;   // jac_batch measures row 0 from its own input T; the equation is T - T_set
        // (I/dt + J) dx = -F; a Newton iteration is the same system without the shift
        const double shift = newton ? 0.0 : 1.0 / dt;
        for (int j = 0; j < n; ++j)
          for (int i = 0; i < n; ++i) A[(size_t)j * n + i] = J[(size_t)j * n + i] + (i == j ? shift : 0.0);
        for (int i = 0; i < n; ++i) b[i] = -F[i];
        const int info = lu_solve_one<double>(n, A.data(), b.data(), dx.data());
        bool ok = info == 0;
        for (int i = 0; ok && i < n; ++i) ok = std::isfinite(dx[i]);
        // the trial estimate; admissible when dx is finite and every mass fraction stays >= -y_floor
        double err = 0.0;
        bool admissible = ok;
        if (ok) {
          for (int i = 0; i < n; ++i) {
            err = std::fmax(err, std::fabs(dx[i]) / (o->atol + o->rtol * std::fabs(x[i])));
            xt[i] = x[i] + dx[i];
          }
          for (int i = 1; i < n; ++i) admissible = admissible && xt[i] >= -o->y_floor;
        }
        if (newton) {
          ++nn;
          if (admissible && err <= 1.0) {
            x = xt;
            converged = true;
          } else if (admissible) {
            x = xt;
            if (++it >= o->max_newton) {   // the stage is over without convergence: condition the estimate
              newton = false;
              it = 0;
            }
          } else {
            newton = false;
            it = 0;
          }
        } else {
          ++np;
          if (admissible) {
            x = xt;
            dt *= o->dt_grow;
          } else {
            dt *= o->dt_shrink;
          }
          if (++it >= o->max_ptc) {   // back to the Newton iteration from the conditioned estimate
            newton = true;
            it = 0;
          }
        }
      }
      T[r] = x[0];
      for (int i = 0; i < K; ++i) Y[(int64_t)i * ld + r] = x[1 + i];
      status[r] = converged ? 0 : 1;
      if (n_newton) n_newton[r] = nn;
      if (n_ptc) n_ptc[r] = np;
    }
  }
  return 0;
}
}
