// marut_physics.cuh -- pointwise physics of the CUDA path: equation of state, inviscid and
// viscous fluxes, Rusanov flux, NASA-7 thermodynamics and finite-rate chemistry.
// All FP64, IEEE division and square root (no fast-math); FMA contraction is allowed.
#pragma once
#include "marut_common.cuh"

namespace marut {

// ---------------------------------------------------------------- NASA-7 (PAPER.md:134, 288(i))
struct Thermo {
  // e_s(T) and cv_s(T) per unit mass for species s from the NASA-7 table
  __device__ static __forceinline__ const double *range(const MechDev &m, int s, double T) {
    return m.nasa[s][T < m.T_mid ? 0 : 1];
  }
  __device__ static __forceinline__ double cp_R(const double *a, double T) {
    return a[0] + T * (a[1] + T * (a[2] + T * (a[3] + T * a[4])));
  }
  __device__ static __forceinline__ double h_RT(const double *a, double T) {
    return a[0] + T * (a[1] * 0.5 + T * (a[2] * (1.0 / 3.0) + T * (a[3] * 0.25 + T * (a[4] * 0.2)))) + a[5] / T;
  }
  __device__ static __forceinline__ double s_R(const double *a, double T, double lnT) {
    return a[0] * lnT + T * (a[1] + T * (a[2] * 0.5 + T * (a[3] * (1.0 / 3.0) + T * (a[4] * 0.25)))) + a[6];
  }
};

// Newton for T on sum_s rho_s e_s(T) = e_int (PAPER.md:288(i); R12: T0 = 4000 K,
// stop |dT| <= 1e-13 T, cap 50 iterations).
template <int NSP>
__device__ inline double temperature_newton(const MechDev &m, const double *rho_s, double e_int, double T_start = 4000.0) {
  double T = T_start;
  double rR[NSP];
#pragma unroll
  for (int s = 0; s < NSP; ++s) rR[s] = rho_s[s] * m.Rs[s];
  for (int it = 0; it < 50; ++it) {
    double f = -e_int, df = 0.0;
#pragma unroll
    for (int s = 0; s < NSP; ++s) {
      const double *a = Thermo::range(m, s, T);
      f += rR[s] * T * (Thermo::h_RT(a, T) - 1.0);
      df += rR[s] * (Thermo::cp_R(a, T) - 1.0);
    }
    double dT = f / df;
    T -= dT;
    if (fabs(dT) <= 1e-13 * T) break;
  }
  return T;
}

// ---------------------------------------------------------------- primitives
template <int DIM>
struct Prim {
  double rho, irho, p, a, T;
  double v[DIM];
};

// ideal gas; T = p/rho with R = 1
template <int DIM, bool WANT_A>
__device__ __forceinline__ Prim<DIM> prim_ideal(const double *U, double gamma) {
  Prim<DIM> q;
  q.rho = U[0];
  q.irho = 1.0 / U[0];
  double ke = 0.0;
#pragma unroll
  for (int c = 0; c < DIM; ++c) {
    q.v[c] = U[1 + c] * q.irho;
    ke += q.v[c] * U[1 + c];
  }
  q.p = (gamma - 1.0) * (U[DIM + 1] - 0.5 * ke);
  q.T = q.p * q.irho;
  q.a = WANT_A ? sqrt(gamma * q.p * q.irho) : 0.0;
  return q;
}

// reacting mixture with known T: p = rho R T, R = sum_s Y_s R_s; frozen sound speed
template <int DIM, int NSP, bool WANT_A>
__device__ inline Prim<DIM> prim_mixture(const double *U, double T, const MechDev &m) {
  Prim<DIM> q;
  double rho = 0.0, rhoR = 0.0, rhocp = 0.0;
#pragma unroll
  for (int s = 0; s < NSP; ++s) {
    const double Rs = m.Rs[s];
    rho += U[s];
    rhoR += U[s] * Rs;
    if (WANT_A) rhocp += U[s] * Rs * Thermo::cp_R(Thermo::range(m, s, T), T);
  }
  q.rho = rho;
  q.irho = 1.0 / rho;
#pragma unroll
  for (int c = 0; c < DIM; ++c) q.v[c] = U[NSP + c] * q.irho;
  q.T = T;
  q.p = rhoR * T;
  if (WANT_A) {
    double R = rhoR * q.irho, cp = rhocp * q.irho;
    q.a = sqrt(cp / (cp - R) * R * T);
  } else q.a = 0.0;
  return q;
}

// |v| + a of an ideal-gas state (eq. 18; R11): the ONE expression both wave_speed_kernel and the
// fused reduction of the stage kernels evaluate, so that marut_max_dt, marut_max_dt_async and marut_ssprk33_step_cfl give
// the same time step bit for bit.  A state with rho <= 0 < p or p < 0 < rho gives NaN (caught by the callers).
template <int DIM>
__device__ __forceinline__ double wave_speed_ideal(const double *U, double gamma) {
  const double rinv = rcp_pos(U[0]);
  double m2 = 0.0;
#pragma unroll
  for (int c = 0; c < DIM; ++c) m2 += U[1 + c] * U[1 + c];
  const double p = (gamma - 1.0) * (U[DIM + 1] - 0.5 * m2 * rinv);
  const double vabs = (m2 > 0.0) ? sqrt_pos(m2) * fabs(rinv) : 0.0;     // a fluid at rest: sqrt_pos(0) is not defined
  return vabs + sqrt_pos(gamma * p * rinv);
}

// reacting mixture with pressure and sound speed already known (eos_kernel): only the velocity is formed here
template <int DIM, int NSP>
__device__ __forceinline__ Prim<DIM> prim_given_pa(const double *U, double p, double a) {
  Prim<DIM> q;
  double rho = 0.0;
#pragma unroll
  for (int s = 0; s < NSP; ++s) rho += U[s];
  q.rho = rho;
  q.irho = 1.0 / rho;
#pragma unroll
  for (int c = 0; c < DIM; ++c) q.v[c] = U[NSP + c] * q.irho;
  q.p = p;
  q.a = a;
  q.T = 0.0;
  return q;
}

// e_int = E - 1/2 rho |v|^2 of a reacting state
template <int DIM, int NSP>
__device__ __forceinline__ double internal_energy(const double *U) {
  double rho = 0.0;
#pragma unroll
  for (int s = 0; s < NSP; ++s) rho += U[s];
  double m2 = 0.0;
#pragma unroll
  for (int c = 0; c < DIM; ++c) m2 += U[NSP + c] * U[NSP + c];
  return U[NSP + DIM] - 0.5 * m2 / rho;
}

// F_inv(U) . nv for a scaled vector nv
template <int DIM, int NSP>
__device__ __forceinline__ void flux_dot(const double *U, const Prim<DIM> &q, const double *nv, double *F) {
  double vn = 0.0;
#pragma unroll
  for (int c = 0; c < DIM; ++c) vn += q.v[c] * nv[c];
#pragma unroll
  for (int s = 0; s < NSP; ++s) F[s] = U[s] * vn;
#pragma unroll
  for (int c = 0; c < DIM; ++c) F[NSP + c] = U[NSP + c] * vn + q.p * nv[c];
  F[NSP + DIM] = (U[NSP + DIM] + q.p) * vn;
}

// Rusanov / local Lax-Friedrichs flux with the scaled outward normal nv (R5):
//   F* = 1/2 (F(U-) + F(U+)).nv - 1/2 lambda |nv| (U+ - U-), lambda = max(|v-.n|+a-, |v+.n|+a+)
// Fm = F(U-).nv is passed in when the caller already has it.
template <int DIM, int NSP>
__device__ __forceinline__ void rusanov(const double *Um, const Prim<DIM> &qm, const double *Fm, const double *Up,
                                        const Prim<DIM> &qp, const double *nv, double *Fs) {
  constexpr int NVAR = NSP + DIM + 1;
  double n2 = 0.0, vnm = 0.0, vnp = 0.0;
#pragma unroll
  for (int c = 0; c < DIM; ++c) {
    n2 += nv[c] * nv[c];
    vnm += qm.v[c] * nv[c];
    vnp += qp.v[c] * nv[c];
  }
  const double nrm = sqrt(n2), inrm = 1.0 / nrm;
  const double lam = fmax(fabs(vnm * inrm) + qm.a, fabs(vnp * inrm) + qp.a);
  double Fp[NVAR];
  flux_dot<DIM, NSP>(Up, qp, nv, Fp);
  const double hl = 0.5 * lam * nrm;
#pragma unroll
  for (int v = 0; v < NVAR; ++v) Fs[v] = 0.5 * (Fm[v] + Fp[v]) - hl * (Up[v] - Um[v]);
}

// Rusanov lift of one face node from the two states (Euler; eq. 12; R5, R6), with a
// scaled normal and division-free apart from 1/rho+:
//   lambda |nv| = max(|v-.nv| + a- |nv|, |v+.nv| + a+ |nv|);  lift = (F*(U-,U+;nv) - F(U-).nv)/w_b
// Fm_out = F(U-).nv (for the faces whose F* comes from elsewhere, e.g. mortars).
template <int DIM>
__device__ __forceinline__ void rusanov_lift(const double *Um, double irhom, double pm, double am, const double *Up,
                                             const double *nv, double nrm, double gamma, double inv_wb, double *lift,
                                             double *Fm_out) {
  constexpr int NVAR = DIM + 2;
  double mnm = 0.0, mnp = 0.0, kep = 0.0;
#pragma unroll
  for (int c = 0; c < DIM; ++c) {
    mnm += Um[1 + c] * nv[c];
    mnp += Up[1 + c] * nv[c];
    kep += Up[1 + c] * Up[1 + c];
  }
  const double irhop = 1.0 / Up[0];
  const double vnm = mnm * irhom;
  const double pp = (gamma - 1.0) * (Up[DIM + 1] - 0.5 * kep * irhop);
  const double ap = sqrt(gamma * pp * irhop);
  const double vnp = mnp * irhop;
  const double hl = 0.5 * fmax(fabs(vnm) + am * nrm, fabs(vnp) + ap * nrm);
  double Fm[NVAR], Fp[NVAR];
  Fm[0] = mnm;
  Fp[0] = mnp;
#pragma unroll
  for (int c = 0; c < DIM; ++c) {
    Fm[1 + c] = Um[1 + c] * vnm + pm * nv[c];
    Fp[1 + c] = Up[1 + c] * vnp + pp * nv[c];
  }
  Fm[DIM + 1] = (Um[DIM + 1] + pm) * vnm;
  Fp[DIM + 1] = (Up[DIM + 1] + pp) * vnp;
#pragma unroll
  for (int v = 0; v < NVAR; ++v) {
    lift[v] = inv_wb * (0.5 * (Fp[v] - Fm[v]) - hl * (Up[v] - Um[v]));
    Fm_out[v] = Fm[v];
  }
}

// viscous flux F_v(U,S).nv (eq. 15; q = -k grad T, k = gamma mu/(Pr (gamma-1)))
// S[w*DIM + c] = d W_w / d x_c, W = (rho, v_1..v_d, T); F has DIM+2 entries, F[0] = 0.
template <int DIM>
__device__ __forceinline__ void viscous_flux_dot(const double *vel, const double *S, const double *nv, double mu,
                                                 double kappa, double *F) {
  double divu = 0.0;
#pragma unroll
  for (int i = 0; i < DIM; ++i) divu += S[(1 + i) * DIM + i];
  double Fe = 0.0;
  F[0] = 0.0;
#pragma unroll
  for (int i = 0; i < DIM; ++i) {
    double ti = 0.0;
#pragma unroll
    for (int j = 0; j < DIM; ++j) {
      double tau = (i == j) ? mu * (2.0 * S[(1 + i) * DIM + i] - (2.0 / 3.0) * divu)
                            : mu * (S[(1 + i) * DIM + j] + S[(1 + j) * DIM + i]);
      ti += tau * nv[j];
    }
    F[1 + i] = ti;
    Fe += vel[i] * ti;   // sum_j (sum_i v_i tau_ij) n_j  (tau symmetric)
  }
#pragma unroll
  for (int j = 0; j < DIM; ++j) Fe += kappa * S[(1 + DIM) * DIM + j] * nv[j];
  F[1 + DIM] = Fe;
}

// Compact form of the BR1 gradient for the viscous flux (eq. 15): the symmetric stress tensor and
// the heat-flux vector, NTAU = d(d+1)/2 + d doubles per node instead of the (d+2) d gradient components.
//   tau[0..d)      = tau_ii = mu (2 S_ii - 2/3 div u)
//   tau[d..d(d+1)/2) = tau_ij (i<j) = mu (S_ij + S_ji)   order: 2-D xy ; 3-D xy, xz, yz
//   tau[last d]    = kappa dT/dx_j
// Same expressions, in the same order, as viscous_flux_dot: the two forms give identical results.
template <int DIM>
struct Tau {
  static constexpr int NTAU = DIM * (DIM + 1) / 2 + DIM;
  __host__ __device__ static constexpr int off(int i, int j) {   // i < j
    return (DIM == 2) ? 2 : ((i == 0) ? ((j == 1) ? 3 : 4) : 5);
  }
};
template <int DIM>
__device__ __forceinline__ void gradient_to_tau(const double *S, double mu, double kappa, double *tau) {
  double divu = 0.0;
#pragma unroll
  for (int i = 0; i < DIM; ++i) divu += S[(1 + i) * DIM + i];
#pragma unroll
  for (int i = 0; i < DIM; ++i) {
    tau[i] = mu * (2.0 * S[(1 + i) * DIM + i] - (2.0 / 3.0) * divu);
#pragma unroll
    for (int j = i + 1; j < DIM; ++j) tau[Tau<DIM>::off(i, j)] = mu * (S[(1 + i) * DIM + j] + S[(1 + j) * DIM + i]);
  }
#pragma unroll
  for (int j = 0; j < DIM; ++j) tau[DIM * (DIM + 1) / 2 + j] = kappa * S[(1 + DIM) * DIM + j];
}
template <int DIM>
__device__ __forceinline__ void viscous_flux_dot_tau(const double *vel, const double *tau, const double *nv, double *F) {
  double Fe = 0.0;
  F[0] = 0.0;
#pragma unroll
  for (int i = 0; i < DIM; ++i) {
    double ti = 0.0;
#pragma unroll
    for (int j = 0; j < DIM; ++j) {
      const double t = (i == j) ? tau[i] : tau[Tau<DIM>::off(i < j ? i : j, i < j ? j : i)];
      ti += t * nv[j];
    }
    F[1 + i] = ti;
    Fe += vel[i] * ti;
  }
#pragma unroll
  for (int j = 0; j < DIM; ++j) Fe += tau[DIM * (DIM + 1) / 2 + j] * nv[j];
  F[1 + DIM] = Fe;
}

// ---------------------------------------------------------------- chemistry (eq. 21-22)
// omega_s [kg m^-3 s^-1] from T and partial densities; concentrations in mol/cm^3 inside the rate law,
// K_c = exp(-sum dnu g_s/(R_u T)) (p_ref/(R_u T) 1e-6)^(sum dnu)  (R12)
template <int NSP>
__device__ inline void production_rates(const MechDev &m, double T, const double *rho_s, double *omega) {
  // k_f = A exp(b ln T - Ea/T);  k_b = k_f / K_c = A exp(b ln T - Ea/T + dG - dnu ln c0): two exponentials per
  // reaction, no pow() and no division (same value as the definition up to rounding)
  double X[NSP], g[NSP];
  const double lnT = log(T), invT = 1.0 / T;
#pragma unroll
  for (int s = 0; s < NSP; ++s) {
    X[s] = rho_s[s] / m.W[s] * 1.0e-6;
    const double *a = Thermo::range(m, s, T);
    g[s] = Thermo::h_RT(a, T) - Thermo::s_R(a, T, lnT);
    omega[s] = 0.0;
  }
  const double lnc0 = log(P_REF / (R_UNIVERSAL * T) * 1.0e-6);
  double ikc = 1.0;   // 1 / K_c of the current group of reactions (same net stoichiometric vector)
  for (int r = 0; r < m.nr; ++r) {
    double dG = 0.0, pf = 1.0, pb = 1.0;
    int dnu = 0;
#pragma unroll
    for (int s = 0; s < NSP; ++s) {
      const int nr_ = m.nu_r[r][s], np_ = m.nu_p[r][s];
      const int d = np_ - nr_;
      if (d != 0) { dG += d * g[s]; dnu += d; }
      if (nr_ > 0) pf *= (nr_ == 1) ? X[s] : ((nr_ == 2) ? X[s] * X[s] : X[s] * X[s] * X[s]);
      if (np_ > 0) pb *= (np_ == 1) ? X[s] : ((np_ == 2) ? X[s] * X[s] : X[s] * X[s] * X[s]);
    }
    if (m.new_group[r]) ikc = exp(dG - dnu * lnc0);
    const double kf = m.A[r] * exp(m.b[r] * lnT - m.Ea[r] * invT);
    const double kb = kf * ikc;
    const double Rr = kf * pf - kb * pb;
#pragma unroll
    for (int s = 0; s < NSP; ++s) {
      const int d = m.nu_p[r][s] - m.nu_r[r][s];
      if (d != 0) omega[s] += d * Rr;
    }
  }
#pragma unroll
  for (int s = 0; s < NSP; ++s) omega[s] = m.W[s] * omega[s] * 1.0e6;
}

// The same rates for the fused stage kernel: the concentrations X_s go through a per-thread shared-memory column
// (Xs[s * stride]) so that the rate products can index the species listed per reaction (fr / br) instead of
// looping over all species with runtime exponents.
template <int NSP>
__device__ inline void production_rates_listed(const MechDev &m, double T, const double *rho_s, double *Xs, int stride,
                                               double *omega) {
  double g[NSP];
  const double lnT = log(T), invT = 1.0 / T;
#pragma unroll
  for (int s = 0; s < NSP; ++s) {
    Xs[s * stride] = rho_s[s] / m.W[s] * 1.0e-6;
    const double *a = Thermo::range(m, s, T);
    g[s] = Thermo::h_RT(a, T) - Thermo::s_R(a, T, lnT);
    omega[s] = 0.0;
  }
  const double lnc0 = log(P_REF / (R_UNIVERSAL * T) * 1.0e-6);
  double ikc = 1.0;
  for (int r = 0; r < m.nr; ++r) {
    if (m.new_group[r]) {
      double dG = 0.0;
#pragma unroll
      for (int s = 0; s < NSP; ++s) dG += m.dnu[r][s] * g[s];
      ikc = exp(dG - m.dnu_sum[r] * lnc0);
    }
    double pf = 1.0, pb = 1.0;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const int a = m.fr[r][q], b = m.br[r][q];
      if (a >= 0) pf *= Xs[a * stride];
      if (b >= 0) pb *= Xs[b * stride];
    }
    const double kf = m.A[r] * exp(m.b[r] * lnT - m.Ea[r] * invT);
    const double Rr = kf * (pf - ikc * pb);
#pragma unroll
    for (int s = 0; s < NSP; ++s) omega[s] += m.dnu[r][s] * Rr;
  }
#pragma unroll
  for (int s = 0; s < NSP; ++s) omega[s] = m.W[s] * omega[s] * 1.0e6;
}

}  // namespace marut
