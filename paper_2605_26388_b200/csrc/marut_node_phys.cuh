// marut_node_phys.cuh -- the node kernel (marut_node.cuh) for the physics with extra per-node work:
// Navier-Stokes with BR1 viscous fluxes (eq. 15-16) and the reacting
// mixture with its chemistry source (a8, a9; eq. 20-22).  Same structure: thread-per-node
// flux evaluation, balanced line-task derivative passes, densely mapped face tasks, last pass fused with the
// lift + 1/J + source + SSP-RK combination.  Differences from the Euler instance: the derivative passes write
// a separate result plane set (the flux planes stay intact because the viscous face tasks read the own
// normal flux from them), and the face tasks gather the neighbour's BR1 gradient (NS) or pressure and sound speed
// (reacting) as well.  Reacting: pressure, frozen sound speed and the chemistry source of every node come from the
// aux array eos_kernel fills ahead of the stage, so this kernel carries no mechanism table.  Interior faces: conforming;
// Navier-Stokes in 2-D also 2:1 mortars (reading R23).
//
// Product code; shares nothing with oracle/.
#pragma once
#include "marut_node.cuh"

#ifndef MARUT_PHYS_MINB128
#define MARUT_PHYS_MINB128 5
#endif

namespace marut {

template <int DIM, int NP, int NSP, int PHYS, int EB>
struct PhysCfg {
  using G = Geo<DIM, NP>;
  static constexpr int NVAR = NSP + DIM + 1, NW = DIM + 2;
  static constexpr int NN = G::NN, NF = G::NF;
  static constexpr int TILE = EB * NN;
  static constexpr int NFN = 2 * DIM * NF, NTASK = EB * NFN;
  static constexpr int NT = ((TILE + 31) / 32) * 32;
  static constexpr int NST = NVAR + 3;                       // stash planes: U, 1/rho, p, a
  // plane strides.  3-D, n = 4: lines of four doubles at row stride 4 / plane stride 16 put a half-warp's line tasks on 4
  // of the 16 banks in the xi and eta passes (57 % of the kernel's shared-memory wavefronts were conflicts,
  // profiles/r02_c3_stage.md); a k-plane stride of 17 and a variable-plane stride of 70 make the xi pass conflict-free and
  // leave the eta pass at 1.6x the minimum (brute-force count over the strides, as for NodeLayout)
  static constexpr bool PAD4 = (DIM == 3 && NP == 4);
  static constexpr int KS = PAD4 ? 17 : NP * NP, PS = PAD4 ? 70 : (NN | 1);
  static constexpr int NFP = DIM * NVAR * EB;                // flux planes
  // result planes of the derivative passes.  Navier-Stokes keeps them apart from the flux planes (its face tasks read the
  // own normal flux there); the reacting stage accumulates in place in the xi flux planes (a line belongs to one
  // thread): 66 -> 57 KB of shared memory per CTA, four CTAs per SM instead of three
  static constexpr int NRP = (PHYS == PH_NS) ? NVAR * EB : 0;
  static constexpr int NSRC = 0;                             // (the chemistry source comes from eos_kernel's aux array)
  static constexpr int MDP = ((G::MD + DIM + 1) / 2) * 2;
  static constexpr size_t smem_doubles(bool affine) {
    return (size_t)(NFP + NRP) * PS + (size_t)NST * TILE + (size_t)NVAR * NTASK + NSRC + (affine ? EB * MDP : 0);
  }
};

// Viscous numerical flux F_v* (outward, own normal) at face node a0 of a 2-D mortar face f of element e (PAPER.md:223,
// 234; reading R23): the central flux of eq. 16 on the mortar.  The coarse side's state and its BR1 gradient
// (stored as stress tensor + heat flux, linear in the gradient) are interpolated to the mortar with P_fwd; fine side:
// F_v* = (F_v,own + F_v(P U_C, P tau_C).n)/2; coarse side: sum_m P_rev^m (2 (-(F_v(U_F, tau_F) + F_v(P U_C, P tau_C)).n_F / 2)).
// Fvm: the own viscous normal flux.  Rare path, kept out of line.
template <int NP>
__device__ __noinline__ void ns_mortar_viscous_2d(const StageParams &P, long e, int f, int a0, int2 cn, const double *Fvm,
                                                  const double *nv, double *Fvs) {
  using G = Geo<2, NP>;
  constexpr int NVAR = 4, NN = NP * NP, NTAU = Tau<2>::NTAU;
  const int kind = cn.y & 3, fR = (cn.y >> 2) & 7, sub = (cn.y >> 8) & 1;
  const double *Pf = P.mortar_mat, *Prv = P.mortar_mat + 2 * NP * NP;
  if (kind == FK_MORTAR_FINE) {
    double Ui[NVAR] = {0.0, 0.0, 0.0, 0.0}, ti[NTAU], Fvp[NVAR];
#pragma unroll
    for (int k = 0; k < NTAU; ++k) ti[k] = 0.0;
    for (int j = 0; j < NP; ++j) {
      const double w = __ldg(&Pf[(sub * NP + a0) * NP + j]);
      const int pC = G::face_node(fR, j, 0);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Ui[v] += w * __ldg(P.u_in + ((long)cn.x * NVAR + v) * NN + pC);
#pragma unroll
      for (int k = 0; k < NTAU; ++k) ti[k] += w * __ldg(P.S + ((long)cn.x * NTAU + k) * NN + pC);
    }
    const Prim<2> qi = prim_ideal<2, false>(Ui, P.gamma);
    viscous_flux_dot_tau<2>(qi.v, ti, nv, Fvp);
    Fvs[0] = 0.0;
#pragma unroll
    for (int v = 1; v < NVAR; ++v) Fvs[v] = 0.5 * (Fvm[v] + Fvp[v]);
  } else {
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Fvs[v] = 0.0;
    const int lF = fR >> 1;
    const double sF = (fR & 1) ? 1.0 : -1.0;
    const bool aff = P.affine_flag != 0;
    for (int m = 0; m < 2; ++m) {
      const long eF = __ldg(&P.mortar_fine[cn.x * 2 + m]);
      for (int a = 0; a < NP; ++a) {
        const int pF = G::face_node(fR, a, 0);
        double UF[NVAR], tF[NTAU], Ui[NVAR] = {0.0, 0.0, 0.0, 0.0}, ti[NTAU], nF[2], FvF[NVAR], FvC[NVAR];
#pragma unroll
        for (int v = 0; v < NVAR; ++v) UF[v] = __ldg(P.u_in + (eF * NVAR + v) * NN + pF);
#pragma unroll
        for (int k = 0; k < NTAU; ++k) {
          tF[k] = __ldg(P.S + (eF * NTAU + k) * NN + pF);
          ti[k] = 0.0;
        }
        for (int j = 0; j < NP; ++j) {
          const double w = __ldg(&Pf[(m * NP + a) * NP + j]);
          const int pC = G::face_node(f, j, 0);
#pragma unroll
          for (int v = 0; v < NVAR; ++v) Ui[v] += w * __ldg(P.u_in + (e * NVAR + v) * NN + pC);
#pragma unroll
          for (int k = 0; k < NTAU; ++k) ti[k] += w * __ldg(P.S + (e * NTAU + k) * NN + pC);
        }
#pragma unroll
        for (int c = 0; c < 2; ++c)
          nF[c] = sF * (aff ? __ldg(&P.metric[eF * 5 + lF * 2 + c]) : __ldg(&P.metric[(eF * 5 + lF * 2 + c) * NN + pF]));
        const Prim<2> qF = prim_ideal<2, false>(UF, P.gamma);
        const Prim<2> qi = prim_ideal<2, false>(Ui, P.gamma);
        viscous_flux_dot_tau<2>(qF.v, tF, nF, FvF);
        viscous_flux_dot_tau<2>(qi.v, ti, nF, FvC);
        const double w2 = -2.0 * __ldg(&Prv[(m * NP + a0) * NP + a]);
#pragma unroll
        for (int v = 1; v < NVAR; ++v) Fvs[v] += w2 * (0.5 * (FvF[v] + FvC[v]));
      }
    }
  }
}

// Navier-Stokes across 3-D 4:1 mortars (readings R21 + R23): the TOTAL numerical flux T = F*_hyp - F_v* at the 4 n^2 fine
// face nodes of every mortar (outward for the fine side, its normal), evaluated once per mortar ahead of the stage -- the
// Rusanov flux of mortar_flux3d_kernel minus the central viscous flux (F_v(U_F, tau_F) + F_v(P U_C, P tau_C)).n_F / 2,
// P = Pf[s0] x Pf[s1] applied to the coarse face's state and stored stress tensor / heat flux.  HYP = false: -F_v* alone
// (the viscous-only launch after stage_split_kernel).  The stage then treats T exactly as the Euler kernels treat the
// stored Rusanov flux (node_mortar_flux_3d).  One CTA per mortar, one thread per (sub-face, fine face node).  Affine.
template <int NP, bool HYP>
__global__ void __launch_bounds__(4 * NP * NP) mortar_flux3d_ns_kernel(const double *__restrict__ u, const double *__restrict__ S,
                                                                       const double *__restrict__ metric, const int *__restrict__ info,
                                                                       const int *__restrict__ mortar_fine,
                                                                       const double *__restrict__ mortar_mat, double gamma,
                                                                       double *__restrict__ mflux) {
  using G = Geo<3, NP>;
  constexpr int NVAR = 5, NN = NP * NP * NP, NF = NP * NP, MD = 10, NTAU = Tau<3>::NTAU, NC = NVAR + NTAU;
  __shared__ double UC[NF * NC], Pfs[2 * NP * NP];      // coarse face: state and stored viscous tensor per face node
  const long m = blockIdx.x;
  const int tid = threadIdx.x;
  const int eC = info[m * 3], fC = info[m * 3 + 1], fF = info[m * 3 + 2];
  for (int i = tid; i < NF * NC; i += 4 * NF) {
    const int j = i / NC, k = i - j * NC;
    const int pC = G::face_node(fC, j % NP, j / NP);
    UC[i] = (k < NVAR) ? __ldg(u + ((long)eC * NVAR + k) * NN + pC) : __ldg(S + ((long)eC * NTAU + (k - NVAR)) * NN + pC);
  }
  for (int i = tid; i < 2 * NP * NP; i += 4 * NF) Pfs[i] = __ldg(&mortar_mat[i]);
  __syncthreads();
  const int s = tid / NF, b = tid - s * NF, b0 = b % NP, b1 = b / NP, s0 = s & 1, s1 = s >> 1;
  const long eF = mortar_fine[m * 4 + s];
  const int pF = G::face_node(fF, b0, b1), lF = fF >> 1;
  const double sF = (fF & 1) ? 1.0 : -1.0;
  double UF[NVAR], tF[NTAU], Ci[NC], nF[3], T[NVAR];
#pragma unroll
  for (int v = 0; v < NVAR; ++v) UF[v] = __ldg(u + (eF * NVAR + v) * NN + pF);
#pragma unroll
  for (int k = 0; k < NTAU; ++k) tF[k] = __ldg(S + (eF * NTAU + k) * NN + pF);
#pragma unroll
  for (int k = 0; k < NC; ++k) Ci[k] = 0.0;
  for (int j1 = 0; j1 < NP; ++j1) {
    const double w1 = Pfs[(s1 * NP + b1) * NP + j1];
    for (int j0 = 0; j0 < NP; ++j0) {
      const double w = Pfs[(s0 * NP + b0) * NP + j0] * w1;
#pragma unroll
      for (int k = 0; k < NC; ++k) Ci[k] += w * UC[(j0 + NP * j1) * NC + k];
    }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) nF[c] = sF * __ldg(&metric[eF * MD + lF * 3 + c]);
  const Prim<3> qF = prim_ideal<3, true>(UF, gamma);
  const Prim<3> qC = prim_ideal<3, true>(Ci, gamma);
  if constexpr (HYP) {
    double FmF[NVAR];
    flux_dot<3, 1>(UF, qF, nF, FmF);
    rusanov<3, 1>(UF, qF, FmF, Ci, qC, nF, T);
  } else {
#pragma unroll
    for (int v = 0; v < NVAR; ++v) T[v] = 0.0;
  }
  double FvF[NVAR], FvC[NVAR];
  viscous_flux_dot_tau<3>(qF.v, tF, nF, FvF);
  viscous_flux_dot_tau<3>(qC.v, Ci + NVAR, nF, FvC);
#pragma unroll
  for (int v = 1; v < NVAR; ++v) T[v] -= 0.5 * (FvF[v] + FvC[v]);
#pragma unroll
  for (int v = 0; v < NVAR; ++v) mflux[((m * 4 + s) * NF + b) * NVAR + v] = T[v];
}
template <int NP>
cudaError_t launch_mortar_flux3d_ns_t(bool hyp, const double *u, const double *S, const double *metric, const int *info,
                                      const int *fine, const double *mat, double gamma, double *mflux, long n_mortar,
                                      cudaStream_t st) {
  if (hyp) mortar_flux3d_ns_kernel<NP, true><<<(unsigned)n_mortar, 4 * NP * NP, 0, st>>>(u, S, metric, info, fine, mat, gamma, mflux);
  else mortar_flux3d_ns_kernel<NP, false><<<(unsigned)n_mortar, 4 * NP * NP, 0, st>>>(u, S, metric, info, fine, mat, gamma, mflux);
  return cudaGetLastError();
}

// BND (Navier-Stokes): the instantiation for meshes with boundary faces -- prescribed states, outflow, slip walls and the
// no-slip adiabatic / isothermal walls of PAPER.md:223 (readings R18, R22); the default one carries no code
// for them.
// VONLY (Navier-Stokes): the parabolic operator alone, ADDED to u_out: u_out += cc * L_visc(u_in).  Second launch of a
// stage whose hyperbolic part ran in stage_split_kernel (split-form / blended volume integral, PAPER.md:183-191, 208:
// the two pipelines "add their contributions into a shared residual buffer").
template <int DIM, int NP, int NSP, int PHYS, bool AFFINE, int EB, int MINB, bool BND = false, bool VONLY = false>
__global__ void __launch_bounds__((PhysCfg<DIM, NP, NSP, PHYS, EB>::NT), MINB)
stage_phys_kernel(const __grid_constant__ StageParams P) {
  using C = PhysCfg<DIM, NP, NSP, PHYS, EB>;
  using G = Geo<DIM, NP>;
  constexpr int NVAR = C::NVAR, NW = C::NW, NN = C::NN, NF = C::NF, TILE = C::TILE, NFN = C::NFN, NTASK = C::NTASK;
  constexpr int NT = C::NT, MD = G::MD, MDP = C::MDP, KS = C::KS, PS = C::PS;
  constexpr int NL = NF, NLT = NVAR * NL;
  extern __shared__ __align__(16) double smem[];
  double *Fsm = smem;                         // [DIM][NVAR][EB] flux planes (kept intact)
  double *Rsm = (PHYS == PH_NS) ? Fsm + C::NFP * PS : Fsm;   // [NVAR][EB] result planes (reacting: the xi flux planes, in place)
  double *Ust = Fsm + (C::NFP + C::NRP) * PS; // [NVAR + 3][TILE]  U, 1/rho, p, a
  double *Lft = Ust + C::NST * TILE;          // [NVAR][NTASK]     lifts of the face nodes
  double *Msm = Lft + NVAR * NTASK;                // affine: [EB][MDP] Ja, 1/J, |Ja^l|

  const int tid = threadIdx.x;
  // P.reverse (Navier-Stokes: set by the library): the blocks are walked from the last element to the first, against the
  // direction of the gradient sweep ahead of this launch -- it starts on the stress planes that sweep wrote last (still
  // in L2) and ends where the next stage's gradient sweep starts reading u_out
  const long e0 = (P.reverse ? (long)gridDim.x - 1 - (long)blockIdx.x : (long)blockIdx.x) * EB;
  const int nel = (int)((P.ne - e0 < EB) ? (P.ne - e0) : EB);
  const int ntask = nel * NFN, nline = nel * NLT;

  // L2 prefetch of the per-node planes that a CTA launched about half a wave later reads in its phase N: turns their DRAM
  // latency into L2 hits (rounded outwards to 16 bytes: kept inside the arrays by stopping one block short of the end).
  // Measured (c5, ms per step): none 1.751, 148 * MINB blocks ahead 1.682, 74 * MINB 1.678, 296 * MINB 1.712, with u_n
  // as well 1.687; c3 (power-capped, DRAM-side) does not move with any of them.
  if (tid == 0) {
    const long ep = e0 + (P.reverse ? -1L : 1L) * (74 * MINB) * EB;
    if (ep >= 0 && ep + EB < P.ne) {
      l2_prefetch(P.u_in + ep * NVAR * NN, (size_t)EB * NVAR * NN * sizeof(double));
      if constexpr (PHYS == PH_NS) l2_prefetch(P.S + ep * Tau<DIM>::NTAU * NN, (size_t)EB * Tau<DIM>::NTAU * NN * sizeof(double));
      if constexpr (!AFFINE) l2_prefetch(P.metric + ep * MD * NN, (size_t)EB * MD * NN * sizeof(double));
      if constexpr (PHYS == PH_REACT) l2_prefetch(P.Taux + ep * (2 + NSP) * NN, (size_t)EB * (2 + NSP) * NN * sizeof(double));
    }
  }
  // first face task of this thread: connectivity load first (the neighbour gather depends on it)
  const bool has0 = tid < ntask;
  const FaceTask t0 = decode_task<DIM, NP>(has0 ? tid : 0);
  int2 cn0 = make_int2(0, 0);
  if (has0) cn0 = __ldg(&P.conn[(e0 + t0.el) * 2 * DIM + t0.f]);

  constexpr int NA = 2 + NSP;                 // reacting: planes of the aux array (p, a, omega_s)
  if constexpr (AFFINE) {
    for (int i = tid; i < nel * MDP; i += NT) {
      const int me = i / MDP, k = i - me * MDP;
      Msm[i] = (k < MD) ? __ldg(&P.metric[(e0 + me) * MD + k]) : ((k < MD + DIM) ? __ldg(&P.fnorm[(e0 + me) * DIM + (k - MD)]) : 0.0);
    }
  }
  const int el = tid / NN, p = tid - el * NN;
  const long e = e0 + el;
  const bool active = (tid < TILE) && (el < nel);
  double U[NVAR], pA = 0.0, aA = 0.0;         // reacting: pressure and frozen sound speed from eos_kernel
  if (active) {
    const double *up = P.u_in + e * NVAR * NN + p;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) U[v] = __ldg(up + v * NN);
    // what only the last pass reads -- 1/J of curved meshes, u_n -- is brought into L2 now (prefetches hold no registers)
    if constexpr (!AFFINE) asm volatile("prefetch.global.L2 [%0];" ::"l"(&P.metric[(e * MD + DIM * DIM) * NN + p]));
    if (!VONLY && P.ca != 0.0) {
#pragma unroll
      for (int v = 0; v < NVAR; ++v) asm volatile("prefetch.global.L2 [%0];" ::"l"(P.u_n + (e * NVAR + v) * NN + p));
    }
    if constexpr (PHYS == PH_REACT) {
      pA = __ldg(&P.Taux[e * NA * NN + p]);
      aA = __ldg(&P.Taux[(e * NA + 1) * NN + p]);
    }
  }
  // neighbour trace of the first face task: in flight during phase N
  double Up0[NVAR], pp0 = 0.0, ap0 = 0.0;
  int pR0 = 0;
  if (has0 && (!BND || (cn0.y & 3) == FK_CONFORMING)) {
    const int fR = (cn0.y >> 2) & 7, orient = (cn0.y >> 5) & 7;
    int b0, b1;
    partner_index<DIM, NP>(orient, t0.a0, t0.a1, b0, b1);
    pR0 = face_node_of<DIM, NP>(fR, b0, b1);
    const double *un = P.u_in + (long)cn0.x * NVAR * NN + pR0;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Up0[v] = __ldg(un + v * NN);
    if constexpr (PHYS == PH_REACT) {
      pp0 = __ldg(&P.Taux[(long)cn0.x * NA * NN + pR0]);
      ap0 = __ldg(&P.Taux[((long)cn0.x * NA + 1) * NN + pR0]);
    }
  }

  // ---- phase N: own node
  if (active) {
    const int qk = (DIM == 3) ? p / (NP * NP) : 0;
    const int sp = p + (KS - NP * NP) * qk;
    double Ja[DIM * DIM];
#pragma unroll
    for (int k = 0; k < DIM * DIM; ++k) Ja[k] = metric_at<DIM, NP, AFFINE>(P.metric, e, k, p);
    Prim<DIM> pr;
    if constexpr (PHYS == PH_REACT) pr = prim_given_pa<DIM, NSP>(U, pA, aA);
    else pr = prim_ideal<DIM, true>(U, P.gamma);
    double Sg[(PHYS == PH_NS) ? NW * DIM : 1];
    if constexpr (PHYS == PH_NS) {
#pragma unroll
      for (int k = 0; k < Tau<DIM>::NTAU; ++k) Sg[k] = __ldg(&P.S[(e * Tau<DIM>::NTAU + k) * NN + p]);
    }
#pragma unroll
    for (int l = 0; l < DIM; ++l) {
      double F[NVAR];
      if constexpr (VONLY) {
#pragma unroll
        for (int v = 0; v < NVAR; ++v) F[v] = 0.0;
      } else flux_dot<DIM, NSP>(U, pr, &Ja[l * DIM], F);
      if constexpr (PHYS == PH_NS) {
        double Fv[NW];
        viscous_flux_dot_tau<DIM>(pr.v, Sg, &Ja[l * DIM], Fv);
#pragma unroll
        for (int v = 0; v < NVAR; ++v) F[v] -= Fv[v];
      }
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Fsm[((l * NVAR + v) * EB + el) * PS + sp] = F[v];
    }
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Ust[v * TILE + tid] = U[v];
    Ust[NVAR * TILE + tid] = pr.irho;
    Ust[(NVAR + 1) * TILE + tid] = pr.p;
    Ust[(NVAR + 2) * TILE + tid] = pr.a;
  }
  __syncthreads();

  // ---- xi pass (eq. 9): lines (j,k) of variable v -> result planes
  for (int t = tid; t < nline; t += NT) {
    const int le = t / NLT, r = t - le * NLT;
    const int v = r / NL, ln = r - v * NL;
    const int lj = ln % NP, lk = ln / NP;
    const int off = (v * EB + le) * PS + NP * lj + KS * lk;
    double f[NP], acc[NP];
#pragma unroll
    for (int m = 0; m < NP; ++m) { f[m] = Fsm[off + m]; acc[m] = 0.0; }
    line_deriv<NP>(P, f, acc);
#pragma unroll
    for (int i = 0; i < NP; ++i) Rsm[off + i] = acc[i];
  }

  // ---- face tasks, densely mapped (a2; NS: + BR1 viscous interface flux, eq. 16)
  for (int g = tid; g < ntask; g += NT) {
    FaceTask t;
    int2 cn;
    double Up[NVAR], pp = 0.0, ap = 0.0;
    int pR;
    if (g == tid) {
      t = t0; cn = cn0; pR = pR0; pp = pp0; ap = ap0;
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Up[v] = Up0[v];
    } else {
      t = decode_task<DIM, NP>(g);
      cn = __ldg(&P.conn[(e0 + t.el) * 2 * DIM + t.f]);
      pR = 0;
      if (!BND || (cn.y & 3) == FK_CONFORMING) {
        const int fR = (cn.y >> 2) & 7, orient = (cn.y >> 5) & 7;
        int b0, b1;
        partner_index<DIM, NP>(orient, t.a0, t.a1, b0, b1);
        pR = face_node_of<DIM, NP>(fR, b0, b1);
        const double *un = P.u_in + (long)cn.x * NVAR * NN + pR;
#pragma unroll
        for (int v = 0; v < NVAR; ++v) Up[v] = __ldg(un + v * NN);
        if constexpr (PHYS == PH_REACT) {
          pp = __ldg(&P.Taux[(long)cn.x * NA * NN + pR]);
          ap = __ldg(&P.Taux[((long)cn.x * NA + 1) * NN + pR]);
        }
      }
    }
    const bool bnd = BND && (cn.y & 3) == FK_BOUNDARY;
    const int bk = (cn.y >> 2) & 7;                 // boundary kind (boundary faces only)
    const int l = t.f >> 1;
    const double sgn = (t.f & 1) ? 1.0 : -1.0;
    const int idx = t.el * NN + t.p;
    const long ee = e0 + t.el;
    double Um[NVAR], nv[DIM], nrm;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Um[v] = Ust[v * TILE + idx];
    const double irhom = Ust[NVAR * TILE + idx], pm = Ust[(NVAR + 1) * TILE + idx], am = Ust[(NVAR + 2) * TILE + idx];
    if constexpr (AFFINE) {
#pragma unroll
      for (int c = 0; c < DIM; ++c) nv[c] = sgn * Msm[t.el * MDP + l * DIM + c];
      nrm = Msm[t.el * MDP + MD + l];
    } else {
      double n2 = 0.0;
#pragma unroll
      for (int c = 0; c < DIM; ++c) {
        nv[c] = sgn * __ldg(&P.metric[(ee * MD + l * DIM + c) * NN + t.p]);
        n2 += nv[c] * nv[c];
      }
      nrm = sqrt(n2);
    }
    const bool mort = BND && PHYS == PH_NS && (cn.y & 3) >= FK_MORTAR_FINE;   // 2:1 / 4:1 mortar face (readings R23, R21)
    if constexpr (BND) {
      if (mort) {
#pragma unroll
        for (int v = 0; v < NVAR; ++v) Up[v] = Um[v];       // (placeholder: the mortar flux replaces the lift below)
      }
      if (bnd) {
        // exterior state of the hyperbolic surface flux (R8, R18, R22): prescribed state; outflow: the interior
        // state; slip wall and the two no-slip walls: the interior state with the normal momentum reflected
#pragma unroll
        for (int v = 0; v < NVAR; ++v) Up[v] = (bk == BC_PRESCRIBED) ? __ldg(&P.bc_state[cn.x * NVAR + v]) : Um[v];
        if (bk >= BC_SLIP_WALL) {
          double mn = 0.0;
#pragma unroll
          for (int c = 0; c < DIM; ++c) mn += Um[NSP + c] * (nv[c] / nrm);
#pragma unroll
          for (int c = 0; c < DIM; ++c) Up[NSP + c] = Um[NSP + c] - 2.0 * mn * (nv[c] / nrm);
        }
      }
    }
    Prim<DIM> qp;
    if constexpr (PHYS == PH_REACT) qp = prim_given_pa<DIM, NSP>(Up, pp, ap);
    else qp = prim_ideal<DIM, true>(Up, P.gamma);
    double mnm = 0.0, vnp = 0.0;
#pragma unroll
    for (int c = 0; c < DIM; ++c) {
      mnm += Um[NSP + c] * nv[c];
      vnp += qp.v[c] * nv[c];
    }
    const double vnm = mnm * irhom;
    const double hl = 0.5 * fmax(fabs(vnm) + am * nrm, fabs(vnp) + qp.a * nrm);
    double Fm[NVAR], Fp[NVAR], lift[NVAR];
#pragma unroll
    for (int s = 0; s < NSP; ++s) {
      Fm[s] = Um[s] * vnm;
      Fp[s] = Up[s] * vnp;
    }
#pragma unroll
    for (int c = 0; c < DIM; ++c) {
      Fm[NSP + c] = Um[NSP + c] * vnm + pm * nv[c];
      Fp[NSP + c] = Up[NSP + c] * vnp + qp.p * nv[c];
    }
    Fm[NSP + DIM] = (Um[NSP + DIM] + pm) * vnm;
    Fp[NSP + DIM] = (Up[NSP + DIM] + qp.p) * vnp;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) lift[v] = 0.5 * (Fp[v] - Fm[v]) - hl * (Up[v] - Um[v]);
    if constexpr (VONLY) {      // no hyperbolic surface term; the flux planes hold -F_v . Ja, so the own F_v.n = -(plane) sgn
#pragma unroll
      for (int v = 0; v < NVAR; ++v) { lift[v] = 0.0; Fm[v] = 0.0; }
    }
    if constexpr (PHYS == PH_NS) {
      // viscous part: F_v* = mean of the two sides; own F_v.n = F_inv(U-).n - (own total normal flux in the plane)
      const int qk = (DIM == 3) ? t.p / (NP * NP) : 0;
      const int sp = t.p + (KS - NP * NP) * qk;
      if constexpr (BND && DIM == 2) {
        if (mort) {
          double Fvm[NVAR], Fvs[NVAR];
          Fvm[0] = 0.0;
#pragma unroll
          for (int v = 1; v < NVAR; ++v) Fvm[v] = Fm[v] - sgn * Fsm[((l * NVAR + v) * EB + t.el) * PS + sp];
          if constexpr (!VONLY) {
            double Fs[NVAR];
            node_mortar_flux_2d<NP>(P, ee, t.f, t.a0, cn, Um, nv, Fs);
#pragma unroll
            for (int v = 0; v < NVAR; ++v) lift[v] = Fs[v] - Fm[v];
          }
          ns_mortar_viscous_2d<NP>(P, ee, t.f, t.a0, cn, Fvm, nv, Fvs);
#pragma unroll
          for (int v = 1; v < NVAR; ++v) lift[v] -= Fvs[v] - Fvm[v];
        }
      }
      if constexpr (BND && DIM == 3 && AFFINE) {
        if (mort) {
          // the stored total flux T = F*_hyp - F_v* (mortar_flux3d_ns_kernel) against the own total normal flux
          double Fs[NVAR];
          node_mortar_flux_3d<NP>(P, t.a0, t.a1, cn, Fs);
#pragma unroll
          for (int v = 0; v < NVAR; ++v) lift[v] = Fs[v] - sgn * Fsm[((l * NVAR + v) * EB + t.el) * PS + sp];
        }
      }
      if (mort) {
      } else if (bnd) {
        // viscous wall flux F_v*(U_w, S-) (reading R22): momentum rows = the wall shear stress, as the element's own;
        // energy row: no stress work (v_w = 0), the heat flux k grad T . n at an isothermal wall, nothing at an
        // adiabatic one.  Prescribed / outflow / slip faces: F_v* = F_v(U-, S-), no viscous surface term.
        if (bk >= BC_WALL_ADIABATIC) {
          double FwE = 0.0;
          if (bk == BC_WALL_ISOTHERMAL) {
#pragma unroll
            for (int j = 0; j < DIM; ++j)
              FwE += __ldg(&P.S[(ee * Tau<DIM>::NTAU + DIM * (DIM + 1) / 2 + j) * NN + t.p]) * nv[j];
          }
          const double FvmE = Fm[NVAR - 1] - sgn * Fsm[((l * NVAR + NVAR - 1) * EB + t.el) * PS + sp];
          lift[NVAR - 1] -= FwE - FvmE;
        }
      } else {
        double Sp[NW * DIM], Fvp[NW];
#pragma unroll
        for (int k = 0; k < Tau<DIM>::NTAU; ++k) Sp[k] = __ldg(&P.S[((long)cn.x * Tau<DIM>::NTAU + k) * NN + pR]);
        viscous_flux_dot_tau<DIM>(qp.v, Sp, nv, Fvp);
#pragma unroll
        for (int v = 1; v < NVAR; ++v) {
          const double Fvm = Fm[v] - sgn * Fsm[((l * NVAR + v) * EB + t.el) * PS + sp];
          lift[v] -= 0.5 * (Fvp[v] - Fvm);
        }
      }
    }
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Lft[v * NTASK + g] = P.inv_wb * lift[v];
  }
  __syncthreads();

  if constexpr (DIM == 3) {
    // ---- eta pass: lines (i,k) of variable v; lane order (k, v, i)
    for (int t = tid; t < nline; t += NT) {
      const int le = t / NLT, r = t - le * NLT;
      const int lk = r % NP, r2 = r / NP;
      const int v = r2 % NVAR, li = r2 / NVAR;
      const int off = (v * EB + le) * PS + li + KS * lk;
      const double *pe = Fsm + NVAR * EB * PS + off;
      double f[NP], acc[NP];
#pragma unroll
      for (int m = 0; m < NP; ++m) { f[m] = pe[m * NP]; acc[m] = Rsm[off + m * NP]; }
      line_deriv<NP>(P, f, acc);
#pragma unroll
      for (int j = 0; j < NP; ++j) Rsm[off + j * NP] = acc[j];
    }
    __syncthreads();
  }

  // ---- last pass (zeta in 3-D, eta in 2-D) fused with phase D: lifts, 1/J, source, SSP-RK combination
  const bool use_un = !VONLY && (P.ca != 0.0);
  for (int t = tid; t < nline; t += NT) {
    const int le = t / NLT, r = t - le * NLT;
    const int v = r / NL, ij = r - v * NL;
    constexpr int LS = (DIM == 3) ? KS : NP;
    constexpr int GS = (DIM == 3) ? NP * NP : NP;
    const long ee = e0 + le;
    const int off = (v * EB + le) * PS + ij;
    const double *pl = Fsm + (DIM - 1) * NVAR * EB * PS + off;
    const long gofs = (ee * NVAR + v) * NN + ij;
    double un[NP];
    if (use_un) {
#pragma unroll
      for (int m = 0; m < NP; ++m) un[m] = P.u_n[gofs + m * GS];
    }
    double f[NP], acc[NP];
#pragma unroll
    for (int m = 0; m < NP; ++m) { f[m] = pl[m * LS]; acc[m] = Rsm[off + m * LS]; }
    line_deriv<NP>(P, f, acc);
    const double *lf = Lft + v * NTASK + le * NFN;
    if constexpr (DIM == 3) {
      const int li = ij % NP, lj = ij / NP;
      acc[0] += lf[4 * NF + ij];
      acc[NP - 1] += lf[5 * NF + ij];
      if (li == 0 || li == NP - 1) {
        const double *l2 = lf + ((li == 0) ? 0 : NF) + lj;
#pragma unroll
        for (int m = 0; m < NP; ++m) acc[m] += l2[NP * m];
      }
      if (lj == 0 || lj == NP - 1) {
        const double *l2 = lf + ((lj == 0) ? 2 * NF : 3 * NF) + li;
#pragma unroll
        for (int m = 0; m < NP; ++m) acc[m] += l2[NP * m];
      }
    } else {
      acc[0] += lf[2 * NF + ij];
      acc[NP - 1] += lf[3 * NF + ij];
      if (ij == 0 || ij == NP - 1) {
        const double *l2 = lf + ((ij == 0) ? 0 : NF);
#pragma unroll
        for (int m = 0; m < NP; ++m) acc[m] += l2[m];
      }
    }
    const double *us = Ust + v * TILE + le * NN + ij;
    double invJ = 0.0;
    if constexpr (AFFINE) invJ = Msm[le * MDP + DIM * DIM];
#pragma unroll
    for (int m = 0; m < NP; ++m) {
      if constexpr (!AFFINE) invJ = __ldg(&P.metric[(ee * MD + DIM * DIM) * NN + ij + m * GS]);
      double src = 0.0;
      if constexpr (PHYS == PH_REACT) {
        if (v < NSP && P.explicit_source) src = __ldg(&P.Taux[(ee * NA + 2 + v) * NN + ij + m * GS]);
      }
      if constexpr (VONLY) {
        P.u_out[gofs + m * GS] += stage_cc(P) * (0.0 - invJ * acc[m]);
      } else {
        const double val = P.cb * us[m * GS] + stage_cc(P) * (src - invJ * acc[m]);
        P.u_out[gofs + m * GS] = use_un ? (P.ca * un[m] + val) : val;
      }
    }
  }
}

template <int DIM, int NP, int NSP, int PHYS, bool AFFINE, bool BND = false, bool VONLY = false>
cudaError_t launch_stage_phys_t(const StageParams &P, cudaStream_t st) {
  if constexpr (PHYS == PH_NS && !VONLY) {
    if (P.visc_only) return launch_stage_phys_t<DIM, NP, NSP, PHYS, AFFINE, true, true>(P, st);   // (one instantiation: with boundary code)
  }
  if constexpr (PHYS == PH_NS && !BND) {
    if (P.bc_kinds) return launch_stage_phys_t<DIM, NP, NSP, PHYS, AFFINE, true>(P, st);
  }
  constexpr int NN = Geo<DIM, NP>::NN, EB = node_eb<NN>();
  using C = PhysCfg<DIM, NP, NSP, PHYS, EB>;
  constexpr size_t smem = C::smem_doubles(AFFINE) * sizeof(double);
  constexpr int MINB = (C::NT <= 128) ? MARUT_PHYS_MINB128 : ((C::NT <= 256) ? 2 : 1);
  auto k = stage_phys_kernel<DIM, NP, NSP, PHYS, AFFINE, EB, MINB, BND, VONLY>;
  static std::atomic<unsigned long long> attr_done{0};
  if (cudaError_t err = set_smem_once((const void *)k, smem, attr_done); err != cudaSuccess) return err;
  const long grid = (P.ne + EB - 1) / EB;
  k<<<(unsigned)grid, C::NT, smem, st>>>(P);
  return cudaGetLastError();
}

}  // namespace marut
