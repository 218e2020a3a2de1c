// marut_line.cuh -- the fast fused stage kernel (Euler, 2-D / 3-D, affine or curved, conforming +
// boundary + 2-D mortar faces): one thread per xi-LINE of LGL nodes, EB elements per CTA.
//
//   phase 0  TMA bulk copies (cp.async.bulk + mbarrier) land the CTA's contiguous u_in tile and u_n tile
//            in shared memory (one pass over u per stage)
//   phase A  per line: primitives and contravariant fluxes (eq. 9); F^xi stays in registers, F^eta / F^zeta
//            go to shared memory in padded lines (128-bit, conflict-free)
//   phase B  volume term: xi from registers with compile-time D, eta / zeta from broadcast line reads
//   phase C  interface flux (a2-a4): xi faces from the owner's registers; eta / zeta faces densely mapped
//            (every thread one face node per face), result written in place of the own normal flux
//   phase D  surface lift + 1/J + SSP-RK combination (eq. 12, 45) in place of the u_n tile, then one TMA
//            bulk store of the u_out tile
//
// Product code; shares nothing with oracle/.
#pragma once
#include "marut_kernels.cuh"

namespace marut {

// ---------------------------------------------------------------- PTX wrappers (sm_100a)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!ok);
}
__device__ __forceinline__ void bulk_load(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void bulk_store(void *dst_gmem, const void *src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_commit_wait_read() {
  asm volatile("cp.async.bulk.commit_group;\n\tcp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---------------------------------------------------------------- compile-time geometry of the line kernel
template <int DIM, int NP, int NSP, int EB>
struct LineCfg {
  static constexpr int NVAR = NSP + DIM + 1;
  static constexpr int NL = (DIM == 2) ? NP : NP * NP;   // xi-lines per element
  static constexpr int NN = NL * NP;
  static constexpr int NPP = NP + (NP & 1);              // padded line length (even -> 16-byte lines)
  static constexpr int NNP = NL * NPP;
  static constexpr int ESZ = NVAR * NN;                  // doubles per element in global memory
  static constexpr int TILE = (EB * ESZ + 2) & ~1;       // u tile incl. alignment slack (even)
  static constexpr int NT = ((EB * NL + 31) / 32) * 32;
  static constexpr int F_DOUBLES = (DIM - 1) * NVAR * EB * NNP;
  static constexpr int AUX_DOUBLES = 2 * EB * NN;        // 1/rho and a per node
  static constexpr size_t SMEM = sizeof(double) * (size_t)(2 * TILE + F_DOUBLES + AUX_DOUBLES + NP * NP) + 16;
};

// 2-D mortar faces: the numerical flux of face node a0 on face f of element e, by the rules of
// the generic kernel (fine side: coarse trace interpolated; coarse side: both mortars projected back, factor 2).
// Rare path, kept out of line.
template <int NP>
__device__ __noinline__ void mortar_flux_2d(const StageParams &P, long e, int f, int a0, int2 cn, const double *U,
                                            const double *nv, double *Fs) {
  using G = Geo<2, NP>;
  constexpr int NVAR = 4, NN = NP * NP;
  const int kind = cn.y & 3, fR = (cn.y >> 2) & 7, sub = (cn.y >> 8) & 1;
  const double *Pf = P.mortar_mat, *Prv = P.mortar_mat + 2 * NP * NP;
  const Prim<2> pr = prim_ideal<2, true>(U, P.gamma);
  if (kind == FK_MORTAR_FINE) {
    double Up[NVAR] = {0.0, 0.0, 0.0, 0.0};
    for (int j = 0; j < NP; ++j) {
      const double w = __ldg(&Pf[(sub * NP + a0) * NP + j]);
      const double *uc = P.u_in + (long)cn.x * NVAR * NN + G::face_node(fR, j, 0);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Up[v] += w * __ldg(uc + v * NN);
    }
    const Prim<2> qp = prim_ideal<2, true>(Up, P.gamma);
    double Fm[NVAR];
    flux_dot<2, 1>(U, pr, nv, Fm);
    rusanov<2, 1>(U, pr, Fm, Up, qp, nv, Fs);
  } else {
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Fs[v] = 0.0;
    for (int m = 0; m < 2; ++m) {
      const long eF = __ldg(&P.mortar_fine[cn.x * 2 + m]);
      const int lF = fR >> 1;
      const double sF = (fR & 1) ? 1.0 : -1.0;
      for (int a = 0; a < NP; ++a) {
        const int pF = G::face_node(fR, a, 0);
        double UF[NVAR], UC[NVAR], nF[2], FmF[NVAR], Fm_[NVAR];
#pragma unroll
        for (int v = 0; v < NVAR; ++v) {
          UF[v] = __ldg(P.u_in + (eF * NVAR + v) * NN + pF);
          UC[v] = 0.0;
        }
        for (int j = 0; j < NP; ++j) {
          const double w = __ldg(&Pf[(m * NP + a) * NP + j]);
          const double *uc = P.u_in + e * NVAR * NN + G::face_node(f, j, 0);
#pragma unroll
          for (int v = 0; v < NVAR; ++v) UC[v] += w * __ldg(uc + v * NN);
        }
        // fine-side normal (the mesh is affine or curved: read the fine element's metric at its face node)
        const bool aff = P.affine_flag != 0;
#pragma unroll
        for (int c = 0; c < 2; ++c)
          nF[c] = sF * (aff ? __ldg(&P.metric[eF * 5 + lF * 2 + c]) : __ldg(&P.metric[(eF * 5 + lF * 2 + c) * NN + pF]));
        const Prim<2> qF = prim_ideal<2, true>(UF, P.gamma);
        const Prim<2> qC = prim_ideal<2, true>(UC, P.gamma);
        flux_dot<2, 1>(UF, qF, nF, FmF);
        rusanov<2, 1>(UF, qF, FmF, UC, qC, nF, Fm_);
        const double w2 = -2.0 * __ldg(&Prv[(m * NP + a0) * NP + a]);
#pragma unroll
        for (int v = 0; v < NVAR; ++v) Fs[v] += w2 * Fm_[v];
      }
    }
  }
}

// Rusanov flux with a scaled normal, division-free (R5):
//   lambda |nv| = max(|v-.nv| + a- |nv|, |v+.nv| + a+ |nv|)
// Fm = F(U-).nv is passed in (the owner already has it from the volume flux).
template <int DIM, int NVAR>
__device__ __forceinline__ void rusanov_scaled(const double *Um, double irhom, double am, const double *Fm, const double *Up,
                                               double gamma, const double *nv, double nrm, double *Fs) {
  const double irhop = 1.0 / Up[0];
  double mnm = 0.0, mnp = 0.0, kep = 0.0;
#pragma unroll
  for (int c = 0; c < DIM; ++c) {
    mnm += Um[1 + c] * nv[c];
    mnp += Up[1 + c] * nv[c];
    kep += Up[1 + c] * Up[1 + c];
  }
  const double pp = (gamma - 1.0) * (Up[DIM + 1] - 0.5 * kep * irhop);
  const double ap = sqrt(gamma * pp * irhop);
  const double vnm = mnm * irhom, vnp = mnp * irhop;
  const double hl = 0.5 * fmax(fabs(vnm) + am * nrm, fabs(vnp) + ap * nrm);
  double Fp[NVAR];
  Fp[0] = mnp;
#pragma unroll
  for (int c = 0; c < DIM; ++c) Fp[1 + c] = Up[1 + c] * vnp + pp * nv[c];
  Fp[DIM + 1] = (Up[DIM + 1] + pp) * vnp;
#pragma unroll
  for (int v = 0; v < NVAR; ++v) Fs[v] = 0.5 * (Fm[v] + Fp[v]) - hl * (Up[v] - Um[v]);
}

// numerical flux at one face node of element e, face f (all face kinds)
template <int DIM, int NP>
__device__ __forceinline__ void face_flux(const StageParams &P, long e, int f, int a0, int a1, const double *Um, double irhom,
                                          double am, const double *Fm, const double *nv, double nrm, double *Fs) {
  using G = Geo<DIM, NP>;
  constexpr int NVAR = DIM + 2, NN = G::NN;
  const int2 cn = __ldg(&P.conn[e * 2 * DIM + f]);
  const int kind = cn.y & 3;
  if (kind == FK_CONFORMING || kind == FK_BOUNDARY) {
    double Up[NVAR];
    if (kind == FK_CONFORMING) {
      const int fR = (cn.y >> 2) & 7, orient = (cn.y >> 5) & 7;
      int b0, b1;
    partner_index<DIM, NP>(orient, a0, a1, b0, b1);
      const double *un = P.u_in + (long)cn.x * NVAR * NN + G::face_node(fR, b0, b1);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Up[v] = __ldg(un + v * NN);
    } else {
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Up[v] = __ldg(&P.bc_state[cn.x * NVAR + v]);
    }
    rusanov_scaled<DIM, NVAR>(Um, irhom, am, Fm, Up, P.gamma, nv, nrm, Fs);
  } else {
    if constexpr (DIM == 2) mortar_flux_2d<NP>(P, e, f, a0, cn, Um, nv, Fs);
  }
}

template <int DIM, int NP, bool AFFINE, int EB>
__global__ void __launch_bounds__((LineCfg<DIM, NP, 1, EB>::NT)) stage_line_kernel(const __grid_constant__ StageParams P) {
  using C = LineCfg<DIM, NP, 1, EB>;
  using G = Geo<DIM, NP>;
  constexpr int NVAR = C::NVAR, NL = C::NL, NN = C::NN, NPP = C::NPP, NNP = C::NNP, ESZ = C::ESZ, MD = G::MD;
  constexpr int FPL = NVAR * EB * NNP;   // doubles per flux direction plane set
  extern __shared__ __align__(16) double smem[];
  double *Ubuf = smem, *Nbuf = Ubuf + C::TILE, *Fsm = Nbuf + C::TILE, *Aux = Fsm + C::F_DOUBLES, *Dsm = Aux + C::AUX_DOUBLES;
  uint64_t *bars = reinterpret_cast<uint64_t *>(Dsm + NP * NP);

  const int tid = threadIdx.x;
  const long e0 = (long)blockIdx.x * EB;
  const int nel = (int)((P.ne - e0 < EB) ? (P.ne - e0) : EB);
  const long g0 = e0 * ESZ;
  const int len = nel * ESZ, head = (int)(g0 & 1), alen = (len - head) & ~1;
  double *Ut = Ubuf + head, *Nt = Nbuf + head;   // tile bases: global double g -> Ut[g - g0]
  const bool use_un = (P.ca != 0.0);

  // ---- phase 0: TMA bulk loads of the u_in and u_n tiles
  if (tid == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
    mbar_expect_tx(&bars[0], (uint32_t)alen * 8u);
    bulk_load(Ut + head, P.u_in + g0 + head, (uint32_t)alen * 8u, &bars[0]);
    if (head) Ut[0] = __ldg(P.u_in + g0);
    if (head + alen < len) Ut[len - 1] = __ldg(P.u_in + g0 + len - 1);
    if (use_un) {
      mbar_expect_tx(&bars[1], (uint32_t)alen * 8u);
      bulk_load(Nt + head, P.u_n + g0 + head, (uint32_t)alen * 8u, &bars[1]);
      if (head) Nt[0] = P.u_n[g0];
      if (head + alen < len) Nt[len - 1] = P.u_n[g0 + len - 1];
    }
  }
  for (int i = tid; i < NP * NP; i += C::NT) Dsm[i] = P.D[i];

  const int el = tid / NL, ln = tid - el * NL;
  const int j = ln % NP, k = ln / NP;   // k = 0 in 2-D
  const bool active = (tid < EB * NL) && (el < nel);
  const long e = e0 + el;
  double Ja[DIM * DIM], invJ = 0.0, fn[DIM];
  if (AFFINE && active) {
#pragma unroll
    for (int q = 0; q < DIM * DIM; ++q) Ja[q] = __ldg(&P.metric[e * MD + q]);
    invJ = __ldg(&P.metric[e * MD + DIM * DIM]);
#pragma unroll
    for (int l = 0; l < DIM; ++l) fn[l] = __ldg(&P.fnorm[e * DIM + l]);
  }
  mbar_wait(&bars[0], 0);
  __syncthreads();

  // ---- phase A: primitives and contravariant fluxes of the own line
  double Fx[NP][NVAR];
  double irho_e[2] = {0.0, 0.0}, a_e[2] = {0.0, 0.0};   // line end points (xi faces)
  if (active) {
    const double *ul = Ut + (el * NVAR) * NN + ln * NP;
    double *fl = Fsm + el * NNP + ln * NPP;
    double *ax = Aux + el * NN + ln * NP;
#pragma unroll
    for (int i2 = 0; i2 < NPP / 2; ++i2) {
      double Fo[2][(DIM - 1) * NVAR];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int i = 2 * i2 + h;
        if (i < NP) {
          double U[NVAR];
#pragma unroll
          for (int v = 0; v < NVAR; ++v) U[v] = ul[v * NN + i];
          if constexpr (!AFFINE) {
#pragma unroll
            for (int q = 0; q < DIM * DIM; ++q) Ja[q] = __ldg(&P.metric[(e * MD + q) * NN + ln * NP + i]);
          }
          const Prim<DIM> pr = prim_ideal<DIM, true>(U, P.gamma);
          flux_dot<DIM, 1>(U, pr, &Ja[0], Fx[i]);
#pragma unroll
          for (int l = 1; l < DIM; ++l) flux_dot<DIM, 1>(U, pr, &Ja[l * DIM], &Fo[h][(l - 1) * NVAR]);
          ax[i] = pr.irho;
          ax[EB * NN + i] = pr.a;
          if (i == 0) { irho_e[0] = pr.irho; a_e[0] = pr.a; }
          if (i == NP - 1) { irho_e[1] = pr.irho; a_e[1] = pr.a; }
        } else {
#pragma unroll
          for (int q = 0; q < (DIM - 1) * NVAR; ++q) Fo[h][q] = 0.0;
        }
      }
#pragma unroll
      for (int q = 0; q < (DIM - 1) * NVAR; ++q)
        *reinterpret_cast<double2 *>(fl + (q / NVAR) * FPL + (q % NVAR) * EB * NNP + 2 * i2) = make_double2(Fo[0][q], Fo[1][q]);
    }
  }
  __syncthreads();

  // ---- phase B: volume term  sum_l D_l Ftilde^l  (eq. 9)
  double R[NP][NVAR];
  if (active) {
#pragma unroll
    for (int i = 0; i < NP; ++i)
#pragma unroll
      for (int v = 0; v < NVAR; ++v) {
        double acc = 0.0;
#pragma unroll
        for (int m = 0; m < NP; ++m) acc += P.D[i * NP + m] * Fx[m][v];
        R[i][v] = acc;
      }
#pragma unroll
    for (int l = 1; l < DIM; ++l) {
      const int jl = (l == 1) ? j : k;
#pragma unroll
      for (int m = 0; m < NP; ++m) {
        const double d = Dsm[jl * NP + m];
        const int lnm = (l == 1) ? (k * NP + m) : (m * NP + j);
        const double *src = Fsm + (l - 1) * FPL + el * NNP + lnm * NPP;
#pragma unroll
        for (int v = 0; v < NVAR; ++v) {
          double line[NPP];
#pragma unroll
          for (int i2 = 0; i2 < NPP / 2; ++i2) {
            const double2 t = *reinterpret_cast<const double2 *>(src + v * EB * NNP + 2 * i2);
            line[2 * i2] = t.x;
            line[2 * i2 + 1] = t.y;
          }
#pragma unroll
          for (int i = 0; i < NP; ++i) R[i][v] += d * line[i];
        }
      }
    }

    // ---- phase C (xi faces): both end points of the own line, from registers
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      const int i = side ? NP - 1 : 0;
      const double sgn = side ? 1.0 : -1.0;
      double Um[NVAR], nv[DIM], Fm[NVAR], Fs[NVAR], nrm;
#pragma unroll
      for (int v = 0; v < NVAR; ++v) {
        Um[v] = Ut[(el * NVAR + v) * NN + ln * NP + i];
        Fm[v] = sgn * Fx[i][v];
      }
      if constexpr (AFFINE) {
#pragma unroll
        for (int c = 0; c < DIM; ++c) nv[c] = sgn * Ja[c];
        nrm = fn[0];
      } else {
        double n2 = 0.0;
#pragma unroll
        for (int c = 0; c < DIM; ++c) {
          nv[c] = sgn * __ldg(&P.metric[(e * MD + c) * NN + ln * NP + i]);
          n2 += nv[c] * nv[c];
        }
        nrm = sqrt(n2);
      }
      face_flux<DIM, NP>(P, e, side, j, k, Um, irho_e[side], a_e[side], Fm, nv, nrm, Fs);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) R[i][v] += P.inv_wb * (Fs[v] - Fm[v]);
    }
  }
  __syncthreads();   // every line read of phase B is done: the flux planes may be overwritten

  // ---- phase C (eta / zeta faces): thread ln owns face node ln of each face; the lift contribution
  //      (F* - Ftilde.n)/w_b replaces the own normal flux in the flux plane
  if (active) {
#pragma unroll
    for (int f = 2; f < 2 * DIM; ++f) {
      const int l = f >> 1, side = f & 1;
      const double sgn = side ? 1.0 : -1.0;
      const int a0 = j, a1 = k;                 // face node (a0, a1) = (ln % NP, ln / NP)
      int p, pq;                                // volume node: unpadded / padded index
      if (DIM == 2) { p = a0 + NP * (side * (NP - 1)); pq = (side * (NP - 1)) * NPP + a0; }
      else if (l == 1) { p = a0 + NP * (side * (NP - 1) + NP * a1); pq = (a1 * NP + side * (NP - 1)) * NPP + a0; }
      else { p = a0 + NP * (a1 + NP * (side * (NP - 1))); pq = ((side * (NP - 1)) * NP + a1) * NPP + a0; }
      double Um[NVAR], nv[DIM], Fm[NVAR], Fs[NVAR], nrm;
      double *fp = Fsm + (l - 1) * FPL + el * NNP + pq;
#pragma unroll
      for (int v = 0; v < NVAR; ++v) {
        Um[v] = Ut[(el * NVAR + v) * NN + p];
        Fm[v] = sgn * fp[v * EB * NNP];
      }
      const double irhom = Aux[el * NN + p], am = Aux[EB * NN + el * NN + p];
      if constexpr (AFFINE) {
#pragma unroll
        for (int c = 0; c < DIM; ++c) nv[c] = sgn * Ja[l * DIM + c];
        nrm = fn[l];
      } else {
        double n2 = 0.0;
#pragma unroll
        for (int c = 0; c < DIM; ++c) {
          nv[c] = sgn * __ldg(&P.metric[(e * MD + l * DIM + c) * NN + p]);
          n2 += nv[c] * nv[c];
        }
        nrm = sqrt(n2);
      }
      face_flux<DIM, NP>(P, e, f, a0, a1, Um, irhom, am, Fm, nv, nrm, Fs);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) fp[v * EB * NNP] = P.inv_wb * (Fs[v] - Fm[v]);
    }
  }
  if (use_un) mbar_wait(&bars[1], 0);
  __syncthreads();

  // ---- phase D: lift of the eta / zeta faces, 1/J, SSP-RK combination (eq. 12, 45), in place of the u_n tile
  if (active) {
    const bool on_eta = (j == 0 || j == NP - 1), on_zeta = (DIM == 3) && (k == 0 || k == NP - 1);
    const double *ul = Ut + (el * NVAR) * NN + ln * NP;
    double *nl = Nt + (el * NVAR) * NN + ln * NP;
    const double *fl = Fsm + el * NNP + ln * NPP;
#pragma unroll
    for (int i = 0; i < NP; ++i) {
      if constexpr (!AFFINE) invJ = __ldg(&P.metric[(e * MD + DIM * DIM) * NN + ln * NP + i]);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) {
        double r = R[i][v];
        if (on_eta) r += fl[v * EB * NNP + i];
        if (on_zeta) r += fl[FPL + v * EB * NNP + i];
        const double val = P.cb * ul[v * NN + i] + stage_cc(P) * (0.0 - invJ * r);
        nl[v * NN + i] = use_un ? (P.ca * nl[v * NN + i] + val) : val;
      }
    }
  }
  fence_async_smem();
  __syncthreads();
  if (tid == 0) {
    bulk_store(P.u_out + g0 + head, Nt + head, (uint32_t)alen * 8u);
    if (head) P.u_out[g0] = Nt[0];
    if (head + alen < len) P.u_out[g0 + len - 1] = Nt[len - 1];
    bulk_commit_wait_read();
  }
}

// launch helper: EB elements per CTA chosen for ~100 KB of shared memory per CTA (2 CTAs / SM)
template <int DIM, int NP>
constexpr int line_eb() {
  constexpr int NL = (DIM == 2) ? NP : NP * NP, NN = NL * NP, NPP = NP + (NP & 1), NVAR = DIM + 2;
  constexpr int per = 8 * (2 * NVAR * NN + (DIM - 1) * NVAR * NL * NPP + 2 * NN);
  int eb = 128 / NL;
  if (eb > 100000 / per) eb = 100000 / per;
  return eb < 1 ? 1 : eb;
}

template <int DIM, int NP, bool AFFINE>
cudaError_t launch_stage_line_t(const StageParams &P, cudaStream_t st) {
  constexpr int EB = line_eb<DIM, NP>();
  using C = LineCfg<DIM, NP, 1, EB>;
  auto k = stage_line_kernel<DIM, NP, AFFINE, EB>;
  static bool attr = false;
  if (!attr) {
    cudaError_t err = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (err != cudaSuccess) return err;
    attr = true;
  }
  const long grid = (P.ne + EB - 1) / EB;
  k<<<(unsigned)grid, C::NT, C::SMEM, st>>>(P);
  return cudaGetLastError();
}

}  // namespace marut
