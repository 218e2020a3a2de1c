// marut_node.cuh -- the fused stage kernel of the CUDA path, any dim / degree /
// physics: one thread per LGL node, EB elements per CTA, small register and shared-memory footprint so that
// 20-30 warps are resident per SM (the stage is latency-bound otherwise; profiles/r01_c2_stage_line_kernel.md).
//
//   phase N  per node: U from global (coalesced), primitives, contravariant fluxes (eq. 9) -> shared flux
//            planes; U and (1/rho, p, a) stashed in shared memory for the face phase
//   phase V  per node: volume term sum_l D_l Ftilde^l from the flux planes (broadcast line reads)
//   phase S  per FACE node, densely mapped (task g = tid, tid + NT, ...: every lane of a warp has a face
//            node): neighbour trace gathered from global (issued before phase V, consumed after), Rusanov /
//            mortar / boundary flux (a2-a4), lift (F* - Ftilde.n)/w_b -> shared lift buffer
//   phase D  per node: lifts of the faces the node lies on, 1/J, source, SSP-RK combination (eq. 12, 45),
//            u_n read and u_out written straight from / to global (coalesced): one pass over u per stage
//
// Product code; shares nothing with oracle/.
#pragma once
#include "marut_kernels.cuh"

namespace marut {

// shared-memory layout of one variable plane of one element: node (i,j,k) at i + NP*j + KS*k, planes PS apart.
// KS / PS / the lane order of the plane tasks are chosen so that the node threads (consecutive nodes), the
// (v,k)-plane tasks (offset k*KS) and the (v,i)-plane tasks (offset i) all hit 16 distinct 8-byte banks per
// half-warp (brute-force search over the strides).
template <int DIM, int NP, int EB>
struct NodeLayout {
  static constexpr int KS = NP * NP;
  static constexpr int PS = (DIM == 2) ? (NP * NP + 1) : ((NP * KS) | 1);
  static constexpr bool K_FASTEST = true;
};
template <int EB>
struct NodeLayout<3, 5, EB> {
  static constexpr int KS = 25, PS = 125;   // unpadded: with the lane orders of the three passes below every
  static constexpr bool K_FASTEST = false;  // half-warp hits 16 distinct banks in the xi and eta passes
};
template <int EB>
struct NodeLayout<3, 4, EB> {
  static constexpr int KS = 17, PS = (EB == 1) ? 68 : 70;
  static constexpr bool K_FASTEST = true;
};

template <int DIM, int NP, int NSP, int EB>
struct NodeCfg {
  using G = Geo<DIM, NP>;
  using L = NodeLayout<DIM, NP, EB>;
  static constexpr int NVAR = NSP + DIM + 1;
  static constexpr int NN = G::NN, NF = G::NF;
  static constexpr int TILE = EB * NN;
  static constexpr int NFN = 2 * DIM * NF;          // face nodes per element
  static constexpr int NTASK = EB * NFN;            // face tasks per CTA
  static constexpr int LFS = (DIM == 3 && NP == 5 && EB == 1) ? 160 : NTASK;   // stride of a variable in the lift buffer
  static constexpr int NT = ((TILE + 31) / 32) * 32;
  static constexpr int NW = NT / 32;
  static constexpr int NST = NVAR + 3;              // stash planes: U, 1/rho, p, a
  // plane of (variable, element) inside one direction's plane set: variable-major in 3-D, element-major in 2-D
  __host__ __device__ static constexpr int plane(int v, int el) { return (DIM == 2) ? el * NVAR + v : v * EB + el; }
  static constexpr int KS = L::KS, PS = L::PS;
  static constexpr int NPL = DIM * NVAR * EB;       // flux planes
  static constexpr int NVT = EB * NVAR * NP;        // plane tasks per derivative pass (3-D)
  static constexpr int MDP = ((G::MD + DIM + 1) / 2) * 2;   // per-element affine metric slot (Ja, 1/J, |Ja^l|)
  static constexpr size_t smem_doubles(bool affine) {
    return (size_t)NPL * PS + (size_t)NST * TILE + (size_t)NVAR * LFS + (affine ? EB * MDP : 0);
  }
};

// 2-D mortar faces (R7): numerical flux F* (outward, own normal) at face node a0 of
// face f of element e.  Fine side: coarse trace interpolated to this half of the coarse face; coarse side:
// Riemann problem on both mortars with the fine-side normal, projected back with the area factor 2.
// Rare path, kept out of line.
template <int NP>
__device__ __noinline__ void node_mortar_flux_2d(const StageParams &P, long e, int f, int a0, int2 cn, const double *U,
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


// The 2-D mortar fluxes evaluated ONCE per mortar ahead of the stage (the line kernel's path; same arithmetic as
// node_mortar_flux_2d, in the same order): F*(U_F, P_fwd^s U_C; n_F) at the 2 n fine face nodes of every mortar,
// mflux[m][s][a][v], outward for the fine side.  One thread per (mortar, half s, fine face node a).  info[m] = (eC, fC, fF).
// Evaluated inside the stage kernel, every coarse face node repeated all 2 n of them in a loop of dependent loads: a tile
// with a mortar face took 26 us (profiles/r02_launches.md).
template <int NP>
__global__ void __launch_bounds__(128) mortar_flux2d_kernel(const double *__restrict__ u, const double *__restrict__ metric,
                                                            int affine, const int *__restrict__ info,
                                                            const int *__restrict__ mortar_fine,
                                                            const double *__restrict__ mortar_mat, double gamma, long n_mortar,
                                                            double *__restrict__ mflux) {
  using G = Geo<2, NP>;
  constexpr int NVAR = 4, NN = NP * NP;
  const long g = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n_mortar * 2 * NP) return;
  const long m = g / (2 * NP);
  const int r = (int)(g - m * 2 * NP), s = r / NP, a = r - s * NP;
  const int eC = __ldg(&info[m * 3]), fC = __ldg(&info[m * 3 + 1]), fF = __ldg(&info[m * 3 + 2]);
  const long eF = __ldg(&mortar_fine[m * 2 + s]);
  const int pF = G::face_node(fF, a, 0), lF = fF >> 1;
  const double sF = (fF & 1) ? 1.0 : -1.0;
  double UF[NVAR], UC[NVAR], nF[2], FmF[NVAR], Fs[NVAR];
#pragma unroll
  for (int v = 0; v < NVAR; ++v) {
    UF[v] = __ldg(u + (eF * NVAR + v) * NN + pF);
    UC[v] = 0.0;
  }
#pragma unroll
  for (int j = 0; j < NP; ++j) {
    const double w = __ldg(&mortar_mat[(s * NP + a) * NP + j]);
    const double *uc = u + (long)eC * NVAR * NN + G::face_node(fC, j, 0);
#pragma unroll
    for (int v = 0; v < NVAR; ++v) UC[v] += w * __ldg(uc + v * NN);
  }
#pragma unroll
  for (int c = 0; c < 2; ++c)
    nF[c] = sF * (affine ? __ldg(&metric[eF * 5 + lF * 2 + c]) : __ldg(&metric[(eF * 5 + lF * 2 + c) * NN + pF]));
  const Prim<2> qF = prim_ideal<2, true>(UF, gamma);
  const Prim<2> qC = prim_ideal<2, true>(UC, gamma);
  flux_dot<2, 1>(UF, qF, nF, FmF);
  rusanov<2, 1>(UF, qF, FmF, UC, qC, nF, Fs);
#pragma unroll
  for (int v = 0; v < NVAR; ++v) mflux[g * NVAR + v] = Fs[v];
}
template <int NP>
cudaError_t launch_mortar_flux2d_t(const double *u, const double *metric, int affine, const int *info, const int *fine,
                                   const double *mat, double gamma, double *mflux, long n_mortar, cudaStream_t st) {
  const long n = n_mortar * 2 * NP;
  mortar_flux2d_kernel<NP><<<(unsigned)((n + 127) / 128), 128, 0, st>>>(u, metric, affine, info, fine, mat, gamma, n_mortar, mflux);
  return cudaGetLastError();
}
// numerical flux F* (outward, own normal) at face node a0 of a 2-D mortar face from the stored fluxes: fine side (mortar
// index in conn.y bits 10..): its own; coarse side (conn.x = mortar index): projection sum_s P_rev^s (2 (-F*_s)) in the
// order of node_mortar_flux_2d.  Cheap enough to sit inline in the line kernel.
template <int NP>
__device__ __forceinline__ void node_mortar_flux_2d_stored(const StageParams &P, int a0, int2 cn, double *Fs) {
  constexpr int NVAR = 4;
  const int kind = cn.y & 3, sub = (cn.y >> 8) & 1;
  if (kind == FK_MORTAR_FINE) {
    const double *F = P.mflux + (((long)(cn.y >> 10) * 2 + sub) * NP + a0) * NVAR;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Fs[v] = __ldg(F + v);
  } else {
    const double *Prv = P.mortar_mat + 2 * NP * NP;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Fs[v] = 0.0;
#pragma unroll
    for (int m = 0; m < 2; ++m) {
#pragma unroll
      for (int a = 0; a < NP; ++a) {
        const double w2 = -2.0 * __ldg(&Prv[(m * NP + a0) * NP + a]);
        const double *F = P.mflux + (((long)cn.x * 2 + m) * NP + a) * NVAR;
#pragma unroll
        for (int v = 0; v < NVAR; ++v) Fs[v] += w2 * __ldg(F + v);
      }
    }
  }
}

// 3-D 4:1 mortar faces (R21): the tensor product of the 2-D construction.  The Riemann fluxes
// F*(U_F, U_i; n_F) at the 4 n^2 fine face nodes of every mortar are evaluated once by mortar_flux3d_kernel before the
// stage (every coarse face node needs all of them); cn.x = mortar index on both sides, sub = s0 + 2 s1 names the half
// of the coarse face's first / second face-local direction.  Fine side: its own flux is the stored one.  Coarse side:
// L2 projection (Pr[s0] x Pr[s1]) of the outward flux -F*, times the area ratio 4.
template <int NP>
__device__ __forceinline__ void node_mortar_flux_3d(const StageParams &P, int a0, int a1, int2 cn, double *Fs) {
  constexpr int NVAR = 5, NF = NP * NP;
  const int kind = cn.y & 3, sub = (cn.y >> 8) & 3;
  if (kind == FK_MORTAR_FINE) {
    const double *F = P.mflux + (((long)cn.x * 4 + sub) * NF + a0 + NP * a1) * NVAR;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Fs[v] = __ldg(F + v);
  } else {
    const double *Prv = P.mortar_mat + 2 * NP * NP;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Fs[v] = 0.0;
    for (int m = 0; m < 4; ++m) {
      const int s0 = m & 1, s1 = m >> 1;
      const double *Fm_ = P.mflux + ((long)cn.x * 4 + m) * NF * NVAR;
      for (int b1 = 0; b1 < NP; ++b1) {
        const double r1 = -4.0 * __ldg(&Prv[(s1 * NP + a1) * NP + b1]);
        for (int b0 = 0; b0 < NP; ++b0) {
          const double w2 = r1 * __ldg(&Prv[(s0 * NP + a0) * NP + b0]);
          const double *F = Fm_ + (b0 + NP * b1) * NVAR;
#pragma unroll
          for (int v = 0; v < NVAR; ++v) Fs[v] += w2 * __ldg(F + v);
        }
      }
    }
  }
}

// F* at the fine face nodes of every 3-D mortar (R21): one CTA per mortar, one thread per (sub-face, fine face
// node).  The coarse trace is staged in shared memory, interpolated to the thread's node (Pf[s0] x Pf[s1]), and the
// Rusanov flux is evaluated with the fine element's own normal.  info[m] = (eC, fC, fF).  Affine meshes.
template <int NP>
__global__ void __launch_bounds__(4 * NP * NP) mortar_flux3d_kernel(const double *__restrict__ u, const double *__restrict__ metric,
                                                                    const int *__restrict__ info, const int *__restrict__ mortar_fine,
                                                                    const double *__restrict__ mortar_mat, double gamma,
                                                                    double *__restrict__ mflux) {
  using G = Geo<3, NP>;
  constexpr int NVAR = 5, NN = NP * NP * NP, NF = NP * NP, MD = 10;
  __shared__ double UC[NF * NVAR], Pfs[2 * NP * NP];
  const long m = blockIdx.x;
  const int tid = threadIdx.x;
  const int eC = info[m * 3], fC = info[m * 3 + 1], fF = info[m * 3 + 2];
  for (int i = tid; i < NF * NVAR; i += 4 * NF) {
    const int j = i / NVAR, v = i - j * NVAR;
    UC[i] = __ldg(u + ((long)eC * NVAR + v) * NN + G::face_node(fC, j % NP, j / NP));
  }
  for (int i = tid; i < 2 * NP * NP; i += 4 * NF) Pfs[i] = __ldg(&mortar_mat[i]);
  __syncthreads();
  const int s = tid / NF, b = tid - s * NF, b0 = b % NP, b1 = b / NP, s0 = s & 1, s1 = s >> 1;
  const long eF = mortar_fine[m * 4 + s];
  const int pF = G::face_node(fF, b0, b1), lF = fF >> 1;
  const double sF = (fF & 1) ? 1.0 : -1.0;
  double UF[NVAR], Ui[NVAR], nF[3], FmF[NVAR], Fs[NVAR];
#pragma unroll
  for (int v = 0; v < NVAR; ++v) {
    UF[v] = __ldg(u + (eF * NVAR + v) * NN + pF);
    Ui[v] = 0.0;
  }
  for (int j1 = 0; j1 < NP; ++j1) {
    const double w1 = Pfs[(s1 * NP + b1) * NP + j1];
    for (int j0 = 0; j0 < NP; ++j0) {
      const double w = w1 * Pfs[(s0 * NP + b0) * NP + j0];
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Ui[v] += w * UC[(j0 + NP * j1) * NVAR + v];
    }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) nF[c] = sF * __ldg(&metric[eF * MD + lF * 3 + c]);
  const Prim<3> qF = prim_ideal<3, true>(UF, gamma);
  const Prim<3> qC = prim_ideal<3, true>(Ui, gamma);
  flux_dot<3, 1>(UF, qF, nF, FmF);
  rusanov<3, 1>(UF, qF, FmF, Ui, qC, nF, Fs);
#pragma unroll
  for (int v = 0; v < NVAR; ++v) mflux[((m * 4 + s) * NF + b) * NVAR + v] = Fs[v];
}
template <int NP>
cudaError_t launch_mortar_flux3d_t(const double *u, const double *metric, const int *info, const int *fine, const double *mat,
                                   double gamma, double *mflux, long n_mortar, cudaStream_t st) {
  mortar_flux3d_kernel<NP><<<(unsigned)n_mortar, 4 * NP * NP, 0, st>>>(u, metric, info, fine, mat, gamma, mflux);
  return cudaGetLastError();
}

// decoded face task (no dynamically indexed local arrays: they would go to local memory)
struct FaceTask {
  int el, f, a0, a1, p;   // element in tile, face, face-node coordinates, volume node
};
template <int DIM, int NP>
__device__ __forceinline__ int face_node_of(int f, int a0, int a1) {
  const int l = f >> 1, s = (f & 1) ? NP - 1 : 0;
  if (DIM == 2) return (l == 0) ? s + NP * a0 : a0 + NP * s;
  return (l == 0) ? s + NP * (a0 + NP * a1) : ((l == 1) ? a0 + NP * (s + NP * a1) : a0 + NP * (a1 + NP * s));
}
template <int DIM, int NP>
__device__ __forceinline__ FaceTask decode_task(int g) {
  constexpr int NF = Geo<DIM, NP>::NF, NFN = 2 * DIM * NF;
  FaceTask t;
  t.el = g / NFN;
  const int r = g - t.el * NFN;
  t.f = r / NF;
  const int a = r - t.f * NF;
  t.a1 = (DIM == 3) ? a / NP : 0;
  t.a0 = a - t.a1 * NP;
  t.p = face_node_of<DIM, NP>(t.f, t.a0, t.a1);
  return t;
}

// exterior state of a conforming / boundary face node (mortar faces: nothing to gather here)
template <int DIM, int NP, int NVAR>
__device__ __forceinline__ void gather_exterior(const StageParams &P, const FaceTask &t, int2 cn, double *Up) {
  constexpr int NN = Geo<DIM, NP>::NN;
  const int kind = cn.y & 3;
  if (kind == FK_CONFORMING) {
    const int fR = (cn.y >> 2) & 7, orient = (cn.y >> 5) & 7;
    int b0, b1;
    partner_index<DIM, NP>(orient, t.a0, t.a1, b0, b1);
    const double *un = P.u_in + (long)cn.x * NVAR * NN + face_node_of<DIM, NP>(fR, b0, b1);
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Up[v] = __ldg(un + v * NN);
  } else if (kind == FK_BOUNDARY) {
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Up[v] = __ldg(&P.bc_state[cn.x * NVAR + v]);
  } else {
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Up[v] = 1.0;
  }
}

// lift (F* - Ftilde.n)/w_b of one face node (Euler), written to the lift buffer.  BCK: the instantiation that knows
// outflow / slip-wall faces and 3-D mortar faces (selected by StageParams::bc_kinds; the default one carries no code
// for them: the out-of-line 3-D mortar call alone costs the default 3-D kernel 30 %).  Up = exterior state of a
// conforming / boundary face (ignored for mortar faces).
template <int DIM, int NP, bool AFFINE, int EB, bool BCK = false>
__device__ __forceinline__ void euler_face_task(const StageParams &P, const double *Ust, const double *Msm, double *Lft,
                                                long e0, int g, const FaceTask &t, int2 cn, const double *Up) {
  using C = NodeCfg<DIM, NP, 1, EB>;
  constexpr int NVAR = C::NVAR, NN = C::NN, TILE = C::TILE, NTASK = C::NTASK, MD = Geo<DIM, NP>::MD, MDP = C::MDP;
  const int l = t.f >> 1;
  const double sgn = (t.f & 1) ? 1.0 : -1.0;
  const int idx = t.el * NN + t.p;
  const long e = e0 + t.el;
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
      nv[c] = sgn * __ldg(&P.metric[(e * MD + l * DIM + c) * NN + t.p]);
      n2 += nv[c] * nv[c];
    }
    nrm = sqrt(n2);
  }
  // own normal flux F(U-).nv, recomputed from the stash (cheaper than five more shared loads)
  double mnm = 0.0;
#pragma unroll
  for (int c = 0; c < DIM; ++c) mnm += Um[1 + c] * nv[c];
  const double vnm = mnm * irhom;
  double Fm[NVAR], lift[NVAR];
  Fm[0] = mnm;
#pragma unroll
  for (int c = 0; c < DIM; ++c) Fm[1 + c] = Um[1 + c] * vnm + pm * nv[c];
  Fm[DIM + 1] = (Um[DIM + 1] + pm) * vnm;
  const int kind = cn.y & 3;
  if (BCK && kind == FK_BOUNDARY && ((cn.y >> 2) & 7) != BC_PRESCRIBED) {
    // outflow / slip-wall face (marut_set_boundary_kinds; R18), the Rusanov flux in closed form:
    // outflow U+ = U-: F* = F(U-).nv, no lift.  Slip wall U+ = U- with m+ = m- - 2 (m-.nhat) nhat: same rho, E, p, a and
    // v+.nv = -v-.nv, so the mass and energy components of F* vanish.
#pragma unroll
    for (int v = 0; v < NVAR; ++v) lift[v] = 0.0;
    if (((cn.y >> 2) & 7) >= BC_SLIP_WALL) {      // slip wall; the no-slip walls of a Navier-Stokes mesh use its hyperbolic flux (R22)
      const double hl = 0.5 * (fabs(vnm) + am * nrm);
      const double r = 2.0 * mnm / (nrm * nrm);
      lift[0] = -P.inv_wb * Fm[0];
      lift[DIM + 1] = -P.inv_wb * Fm[DIM + 1];
#pragma unroll
      for (int c = 0; c < DIM; ++c) {
        const double dm = -r * nv[c];                                      // m+ - m-
        const double Fp = (Um[1 + c] + dm) * (0.0 - vnm) + pm * nv[c];
        lift[1 + c] = P.inv_wb * (0.5 * (Fp - Fm[1 + c]) - hl * dm);
      }
    }
  } else if (kind == FK_CONFORMING || kind == FK_BOUNDARY) {
    // Rusanov with a scaled normal, division-free apart from 1/rho+ (R5):
    //   lambda |nv| = max(|v-.nv| + a- |nv|, |v+.nv| + a+ |nv|);  lift = (F* - F-.nv)/w_b
    const double irhop = 1.0 / Up[0];
    double mnp = 0.0, kep = 0.0;
#pragma unroll
    for (int c = 0; c < DIM; ++c) {
      mnp += Up[1 + c] * nv[c];
      kep += Up[1 + c] * Up[1 + c];
    }
    const double pp = (P.gamma - 1.0) * (Up[DIM + 1] - 0.5 * kep * irhop);
    const double ap = sqrt(P.gamma * pp * irhop);
    const double vnp = mnp * irhop;
    const double hl = 0.5 * fmax(fabs(vnm) + am * nrm, fabs(vnp) + ap * nrm);
    double Fp[NVAR];
    Fp[0] = mnp;
#pragma unroll
    for (int c = 0; c < DIM; ++c) Fp[1 + c] = Up[1 + c] * vnp + pp * nv[c];
    Fp[DIM + 1] = (Up[DIM + 1] + pp) * vnp;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) lift[v] = P.inv_wb * (0.5 * (Fp[v] - Fm[v]) - hl * (Up[v] - Um[v]));
  } else {
    if constexpr (DIM == 2) {
      double Fs[NVAR];
      node_mortar_flux_2d<NP>(P, e, t.f, t.a0, cn, Um, nv, Fs);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) lift[v] = P.inv_wb * (Fs[v] - Fm[v]);
    } else if constexpr (BCK) {
      double Fs[NVAR];
      node_mortar_flux_3d<NP>(P, t.a0, t.a1, cn, Fs);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) lift[v] = P.inv_wb * (Fs[v] - Fm[v]);
    } else {
#pragma unroll
      for (int v = 0; v < NVAR; ++v) lift[v] = 0.0;     // 3-D mortar faces run in the BCK instantiation only
    }
  }
#pragma unroll
  for (int v = 0; v < NVAR; ++v) Lft[v * C::LFS + g] = lift[v];
}

// ---------------------------------------------------------------- derivative passes (line tasks)
// One task = one line of NP nodes of one variable: NP shared loads feed NP*NP FMAs whose D operands are
// compile-time-indexed constant-bank values.  Tasks per pass = NVAR * NP^(DIM-1) per element (= the node count
// for Euler at NP = 5): every warp of the CTA takes part with all lanes, so the passes are balanced.
// The xi pass overwrites Ftilde^xi with D_xi Ftilde^xi; the eta pass adds D_eta Ftilde^eta to it; the last
// pass (zeta in 3-D, eta in 2-D) keeps its NP results in registers and finishes those NP degrees of freedom.
template <int NP>
__device__ __forceinline__ void line_deriv(const StageParams &P, const double *f, double *acc) {
#pragma unroll
  for (int i = 0; i < NP; ++i) {
#pragma unroll
    for (int m = 0; m < NP; ++m) acc[i] += P.D[i * NP + m] * f[m];
  }
}

// L2 bulk prefetch of the tile this many CTAs ahead (measured: -3 % on c2) and the CTAs of 128 threads per SM the
// register allocation is sized for
constexpr int NODE_L2_PREFETCH = 1024;
constexpr int NODE_MINB128 = 6;
// last-pass task t -> (element in tile, variable, line): 3-D: ij = i + NP*j, lanes run over ij first;
// 2-D: ij = i, lane order (i, element, v)
template <int DIM, int NP>
struct LastPass {
  static constexpr int NL = (DIM == 3) ? NP * NP : NP;
  // lanes per (element, variable) plane.  A 32-lane slot for NP = 5 (25 of 32 lanes active, no warp straddling two
  // planes) removes the remaining bank conflicts of the last pass but needs a second round on one warp: slower.
  static constexpr int SLOT = NL;
};
template <int DIM, int NP, int NVAR, int EB>
__device__ __forceinline__ void last_pass_task(int t, int &el, int &v, int &ij) {
  constexpr int NL = LastPass<DIM, NP>::NL, SLOT = LastPass<DIM, NP>::SLOT;
  if constexpr (DIM == 3) {
    const int w = t / SLOT;
    ij = t - w * SLOT;
    el = w / NVAR;
    v = w - el * NVAR;
    if (ij >= NL) el = EB;   // padding lane
  } else {
    ij = t % NP;
    el = (t / NP) % EB;
    v = t / (NP * EB);
  }
}

template <int DIM, int NP, bool AFFINE, int EB, int MINB, bool BCK = false>
__global__ void __launch_bounds__((NodeCfg<DIM, NP, 1, EB>::NT), MINB)
stage_node_kernel(const __grid_constant__ StageParams P) {
  using C = NodeCfg<DIM, NP, 1, EB>;
  using G = Geo<DIM, NP>;
  constexpr int NVAR = C::NVAR, NN = C::NN, NF = C::NF, TILE = C::TILE, NFN = C::NFN, NTASK = C::NTASK, NT = C::NT;
  constexpr int MD = G::MD, MDP = C::MDP, KS = C::KS, PS = C::PS, NW = C::NW;
  constexpr int NL = NF;                    // lines per direction and element
  constexpr int NLT = NVAR * NL;            // line tasks per pass and element
  extern __shared__ __align__(16) double smem[];
  double *Fsm = smem;                       // [DIM][NVAR][EB] planes of PS doubles: contravariant fluxes
  double *Ust = Fsm + C::NPL * PS;          // [NVAR + 3][TILE]  U, 1/rho, p, a
  double *Lft = Ust + C::NST * TILE;        // [NVAR][NTASK]     lifts of the face nodes
  double *Msm = Lft + NVAR * C::LFS;         // affine: [EB][MDP] Ja, 1/J, |Ja^l|

  const int tid = threadIdx.x;
  const long e0 = (long)blockIdx.x * EB;
  const int nel = (int)((P.ne - e0 < EB) ? (P.ne - e0) : EB);
  const int ntask = nel * NFN, nline = nel * NLT;

  // L2 prefetch of the tile a CTA launched ~one wave later will read (u_in and u_n): turns its DRAM latency into an
  // L2 hit.  Bulk prefetch needs 16-byte alignment and size: round outwards, stay inside the array.
  if (tid == 0) {
    const long ep = e0 + (long)NODE_L2_PREFETCH * EB;
    if (ep + EB < P.ne) {
      const size_t bytes = (size_t)EB * NVAR * NN * sizeof(double);
      l2_prefetch(P.u_in + ep * NVAR * NN, bytes);
      if (P.ca != 0.0) l2_prefetch(P.u_n + ep * NVAR * NN, bytes);
    }
  }
  // first face task of this thread: connectivity load issued first (the neighbour gather depends on it)
  const bool has0 = tid < ntask;
  const FaceTask t0 = decode_task<DIM, NP>(has0 ? tid : 0);
  int2 cn0 = make_int2(0, FK_BOUNDARY);
  if (has0) cn0 = __ldg(&P.conn[(e0 + t0.el) * 2 * DIM + t0.f]);

  if constexpr (AFFINE) {
    for (int i = tid; i < nel * MDP; i += NT) {
      const int el = i / MDP, k = i - el * MDP;
      Msm[i] = (k < MD) ? __ldg(&P.metric[(e0 + el) * MD + k]) : ((k < MD + DIM) ? __ldg(&P.fnorm[(e0 + el) * DIM + (k - MD)]) : 0.0);
    }
  }

  const bool use_un = (P.ca != 0.0);
  // neighbour trace of the first face task: issued in phase N, consumed after the xi pass
  double Up0[NVAR];
  // ---- phase N: own node
  {
    const int el = tid / NN, p = tid - el * NN;
    const long e = e0 + el;
    const bool active = (tid < TILE) && (el < nel);
    double U[NVAR];
    if (active) {
      const double *up = P.u_in + e * NVAR * NN + p;
#pragma unroll
      for (int v = 0; v < NVAR; ++v) U[v] = __ldg(up + v * NN);
    }
    if (active) {
      const int qk = (DIM == 3) ? p / (NP * NP) : 0;
      const int sp = p + (KS - NP * NP) * qk;   // node offset inside a flux plane
      double Ja[DIM * DIM];
#pragma unroll
      for (int k = 0; k < DIM * DIM; ++k) Ja[k] = metric_at<DIM, NP, AFFINE>(P.metric, e, k, p);
      const Prim<DIM> pr = prim_ideal<DIM, true>(U, P.gamma);
#pragma unroll
      for (int l = 0; l < DIM; ++l) {
        double F[NVAR];
        flux_dot<DIM, 1>(U, pr, &Ja[l * DIM], F);
#pragma unroll
        for (int v = 0; v < NVAR; ++v) Fsm[(l * NVAR * EB + C::plane(v, el)) * PS + sp] = F[v];
      }
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Ust[v * TILE + tid] = U[v];
      Ust[NVAR * TILE + tid] = pr.irho;
      Ust[(NVAR + 1) * TILE + tid] = pr.p;
      Ust[(NVAR + 2) * TILE + tid] = pr.a;
    }
  }
  if (has0) gather_exterior<DIM, NP, NVAR>(P, t0, cn0, Up0);
  __syncthreads();

  // ---- xi pass (eq. 9): lines (j,k) of variable v; lanes run over the lines first
  for (int t = tid; t < EB * NLT; t += NT) {
    int el, v, lj, lk = 0;
    if constexpr (DIM == 3) {
      el = t / NLT;
      const int r = t - el * NLT;
      v = r / NL;
      const int ln = r - v * NL;
      lj = ln % NP;
      lk = ln / NP;
    } else {   // 2-D lane order (v, element, j): bank-conflict-free with element-major planes
      v = t % NVAR;
      el = (t / NVAR) % EB;
      lj = t / (NVAR * EB);
    }
    if (el >= nel) continue;
    double *px = Fsm + C::plane(v, el) * PS + NP * lj + KS * lk;
    double f[NP], acc[NP];
#pragma unroll
    for (int m = 0; m < NP; ++m) { f[m] = px[m]; acc[m] = 0.0; }
    line_deriv<NP>(P, f, acc);
#pragma unroll
    for (int i = 0; i < NP; ++i) px[i] = acc[i];
  }

  // ---- face phase, first round: face nodes densely mapped
  if (has0) euler_face_task<DIM, NP, AFFINE, EB, BCK>(P, Ust, Msm, Lft, e0, tid, t0, cn0, Up0);
  __syncthreads();

  if constexpr (DIM == 3) {
    // ---- eta pass: lines (i,k) of variable v; lane order (k, v, i) is bank-conflict-free
    for (int t = tid; t < nline; t += NT) {
      const int el = t / NLT, r = t - el * NLT;
      const int lk = r % NP, r2 = r / NP;
      const int v = r2 % NVAR, li = r2 / NVAR;
      double *px = Fsm + C::plane(v, el) * PS + li + KS * lk;
      const double *pe = px + NVAR * EB * PS;
      double f[NP], acc[NP];
#pragma unroll
      for (int m = 0; m < NP; ++m) { f[m] = pe[m * NP]; acc[m] = px[m * NP]; }
      line_deriv<NP>(P, f, acc);
#pragma unroll
      for (int j = 0; j < NP; ++j) px[j * NP] = acc[j];
    }
  }
  // ---- face phase, remaining rounds
  for (int g = tid + NT; g < ntask; g += NT) {
    const FaceTask t = decode_task<DIM, NP>(g);
    const int2 cn = __ldg(&P.conn[(e0 + t.el) * 2 * DIM + t.f]);
    double Up[NVAR];
    gather_exterior<DIM, NP, NVAR>(P, t, cn, Up);
    euler_face_task<DIM, NP, AFFINE, EB, BCK>(P, Ust, Msm, Lft, e0, g, t, cn, Up);
  }
  if constexpr (DIM == 3 || (NTASK > NT)) __syncthreads();

  // ---- last pass (zeta in 3-D, eta in 2-D) fused with phase D: lifts, 1/J, SSP-RK combination (eq. 12, 45)
  for (int t = tid; t < EB * NVAR * LastPass<DIM, NP>::SLOT; t += NT) {
    int el, v, ij;                               // 3-D: ij = i + NP*j ; 2-D: ij = i
    last_pass_task<DIM, NP, NVAR, EB>(t, el, v, ij);
    if (el >= nel) continue;
    constexpr int LS = (DIM == 3) ? KS : NP;      // stride of the line in the flux plane
    constexpr int GS = (DIM == 3) ? NP * NP : NP; // stride of the line in global memory
    const long e = e0 + el;
    const double *px = Fsm + C::plane(v, el) * PS + ij;
    const double *pl = px + (DIM - 1) * NVAR * EB * PS;
    const long gofs = (e * NVAR + v) * NN + ij;
    double un[NP];
    if (use_un) {
#pragma unroll
      for (int m = 0; m < NP; ++m) un[m] = P.u_n[gofs + m * GS];
    }
    double f[NP], acc[NP];
#pragma unroll
    for (int m = 0; m < NP; ++m) { f[m] = pl[m * LS]; acc[m] = px[m * LS]; }
    line_deriv<NP>(P, f, acc);
    // lifts of the faces the nodes of this line lie on
    const double *lf = Lft + v * C::LFS + el * NFN;
    if constexpr (DIM == 3) {
      const int qi = ij % NP, qj = ij / NP;
      acc[0] += lf[4 * NF + ij];
      acc[NP - 1] += lf[5 * NF + ij];
      if (qi == 0 || qi == NP - 1) {
        const double *l2 = lf + ((qi == 0) ? 0 : NF) + qj;
#pragma unroll
        for (int m = 0; m < NP; ++m) acc[m] += l2[NP * m];
      }
      if (qj == 0 || qj == NP - 1) {
        const double *l2 = lf + ((qj == 0) ? 2 * NF : 3 * NF) + qi;
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
    const double *us = Ust + v * TILE + el * NN + ij;
    double invJ = 0.0;
    if constexpr (AFFINE) invJ = Msm[el * MDP + DIM * DIM];
#pragma unroll
    for (int m = 0; m < NP; ++m) {
      if constexpr (!AFFINE) invJ = __ldg(&P.metric[(e * MD + DIM * DIM) * NN + ij + m * GS]);
      const double val = P.cb * us[m * GS] + stage_cc(P) * (0.0 - invJ * acc[m]);
      P.u_out[gofs + m * GS] = use_un ? (P.ca * un[m] + val) : val;
    }
  }
}

// elements per CTA: ~128 threads
template <int NN>
constexpr int node_eb() { return (NN >= 96) ? 1 : 128 / NN; }

template <int DIM, int NP, bool AFFINE, bool BCK = false>
cudaError_t launch_stage_node_t(const StageParams &P, cudaStream_t st) {
  if constexpr (!BCK) {
    if (P.bc_kinds) return launch_stage_node_t<DIM, NP, AFFINE, true>(P, st);
  }
  constexpr int NN = Geo<DIM, NP>::NN, EB = node_eb<NN>();
  using C = NodeCfg<DIM, NP, 1, EB>;
  constexpr size_t smem = C::smem_doubles(AFFINE) * sizeof(double);
  constexpr int MINB = (C::NT <= 128) ? NODE_MINB128 : ((C::NT <= 256) ? 3 : 1);
  auto k = stage_node_kernel<DIM, NP, AFFINE, EB, MINB, BCK>;
  static std::atomic<unsigned long long> attr_done{0};
  if (cudaError_t err = set_smem_once((const void *)k, smem, attr_done); err != cudaSuccess) return err;
  const long grid = (P.ne + EB - 1) / EB;
  k<<<(unsigned)grid, C::NT, smem, st>>>(P);
  return cudaGetLastError();
}

}  // namespace marut
