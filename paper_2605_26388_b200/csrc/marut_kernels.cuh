// marut_kernels.cuh -- the per-node kernels of the CUDA path around the fused stage kernels:
//   gradient_kernel : BR1 gradient S = grad W (a6)
//   eos_kernel      : mixture temperature by Newton (a8)
//   chem_kernel     : chemistry source alone (marut_chem_source)
//   wave_speed_kernel: max-wave-speed / max-diffusivity reduction (a10)
//   metrics_kernel  : GCL-preserving metric terms (a0)
// Thread mapping: one thread per LGL node, EB consecutive elements per CTA.
#pragma once
#include "marut_common.cuh"
#include "marut_physics.cuh"

namespace marut {

template <int DIM, int NP>
struct Geo {
  static constexpr int NN = (DIM == 2) ? NP * NP : NP * NP * NP;
  static constexpr int NF = (DIM == 2) ? NP : NP * NP;   // nodes per face
  static constexpr int MD = DIM * DIM + 1;               // metric planes: Ja^l_c (l-major) and 1/J
  __device__ static __forceinline__ void ijk(int p, int *q) {
    q[0] = p % NP;
    q[1] = (p / NP) % NP;
    if (DIM == 3) q[2] = p / (NP * NP);
  }
  __device__ static __forceinline__ int node(const int *q) {
    return (DIM == 2) ? q[0] + NP * q[1] : q[0] + NP * (q[1] + NP * q[2]);
  }
  // stride of reference direction l in the node index
  __device__ static __forceinline__ int stride(int l) { return l == 0 ? 1 : (l == 1 ? NP : NP * NP); }
  // volume node of face node (a0,a1) on face f
  __device__ static __forceinline__ int face_node(int f, int a0, int a1) {
    const int l = f >> 1, s = (f & 1) ? NP - 1 : 0;
    int q[3];
    if (DIM == 2) {
      q[l] = s;
      q[1 - l] = a0;
    } else {
      q[l] = s;
      q[l == 0 ? 1 : 0] = a0;
      q[l == 2 ? 1 : 2] = a1;
    }
    return node(q);
  }
  // face-node coordinates of volume node q on a face normal to l
  __device__ static __forceinline__ void face_coords(const int *q, int l, int &a0, int &a1) {
    if (DIM == 2) {
      a0 = q[1 - l];
      a1 = 0;
    } else {
      a0 = q[l == 0 ? 1 : 0];
      a1 = q[l == 2 ? 1 : 2];
    }
  }
};

template <int DIM, int NP, bool AFFINE>
__device__ __forceinline__ double metric_at(const double *__restrict__ metric, long e, int plane, int p) {
  using G = Geo<DIM, NP>;
  return AFFINE ? __ldg(&metric[e * G::MD + plane]) : __ldg(&metric[(e * G::MD + plane) * G::NN + p]);
}

// state (+T for reacting) -> primitives
template <int DIM, int NSP, int PHYS, bool WANT_A>
__device__ __forceinline__ Prim<DIM> make_prim(const double *U, double T, double gamma, const MechDev *mech) {
  if constexpr (PHYS == PH_REACT) return prim_mixture<DIM, NSP, WANT_A>(U, T, *mech);
  else return prim_ideal<DIM, WANT_A>(U, gamma);
}

// ======================================================================================
// BR1 gradient  S = (1/J) [ sum_l D_l(Ja^l_c W) + (1/w_b) (What - W) n_c ]  (eq. 13)
// ======================================================================================
struct GradParams {
  const double *__restrict__ u;
  double *__restrict__ S;
  const double *__restrict__ metric;
  const int2 *__restrict__ conn;
  double gamma, inv_wb, mu, kappa;
  long ne;
  double D[MAX_NP * MAX_NP];
  int oriented;                        // 3-D: some interface has a non-trivial orientation code
  const double *__restrict__ bc_state; // [bc][nvar] prescribed states of the boundary ids (kind 0; kind 4: their T is T_wall)
  int boundary;                        // the mesh has boundary or mortar faces: launch the instantiation that knows them
  const int *__restrict__ mortar_fine; // 2-D mortars: [m][2] fine elements (lo, up)
  const double *__restrict__ mortar_mat; // [4][n*n]: Pf_lo, Pf_up, Pr_lo, Pr_up
  const double *__restrict__ mW;       // 3-D mortars: the central trace What at the fine face nodes of every mortar,
                                       //    [m][4][n*n][d+2] (mortar_trace3d_kernel, launched before this kernel); else NULL
};

// BR1 trace jump What - W at a boundary face node (reading R22).  kind: 0 prescribed state
// (central trace with W(U_bc)), 1 outflow (no jump), 2 slip wall (velocity mirrored across the normal), 3 no-slip
// adiabatic wall (What = (rho-, 0, T-)), 4 isothermal wall (What = (rho-, 0, T_wall), T_wall = T of the prescribed state)
template <int DIM>
__device__ __forceinline__ void br1_boundary_jump(int kind, const double *W, const double *Ub, const double *nv, double gamma,
                                                  double *jump) {
  constexpr int NW = DIM + 2;
#pragma unroll
  for (int w = 0; w < NW; ++w) jump[w] = 0.0;
  if (kind == BC_PRESCRIBED || kind == BC_WALL_ISOTHERMAL) {
    const Prim<DIM> qb = prim_ideal<DIM, false>(Ub, gamma);
    if (kind == BC_PRESCRIBED) {
      jump[0] = 0.5 * (W[0] + qb.rho) - W[0];
#pragma unroll
      for (int c = 0; c < DIM; ++c) jump[1 + c] = 0.5 * (W[1 + c] + qb.v[c]) - W[1 + c];
      jump[1 + DIM] = 0.5 * (W[1 + DIM] + qb.T) - W[1 + DIM];
    } else jump[1 + DIM] = qb.T - W[1 + DIM];
  }
  if (kind == BC_SLIP_WALL) {
    double n2 = 0.0, vn = 0.0;
#pragma unroll
    for (int c = 0; c < DIM; ++c) n2 += nv[c] * nv[c];
    const double inrm = 1.0 / sqrt(n2);
#pragma unroll
    for (int c = 0; c < DIM; ++c) vn += W[1 + c] * (nv[c] * inrm);
#pragma unroll
    for (int c = 0; c < DIM; ++c) jump[1 + c] = 0.5 * (W[1 + c] + (W[1 + c] - 2.0 * vn * (nv[c] * inrm))) - W[1 + c];
  }
  if (kind == BC_WALL_ADIABATIC || kind == BC_WALL_ISOTHERMAL) {
#pragma unroll
    for (int c = 0; c < DIM; ++c) jump[1 + c] = 0.0 - W[1 + c];
  }
}

// W = (rho, v, T) of a conserved state (the BR1 gradient variables)
template <int DIM>
__device__ __forceinline__ void br1_vars(const double *U, double gamma, double *W) {
  const Prim<DIM> q = prim_ideal<DIM, false>(U, gamma);
  W[0] = q.rho;
#pragma unroll
  for (int c = 0; c < DIM; ++c) W[1 + c] = q.v[c];
  W[1 + DIM] = q.T;
}

// BR1 surface term of the gradient at face node a0 of a 2-D mortar face f of element e ("Non-conforming
// faces use the same forward and reverse projections as the hyperbolic side"; reading R23): the hyperbolic
// mortar with the flux replaced by the central trace.  add[w][c] = (What - W) n_c on the fine side (What = mean of the
// own W and the coarse trace interpolated to this half), and  sum_m P_rev^m (2 (-What_m n_F)) - W n_c  on the coarse
// side.  Wc: the own element's W planes in shared memory (plane stride wstride), used for the coarse trace.
// Rare path, kept out of line.
template <int NP, bool AFFINE>
__device__ __noinline__ void br1_mortar_jump_2d(const GradParams &P, long e, int f, int a0, int2 cn, const double *W,
                                                const double *Wc, int wstride, const double *nv, double *add) {
  using G = Geo<2, NP>;
  constexpr int NVAR = 4, NW = 4, NN = NP * NP;
  const int kind = cn.y & 3, fR = (cn.y >> 2) & 7, sub = (cn.y >> 8) & 1;
  const double *Pf = P.mortar_mat, *Prv = P.mortar_mat + 2 * NP * NP;
  if (kind == FK_MORTAR_FINE) {
    double Wi[NW] = {0.0, 0.0, 0.0, 0.0};
    for (int j = 0; j < NP; ++j) {
      const double pw = __ldg(&Pf[(sub * NP + a0) * NP + j]);
      const double *uc = P.u + (long)cn.x * NVAR * NN + G::face_node(fR, j, 0);
      double UC[NVAR], WC[NW];
#pragma unroll
      for (int v = 0; v < NVAR; ++v) UC[v] = __ldg(uc + v * NN);
      br1_vars<2>(UC, P.gamma, WC);
#pragma unroll
      for (int w = 0; w < NW; ++w) Wi[w] += pw * WC[w];
    }
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const double What = 0.5 * (W[w] + Wi[w]);
#pragma unroll
      for (int c = 0; c < 2; ++c) add[w * 2 + c] = (What - W[w]) * nv[c];
    }
  } else {
    double GC[NW * 2];
#pragma unroll
    for (int k = 0; k < NW * 2; ++k) GC[k] = 0.0;
    const int lF = fR >> 1;
    const double sF = (fR & 1) ? 1.0 : -1.0;
    for (int m = 0; m < 2; ++m) {
      const long eF = __ldg(&P.mortar_fine[cn.x * 2 + m]);
      for (int a = 0; a < NP; ++a) {
        const int pF = G::face_node(fR, a, 0);
        double UF[NVAR], WF[NW], nF[2];
#pragma unroll
        for (int v = 0; v < NVAR; ++v) UF[v] = __ldg(P.u + (eF * NVAR + v) * NN + pF);
        br1_vars<2>(UF, P.gamma, WF);
#pragma unroll
        for (int c = 0; c < 2; ++c) nF[c] = sF * metric_at<2, NP, AFFINE>(P.metric, eF, lF * 2 + c, pF);
        const double pr = __ldg(&Prv[(m * NP + a0) * NP + a]);
#pragma unroll
        for (int w = 0; w < NW; ++w) {
          double Wi = 0.0;
          for (int j = 0; j < NP; ++j) Wi += __ldg(&Pf[(m * NP + a) * NP + j]) * Wc[w * wstride + G::face_node(f, j, 0)];
          const double What = 0.5 * (WF[w] + Wi);
#pragma unroll
          for (int c = 0; c < 2; ++c) GC[w * 2 + c] += pr * (2.0 * (-(What * nF[c])));
        }
      }
    }
#pragma unroll
    for (int w = 0; w < NW; ++w)
#pragma unroll
      for (int c = 0; c < 2; ++c) add[w * 2 + c] = GC[w * 2 + c] - W[w] * nv[c];
  }
}

// 3-D 4:1 mortars (readings R21 + R23): What = (W_F + (Pf[s0] x Pf[s1]) W_C)/2 at the 4 n^2 fine face nodes of every
// mortar, evaluated once per mortar ahead of gradient_kernel (every coarse face node needs all of them).  One CTA per
// mortar, one thread per (sub-face, fine face node); info[m] = (eC, fC, fF).
template <int NP>
__global__ void __launch_bounds__(4 * NP * NP) mortar_trace3d_kernel(const double *__restrict__ u, const int *__restrict__ info,
                                                                     const int *__restrict__ mortar_fine,
                                                                     const double *__restrict__ mortar_mat, double gamma,
                                                                     double *__restrict__ mW) {
  using G = Geo<3, NP>;
  constexpr int NVAR = 5, NW = 5, NN = NP * NP * NP, NF = NP * NP;
  __shared__ double WC[NF * NW], Pfs[2 * NP * NP];
  const long m = blockIdx.x;
  const int tid = threadIdx.x;
  const int eC = info[m * 3], fC = info[m * 3 + 1], fF = info[m * 3 + 2];
  if (tid < NF) {
    double U[NVAR], W[NW];
#pragma unroll
    for (int v = 0; v < NVAR; ++v) U[v] = __ldg(u + ((long)eC * NVAR + v) * NN + G::face_node(fC, tid % NP, tid / NP));
    br1_vars<3>(U, gamma, W);
#pragma unroll
    for (int w = 0; w < NW; ++w) WC[tid * NW + w] = W[w];
  }
  for (int i = tid; i < 2 * NP * NP; i += 4 * NF) Pfs[i] = __ldg(&mortar_mat[i]);
  __syncthreads();
  const int s = tid / NF, b = tid - s * NF, b0 = b % NP, b1 = b / NP, s0 = s & 1, s1 = s >> 1;
  const long eF = mortar_fine[m * 4 + s];
  double UF[NVAR], WF[NW], Wi[NW];
#pragma unroll
  for (int v = 0; v < NVAR; ++v) UF[v] = __ldg(u + (eF * NVAR + v) * NN + G::face_node(fF, b0, b1));
  br1_vars<3>(UF, gamma, WF);
#pragma unroll
  for (int w = 0; w < NW; ++w) Wi[w] = 0.0;
  for (int j1 = 0; j1 < NP; ++j1) {
    const double w1 = Pfs[(s1 * NP + b1) * NP + j1];
    for (int j0 = 0; j0 < NP; ++j0) {
      const double pw = Pfs[(s0 * NP + b0) * NP + j0] * w1;
#pragma unroll
      for (int w = 0; w < NW; ++w) Wi[w] += pw * WC[(j0 + NP * j1) * NW + w];
    }
  }
#pragma unroll
  for (int w = 0; w < NW; ++w) mW[((m * 4 + s) * NF + b) * NW + w] = 0.5 * (WF[w] + Wi[w]);
}
template <int NP>
cudaError_t launch_mortar_trace3d_t(const double *u, const int *info, const int *fine, const double *mat, double gamma, double *mW,
                                    long n_mortar, cudaStream_t st) {
  mortar_trace3d_kernel<NP><<<(unsigned)n_mortar, 4 * NP * NP, 0, st>>>(u, info, fine, mat, gamma, mW);
  return cudaGetLastError();
}

// BR1 surface term of the gradient at face node (a0, a1) of a 3-D mortar face (readings R21 + R23), from the stored
// traces: fine side (What - W) n_c; coarse side  sum_s (Pr[s0] x Pr[s1]) (4 (-What_s n_F,s)) - W n_c.  Affine meshes
// (the fine elements' normals are constant per face).  cn.x = mortar index, fR = the fine elements' face.
template <int NP>
__device__ __noinline__ void br1_mortar_jump_3d(const GradParams &P, int2 cn, int a0, int a1, const double *W, const double *nv,
                                                double *add) {
  constexpr int NW = 5, NF = NP * NP, MD = 10;
  const int kind = cn.y & 3, fR = (cn.y >> 2) & 7, sub = (cn.y >> 8) & 3;
  if (kind == FK_MORTAR_FINE) {
    const double *Wh = P.mW + (((long)cn.x * 4 + sub) * NF + a0 + NP * a1) * NW;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const double jump = __ldg(Wh + w) - W[w];
#pragma unroll
      for (int c = 0; c < 3; ++c) add[w * 3 + c] = jump * nv[c];
    }
  } else {
    const double *Prv = P.mortar_mat + 2 * NP * NP;
    double GC[NW * 3];
#pragma unroll
    for (int k = 0; k < NW * 3; ++k) GC[k] = 0.0;
    const int lF = fR >> 1;
    const double sF = (fR & 1) ? 1.0 : -1.0;
    for (int m = 0; m < 4; ++m) {
      const int s0 = m & 1, s1 = m >> 1;
      const long eF = __ldg(&P.mortar_fine[cn.x * 4 + m]);
      double nF[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) nF[c] = sF * __ldg(&P.metric[eF * MD + lF * 3 + c]);
      const double *Wm = P.mW + ((long)cn.x * 4 + m) * NF * NW;
      for (int b1 = 0; b1 < NP; ++b1) {
        const double r1 = __ldg(&Prv[(s1 * NP + a1) * NP + b1]);
        for (int b0 = 0; b0 < NP; ++b0) {
          const double pr = __ldg(&Prv[(s0 * NP + a0) * NP + b0]) * r1;
          const double *Wh = Wm + (b0 + NP * b1) * NW;
#pragma unroll
          for (int w = 0; w < NW; ++w) {
            const double What = __ldg(Wh + w);
#pragma unroll
            for (int c = 0; c < 3; ++c) GC[w * 3 + c] += pr * (4.0 * (-(What * nF[c])));
          }
        }
      }
    }
#pragma unroll
    for (int w = 0; w < NW; ++w)
#pragma unroll
      for (int c = 0; c < 3; ++c) add[w * 3 + c] = GC[w * 3 + c] - W[w] * nv[c];
  }
}

// ORIENT3: the instantiation for 3-D meshes with non-trivial face orientation codes (R20); the default one
// keeps the identity pairing folded at compile time (the decode costs 12 registers here: 64 -> 76, one CTA less per SM)
// BND: the instantiation for meshes with boundary faces (prescribed states, outflow, walls; reading R22) or 2-D mortars
// (reading R23)
template <int DIM, int NP, bool AFFINE, int EB, bool ORIENT3 = false, bool BND = false>
__global__ void __launch_bounds__(((EB * Geo<DIM, NP>::NN + 31) / 32) * 32)
gradient_kernel(const __grid_constant__ GradParams P) {
  using G = Geo<DIM, NP>;
  constexpr int NN = G::NN, NVAR = DIM + 2, NW = DIM + 2, MD = G::MD, TILE = EB * NN;
  extern __shared__ double smem[];
  double *Wsm = smem;                 // [NW][TILE]
  double *Dsm = smem + NW * TILE;     // [NP*NP]
  // curved meshes: the node's own metric terms Ja^l_c go through shared memory, [DIM*DIM][TILE] -- one coalesced load
  // per plane, in flight together with the state, instead of DIM * NP * DIM dependent loads inside the derivative loops
  // (the kernel sat on them: long-scoreboard stalls 9.6 per issued instruction, profiles/r02_c3_stage.md)
  double *Jsm = Dsm + ((NP * NP + 1) & ~1);
  const int tid = threadIdx.x;
  for (int i = tid; i < NP * NP; i += blockDim.x) Dsm[i] = P.D[i];
  const int el = tid / NN, p = tid - el * NN;
  const long e = (long)blockIdx.x * EB + el;
  const bool active = (tid < TILE) && (e < P.ne);
  int q[3] = {0, 0, 0};
  G::ijk(p, q);
  double W[NW];
  if (active) {
    // 1/J (used last) and the connectivity entries of the node's faces (used right behind the barrier) are brought
    // towards the SM now -- prefetches hold no registers across the barrier
    if constexpr (!AFFINE) asm volatile("prefetch.global.L2 [%0];" ::"l"(&P.metric[(e * MD + DIM * DIM) * NN + p]));
#pragma unroll
    for (int l = 0; l < DIM; ++l)
      if (q[l] == 0 || q[l] == NP - 1) asm volatile("prefetch.global.L2 [%0];" ::"l"(&P.conn[e * 2 * DIM + 2 * l + ((q[l] == 0) ? 0 : 1)]));
    double U[NVAR];
#pragma unroll
    for (int v = 0; v < NVAR; ++v) U[v] = __ldg(P.u + (e * NVAR + v) * NN + p);
    if constexpr (!AFFINE) {
      double Jo[DIM * DIM];
#pragma unroll
      for (int k = 0; k < DIM * DIM; ++k) Jo[k] = __ldg(&P.metric[(e * MD + k) * NN + p]);
#pragma unroll
      for (int k = 0; k < DIM * DIM; ++k) Jsm[k * TILE + tid] = Jo[k];
    }
    const Prim<DIM> pr = prim_ideal<DIM, false>(U, P.gamma);
    W[0] = pr.rho;
#pragma unroll
    for (int c = 0; c < DIM; ++c) W[1 + c] = pr.v[c];
    W[1 + DIM] = pr.T;
#pragma unroll
    for (int w = 0; w < NW; ++w) Wsm[w * TILE + tid] = W[w];
  }
  __syncthreads();
  if (!active) return;
  double Sg[NW * DIM];
#pragma unroll
  for (int k = 0; k < NW * DIM; ++k) Sg[k] = 0.0;
#pragma unroll
  for (int l = 0; l < DIM; ++l) {
    const int st = G::stride(l), base = tid - q[l] * st, pbase = p - q[l] * st;
    for (int m = 0; m < NP; ++m) {
      const double d = Dsm[q[l] * NP + m];
      double Jm[DIM];
#pragma unroll
      for (int c = 0; c < DIM; ++c)
        Jm[c] = d * (AFFINE ? metric_at<DIM, NP, AFFINE>(P.metric, e, l * DIM + c, pbase + m * st) : Jsm[(l * DIM + c) * TILE + base + m * st]);
#pragma unroll
      for (int w = 0; w < NW; ++w) {
        const double Wm = Wsm[w * TILE + base + m * st];
#pragma unroll
        for (int c = 0; c < DIM; ++c) Sg[w * DIM + c] += Jm[c] * Wm;
      }
    }
  }
#pragma unroll
  for (int l = 0; l < DIM; ++l) {
    if (q[l] != 0 && q[l] != NP - 1) continue;
    const int side = (q[l] == 0) ? 0 : 1, f = 2 * l + side;
    const double sgn = side ? 1.0 : -1.0;
    const int2 cn = __ldg(&P.conn[e * 2 * DIM + f]);
    if constexpr (BND) {
      if ((cn.y & 3) == FK_BOUNDARY) {
        double nv[DIM], Ub[NVAR], jump[NW];
#pragma unroll
        for (int c = 0; c < DIM; ++c) nv[c] = sgn * metric_at<DIM, NP, AFFINE>(P.metric, e, l * DIM + c, p);
#pragma unroll
        for (int v = 0; v < NVAR; ++v) Ub[v] = __ldg(&P.bc_state[cn.x * NVAR + v]);
        br1_boundary_jump<DIM>((cn.y >> 2) & 7, W, Ub, nv, P.gamma, jump);
#pragma unroll
        for (int c = 0; c < DIM; ++c) {
          const double nc = nv[c] * P.inv_wb;
#pragma unroll
          for (int w = 0; w < NW; ++w) Sg[w * DIM + c] += jump[w] * nc;
        }
        continue;
      }
      if constexpr (DIM == 2) {
        if ((cn.y & 3) != FK_CONFORMING) {          // 2:1 mortar face (reading R23)
          double nv[DIM], add[NW * DIM];
#pragma unroll
          for (int c = 0; c < DIM; ++c) nv[c] = sgn * metric_at<DIM, NP, AFFINE>(P.metric, e, l * DIM + c, p);
          br1_mortar_jump_2d<NP, AFFINE>(P, e, f, q[1 - l], cn, W, Wsm + el * NN, TILE, nv, add);
#pragma unroll
          for (int k = 0; k < NW * DIM; ++k) Sg[k] += add[k] * P.inv_wb;
          continue;
        }
      }
      if constexpr (DIM == 3 && AFFINE) {
        if ((cn.y & 3) != FK_CONFORMING) {          // 4:1 mortar face (readings R21 + R23)
          double nv[DIM], add[NW * DIM];
#pragma unroll
          for (int c = 0; c < DIM; ++c) nv[c] = sgn * metric_at<DIM, NP, AFFINE>(P.metric, e, l * DIM + c, p);
          int a0, a1;
          G::face_coords(q, l, a0, a1);
          br1_mortar_jump_3d<NP>(P, cn, a0, a1, W, nv, add);
#pragma unroll
          for (int k = 0; k < NW * DIM; ++k) Sg[k] += add[k] * P.inv_wb;
          continue;
        }
      }
    }
    const int fR = (cn.y >> 2) & 7, orient = (DIM == 2 || ORIENT3) ? ((cn.y >> 5) & 7) : 0;
    int a0, a1;
    G::face_coords(q, l, a0, a1);
    int b0, b1;
    partner_index<DIM, NP>(orient, a0, a1, b0, b1);
    const int pR = G::face_node(fR, b0, b1);
    double Up[NVAR];
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Up[v] = __ldg(P.u + ((long)cn.x * NVAR + v) * NN + pR);
    const Prim<DIM> qp = prim_ideal<DIM, false>(Up, P.gamma);
    double Wp[NW];
    Wp[0] = qp.rho;
#pragma unroll
    for (int c = 0; c < DIM; ++c) Wp[1 + c] = qp.v[c];
    Wp[1 + DIM] = qp.T;
#pragma unroll
    for (int c = 0; c < DIM; ++c) {
      const double nc = sgn * metric_at<DIM, NP, AFFINE>(P.metric, e, l * DIM + c, p) * P.inv_wb;
#pragma unroll
      for (int w = 0; w < NW; ++w) Sg[w * DIM + c] += 0.5 * (Wp[w] - W[w]) * nc;
    }
  }
  const double invJ = metric_at<DIM, NP, AFFINE>(P.metric, e, DIM * DIM, p);
#pragma unroll
  for (int k = 0; k < NW * DIM; ++k) Sg[k] = invJ * Sg[k];
  // stored in the compact form the viscous flux needs: stress tensor + heat flux (Tau<DIM>)
  constexpr int NTAU = Tau<DIM>::NTAU;
  double tau[NTAU];
  gradient_to_tau<DIM>(Sg, P.mu, P.kappa, tau);
#pragma unroll
  for (int k = 0; k < NTAU; ++k) P.S[(e * NTAU + k) * NN + p] = tau[k];
}

// ======================================================================================
// per-node kernels for the reacting mixture
// ======================================================================================
__device__ __forceinline__ void load_mech(MechDev *dst_s, const MechDev *src_g) {
  const int *src = reinterpret_cast<const int *>(src_g);
  int *dst = reinterpret_cast<int *>(dst_s);
  for (int i = threadIdx.x; i < (int)(sizeof(MechDev) / sizeof(int)); i += blockDim.x) dst[i] = src[i];
  __syncthreads();
}

// Per-node thermochemistry of the reacting stage (a8, a9), evaluated ONCE per stage call ahead of the fused stage
// kernel: T by Newton, then p = rho R T and the frozen sound speed (R12) and -- when the
// explicit source is on -- the production rates omega_s (eq. 21-22).  aux[e][2 + NSP][node] = p, a, omega_1..NSP.
// The stage kernel then needs no mechanism table, no exponentials and no Newton: it keeps the footprint of the Euler
// stage (the chemistry is purely per node, "no inter-thread communication").
// RED (marut_ssprk33_step_dt): the kernel also reduces the wave speed |v| + a of the state it evaluates into red[0]
// (and a bad-state count into red[2]) -- wave_speed_kernel's expressions on the same T and a, so the time step that
// dt_finalize_kernel forms from them equals marut_max_dt's bit for bit, without another pass over the state.
template <int DIM, int NSP, bool RED = false>
__global__ void __launch_bounds__(256, 3) eos_kernel(const double *__restrict__ u, double *__restrict__ aux,
                                                  const MechDev *__restrict__ mech_g, long ne, int nn, int with_source,
                                                  unsigned long long *__restrict__ red = nullptr) {
  constexpr int NVAR = NSP + DIM + 1, NA = 2 + NSP;
  __shared__ MechDev mech;
  __shared__ double Xs[NSP * 256];           // per-thread concentration columns of production_rates_listed
  load_mech(&mech, mech_g);
  double lam = 0.0;
  int bad = 0;
  const long total = ne * nn;
  for (long g = (long)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (long)gridDim.x * blockDim.x) {
    const long e = g / nn;
    const int p = (int)(g - e * nn);
    double U[NVAR];
#pragma unroll
    for (int v = 0; v < NVAR; ++v) U[v] = __ldg(u + (e * NVAR + v) * nn + p);
    const double T = temperature_newton<NSP>(mech, U, internal_energy<DIM, NSP>(U));
    const Prim<DIM> q = prim_mixture<DIM, NSP, true>(U, T, mech);
    double *a = aux + e * NA * nn + p;
    a[0] = q.p;
    a[nn] = q.a;
    if constexpr (RED) {
      double v2 = 0.0;
#pragma unroll
      for (int c = 0; c < DIM; ++c) v2 += q.v[c] * q.v[c];
      const double l = sqrt(v2) + q.a;
      if (!(l > 0.0) || !isfinite(l)) bad = 1;
      lam = fmax(lam, l);
    }
    if (with_source) {
      double om[NSP];
      production_rates_listed<NSP>(mech, T, U, Xs + threadIdx.x, 256, om);
#pragma unroll
      for (int s = 0; s < NSP; ++s) a[(2 + s) * nn] = om[s];
    }
  }
  if constexpr (RED) {
    lam = warp_max(lam);
    bad = __any_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0) {
      atomicMax(&red[0], (unsigned long long)__double_as_longlong(lam));
      if (bad) atomicAdd(&red[2], 1ULL);
    }
  }
}

// s = S(u): omega_s for the species rows, 0 for momentum and energy (eq. 20-22)
template <int DIM, int NSP>
__global__ void __launch_bounds__(256) chem_kernel(const double *__restrict__ u, double *__restrict__ s,
                                                   const MechDev *__restrict__ mech_g, long ne, int nn) {
  constexpr int NVAR = NSP + DIM + 1;
  __shared__ MechDev mech;
  load_mech(&mech, mech_g);
  const long total = ne * nn;
  for (long g = (long)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (long)gridDim.x * blockDim.x) {
    const long e = g / nn;
    const int p = (int)(g - e * nn);
    double U[NVAR], om[NSP];
#pragma unroll
    for (int v = 0; v < NVAR; ++v) U[v] = __ldg(u + (e * NVAR + v) * nn + p);
    const double T = temperature_newton<NSP>(mech, U, internal_energy<DIM, NSP>(U));
    production_rates<NSP>(mech, T, U, om);
#pragma unroll
    for (int v = 0; v < NVAR; ++v) s[(e * NVAR + v) * nn + p] = (v < NSP) ? om[v] : 0.0;
  }
}

// Implicit source substep S_dt (eq. 24-25; R14): per node, Newton on
// the backward-Euler residual R(Y*) = Y* - Y^n - dt omega(T(Y*), Y*) of the partial densities, with total density,
// momentum and total energy fixed.  One sweep = residual, NSP forward-difference Jacobian columns
// (eps_k = max(1e-7 |Y_k|, 1e-12)), Gauss-Jordan with partial pivoting -- all in registers; the only global traffic
// is one read of the nodal state and one write of its species rows.  In place.
template <int NSP>
__device__ __forceinline__ double implicit_residual(const MechDev &m, const double *Y, const double *Yn, double dt, double e_int,
                                                    double T_start, double *Xs, int stride, double *R) {
  // the caloric Newton converges to the same root (|dT| <= 1e-13 T) from any start in the table range: warm starts
  // from the temperature of the previous evaluation save most of its iterations
  const double T = temperature_newton<NSP>(m, Y, e_int, T_start);
  double om[NSP];
  production_rates_listed<NSP>(m, T, Y, Xs, stride, om);
#pragma unroll
  for (int s = 0; s < NSP; ++s) R[s] = Y[s] - Yn[s] - dt * om[s];
  return T;
}
template <int DIM, int NSP>
__global__ void __launch_bounds__(128) chem_implicit_kernel(double *__restrict__ u, const MechDev *__restrict__ mech_g, double dt,
                                                            long ne, int nn, int *__restrict__ max_sweeps) {
  constexpr int NVAR = NSP + DIM + 1;
  __shared__ MechDev mech;
  __shared__ double Xs[NSP * 128];
  load_mech(&mech, mech_g);
  const long total = ne * nn;
  int worst = 0;
  for (long g = (long)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (long)gridDim.x * blockDim.x) {
    const long e = g / nn;
    const int p = (int)(g - e * nn);
    double U[NVAR], Y[NSP], Yn[NSP];
#pragma unroll
    for (int v = 0; v < NVAR; ++v) U[v] = u[(e * NVAR + v) * nn + p];
    const double e_int = internal_energy<DIM, NSP>(U);
    double rho = 0.0;
#pragma unroll
    for (int s = 0; s < NSP; ++s) { Y[s] = Yn[s] = U[s]; rho += U[s]; }
    int it = 1;
    double Tc = 4000.0;
    for (; it <= 50; ++it) {
      double R[NSP], A[NSP][NSP + 1];
      Tc = implicit_residual<NSP>(mech, Y, Yn, dt, e_int, Tc, Xs + threadIdx.x, 128, R);
#pragma unroll
      for (int c = 0; c < NSP; ++c) {
        const double eps = fmax(1e-7 * fabs(Y[c]), 1e-12);
        double Yp[NSP], Rp[NSP];
#pragma unroll
        for (int s = 0; s < NSP; ++s) Yp[s] = (s == c) ? Y[s] + eps : Y[s];
        implicit_residual<NSP>(mech, Yp, Yn, dt, e_int, Tc, Xs + threadIdx.x, 128, Rp);
#pragma unroll
        for (int s = 0; s < NSP; ++s) A[s][c] = (Rp[s] - R[s]) / eps;
      }
#pragma unroll
      for (int s = 0; s < NSP; ++s) A[s][NSP] = R[s];
      // Gauss-Jordan with partial pivoting; row swaps as predicated exchanges (no dynamically indexed registers)
#pragma unroll
      for (int c = 0; c < NSP; ++c) {
        int piv = c;
        double best = fabs(A[c][c]);
#pragma unroll
        for (int r = c + 1; r < NSP; ++r)
          if (fabs(A[r][c]) > best) { best = fabs(A[r][c]); piv = r; }
#pragma unroll
        for (int r = c + 1; r < NSP; ++r)
          if (r == piv) {
#pragma unroll
            for (int q = 0; q <= NSP; ++q) { const double t = A[c][q]; A[c][q] = A[r][q]; A[r][q] = t; }
          }
        const double inv = 1.0 / A[c][c];
#pragma unroll
        for (int q = c; q <= NSP; ++q) A[c][q] *= inv;
#pragma unroll
        for (int r = 0; r < NSP; ++r) {
          if (r == c) continue;
          const double f = A[r][c];
#pragma unroll
          for (int q = c; q <= NSP; ++q) A[r][q] -= f * A[c][q];
        }
      }
      double dmax = 0.0;
#pragma unroll
      for (int s = 0; s < NSP; ++s) { Y[s] -= A[s][NSP]; dmax = fmax(dmax, fabs(A[s][NSP])); }
      if (dmax <= 1e-13 * rho) break;
    }
    worst = max(worst, it);
    // a node whose Newton iteration did not converge within 50 sweeps (it == 51) is poisoned, so that an unchecked call
    // (sweeps_out == NULL) cannot carry an unconverged state forward silently: the next marut_max_dt reports it
    const bool failed = it > 50;
#pragma unroll
    for (int s = 0; s < NSP; ++s) u[(e * NVAR + s) * nn + p] = failed ? __longlong_as_double(0x7ff8000000000000LL) : Y[s];
  }
  worst = __reduce_max_sync(0xffffffffu, worst);
  if ((threadIdx.x & 31) == 0) atomicMax(max_sweeps, worst);
}

// ======================================================================================
// Hennemann-Gassner shock indicator (R15).
// indicator_kernel: per element, q = rho p -> modal coefficients (V^-1 along every direction, ping-pong in shared
// memory) -> E = max of the two top-shell energy ratios -> alpha = 1/(1 + exp(-(s/T)(E - T))), clipped.
// indicator_smooth_kernel: alpha_e <- max over the face neighbours (conforming, both sides of a mortar).
// ======================================================================================
template <int DIM, int NP, int EB>
__global__ void __launch_bounds__(((EB * Geo<DIM, NP>::NN + 31) / 32) * 32)
indicator_kernel(const double *__restrict__ u, const double *__restrict__ Vinv_g, double gamma, double s_over_T, double T,
                 double amin, double amax, long ne, double *__restrict__ alpha) {
  using G = Geo<DIM, NP>;
  constexpr int NN = G::NN, NVAR = DIM + 2, TILE = EB * NN;
  __shared__ double A[TILE], B[TILE], Vs[NP * NP];
  const int tid = threadIdx.x;
  for (int i = tid; i < NP * NP; i += blockDim.x) Vs[i] = Vinv_g[i];
  const int el = tid / NN, p = tid - el * NN;
  const long e = (long)blockIdx.x * EB + el;
  const bool active = (tid < TILE) && (e < ne);
  const int qi = p % NP, qj = (p / NP) % NP, qk = (DIM == 3) ? p / (NP * NP) : 0;
  if (active) {
    double U[NVAR];
#pragma unroll
    for (int v = 0; v < NVAR; ++v) U[v] = __ldg(u + (e * NVAR + v) * NN + p);
    const Prim<DIM> pr = prim_ideal<DIM, false>(U, gamma);
    A[tid] = pr.rho * pr.p;
  }
  __syncthreads();
  // xi: A -> B
  if (active) {
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < NP; ++i) acc += Vs[qi * NP + i] * A[tid - qi + i];
    B[tid] = acc;
  }
  __syncthreads();
  // eta: B -> A
  if (active) {
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < NP; ++i) acc += Vs[qj * NP + i] * B[tid - qj * NP + i * NP];
    A[tid] = acc;
  }
  __syncthreads();
  double *src = A;
  if constexpr (DIM == 3) {
    // zeta: A -> B
    if (active) {
      double acc = 0.0;
#pragma unroll
      for (int i = 0; i < NP; ++i) acc += Vs[qk * NP + i] * A[tid - qk * NP * NP + i * NP * NP];
      B[tid] = acc;
    }
    __syncthreads();
    src = B;
  }
  // energies: one thread per element sums its NN modes (fixed order)
  if (active && p == 0) {
    constexpr int N = NP - 1;
    double et0 = 0.0, eh0 = 0.0, et1 = 0.0, eh1 = 0.0;
    int r = 0;
    for (int k = 0; k < ((DIM == 3) ? NP : 1); ++k)
      for (int j = 0; j < NP; ++j)
        for (int i = 0; i < NP; ++i, ++r) {
          int mx = i;
          if (j > mx) mx = j;
          if (k > mx) mx = k;
          const double m2 = src[el * NN + r] * src[el * NN + r];
          et0 += m2;
          if (mx == N) eh0 += m2;
          if (mx <= N - 1) {
            et1 += m2;
            if (mx == N - 1) eh1 += m2;
          }
        }
    double E = eh0 / et0;
    if (et1 > 0.0) E = fmax(E, eh1 / et1);
    double a = 1.0 / (1.0 + exp(-s_over_T * (E - T)));
    if (a < amin) a = 0.0;
    if (a > amax) a = amax;
    alpha[e] = a;
  }
}
// (3-D: a fine element's mortar entry names the mortar, mortar_info[3 m] its coarse element)
template <int DIM>
__global__ void indicator_smooth_kernel(const double *__restrict__ raw, const int2 *__restrict__ conn,
                                        const int *__restrict__ mortar_fine, const int *__restrict__ mortar_info, long ne,
                                        double *__restrict__ alpha) {
  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= ne) return;
  double a = raw[e];
#pragma unroll
  for (int f = 0; f < 2 * DIM; ++f) {
    const int2 cn = __ldg(&conn[e * 2 * DIM + f]);
    const int kind = cn.y & 3;
    if (kind == FK_CONFORMING || (DIM == 2 && kind == FK_MORTAR_FINE)) a = fmax(a, raw[cn.x]);
    else if (kind == FK_MORTAR_FINE) a = fmax(a, raw[__ldg(&mortar_info[cn.x * 3])]);
    else if (kind == FK_MORTAR_COARSE) {
      constexpr int NFINE = (DIM == 2) ? 2 : 4;
#pragma unroll
      for (int k = 0; k < NFINE; ++k) a = fmax(a, raw[__ldg(&mortar_fine[cn.x * NFINE + k])]);
    }
  }
  alpha[e] = a;
}

// ======================================================================================
// Per-stage positivity floor (R17): one thread per node, in place;
// rho <- max(rho, rho_min) with the momentum kept, then E raised so that p >= p_min.  Nodes above both floors are not
// written.  count (may be NULL): number of nodes changed, one atomicAdd per warp that changed any.
// ======================================================================================
template <int DIM>
__global__ void __launch_bounds__(256) positivity_floor_kernel(double *u, double gamma, double rho_min, double p_min, long ne,
                                                               int nn, unsigned long long *count) {
  constexpr int NVAR = DIM + 2;
  const long total = ne * nn;
  const long span = (long)gridDim.x * blockDim.x;
  const long rounds = (total + span - 1) / span;     // whole warps stay in the loop for the ballot
  for (long r = 0; r < rounds; ++r) {
    const long g = r * span + (long)blockIdx.x * blockDim.x + threadIdx.x;
    bool ch = false;
    if (g < total) {
      const long e = g / nn;
      double *U = u + e * NVAR * nn + (g - e * nn);
      double rho = U[0], m2 = 0.0;
      const double E = U[(long)(1 + DIM) * nn];
#pragma unroll
      for (int c = 0; c < DIM; ++c) {
        const double mc = U[(long)(1 + c) * nn];
        m2 += mc * mc;
      }
      if (rho < rho_min) {
        rho = rho_min;
        U[0] = rho;
        ch = true;
      }
      const double ke = 0.5 * m2 / rho;
      if ((gamma - 1.0) * (E - ke) < p_min) {
        U[(long)(1 + DIM) * nn] = p_min / (gamma - 1.0) + ke;
        ch = true;
      }
    }
    if (count != nullptr) {
      const unsigned b = __ballot_sync(0xffffffffu, ch);
      if (b != 0u && (threadIdx.x & 31) == 0) atomicAdd(count, (unsigned long long)__popc(b));
    }
  }
}

// ======================================================================================
// max wave speed / max diffusivity (a10; eq. 17-18): warp-shuffle reduction, one atomicMax per CTA.
// red[0] = max(|u|_2 + a) ; red[1] = max(mu/rho) ; red[2] = count of non-finite/non-positive speeds
// (bit patterns of non-negative doubles order like unsigned integers)
// ======================================================================================
template <int DIM, int NSP, int PHYS>
__global__ void __launch_bounds__(256) wave_speed_kernel(const double *__restrict__ u, const MechDev *__restrict__ mech_g,
                                                         double gamma, double mu, long ne, int nn,
                                                         unsigned long long *__restrict__ red) {
  constexpr int NVAR = NSP + DIM + 1;
  __shared__ MechDev mech;
  __shared__ double wl[8], wn[8];
  __shared__ int wbad[8];
  if constexpr (PHYS == PH_REACT) load_mech(&mech, mech_g);
  double lam = 0.0, nu = 0.0;
  int bad = 0;
  const long total = ne * nn;
  // two nodes per trip (one grid stride apart), all loads of both issued before either is used: twice the bytes in
  // flight per thread; the maxima do not depend on the order
  constexpr int UNR = (PHYS == PH_REACT) ? 1 : 2;
  const long stride = (long)gridDim.x * blockDim.x;
  for (long g0 = (long)blockIdx.x * blockDim.x + threadIdx.x; g0 < total; g0 += UNR * stride) {
    double U[UNR][NVAR];
    bool on[UNR];
#pragma unroll
    for (int k = 0; k < UNR; ++k) {
      const long g = g0 + k * stride;
      on[k] = g < total;
      const long gc = on[k] ? g : g0;
      const long e = gc / nn;
      const int p = (int)(gc - e * nn);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) U[k][v] = __ldg(u + (e * NVAR + v) * nn + p);
    }
#pragma unroll
    for (int k = 0; k < UNR; ++k) {
      if (!on[k]) continue;
      double l;
      if constexpr (PHYS == PH_REACT) {
        const double T = temperature_newton<NSP>(mech, U[k], internal_energy<DIM, NSP>(U[k]));
        const Prim<DIM> q = prim_mixture<DIM, NSP, true>(U[k], T, mech);
        double v2 = 0.0;
#pragma unroll
        for (int c = 0; c < DIM; ++c) v2 += q.v[c] * q.v[c];
        l = sqrt(v2) + q.a;
      } else l = wave_speed_ideal<DIM>(U[k], gamma);
      if (!(l > 0.0) || !isfinite(l)) bad = 1;
      lam = fmax(lam, l);
      if constexpr (PHYS == PH_NS) nu = fmax(nu, mu / U[k][0]);
    }
  }
  lam = warp_max(lam);
  nu = warp_max(nu);
  bad = __any_sync(0xffffffffu, bad);
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) { wl[w] = lam; wn[w] = nu; wbad[w] = bad; }
  __syncthreads();
  if (w == 0) {
    lam = (lane < (int)(blockDim.x >> 5)) ? wl[lane] : 0.0;
    nu = (lane < (int)(blockDim.x >> 5)) ? wn[lane] : 0.0;
    bad = (lane < (int)(blockDim.x >> 5)) ? wbad[lane] : 0;
    lam = warp_max(lam);
    nu = warp_max(nu);
    bad = __any_sync(0xffffffffu, bad);
    if (lane == 0) {
      atomicMax(&red[0], (unsigned long long)__double_as_longlong(lam));
      atomicMax(&red[1], (unsigned long long)__double_as_longlong(nu));
      if (bad) atomicAdd(&red[2], 1ULL);
    }
  }
}

// ======================================================================================
// metric terms (a0; R2).  One CTA per element, one thread per node.
// out: metric_full [e][MD][NN] (Ja^l_c planes then 1/J); elem_info [e][2] = {min J, max relative
// deviation of any metric plane from its node-0 value}
// ======================================================================================
template <int DIM, int NP>
__global__ void metrics_kernel(const double *__restrict__ xyz, double *__restrict__ metric_full,
                               double *__restrict__ elem_info, const double *__restrict__ Dg, long ne) {
  using G = Geo<DIM, NP>;
  constexpr int NN = G::NN, MD = G::MD;
  extern __shared__ double smem[];
  double *X = smem;                    // [DIM][NN]
  double *dX = X + DIM * NN;           // [DIM*DIM][NN]   dX[c*DIM+l] = d X_c / d xi_l
  double *Dsm = dX + DIM * DIM * NN;   // [NP*NP]
  double *ref = Dsm + NP * NP;         // [MD + 1]
  const long e = blockIdx.x;
  const int p = threadIdx.x;
  for (int i = p; i < NP * NP; i += NN) Dsm[i] = Dg[i];
  // coordinates relative to the element's first node (translation invariance of D and of the curl
  // form; round-off ~eps*h instead of ~eps*|X|; R2)
  for (int c = 0; c < DIM; ++c) X[c * NN + p] = xyz[(e * DIM + c) * NN + p] - xyz[(e * DIM + c) * NN];
  __syncthreads();
  int q[3] = {0, 0, 0};
  G::ijk(p, q);
  // Every operation below is a single correctly rounded FP64 operation in a fixed order
  // (__dmul_rn / __dadd_rn are never contracted into FMAs): with the 1-D operators rounded from
  // extended precision the metric terms are reproducible to the last bit, which matters because
  // low-Mach flows amplify metric round-off by p0/(rho u^2) through the discrete GCL residual.
  auto deriv = [&](auto f, int l) {   // sum_m D[q_l][m] f(node with q_l -> m), m ascending
    const int st = G::stride(l), base = p - q[l] * st;
    double acc = 0.0;
    for (int m = 0; m < NP; ++m) acc = __dadd_rn(acc, __dmul_rn(Dsm[q[l] * NP + m], f(base + m * st)));
    return acc;
  };
  for (int c = 0; c < DIM; ++c)
    for (int l = 0; l < DIM; ++l) dX[(c * DIM + l) * NN + p] = deriv([&](int r) { return X[c * NN + r]; }, l);
  __syncthreads();
  double Ja[DIM * DIM], J;
  if constexpr (DIM == 2) {
    const double x_xi = dX[0 * NN + p], x_eta = dX[1 * NN + p], y_xi = dX[2 * NN + p], y_eta = dX[3 * NN + p];
    Ja[0] = y_eta; Ja[1] = -x_eta; Ja[2] = -y_xi; Ja[3] = x_xi;
    J = __dsub_rn(__dmul_rn(x_xi, y_eta), __dmul_rn(x_eta, y_xi));
  } else {
    auto g = [&](int c, int l) { return dX[(c * 3 + l) * NN + p]; };
    auto det2 = [&](double a, double b, double c, double d) { return __dsub_rn(__dmul_rn(a, b), __dmul_rn(c, d)); };
    const double t1 = __dmul_rn(g(0, 0), det2(g(1, 1), g(2, 2), g(1, 2), g(2, 1)));
    const double t2 = __dmul_rn(g(0, 1), det2(g(1, 0), g(2, 2), g(1, 2), g(2, 0)));
    const double t3 = __dmul_rn(g(0, 2), det2(g(1, 0), g(2, 1), g(1, 1), g(2, 0)));
    J = __dadd_rn(__dsub_rn(t1, t2), t3);
    // conservative curl form: (Ja^i)_c = d_k[X_l d_j X_m] - d_j[X_l d_k X_m], (i,j,k), (c,m,l) cyclic
    for (int i = 0; i < 3; ++i) {
      const int j = (i + 1) % 3, k = (i + 2) % 3;
      for (int c = 0; c < 3; ++c) {
        const int mm = (c + 1) % 3, ll = (c + 2) % 3;
        const double A = deriv([&](int r) { return __dmul_rn(X[ll * NN + r], dX[(mm * 3 + j) * NN + r]); }, k);
        const double B = deriv([&](int r) { return __dmul_rn(X[ll * NN + r], dX[(mm * 3 + k) * NN + r]); }, j);
        Ja[i * 3 + c] = __dsub_rn(A, B);
      }
    }
  }
  // element reductions: min J and affinity measure (max relative deviation from the node-0 values)
  if (p == 0) {
    double s = 0.0;
    for (int k = 0; k < DIM * DIM; ++k) { ref[k] = Ja[k]; s = fmax(s, fabs(Ja[k])); }
    ref[DIM * DIM] = J;
    ref[MD] = s;
  }
  __syncthreads();   // also: every thread is done reading X / dX
  double dev = fabs(J - ref[DIM * DIM]) / fabs(ref[DIM * DIM]);
  for (int k = 0; k < DIM * DIM; ++k) dev = fmax(dev, fabs(Ja[k] - ref[k]) / ref[MD]);
  double *redJ = dX, *redD = dX + NN;
  redJ[p] = J;
  redD[p] = dev;
  __syncthreads();
  if (p == 0) {
    double mn = redJ[0], mx = redD[0];
    for (int r = 1; r < NN; ++r) { mn = fmin(mn, redJ[r]); mx = fmax(mx, redD[r]); }
    // affine element (R2b): metric terms constant to 1e-12 -> node-0 values at every node
    if (mx < 1e-12) mn = ref[DIM * DIM];
    elem_info[e * 2 + 0] = mn;
    elem_info[e * 2 + 1] = mx;
    ref[MD] = mx;
  }
  __syncthreads();
  const bool affine = ref[MD] < 1e-12;
  double *out = metric_full + e * MD * NN;
  for (int k = 0; k < DIM * DIM; ++k) out[k * NN + p] = affine ? ref[k] : Ja[k];
  out[DIM * DIM * NN + p] = 1.0 / (affine ? ref[DIM * DIM] : J);
}

// affine meshes: keep one metric set per element (node 0)
template <int DIM, int NP>
__global__ void compact_metrics_kernel(const double *__restrict__ metric_full, double *__restrict__ metric_el, long ne) {
  using G = Geo<DIM, NP>;
  const long g = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= ne * G::MD) return;
  metric_el[g] = metric_full[g * G::NN];
}

// affine meshes: lengths of the scaled face normals |Ja^l| per element (used by the line kernel)
template <int DIM>
__global__ void fnorm_kernel(const double *__restrict__ metric_el, double *__restrict__ fnorm, long ne) {
  const long g = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= ne * DIM) return;
  const long e = g / DIM;
  const int l = (int)(g - e * DIM);
  double n2 = 0.0;
#pragma unroll
  for (int c = 0; c < DIM; ++c) {
    const double x = metric_el[e * (DIM * DIM + 1) + l * DIM + c];
    n2 += x * x;
  }
  fnorm[g] = sqrt(n2);
}

// ---------------------------------------------------------------- launch helpers
template <int NN>
constexpr int elems_per_block() { return (256 / NN) < 1 ? 1 : 256 / NN; }

template <int DIM, int NP, bool AFFINE, bool ORIENT3 = false, bool BND = false>
cudaError_t launch_gradient_t(const GradParams &P, cudaStream_t st) {
  if constexpr (!BND) {
    // meshes with boundary or mortar faces: the general instantiation (orientation decode included)
    if (P.boundary) return launch_gradient_t<DIM, NP, AFFINE, (DIM == 3), true>(P, st);
  }
  if constexpr (DIM == 3 && !ORIENT3 && !BND) {
    if (P.oriented) return launch_gradient_t<DIM, NP, AFFINE, true>(P, st);
  }
  constexpr int NN = Geo<DIM, NP>::NN, EB = elems_per_block<NN>();
  constexpr int threads = ((EB * NN + 31) / 32) * 32;
  constexpr size_t smem = (size_t)((DIM + 2) * EB * NN + ((NP * NP + 1) & ~1) + (AFFINE ? 0 : DIM * DIM * EB * NN)) * sizeof(double);
  auto k = gradient_kernel<DIM, NP, AFFINE, EB, ORIENT3, BND>;
  static std::atomic<unsigned long long> attr_done{0};
  if (cudaError_t err = set_smem_once((const void *)k, smem, attr_done); err != cudaSuccess) return err;
  const long grid = (P.ne + EB - 1) / EB;
  k<<<(unsigned)grid, threads, smem, st>>>(P);
  return cudaGetLastError();
}

}  // namespace marut
