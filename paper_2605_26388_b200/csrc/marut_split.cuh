// marut_split.cuh -- fused Euler stage with the entropy-stable split-form volume integral (
// PAPER.md:183-187 eq. 10, 594-627 eq. 39-41): R_i = -(2/J_i) sum_l sum_m D_{i_l m} F#(U_i, U_m; avg Ja^l), F# the
// two-point flux of Ranocha with logarithmic means (reading R13).  Interface / mortar / boundary flux,
// lift, 1/J and the SSP-RK combination are those of marut_node.cuh (same face tasks, same stash).
//
//   phase N  per node: U from global, primitives; stash U, 1/rho, p, a (face tasks) and ln rho, ln(rho/p)
//            (so that a logarithmic mean costs no logarithm per pair)
//   phase V  per node: for every direction and every node m of the line through the node: two-point flux with
//            the partner's stash entries, accumulated with D from the constant bank -- ALU-bound
//   phase S  face nodes, densely mapped (euler_face_task)
//   phase D  per node: lifts, 1/J, SSP-RK combination, u_n / u_out straight from / to global
//
// Product code; shares nothing with oracle/.
#pragma once
#include "marut_node.cuh"

namespace marut {

// logarithmic mean {{a}}^ln = num/den from the two values and their logarithms, one division for the caller (who
// needs either the mean or its reciprocal).  With d = aL - aR, s = aL + aR, u = (d/s)^2:
//   u >= 1e-2:  num = d, den = ln aL - ln aR                              (the definition)
//   u <  1e-2:  {{a}}^ln = s/(2 (1 + u/3 + u^2/5 + u^3/7)), multiplied through by s^6 (R13)
__device__ __forceinline__ void logmean_nd(double aL, double aR, double lnL, double lnR, double &num, double &den) {
  const double d = aL - aR, s = aL + aR, X = s * s, Y = d * d;
  if (Y < 1.0e-2 * X) {
    const double X2 = X * X, Y2 = Y * Y;
    num = s * X2 * X;
    den = 2.0 * (X2 * X + X2 * Y * (1.0 / 3.0) + X * Y2 * (1.0 / 5.0) + Y2 * Y * (1.0 / 7.0));
  } else {
    num = d;
    den = lnL - lnR;
  }
}

template <int DIM, int NP, bool AFFINE, int EB, int MINB, bool BCK = false>
__global__ void __launch_bounds__((NodeCfg<DIM, NP, 1, EB>::NT), MINB)
stage_split_kernel(const __grid_constant__ StageParams P) {
  using C = NodeCfg<DIM, NP, 1, EB>;
  using G = Geo<DIM, NP>;
  constexpr int NVAR = C::NVAR, NN = C::NN, NF = C::NF, TILE = C::TILE, NFN = C::NFN, NT = C::NT;
  constexpr int MD = G::MD, MDP = C::MDP, NST = C::NST;
  extern __shared__ __align__(16) double smem[];
  double *Ust = smem;                       // [NVAR + 3][TILE]  U, 1/rho, p, a
  double *Lns = Ust + NST * TILE;           // [3 + DIM][TILE]   ln rho, ln(rho/p), rho/p, velocity
  double *Pair = Lns + (3 + DIM) * TILE;    // [DIM][NP/2][NVAR][TILE] two-point fluxes left for the partner node
  double *Lft = Pair + DIM * (NP / 2) * NVAR * TILE;             // [NVAR][LFS]       lifts of the face nodes
  double *Msm = Lft + NVAR * C::LFS;        // affine: [EB][MDP] Ja, 1/J, |Ja^l|

  const int tid = threadIdx.x;
  const long e0 = (P.reverse ? (long)gridDim.x - 1 - (long)blockIdx.x : (long)blockIdx.x) * EB;   // (see stage_phys_kernel)
  const int nel = (int)((P.ne - e0 < EB) ? (P.ne - e0) : EB);
  const int ntask = nel * NFN;
  // L2 prefetch of the state (curved: and metric) planes of the block about half a wave ahead, as in stage_phys_kernel
  if (tid == 0) {
    const long ep = e0 + (P.reverse ? -1L : 1L) * (74 * MINB) * EB;
    if (ep >= 0 && ep + EB < P.ne) {
      l2_prefetch(P.u_in + ep * NVAR * NN, (size_t)EB * NVAR * NN * sizeof(double));
      if constexpr (!AFFINE) l2_prefetch(P.metric + ep * MD * NN, (size_t)EB * MD * NN * sizeof(double));
    }
  }
  const bool has0 = tid < ntask;
  const FaceTask t0 = decode_task<DIM, NP>(has0 ? tid : 0);
  int2 cn0 = make_int2(0, FK_BOUNDARY);
  if (has0) cn0 = __ldg(&P.conn[(e0 + t0.el) * 2 * DIM + t0.f]);
  if constexpr (AFFINE) {
    for (int i = tid; i < nel * MDP; i += NT) {
      const int me = i / MDP, k = i - me * MDP;
      Msm[i] = (k < MD) ? __ldg(&P.metric[(e0 + me) * MD + k]) : ((k < MD + DIM) ? __ldg(&P.fnorm[(e0 + me) * DIM + (k - MD)]) : 0.0);
    }
  }
  const int el = tid / NN, p = tid - el * NN;
  const long e = e0 + el;
  const bool active = (tid < TILE) && (el < nel);
  const int qi = p % NP, qj = (p / NP) % NP, qk = (DIM == 3) ? p / (NP * NP) : 0;

  // ---- phase N
  double U[NVAR], vi[DIM], pi_ = 0.0, lnr = 0.0, lnb = 0.0;
  if (active) {
    const double *up = P.u_in + e * NVAR * NN + p;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) U[v] = __ldg(up + v * NN);
    // u_n, read by the combination at the kernel's end, and 1/J of a curved mesh: into L2 now (no registers held)
    if (P.ca != 0.0) {
#pragma unroll
      for (int v = 0; v < NVAR; ++v) asm volatile("prefetch.global.L2 [%0];" ::"l"(P.u_n + (e * NVAR + v) * NN + p));
    }
    if constexpr (!AFFINE) asm volatile("prefetch.global.L2 [%0];" ::"l"(&P.metric[(e * MD + DIM * DIM) * NN + p]));
    const Prim<DIM> pr = prim_ideal<DIM, true>(U, P.gamma);
#pragma unroll
    for (int c = 0; c < DIM; ++c) vi[c] = pr.v[c];
    pi_ = pr.p;
    lnr = log(U[0]);
    lnb = log(U[0] / pr.p);
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Ust[v * TILE + tid] = U[v];
    Ust[NVAR * TILE + tid] = pr.irho;
    Ust[(NVAR + 1) * TILE + tid] = pr.p;
    Ust[(NVAR + 2) * TILE + tid] = pr.a;
    Lns[tid] = lnr;
    Lns[TILE + tid] = lnb;
    Lns[2 * TILE + tid] = U[0] / pr.p;
#pragma unroll
    for (int c = 0; c < DIM; ++c) Lns[(3 + c) * TILE + tid] = pr.v[c];
  }
  double Up0[NVAR];
  if (has0) gather_exterior<DIM, NP, NVAR>(P, t0, cn0, Up0);
  __syncthreads();

  // ---- phase V: split-form volume term (eq. 10).  F#(U_i, U_m) = F#(U_m, U_i) with the same averaged metric, so every
  // pair of a line is evaluated ONCE: node i takes its partners at cyclic distance s = 1..NP/2 (m = (i + s) mod NP;
  // for even NP the distance NP/2 only from the lower half), adds 2 D_im F# to its own residual and leaves F# in the
  // pair buffer for node m, which adds 2 D_mi F# after the barrier.  Balanced: NP/2 evaluations per direction.
  constexpr int NS = NP / 2;
  double R[NVAR];
#pragma unroll
  for (int v = 0; v < NVAR; ++v) R[v] = 0.0;
  if (active) {
    const double bi = U[0] / pi_, inv_gm1 = 1.0 / (P.gamma - 1.0);
#pragma unroll
    for (int l = 0; l < DIM; ++l) {
      const int ql = (l == 0) ? qi : ((l == 1) ? qj : qk);
      const int st = G::stride(l);
      const int base = tid - ql * st;
      double Ji[DIM];
#pragma unroll
      for (int c = 0; c < DIM; ++c) Ji[c] = AFFINE ? Msm[el * MDP + l * DIM + c] : __ldg(&P.metric[(e * MD + l * DIM + c) * NN + p]);
      if (ql == 0 || ql == NP - 1) {
        // diagonal term 2 D_ii F#(U_i, U_i) = 2 D_ii F_inv(U_i).Ja^l_i (D_ii = 0 at interior LGL nodes)
        const double d = P.D[ql * NP + ql];
        double vn = 0.0;
#pragma unroll
        for (int c = 0; c < DIM; ++c) vn += vi[c] * Ji[c];
        R[0] += d * (U[0] * vn);
#pragma unroll
        for (int c = 0; c < DIM; ++c) R[1 + c] += d * (U[1 + c] * vn + pi_ * Ji[c]);
        R[1 + DIM] += d * ((U[1 + DIM] + pi_) * vn);
      }
#pragma unroll
      for (int sd = 1; sd <= NS; ++sd) {
        if ((NP % 2 == 0) && sd == NS && ql >= NS) continue;
        const int m = (ql + sd >= NP) ? ql + sd - NP : ql + sd;
        const int pm = base + m * st;            // stash index of the partner node
        const double rm = Ust[pm], pmm = Ust[(NVAR + 1) * TILE + pm];
        // energy flux of the cited entropy-conservative flux (R13): kinetic term 1/2 v_i.v_m, pressure work
        // 1/2 (p_i v_m + p_m v_i).n
        double nv[DIM], vavg[DIM], vn = 0.0, v2 = 0.0, pvn = 0.0;
#pragma unroll
        for (int c = 0; c < DIM; ++c) {
          const double vm = Lns[(3 + c) * TILE + pm];
          if constexpr (AFFINE) nv[c] = Ji[c];
          else nv[c] = 0.5 * (Ji[c] + __ldg(&P.metric[(e * MD + l * DIM + c) * NN + (pm - el * NN)]));
          vavg[c] = 0.5 * (vi[c] + vm);
          vn += vavg[c] * nv[c];
          v2 += vi[c] * vm;
          pvn += 0.5 * (pi_ * vm + pmm * vi[c]) * nv[c];
        }
        double nr, dr, nb, db;
        logmean_nd(U[0], rm, lnr, Lns[pm], nr, dr);
        logmean_nd(bi, Lns[2 * TILE + pm], lnb, Lns[TILE + pm], nb, db);
        // one reciprocal for both means: rho_ln = nr/dr, 1/((gamma-1) {{T^-1}}^ln) = db/((gamma-1) nb)
        const double inv = 1.0 / (dr * nb);
        const double rho_ln = nr * (nb * inv);
        const double eint = inv_gm1 * (db * (dr * inv));
        const double pavg = 0.5 * (pi_ + pmm);
        const double mf = rho_ln * vn;
        double F[NVAR];
        F[0] = mf;
#pragma unroll
        for (int c = 0; c < DIM; ++c) F[1 + c] = mf * vavg[c] + pavg * nv[c];
        F[1 + DIM] = (eint + 0.5 * v2) * mf + pvn;
        const double d = P.D[ql * NP + m];
        double *pb = Pair + ((l * NS + (sd - 1)) * NVAR) * TILE + tid;
#pragma unroll
        for (int v = 0; v < NVAR; ++v) {
          R[v] += d * F[v];
          pb[v * TILE] = F[v];
        }
      }
    }
  }
  __syncthreads();
  if (active) {
#pragma unroll
    for (int l = 0; l < DIM; ++l) {
      const int ql = (l == 0) ? qi : ((l == 1) ? qj : qk);
      const int st = G::stride(l);
      const int base = tid - ql * st;
#pragma unroll
      for (int sd = 1; sd <= NS; ++sd) {
        const int i = (ql - sd < 0) ? ql - sd + NP : ql - sd;   // the node that evaluated the pair (i, ql)
        if ((NP % 2 == 0) && sd == NS && i >= NS) continue;
        const double d = P.D[ql * NP + i];
        const double *pb = Pair + ((l * NS + (sd - 1)) * NVAR) * TILE + base + i * st;
#pragma unroll
        for (int v = 0; v < NVAR; ++v) R[v] += d * pb[v * TILE];
      }
    }
#pragma unroll
    for (int v = 0; v < NVAR; ++v) R[v] *= 2.0;
  }

  // ---- phase B (only with a blending field; block-uniform branch): first-order finite-volume residual on the LGL
  // sub-cell grid and the convex blend of eq. 11 / 42 (reading R16).  Node i evaluates the Rusanov flux of the
  // sub-cell interface i+1/2 of each direction from the stash (no division, no square root on affine elements) and
  // leaves it in the pair buffer for node i+1; the outermost interfaces take the element's own flux, which the lift
  // of phase D turns into the interface flux.
  if (P.alpha != nullptr) {
    __syncthreads();                         // the pair buffer is free again
    double *Fv = Pair;                       // [l][v][TILE] at the slices of distance 1
    double Rf[NVAR];
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Rf[v] = 0.0;
    if (active) {
#pragma unroll
      for (int l = 0; l < DIM; ++l) {
        const int ql = (l == 0) ? qi : ((l == 1) ? qj : qk);
        const int st = G::stride(l);
        const double iw = P.inv_w[ql];
        double Ji[DIM];
#pragma unroll
        for (int c = 0; c < DIM; ++c) Ji[c] = AFFINE ? Msm[el * MDP + l * DIM + c] : __ldg(&P.metric[(e * MD + l * DIM + c) * NN + p]);
        if (ql == 0 || ql == NP - 1) {
          const double sg = (ql == 0) ? -iw : iw;
          double vn = 0.0;
#pragma unroll
          for (int c = 0; c < DIM; ++c) vn += vi[c] * Ji[c];
          Rf[0] += sg * (U[0] * vn);
#pragma unroll
          for (int c = 0; c < DIM; ++c) Rf[1 + c] += sg * (U[1 + c] * vn + pi_ * Ji[c]);
          Rf[1 + DIM] += sg * ((U[1 + DIM] + pi_) * vn);
        }
        if (ql < NP - 1) {
          const int pm = tid + st;
          double nv[DIM], nrm;
          if constexpr (AFFINE) {
#pragma unroll
            for (int c = 0; c < DIM; ++c) nv[c] = Ji[c];
            nrm = Msm[el * MDP + MD + l];
          } else {
            double n2 = 0.0;
#pragma unroll
            for (int c = 0; c < DIM; ++c) {
              nv[c] = __ldg(&P.subn[((e * DIM + l) * DIM + c) * NN + p]);
              n2 += nv[c] * nv[c];
            }
            nrm = sqrt(n2);
          }
          double Up[NVAR], vnm = 0.0, vnp = 0.0;
#pragma unroll
          for (int v = 0; v < NVAR; ++v) Up[v] = Ust[v * TILE + pm];
          const double pp = Ust[(NVAR + 1) * TILE + pm], ap = Ust[(NVAR + 2) * TILE + pm];
          const double am = Ust[(NVAR + 2) * TILE + tid];
#pragma unroll
          for (int c = 0; c < DIM; ++c) {
            vnm += vi[c] * nv[c];
            vnp += Lns[(3 + c) * TILE + pm] * nv[c];
          }
          const double hl = 0.5 * fmax(fabs(vnm) + am * nrm, fabs(vnp) + ap * nrm);
          double F[NVAR];
          F[0] = 0.5 * (U[0] * vnm + Up[0] * vnp) - hl * (Up[0] - U[0]);
#pragma unroll
          for (int c = 0; c < DIM; ++c)
            F[1 + c] = 0.5 * ((U[1 + c] * vnm + pi_ * nv[c]) + (Up[1 + c] * vnp + pp * nv[c])) - hl * (Up[1 + c] - U[1 + c]);
          F[1 + DIM] = 0.5 * ((U[1 + DIM] + pi_) * vnm + (Up[1 + DIM] + pp) * vnp) - hl * (Up[1 + DIM] - U[1 + DIM]);
#pragma unroll
          for (int v = 0; v < NVAR; ++v) {
            Rf[v] += iw * F[v];
            Fv[((l * NS) * NVAR + v) * TILE + tid] = F[v];
          }
        }
      }
    }
    __syncthreads();
    if (active) {
#pragma unroll
      for (int l = 0; l < DIM; ++l) {
        const int ql = (l == 0) ? qi : ((l == 1) ? qj : qk);
        if (ql == 0) continue;
        const double iw = P.inv_w[ql];
        const double *fb = Fv + (l * NS) * NVAR * TILE + tid - G::stride(l);
#pragma unroll
        for (int v = 0; v < NVAR; ++v) Rf[v] -= iw * fb[v * TILE];
      }
      const double al = __ldg(&P.alpha[e]);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) R[v] = (1.0 - al) * R[v] + al * Rf[v];
    }
  }

  // u_n for the final combination: issued before the face tasks, consumed after the last barrier (u_out may alias
  // u_n: only this thread writes these locations, later)
  double Un[NVAR];
  const bool use_un = (P.ca != 0.0);
  if (active && use_un) {
    const double *np_ = P.u_n + e * NVAR * NN + p;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Un[v] = np_[v * NN];
  }
  // ---- phase S: face nodes, densely mapped
  if (has0) euler_face_task<DIM, NP, AFFINE, EB, BCK>(P, Ust, Msm, Lft, e0, tid, t0, cn0, Up0);
  for (int g = tid + NT; g < ntask; g += NT) {
    const FaceTask t = decode_task<DIM, NP>(g);
    const int2 cn = __ldg(&P.conn[(e0 + t.el) * 2 * DIM + t.f]);
    double Up[NVAR];
    gather_exterior<DIM, NP, NVAR>(P, t, cn, Up);
    euler_face_task<DIM, NP, AFFINE, EB, BCK>(P, Ust, Msm, Lft, e0, g, t, cn, Up);
  }
  __syncthreads();
  if (!active) return;

  // ---- phase D
  {
    const double *lf = Lft + el * NFN;
    if (qi == 0 || qi == NP - 1) {
      const int g = ((qi == 0) ? 0 : 1) * NF + qj + NP * qk;
#pragma unroll
      for (int v = 0; v < NVAR; ++v) R[v] += lf[v * C::LFS + g];
    }
    if (qj == 0 || qj == NP - 1) {
      const int g = (2 + ((qj == 0) ? 0 : 1)) * NF + qi + NP * qk;
#pragma unroll
      for (int v = 0; v < NVAR; ++v) R[v] += lf[v * C::LFS + g];
    }
    if (DIM == 3 && (qk == 0 || qk == NP - 1)) {
      const int g = (4 + ((qk == 0) ? 0 : 1)) * NF + qi + NP * qj;
#pragma unroll
      for (int v = 0; v < NVAR; ++v) R[v] += lf[v * C::LFS + g];
    }
  }
  const double invJ = AFFINE ? Msm[el * MDP + DIM * DIM] : __ldg(&P.metric[(e * MD + DIM * DIM) * NN + p]);
  double *op = P.u_out + e * NVAR * NN + p;
  if (use_un) {
#pragma unroll
    for (int v = 0; v < NVAR; ++v) op[v * NN] = P.ca * Un[v] + (P.cb * U[v] + stage_cc(P) * (0.0 - invJ * R[v]));
  } else {
#pragma unroll
    for (int v = 0; v < NVAR; ++v) op[v * NN] = P.cb * U[v] + stage_cc(P) * (0.0 - invJ * R[v]);
  }
}

template <int DIM, int NP, bool AFFINE, bool BCK = false>
cudaError_t launch_stage_split_t(const StageParams &P, cudaStream_t st) {
  if constexpr (!BCK) {
    if (P.bc_kinds) return launch_stage_split_t<DIM, NP, AFFINE, true>(P, st);
  }
  constexpr int NN = Geo<DIM, NP>::NN, EB = node_eb<NN>();
  using C = NodeCfg<DIM, NP, 1, EB>;
  constexpr size_t smem = ((size_t)(C::NST + 3 + DIM + DIM * (NP / 2) * C::NVAR) * C::TILE + (size_t)C::NVAR * C::LFS + (AFFINE ? EB * C::MDP : 0)) * sizeof(double);
  constexpr int MINB = (C::NT <= 128) ? 4 : ((C::NT <= 256) ? 2 : 1);
  auto k = stage_split_kernel<DIM, NP, AFFINE, EB, MINB, BCK>;
  static std::atomic<unsigned long long> attr_done{0};
  if (cudaError_t err = set_smem_once((const void *)k, smem, attr_done); err != cudaSuccess) return err;
  const long grid = (P.ne + EB - 1) / EB;
  k<<<(unsigned)grid, C::NT, smem, st>>>(P);
  return cudaGetLastError();
}

}  // namespace marut
