// marut_line2.cuh -- register-tiled fused stage kernel for 3-D Euler on affine meshes:
// the variant with the least traffic through the SM's load/store pipe, which is what bounds the stage
// (profiles/r01_c2_*.md).  One thread per xi-LINE of LGL nodes, EB elements per CTA, two roles per thread.
//
//   phase 0  TMA bulk copies (cp.async.bulk + mbarrier) land the CTA's contiguous u_in and u_n tiles in shared
//            memory; meanwhile every thread loads the connectivity of its six face tasks and issues the
//            neighbour gathers of its two xi-face nodes
//   phase A  line role: primitives and contravariant fluxes of the own line (eq. 9); Ftilde^xi stays in
//            registers (xi derivative with compile-time D), Ftilde^eta / Ftilde^zeta go to shared flux planes;
//            xi-face Rusanov lifts from registers; then the gathers of the four eta / zeta face nodes are issued
//   phase B  plane role: task (element, variable, xi-index): D_eta Ftilde^eta + D_zeta Ftilde^zeta on the
//            (eta,zeta)-plane in registers, result in place of Ftilde^eta (bank-conflict-free plane stride)
//   phase C  eta / zeta faces densely mapped (thread ln owns face node ln of each of the four faces); lifts go
//            to the (now free) Ftilde^zeta planes
//   phase D  line role: volume + lift + 1/J + SSP-RK combination (eq. 12, 45) in place of the u_n tile, then one
//            TMA bulk store of the u_out tile
//
// Product code; shares nothing with oracle/.
#pragma once
#include "marut_line.cuh"
#include "marut_node.cuh"

namespace marut {

template <int NP, int EB>
struct Line2Cfg {
  static constexpr int DIM = 3, NVAR = 5;
  static constexpr int NL = NP * NP, NN = NL * NP;
  static constexpr int ESZ = NVAR * NN;                  // doubles per element in global memory
  static constexpr int TILE = (EB * ESZ + 2) & ~1;       // u tile incl. alignment slack (even)
  static constexpr int NT = ((EB * NL + 31) / 32) * 32;
  static constexpr int PS = (NN | 15) - 10 >= NN ? (NN | 15) - 10 : (NN | 15) + 6;   // plane stride == 5 (mod 16)
  static constexpr int NPLN = 2 * EB * NVAR;             // eta and zeta planes
  static constexpr int NFS = 2 * NL + 2 * (NP - 2) * NP; // nodes on eta / zeta faces (aux slots)
  static constexpr int NPT = NVAR * NP;                  // plane tasks per element
  static constexpr size_t SMEM = sizeof(double) * (size_t)(2 * TILE + NPLN * PS + 2 * EB * NFS) + 16 + sizeof(int) * 6 * NL;
  static_assert(4 * NVAR * NL <= NVAR * PS, "lift buffer must fit the zeta planes of the element");
};

// aux slot of a node on an eta / zeta face (k in {0,N}: the two full planes first; else j in {0,N})
template <int NP>
__device__ __forceinline__ int aux_slot(int i, int j, int k) {
  return (k == 0 || k == NP - 1) ? ((k == 0) ? 0 : NP * NP) + j * NP + i
                                 : 2 * NP * NP + (k - 1) * 2 * NP + ((j == 0) ? 0 : NP) + i;
}

template <int NP, int EB>
__global__ void __launch_bounds__((Line2Cfg<NP, EB>::NT), 2) stage_line2_kernel(const __grid_constant__ StageParams P) {
  using C = Line2Cfg<NP, EB>;
  constexpr int DIM = 3, NVAR = 5, NL = C::NL, NN = C::NN, ESZ = C::ESZ, PS = C::PS, NFS = C::NFS, NT = C::NT, MD = 10;
  extern __shared__ __align__(16) double smem[];
  double *Ubuf = smem, *Nbuf = Ubuf + C::TILE, *Fsm = Nbuf + C::TILE, *Aux = Fsm + C::NPLN * PS;
  uint64_t *bars = reinterpret_cast<uint64_t *>(Aux + 2 * EB * NFS);
  int *lut = reinterpret_cast<int *>(bars + 2);   // [6][NL] volume node of face node ln on face f

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
  for (int i = tid; i < 6 * NL; i += NT) lut[i] = face_node_of<3, NP>(i / NL, (i % NL) % NP, (i % NL) / NP);
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

  const int el = tid / NL, ln = tid - el * NL;
  const int j = ln % NP, k = ln / NP;
  const bool active = (tid < EB * NL) && (el < nel);
  const long e = e0 + el;

  // connectivity of the six face tasks of this thread and the neighbour nodes they read
  const double *nb[6];
  int kind[6];
#pragma unroll
  for (int f = 0; f < 6; ++f) {
    nb[f] = P.u_in;
    kind[f] = FK_BOUNDARY;
    if (active) {
      const int2 cn = __ldg(&P.conn[e * 6 + f]);
      kind[f] = cn.y & 3;
      const int fR = (cn.y >> 2) & 7;
      nb[f] = (kind[f] == FK_CONFORMING) ? P.u_in + (long)cn.x * ESZ + lut[fR * NL + ln]
                                         : P.bc_state + (long)cn.x * NVAR;
    }
  }
  // neighbour traces of the two xi-face nodes: in flight while the tile lands
  double Upx[2][NVAR];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Upx[s][v] = active ? __ldg(nb[s] + ((kind[s] == FK_CONFORMING) ? v * NN : v)) : 1.0;

  double Ja[9], invJ = 0.0, fn[3] = {0.0, 0.0, 0.0};
  if (active) {
#pragma unroll
    for (int q = 0; q < 9; ++q) Ja[q] = __ldg(&P.metric[e * MD + q]);
    invJ = __ldg(&P.metric[e * MD + 9]);
#pragma unroll
    for (int l = 0; l < 3; ++l) fn[l] = __ldg(&P.fnorm[e * 3 + l]);
  }
  mbar_wait(&bars[0], 0);

  // ---- phase A: primitives and contravariant fluxes of the own line; xi derivative and xi faces in registers
  double R[NP][NVAR];
  const bool on_eta = (j == 0 || j == NP - 1), on_zeta = (k == 0 || k == NP - 1);
  if (active) {
    double Fx[NP][NVAR];
    double Ue[2][NVAR], irho_e[2], p_e[2], a_e[2];
    const double *ul = Ut + (el * NVAR) * NN + ln * NP;
    double *fe = Fsm + (el * NVAR) * PS + ln * NP;              // eta planes of the element
    double *fz = fe + EB * NVAR * PS;                           // zeta planes
#pragma unroll
    for (int i = 0; i < NP; ++i) {
      double U[NVAR], F[NVAR];
#pragma unroll
      for (int v = 0; v < NVAR; ++v) U[v] = ul[v * NN + i];
      const Prim<3> pr = prim_ideal<3, false>(U, P.gamma);
      flux_dot<3, 1>(U, pr, &Ja[0], Fx[i]);
      flux_dot<3, 1>(U, pr, &Ja[3], F);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) fe[v * PS + i] = F[v];
      flux_dot<3, 1>(U, pr, &Ja[6], F);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) fz[v * PS + i] = F[v];
      const bool need_a = (i == 0 || i == NP - 1 || on_eta || on_zeta);
      double a = 0.0;
      if (need_a) a = sqrt(P.gamma * pr.p * pr.irho);
      if (on_eta || on_zeta) {
        double *ax = Aux + el * NFS + aux_slot<NP>(i, j, k);
        ax[0] = pr.irho;
        ax[EB * NFS] = a;
      }
      if (i == 0 || i == NP - 1) {
        const int s = (i == 0) ? 0 : 1;
#pragma unroll
        for (int v = 0; v < NVAR; ++v) Ue[s][v] = U[v];
        irho_e[s] = pr.irho; p_e[s] = pr.p; a_e[s] = a;
      }
    }
#pragma unroll
    for (int i = 0; i < NP; ++i)
#pragma unroll
      for (int v = 0; v < NVAR; ++v) {
        double acc = P.D[i * NP] * Fx[0][v];
#pragma unroll
        for (int m = 1; m < NP; ++m) acc += P.D[i * NP + m] * Fx[m][v];
        R[i][v] = acc;
      }
    // xi faces (a2, a4): both end points of the own line, everything from registers
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      const double sgn = s ? 1.0 : -1.0;
      double nv[3], lift[NVAR], Fm[NVAR];
#pragma unroll
      for (int c = 0; c < 3; ++c) nv[c] = sgn * Ja[c];
      rusanov_lift<3>(Ue[s], irho_e[s], p_e[s], a_e[s], Upx[s], nv, fn[0], P.gamma, P.inv_wb, lift, Fm);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) R[s ? NP - 1 : 0][v] += lift[v];
    }
  }
  // neighbour traces of the four eta / zeta face nodes: in flight during phase B
  double Upf[4][NVAR];
#pragma unroll
  for (int f = 2; f < 6; ++f)
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Upf[f - 2][v] = active ? __ldg(nb[f] + ((kind[f] == FK_CONFORMING) ? v * NN : v)) : 1.0;
  __syncthreads();

  // ---- phase B: plane tasks (element, variable, xi-index): eta and zeta derivatives in registers
  for (int t = tid; t < nel * C::NPT; t += NT) {
    double *pe = Fsm + (t / NP) * PS + (t % NP);      // t / NP = el * NVAR + v : plane index; lane t -> bank t mod 16
    const double *pz = pe + EB * NVAR * PS;
    double Rp[NP][NP];                                // [k][j]
#pragma unroll
    for (int kk = 0; kk < NP; ++kk) {
      double f[NP];
#pragma unroll
      for (int m = 0; m < NP; ++m) { f[m] = pe[kk * NL + m * NP]; Rp[kk][m] = 0.0; }
      line_deriv<NP>(P, f, Rp[kk]);
    }
#pragma unroll
    for (int jj = 0; jj < NP; ++jj) {
      double f[NP], acc[NP];
#pragma unroll
      for (int m = 0; m < NP; ++m) { f[m] = pz[m * NL + jj * NP]; acc[m] = Rp[m][jj]; }
      line_deriv<NP>(P, f, acc);
#pragma unroll
      for (int kk = 0; kk < NP; ++kk) pe[kk * NL + jj * NP] = acc[kk];
    }
  }
  __syncthreads();

  // ---- phase C: eta / zeta faces: thread ln owns face node (a0, a1) = (j, k) of each of the four faces;
  //      lifts -> zeta planes of the element: [face - 2][variable][face node]
  if (active) {
    double *lz = Fsm + (EB * NVAR + el * NVAR) * PS;
#pragma unroll
    for (int f = 2; f < 6; ++f) {
      const int l = f >> 1, side = f & 1;
      const double sgn = side ? 1.0 : -1.0;
      const int pi = j, pj = (l == 1) ? side * (NP - 1) : k, pk = (l == 1) ? k : side * (NP - 1);
      const int p = pi + NP * (pj + NP * pk);
      double Um[NVAR], nv[3], lift[NVAR], Fm[NVAR];
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Um[v] = Ut[(el * NVAR + v) * NN + p];
      const double *ax = Aux + el * NFS + aux_slot<NP>(pi, pj, pk);
      const double irhom = ax[0], am = ax[EB * NFS];
      double ke = 0.0;
#pragma unroll
      for (int c = 0; c < 3; ++c) { nv[c] = sgn * Ja[l * 3 + c]; ke += Um[1 + c] * Um[1 + c]; }
      const double pm = (P.gamma - 1.0) * (Um[4] - 0.5 * ke * irhom);
      rusanov_lift<3>(Um, irhom, pm, am, Upf[f - 2], nv, fn[l], P.gamma, P.inv_wb, lift, Fm);
#pragma unroll
      for (int v = 0; v < NVAR; ++v) lz[((f - 2) * NVAR + v) * NL + ln] = lift[v];
    }
  }
  if (use_un) mbar_wait(&bars[1], 0);
  __syncthreads();

  // ---- phase D: volume + lifts + 1/J + SSP-RK combination (eq. 12, 45), in place of the u_n tile
  if (active) {
    const double *ul = Ut + (el * NVAR) * NN + ln * NP;
    double *nl = Nt + (el * NVAR) * NN + ln * NP;
    const double *re = Fsm + (el * NVAR) * PS + ln * NP;
    const double *lz = Fsm + (EB * NVAR + el * NVAR) * PS;
    const double *le = lz + (((j == 0) ? 0 : 1) * NVAR) * NL + NP * k;
    const double *lzz = lz + ((2 + ((k == 0) ? 0 : 1)) * NVAR) * NL + NP * j;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) {
      double r[NP], uu[NP], un[NP];
#pragma unroll
      for (int i = 0; i < NP; ++i) {
        r[i] = re[v * PS + i];
        uu[i] = ul[v * NN + i];
        un[i] = use_un ? nl[v * NN + i] : 0.0;
      }
      if (on_eta) {
#pragma unroll
        for (int i = 0; i < NP; ++i) r[i] += le[v * NL + i];
      }
      if (on_zeta) {
#pragma unroll
        for (int i = 0; i < NP; ++i) r[i] += lzz[v * NL + i];
      }
#pragma unroll
      for (int i = 0; i < NP; ++i) nl[v * NN + i] = P.ca * un[i] + (P.cb * uu[i] + stage_cc(P) * (0.0 - invJ * (R[i][v] + r[i])));
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

template <int NP>
constexpr int line2_eb() { return (NP == 5) ? 5 : ((NP == 4) ? 8 : ((NP == 3) ? 14 : ((NP == 6) ? 3 : 1))); }

template <int NP>
cudaError_t launch_stage_line2_t(const StageParams &P, cudaStream_t st) {
  constexpr int EB = line2_eb<NP>();
  using C = Line2Cfg<NP, EB>;
  auto k = stage_line2_kernel<NP, EB>;
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
