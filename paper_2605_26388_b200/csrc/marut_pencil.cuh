// marut_pencil.cuh -- the fused stage kernel of compressible Euler on affine meshes: persistent
// CTAs, element tiles brought in by TMA bulk copies two tiles ahead (cp.async.bulk + mbarrier), one thread per LINE of
// n nodes with all variables of the line in registers.
//
//   tile   = ET consecutive elements, ET * n^(d-1) <= 128 lines per direction: one line per thread.  The tile's u_in
//            block is contiguous in global memory ([e][v][node]): ONE bulk copy per tile into a two-deep ring; thread 0
//            issues the copy for the tile after next when the current tile is finished.  N = 4 in 3-D has 5000-byte
//            elements: the 16-byte window the copy needs is obtained by starting one double early (`shift`).
//            The tile's connectivity and metric terms come in by 8-byte cp.async one tile ahead; u_n of the tile is
//            L2-prefetched (cp.async.bulk.prefetch.L2) at the start of the tile, one phase before it is read (3-D), or
//            brought into a shared-memory slot of its own by a second bulk copy (2-D, which has the room).
//            Tiles: the first three of a CTA round-robin, then (3-D) drawn from a device-wide counter.  Launches are
//            programmatic dependents of their stream predecessor (the prologue overlaps its tail).
//   phase l (l = 0 .. d-1): the thread owns the line of direction l through (a0, a1): it reads the line's U from the
//            tile, evaluates the contravariant flux Ftilde^l (eq. 9) at its n nodes, applies D along the line in
//            registers, and -- because the line's two end nodes ARE the face nodes (a0, a1) of faces 2l and 2l+1 --
//            evaluates both Rusanov lifts (eq. 12) from registers: no stash, no lift buffer, no divergence.
//            Exterior traces: from the tile itself when the neighbour is one of the tile's elements, else gathered from
//            global memory (L2); issued at the start of the phase, consumed at its end.
//            The partial residual goes through one shared buffer R: phase 0 writes, phase 1 adds (and folds in the
//            u_n term of eq. 45), the last phase adds, applies 1/J and the SSP-RK combination (eq. 45) and writes u_out
//            (zeta lines: coalesced).
//   Per node: 15 shared loads of U and 20 accesses of R, against ~115 shared accesses of the thread-per-node kernel;
//   3 CTA barriers per tile; 1.0/x and sqrt(x) are evaluated by the branch-free sequences of marut_common.cuh.
//
// Selected for MARUT_EULER with the strong form on affine meshes without outflow / slip-wall faces and without 3-D
// mortars (those run stage_node_kernel).  2-D meshes with 2:1 mortars run as TWO launches over tile lists built at
// marut_mesh_create: the tiles without mortar faces through the plain instantiation, the few with mortar faces through
// the MORTAR one (with the mortar path compiled into the kernel every tile ran 63 % slower: 168 registers and a stack
// frame; dispatching per tile inside one kernel, inlined or out of line, did not recover it).  The mortar fluxes themselves
// are evaluated once per mortar by mortar_flux2d_kernel ahead of the stage (marut_node.cuh) and read from there.
// PAPER.md:179-204, 713-725; R4-R8, R10.
// Product code; shares nothing with oracle/.
#pragma once
#include "marut_node.cuh"

namespace marut {

// ---------------------------------------------------------------- PTX wrappers (sm_100a)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
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
__device__ __forceinline__ void bulk_prefetch_l2(const void *src_gmem, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src_gmem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async8(void *dst_smem, const void *src_gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// ---------------------------------------------------------------- compile-time geometry
template <int DIM, int NP>
struct PencilCfg {
  static constexpr int NVAR = DIM + 2;
  static constexpr int NN = Geo<DIM, NP>::NN;
  static constexpr int NL = Geo<DIM, NP>::NF;        // lines per element and direction
  static constexpr int NT = 128;                     // threads per CTA
  static constexpr int ET = NT / NL;                 // elements per tile
  static constexpr int ED = NVAR * NN;               // doubles per element
  static constexpr int TD = ET * ED;                 // doubles per tile
  static constexpr int UB = (TD + 3) & ~1;           // ring slot: tile + the alignment window, itself 16-byte aligned
  // per-tile metadata, prefetched one tile ahead: conn[ET][2d] (int2), metric[ET][d*d+1], fnorm[ET][d]
  static constexpr int NCN = ET * 2 * DIM, NMT = ET * (DIM * DIM + 1), NFN = ET * DIM;
  static constexpr int MW = NCN + NMT + NFN;         // 8-byte words of one metadata slot
  // partial-residual buffer R: element stride ER.  2-D: padded so that the xi and the eta lines of the 128 / n elements of
  // a tile spread over the banks (with ER = ED every half-warp hit 4 of 16; pads by brute-force count over 0..16: 2.7x
  // fewer wavefronts for n = 4).  3-D: unpadded (n = 5 fills the shared memory three CTAs per SM leave).
  static constexpr int RPAD = (DIM != 2) ? 0 : (NP == 2 ? 2 : NP == 3 ? 5 : NP == 4 ? 3 : NP == 5 ? 5 : NP == 6 ? 7 : NP == 7 ? 4 : 1);
  static constexpr int ER = ED + RPAD;
  static constexpr int RD = (ET * ER + 1) & ~1;      // doubles of the R buffer
  // 2-D: the tile's u_n block comes in by a bulk copy of its own (one slot, issued at the start of the tile, consumed in
  // phase 1: phase 0 hides it) -- the 2-D kernels have the shared memory for it, and loading u_n through registers, even
  // two variables ahead, left 15 % of the samples of stages 1 and 2 on the folds' operands.  3-D: no room (n = 5).
  // (only where the slot does not cost a CTA per SM)
  static constexpr size_t base_bytes = (size_t)(2 * UB + RD + 2 * MW) * sizeof(double) + 4 * sizeof(uint64_t);
  static constexpr int UNB0 = (TD + 1) & ~1;
  static constexpr int CTAS0 = (233472 / (int)(base_bytes + 1024)) >= 3 ? 3 : (233472 / (int)(base_bytes + 1024));
  static constexpr bool UN_SMEM = (DIM == 2) && (233472 / (int)(base_bytes + UNB0 * sizeof(double) + 1024)) >= CTAS0;
  static constexpr int UNB = UN_SMEM ? UNB0 : 0;
  static constexpr size_t smem_bytes = base_bytes + (size_t)UNB * sizeof(double);
  static_assert(ET >= 1, "a direction's lines of one element must fit one CTA");
  // CTAs per SM the shared memory allows (228 KB per SM, 1 KB reserved per CTA), at most 3
  static constexpr int MINB = (233472 / (int)(smem_bytes + 1024)) >= 3 ? 3 : ((233472 / (int)(smem_bytes + 1024)) >= 2 ? 2 : 1);
};

// exterior state of face node (a0, a1) across the face described by cn: a conforming neighbour's trace (from the tile
// in shared memory when the neighbour is one of its elements, else from global memory) or a prescribed boundary state
template <int DIM, int NP>
__device__ __forceinline__ void pencil_gather(const StageParams &P, int2 cn, int a0, int a1, const double *__restrict__ Ut,
                                              long e0, int nel, double *Up) {
  constexpr int NVAR = DIM + 2, NN = Geo<DIM, NP>::NN;
  const int kind = cn.y & 3;
  if (kind == FK_CONFORMING) {
    const int fR = (cn.y >> 2) & 7, orient = (cn.y >> 5) & 7;
    int b0, b1;
    partner_index<DIM, NP>(orient, a0, a1, b0, b1);
    const int node = face_node_of<DIM, NP>(fR, b0, b1);
    const long de = (long)cn.x - e0;
    if (de >= 0 && de < nel) {
      const double *us = Ut + (int)de * NVAR * NN + node;
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Up[v] = us[v * NN];
    } else {
      const double *un = P.u_in + (long)cn.x * NVAR * NN + node;
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Up[v] = __ldcg(un + v * NN);
    }
  } else if (kind == FK_BOUNDARY) {
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Up[v] = __ldg(&P.bc_state[cn.x * NVAR + v]);
  } else {
#pragma unroll
    for (int v = 0; v < NVAR; ++v) Up[v] = 1.0;   // mortar faces: F* comes from node_mortar_flux_2d_stored
  }
}

// scalars of one face node that the per-variable lift needs (Rusanov with the scaled normal sgn * Ja^l; R5)
struct PencilFace {
  double hl;        // 1/2 lambda |n|
  double vnp, pp;   // exterior contravariant velocity Ja^l . v+ and pressure
  double mnp;       // Ja^l . m+
};
template <int DIM>
__device__ __forceinline__ PencilFace pencil_face(const double *Up, const double *Ja, double nrm, double gamma, double vnm,
                                                  double pm, double rinvm) {
  PencilFace F;
  const double rinvp = rcp_pos_2ulp(Up[0]);
  double mnp = 0.0, kep = 0.0;
#pragma unroll
  for (int c = 0; c < DIM; ++c) {
    mnp += Up[1 + c] * Ja[c];
    kep += Up[1 + c] * Up[1 + c];
  }
  F.mnp = mnp;
  F.pp = (gamma - 1.0) * (Up[DIM + 1] - 0.5 * kep * rinvp);
  F.vnp = mnp * rinvp;
  const double ap = sqrt_pos_2ulp(gamma * F.pp * rinvp), am = sqrt_pos_2ulp(gamma * pm * rinvm);
  F.hl = 0.5 * fmax(fabs(vnm) + am * nrm, fabs(F.vnp) + ap * nrm);
  return F;
}
// contravariant flux component v of a state (for the exterior side of a face)
template <int DIM>
__device__ __forceinline__ double pencil_flux_comp(int v, const double *Up, const PencilFace &F, const double *Ja) {
  if (v == 0) return F.mnp;
  if (v == DIM + 1) return (Up[DIM + 1] + F.pp) * F.vnp;
  return Up[v] * F.vnp + F.pp * Ja[v - 1];
}

// One phase of one line.  L = direction, FIRST / LAST = position of the phase in the element's sequence.
// Ut: the tile; Rs: partial residual; Md: the tile's metadata slot: conn (int2) | metric | fnorm.
// FUSE (last phase only): the thread also evaluates the wave speed |v| + a of the nodes it finishes, from the values it
// writes to u_out, with the expressions of wave_speed_kernel (eq. 18): lam / bad accumulate the maximum / a bad state.
template <int DIM, int NP, int L, bool MORTAR, bool FUSE = false>
__device__ __forceinline__ void pencil_phase(const StageParams &P, const double *__restrict__ Ut, double *__restrict__ Rs,
                                             const double *__restrict__ Md, long e0, int nel, int t, double cc, double &lam,
                                             int &bad, const double *Un = nullptr) {
  using C = PencilCfg<DIM, NP>;
  constexpr int NVAR = C::NVAR, NN = C::NN, NL = C::NL, ED = C::ED, MD = Geo<DIM, NP>::MD;
  constexpr bool FIRST = (L == 0), LAST = (L == DIM - 1);
  // The u_n term of eq. 45 enters the partial residual in phase 1 (3-D: the middle phase, 2-D: the last one), R += g u_n
  // with g = -ca J / cc, so that  cb U + cc (0 - R / J)  already contains ca u_n; its loads run one variable ahead of their
  // use (loaded where the combination needs them they stalled it: 13 % of the last phase's issue slots in 3-D)
  constexpr bool FOLD_HERE = (L == 1);
  constexpr int SM = (L == 0) ? 1 : ((L == 1) ? NP : NP * NP);
  if (t >= nel * NL) return;
  const int el = t / NL, r = t - el * NL;
  const int a1 = (DIM == 3) ? r / NP : 0, a0 = r - a1 * NP;
  const int p0 = (L == 0) ? NP * r : ((L == 1 && DIM == 3) ? a0 + NP * NP * a1 : r);
  const long e = e0 + el;
  const int2 *cs = reinterpret_cast<const int2 *>(Md) + el * 2 * DIM + 2 * L;
  const int2 c0 = cs[0], c1 = cs[1];
  double Up0[NVAR], Up1[NVAR];
  pencil_gather<DIM, NP>(P, c0, a0, a1, Ut, e0, nel, Up0);
  pencil_gather<DIM, NP>(P, c1, a0, a1, Ut, e0, nel, Up1);
  double U[NVAR][NP];
  const int ofs = el * ED + p0;
  {
    const double *ul = Ut + ofs;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) {
#pragma unroll
      for (int m = 0; m < NP; ++m) U[v][m] = ul[v * NN + m * SM];
    }
  }
  const bool fold_un = FOLD_HERE && (P.ca != 0.0);
  const long gofs = e * ED + p0;
  const double *met = Md + C::NCN + el * MD;
  double Ja[DIM];
#pragma unroll
  for (int c = 0; c < DIM; ++c) Ja[c] = met[L * DIM + c];
  const double nrm = Md[C::NCN + C::NMT + el * DIM + L];
  double invJ = 0.0;
  if constexpr (LAST || FOLD_HERE) invJ = met[DIM * DIM];
  double g = 0.0, unb[3][NP];      // u_n of variable v in unb[v % 3]: loaded while variables v - 2, v - 1 are worked on
  if constexpr (FOLD_HERE) {
    if (fold_un) {
      g = (0.0 - P.ca) / (cc * invJ);
#pragma unroll
      for (int m = 0; m < NP; ++m) unb[0][m] = C::UN_SMEM ? 0.0 : __ldcs(P.u_n + gofs + m * SM);
#pragma unroll
      for (int m = 0; m < NP; ++m) unb[1][m] = C::UN_SMEM ? 0.0 : __ldcs(P.u_n + gofs + NN + m * SM);
    }
  }
  double rinv[NP], pr[NP], vn[NP];
#pragma unroll
  for (int m = 0; m < NP; ++m) {
    rinv[m] = rcp_pos_2ulp(U[0][m]);
    double mn = 0.0, ke = 0.0;
#pragma unroll
    for (int c = 0; c < DIM; ++c) {
      mn += U[1 + c][m] * Ja[c];
      ke += U[1 + c][m] * (U[1 + c][m] * rinv[m]);
    }
    pr[m] = (P.gamma - 1.0) * (U[DIM + 1][m] - 0.5 * ke);
    vn[m] = mn * rinv[m];
  }
  double *rl = Rs + el * C::ER + p0;
  double accE[NVAR][2];
#pragma unroll
  for (int v = 0; v < NVAR; ++v) {
    if constexpr (FOLD_HERE) {
      if (!C::UN_SMEM && fold_un && v + 2 < NVAR) {
#pragma unroll
        for (int m = 0; m < NP; ++m) unb[(v + 2) % 3][m] = __ldcs(P.u_n + gofs + (v + 2) * NN + m * SM);
      }
    }
    double f[NP], acc[NP];
#pragma unroll
    for (int m = 0; m < NP; ++m) {
      if (v == 0) f[m] = U[0][m] * vn[m];
      else if (v == DIM + 1) f[m] = (U[DIM + 1][m] + pr[m]) * vn[m];
      else f[m] = U[v][m] * vn[m] + pr[m] * Ja[v - 1];
    }
    if constexpr (FIRST) {
#pragma unroll
      for (int i = 0; i < NP; ++i) acc[i] = 0.0;
    } else {
#pragma unroll
      for (int i = 0; i < NP; ++i) acc[i] = rl[v * NN + i * SM];
    }
    line_deriv<NP>(P, f, acc);
    if constexpr (FOLD_HERE) {
      if (fold_un) {
#pragma unroll
        for (int i = 0; i < NP; ++i) acc[i] = fma(g, C::UN_SMEM ? Un[el * ED + p0 + v * NN + i * SM] : unb[v % 3][i], acc[i]);
      }
    }
    accE[v][0] = acc[0];
    accE[v][1] = acc[NP - 1];
    if constexpr (!LAST) {
#pragma unroll
      for (int i = 1; i < NP - 1; ++i) rl[v * NN + i * SM] = acc[i];
    } else {
#pragma unroll
      for (int m = 1; m < NP - 1; ++m) {
        const double o = P.cb * U[v][m] + cc * (0.0 - invJ * acc[m]);
        P.u_out[gofs + v * NN + m * SM] = o;
        if constexpr (FUSE) U[v][m] = o;       // the node's new state replaces its old one (no longer needed)
      }
    }
  }
  const int k0 = c0.y & 3, k1 = c1.y & 3;
  {
    // Keep every consumer of the gathered traces below the volume loop: ptxas otherwise schedules the reciprocal of the
    // neighbour's density right behind its load and the warp sits out the gather's latency there (9 % of the samples).
    // The exclusive-or with a zero that is only known at run time and depends on the loop's last result ties them down.
    const int late = __double2loint(accE[NVAR - 1][1]) & P.zero;
#pragma unroll
    for (int v = 0; v < NVAR; ++v) {
      // (the HIGH word: the reciprocal's seed instruction, MUFU.RCP64H, reads nothing else)
      Up0[v] = __hiloint2double(__double2hiint(Up0[v]) ^ late, __double2loint(Up0[v]));
      Up1[v] = __hiloint2double(__double2hiint(Up1[v]) ^ late, __double2loint(Up1[v]));
    }
  }
  const PencilFace F0 = pencil_face<DIM>(Up0, Ja, nrm, P.gamma, vn[0], pr[0], rinv[0]);
  const PencilFace F1 = pencil_face<DIM>(Up1, Ja, nrm, P.gamma, vn[NP - 1], pr[NP - 1], rinv[NP - 1]);
  double Fs0[NVAR], Fs1[NVAR];   // mortar faces only: F* (outward) from the fluxes mortar_flux2d_kernel stored
  if constexpr (MORTAR && DIM == 2) {
    if (k0 >= FK_MORTAR_FINE) node_mortar_flux_2d_stored<NP>(P, a0, c0, Fs0);
    if (k1 >= FK_MORTAR_FINE) node_mortar_flux_2d_stored<NP>(P, a0, c1, Fs1);
  }
#pragma unroll
  for (int v = 0; v < NVAR; ++v) {
    double f0, f1;
    if (v == 0) { f0 = U[0][0] * vn[0]; f1 = U[0][NP - 1] * vn[NP - 1]; }
    else if (v == DIM + 1) { f0 = (U[v][0] + pr[0]) * vn[0]; f1 = (U[v][NP - 1] + pr[NP - 1]) * vn[NP - 1]; }
    else { f0 = U[v][0] * vn[0] + pr[0] * Ja[v - 1]; f1 = U[v][NP - 1] * vn[NP - 1] + pr[NP - 1] * Ja[v - 1]; }
    double lift0, lift1;
    if (MORTAR && DIM == 2 && k0 >= FK_MORTAR_FINE) lift0 = P.inv_wb * (Fs0[v] + f0);
    else lift0 = P.inv_wb * (0.5 * (f0 - pencil_flux_comp<DIM>(v, Up0, F0, Ja)) - F0.hl * (Up0[v] - U[v][0]));
    if (MORTAR && DIM == 2 && k1 >= FK_MORTAR_FINE) lift1 = P.inv_wb * (Fs1[v] - f1);
    else lift1 = P.inv_wb * (0.5 * (pencil_flux_comp<DIM>(v, Up1, F1, Ja) - f1) - F1.hl * (Up1[v] - U[v][NP - 1]));
    const double r0 = accE[v][0] + lift0, r1 = accE[v][1] + lift1;
    if constexpr (!LAST) {
      rl[v * NN] = r0;
      rl[v * NN + (NP - 1) * SM] = r1;
    } else {
      const double o0 = P.cb * U[v][0] + cc * (0.0 - invJ * r0), o1 = P.cb * U[v][NP - 1] + cc * (0.0 - invJ * r1);
      P.u_out[gofs + v * NN] = o0;
      P.u_out[gofs + v * NN + (NP - 1) * SM] = o1;
      if constexpr (FUSE) {
        accE[v][0] = o0;                       // U[v][0], U[v][NP-1] are still read by the later variables' lifts
        accE[v][1] = o1;
      }
    }
  }
  if constexpr (FUSE && LAST) {
#pragma unroll
    for (int m = 0; m < NP; ++m) {
      double Un[NVAR];
#pragma unroll
      for (int v = 0; v < NVAR; ++v) Un[v] = (m == 0) ? accE[v][0] : ((m == NP - 1) ? accE[v][1] : U[v][m]);
      const double l = wave_speed_ideal<DIM>(Un, P.gamma);
      if (!(l > 0.0) || !isfinite(l)) bad = 1;
      lam = fmax(lam, l);
    }
  }
}

// FUSE: the instantiation of the last stage of marut_ssprk33_step_cfl: besides the stage it reduces the maximum wave
// speed of the state it writes (warp shuffle, one atomicMax per CTA) and the CTA that finishes last evaluates eq. 18
// into P.dt_next -- the next step's CFL reduction without another pass over u.
template <int DIM, int NP, bool MORTAR, bool FUSE = false>
__global__ void __launch_bounds__(PencilCfg<DIM, NP>::NT, PencilCfg<DIM, NP>::MINB) stage_pencil_kernel(const __grid_constant__ StageParams P) {
  using C = PencilCfg<DIM, NP>;
  constexpr int ET = C::ET, ED = C::ED, TD = C::TD, UB = C::UB, NT = C::NT, MW = C::MW, MD = Geo<DIM, NP>::MD;
  extern __shared__ __align__(16) double smem[];
  double *Ub = smem;
  double *Rs = smem + 2 * UB;
  double *Mds = Rs + C::RD;
  double *Uns = Mds + 2 * MW;                 // 2-D: the tile's u_n block (C::UNB doubles)
  uint64_t *bars = reinterpret_cast<uint64_t *>(Uns + C::UNB);   // [0], [1]: ring slots, [2]: tile queue word, [3]: u_n slot
  const int tid = threadIdx.x;
  const long ntile = P.tile_list ? P.n_tile_list : (P.ne + ET - 1) / ET;
  const long total = P.ne * ED;
  const bool use_un = (P.ca != 0.0);
  auto window = [&](long tile, long &ws, int &wl, int &shift) -> bool {
    const long b = tile * TD;
    const long nel = (P.ne - tile * ET < ET) ? (P.ne - tile * ET) : ET;
    shift = (int)(b & 1);
    ws = b - shift;
    wl = (int)((nel * ED + shift + 1) & ~1L);
    return ws + wl <= total;
  };
  // P.reverse: the tiles are walked from the last to the first.  Consecutive stage launches alternate the direction, so
  // that a launch starts on the part of its input that the previous launch wrote or read last (still in L2).
  auto phys = [&](long k) -> long {
    const long i = P.reverse ? ntile - 1 - k : k;
    return P.tile_list ? (long)__ldg(&P.tile_list[i]) : i;
  };
  auto issue = [&](long k, int buf) {
    if (k >= ntile) return;                 // (before phys(k): the tile list ends at ntile)
    const long tile = phys(k);
    long ws;
    int wl, shift;
    if (window(tile, ws, wl, shift)) {
      mbar_expect_tx(&bars[buf], (uint32_t)wl * 8u);
      bulk_load(Ub + buf * UB, P.u_in + ws, (uint32_t)wl * 8u, &bars[buf]);
    }
  };
  auto fetch_meta = [&](long k, int buf) {
    if (k >= ntile) return;
    const long tile = phys(k);
    const long e0 = tile * ET;
    const int nel = (int)((P.ne - e0 < ET) ? (P.ne - e0) : ET);
    double *dst = Mds + buf * MW;
    for (int i = tid; i < nel * 2 * DIM; i += NT) cp_async8(dst + i, P.conn + e0 * 2 * DIM + i);
    for (int i = tid; i < nel * MD; i += NT) cp_async8(dst + C::NCN + i, P.metric + e0 * MD + i);
    for (int i = tid; i < nel * DIM; i += NT) cp_async8(dst + C::NCN + C::NMT + i, P.fnorm + e0 * DIM + i);
  };
  // Programmatic dependent launch: the launch that follows on the stream may place its CTAs as soon as this one's leave
  // (it does the same for its own successor), and runs its prologue -- barrier set-up, the first tile's connectivity and
  // metric terms, which no kernel writes -- while the last CTAs of this launch finish; everything a predecessor writes
  // (state, device-resident dt, mortar fluxes, the counter words) is touched only behind griddepcontrol.wait.
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (tid == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    mbar_init(&bars[3], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  fetch_meta(blockIdx.x, 0);
  cp_async_wait_all();
  __syncthreads();
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (tid == 0) {
    issue(blockIdx.x, 0);
    issue((long)blockIdx.x + gridDim.x, 1);
  }
  const double cc = stage_cc(P);
  double lam = 0.0;
  int bad = 0;
  // Tile queue of the CTA: q0 = the tile it works on, q1 = the next (its metadata is fetched now, its state copy is in
  // flight), q2 = the one after (its state copy is issued when q0's ring slot falls free).  The first three are the
  // static round-robin ones; after that the CTAs draw from a device-wide counter (P.tile_ctr), so that a CTA that
  // runs behind (or starts late behind another launch) takes fewer tiles -- no tail of a partly filled last round.
  // (3-D only: c2 -1.1 %.  On the short 2-D tiles warp 0's wait for the atomic at every tile cost more than the tail:
  // c4w +4.6 %; drawing early and publishing a phase later held a register pair across the phase: worse for both.)
  volatile long *qs = reinterpret_cast<volatile long *>(bars + 2);
  long q0 = blockIdx.x, q1 = q0 + gridDim.x, q2 = q1 + gridDim.x;
  int it = 0, nun = 0;
  for (; q0 < ntile; ++it) {
    const long k = q0;
    if (tid == 0) *qs = P.tile_ctr ? 3L * gridDim.x + (long)atomicAdd(&P.tile_ctr[0], 1u) : q2 + gridDim.x;
    const long tile = phys(k);
    const int buf = it & 1;
    const long e0 = tile * ET;
    const int nel = (int)((P.ne - e0 < ET) ? (P.ne - e0) : ET);
    long ws;
    int wl, shift;
    const bool by_tma = window(tile, ws, wl, shift);
    const double *Ut = Ub + buf * UB + shift;
    const double *Md = Mds + buf * MW;
    fetch_meta(q1, buf ^ 1);
    if (by_tma) {
      mbar_wait(&bars[buf], (uint32_t)((it >> 1) & 1));
    } else {
      // A tile that comes in without TMA (the last one of an odd-sized array, which a reversed or counter-drawn walk
      // meets early) still completes one phase of its slot's barrier, so that the parity of the slot's later waits
      // follows from `it` alone (the next wait on this slot lies two iterations, several barriers, ahead).
      if (tid == 0) mbar_arrive(&bars[buf]);
      double *dst = Ub + buf * UB + shift;
      for (int i = tid; i < nel * ED; i += NT) dst[i] = __ldg(P.u_in + e0 * ED + i);
      __syncthreads();
    }
    // u_n of this tile is read by phase 1.  3-D: bring it into L2 one phase ahead (earlier, and part of it is evicted
    // again).  2-D: into its shared-memory slot (free since the barrier that ended the previous tile).
    const bool un_smem = C::UN_SMEM && use_un && by_tma;
    if (tid == 0 && use_un && by_tma) {
      if constexpr (C::UN_SMEM) {
        mbar_expect_tx(&bars[3], (uint32_t)wl * 8u);
        bulk_load(Uns, P.u_n + ws, (uint32_t)wl * 8u, &bars[3]);
      } else bulk_prefetch_l2(P.u_n + ws, (uint32_t)wl * 8u);
    }
    pencil_phase<DIM, NP, 0, MORTAR>(P, Ut, Rs, Md, e0, nel, tid, cc, lam, bad);
    __syncthreads();
    if constexpr (DIM == 3) {
      pencil_phase<DIM, NP, 1, MORTAR>(P, Ut, Rs, Md, e0, nel, tid, cc, lam, bad);
      __syncthreads();
    }
    if constexpr (C::UN_SMEM) {
      if (un_smem) mbar_wait(&bars[3], (uint32_t)(nun & 1));
    }
    pencil_phase<DIM, NP, DIM - 1, MORTAR, FUSE>(P, Ut, Rs, Md, e0, nel, tid, cc, lam, bad, Uns);
    if (un_smem) ++nun;
    cp_async_wait_all();
    const long qn = *qs;                    // (written by thread 0 at the top of the iteration, barriers in between)
    __syncthreads();
    if (tid == 0) issue(q2, buf);
    q0 = q1;
    q1 = q2;
    q2 = qn;
  }
  if (P.tile_ctr && tid == 0) {             // the last CTA to finish leaves the counter words zero for the next launch
    __threadfence();
    if (atomicAdd(&P.tile_ctr[1], 1u) == gridDim.x - 1u) {
      P.tile_ctr[0] = 0u;
      P.tile_ctr[1] = 0u;
      __threadfence();
    }
  }
  if constexpr (FUSE) cfl_reduce_and_finalize(P, lam, bad, tid);
}

template <int DIM, int NP, bool MORTAR, bool FUSE = false>
cudaError_t launch_stage_pencil_t(const StageParams &P, bool force, cudaStream_t st) {
  if constexpr (!FUSE) {
    if (P.red_next) return launch_stage_pencil_t<DIM, NP, MORTAR, true>(P, force, st);
  }
  using C = PencilCfg<DIM, NP>;
  auto k = stage_pencil_kernel<DIM, NP, MORTAR, FUSE>;
  static std::atomic<unsigned long long> attr_done{0};
  if (cudaError_t err = set_smem_once((const void *)k, C::smem_bytes, attr_done); err != cudaSuccess) return err;
  const long ntile = P.tile_list ? P.n_tile_list : (P.ne + C::ET - 1) / C::ET;
  const long nres = (long)C::MINB * P.num_sms;   // one resident wave
  // a mesh that cannot fill the GPU with tiles runs the thread-per-node kernel (its smaller CTAs spread it better),
  // unless the caller insists (marut_debug_stage_kernel: the parity tests of small meshes)
  if (ntile < nres && !force) return cudaErrorNotSupported;
  const long grid = ntile < nres ? ntile : nres;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(C::NT);
  cfg.dynamicSmemBytes = C::smem_bytes;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, k, P);
}

}  // namespace marut
