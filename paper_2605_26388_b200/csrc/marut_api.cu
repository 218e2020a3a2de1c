// marut_api.cu -- the C ABI of include/marut.h: setup, dispatch of the fused stage
// kernels, the CFL reduction and the chemistry source.  Product code; shares nothing with oracle/.
#include "../../include/marut.h"
#include <atomic>
#include "marut_kernels.cuh"
#include "marut_launch.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <new>
#include <vector>

using namespace marut;

// ------------------------------------------------------------------------------------ errors
static thread_local char g_err[512] = "";
static marut_status fail(marut_status st, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return st;
}
#define CUDA_TRY(call)                                                                      \
  do {                                                                                      \
    cudaError_t err__ = (call);                                                             \
    if (err__ != cudaSuccess)                                                               \
      return fail(err__ == cudaErrorMemoryAllocation ? MARUT_ENOMEM : MARUT_ECUDA, "%s: %s", #call, \
                  cudaGetErrorString(err__));                                               \
  } while (0)

// ------------------------------------------------------------------------------------ mesh handle
struct marut_mesh {
  int dim = 0, N = 0, np = 0, nn = 0, nvar = 0, nsp = 1, physics = 0;
  long ne = 0, n_mortar = 0, n_bface = 0;
  int n_bc = 0;
  bool oriented = false;       // some 3-D interface has a non-trivial orientation code (R20)
  bool bc_kinds = false;       // some boundary id is an outflow / slip-wall face
  int pencil_reverse = 0;      // tile / block direction of the next launch of the line kernel or the split-form kernel (alternates)
  unsigned int *d_tile_ctr = nullptr;   // the line kernel's tile counter (two words, zero between launches)
  int *d_tiles_plain = nullptr, *d_tiles_mortar = nullptr;   // 2-D mortar meshes: the line kernel's tiles without / with mortar faces
  long n_tiles_plain = 0, n_tiles_mortar = 0;
  double gamma = 1.4, mu = 0.0, Pr = 0.72, kappa = 0.0;
  bool affine = false;
  double dx_min = 0.0;
  double D[MAX_NP * MAX_NP] = {0}, w[MAX_NP] = {0};
  // device
  double *d_metric = nullptr;
  double *d_fnorm = nullptr;   // affine: [e][dim] |Ja^l|
  int explicit_source = 1;     // reacting: L includes S(U) (default) or is the transport operator only
  int volume_form = 0;         // MARUT_VOLUME_STRONG | MARUT_VOLUME_SPLIT_RANOCHA
  int2 *d_conn = nullptr;
  int *d_mortar_fine = nullptr;
  int *d_mortar_info = nullptr;   // 3-D: [m][3] = eC, fC, fF
  double *d_mflux = nullptr;      // 3-D: F* at the fine face nodes of every mortar, [m][4][n*n][nvar]
  double *d_mortar_mat = nullptr;
  double *d_mW = nullptr;       // Navier-Stokes, 3-D mortars: central BR1 traces at the fine face nodes (mortar_trace3d_kernel)
  double *d_bc = nullptr;
  double *d_S = nullptr;     // NS scratch: stress tensor + heat flux from the BR1 gradient, [e][d(d+1)/2 + d][node]
  double *d_T = nullptr;     // reacting scratch of eos_kernel: [e][2 + n_species][node] = p, a, omega_s
  MechDev *d_mech = nullptr;
  double *d_Vinv = nullptr;  // [n][n] nodal -> orthonormal Legendre modal (shock indicator)
  double *d_araw = nullptr;  // [ne] unsmoothed blending coefficient (allocated on first use)
  const double *d_alpha = nullptr;  // caller-owned blending field of eq. 11 (marut_set_blend), or NULL
  double *d_subn = nullptr;  // curved meshes: sub-cell normals [e][l][c][node] (allocated by the first marut_set_blend)
  unsigned long long *d_red = nullptr;
  unsigned long long *d_red_next = nullptr;   // [4] reduction words of the fused CFL step (zero between uses)
  unsigned long long *h_red = nullptr;  // pinned
  std::atomic<long> launches{0};   // kernels launched through this handle (introspection; any thread)
  int stage_kernel_pref = 0;       // marut_debug_stage_kernel: 0 automatic, 1 thread-per-node kernel, 2 line kernel where eligible
  int ws_occ = 0;                  // resident CTAs per SM of this handle's wave_speed_kernel (queried on first use)
  int device = 0, num_sms = 148;   // the device the handle was created on and its multiprocessor count
};

// ------------------------------------------------------------------------------------ 1-D operators
// LGL nodes as the roots of q(x) = P_{N+1}(x) - P_{N-1}(x), q'(x) = (2N+1) P_N(x);
// w_j = 2 / (N (N+1) P_N(x_j)^2); D_ij = P_N(x_i) / (P_N(x_j) (x_i - x_j)), D_ii = -sum_{j != i} D_ij.
// Evaluated in extended precision and rounded once: x, w, D are the correctly rounded doubles of
// their exact values, so the setup is reproducible to the last bit across implementations.
template <typename T>
static void legendre_three(int N, T x, T &Pm1, T &P0, T &Pp1) {
  // returns P_{N-1}, P_N, P_{N+1}
  T a = 1, b = x;  // P_0, P_1
  if (N == 0) { Pm1 = 0; P0 = 1; Pp1 = x; return; }
  for (int k = 1; k < N; ++k) {
    T c = ((2 * k + 1) * x * b - k * a) / (k + 1);
    a = b; b = c;
  }
  Pm1 = a; P0 = b;
  Pp1 = ((2 * N + 1) * x * b - N * a) / (N + 1);
}
static void build_operators(int N, double *x_out, double *w_out, double *D_out) {
  typedef long double LD;
  const int n = N + 1;
  std::vector<LD> x(n), w(n), PN(n), D((size_t)n * n, 0);
  const LD PI = 3.141592653589793238462643383279502884L;
  for (int j = 0; j < n; ++j) {
    LD xj = -cosl(PI * j / N);
    if (j == 0) xj = -1;
    else if (j == N) xj = 1;
    else
      for (int it = 0; it < 100; ++it) {
        LD a, b, c;
        legendre_three<LD>(N, xj, a, b, c);
        LD dx = (c - a) / ((2 * N + 1) * b);
        xj -= dx;
        if (fabsl(dx) < 1e-20L) break;
      }
    x[j] = xj;
  }
  if (n % 2) x[n / 2] = 0;
  for (int j = 0; j < n; ++j) {
    LD a, b, c;
    legendre_three<LD>(N, x[j], a, b, c);
    PN[j] = b;
    w[j] = 2 / (N * (N + 1) * b * b);
  }
  for (int i = 0; i < n; ++i) {
    LD s = 0;
    for (int j = 0; j < n; ++j)
      if (j != i) { D[i * n + j] = PN[i] / (PN[j] * (x[i] - x[j])); s += D[i * n + j]; }
    D[i * n + i] = -s;
  }
  if (n % 2) D[(n / 2) * n + n / 2] = 0;
  for (int j = 0; j < n; ++j) { x_out[j] = (double)x[j]; w_out[j] = (double)w[j]; }
  for (int k = 0; k < n * n; ++k) D_out[k] = (double)D[k];
}
// barycentric evaluation of the Lagrange basis on nodes x at point y
static void lagrange_row(int n, const double *x, double y, double *row) {
  std::vector<double> lam(n);
  for (int j = 0; j < n; ++j) {
    double p = 1.0;
    for (int k = 0; k < n; ++k) if (k != j) p *= (x[j] - x[k]);
    lam[j] = 1.0 / p;
  }
  for (int j = 0; j < n; ++j)
    if (y == x[j]) { for (int k = 0; k < n; ++k) row[k] = (k == j) ? 1.0 : 0.0; return; }
  double den = 0.0;
  for (int j = 0; j < n; ++j) { row[j] = lam[j] / (y - x[j]); den += row[j]; }
  for (int j = 0; j < n; ++j) row[j] /= den;
}
// 2:1 mortar matrices (R7): P_fwd^m[i][j] = l_j((x_i -/+ 1)/2);
// P_rev^m = 1/2 M^-1 (P_fwd^m)^T M with the EXACT mass matrix M_ij = int l_i l_j (Gauss quadrature),
// i.e. the exact L2 projection onto degree-N polynomials on the coarse face.
static bool build_mortar(int N, const double *x, double *out /*[4][n*n]*/) {
  const int n = N + 1;
  // Gauss-Legendre rule with n points (exact to degree 2N+1)
  std::vector<double> g(n), wg(n);
  for (int q = 0; q < n; ++q) {
    double y = -std::cos(M_PI * (q + 0.75) / (n + 0.5));
    for (int it = 0; it < 100; ++it) {
      double a, b, c;
      legendre_three<double>(n, y, a, b, c);           // b = P_n(y), a = P_{n-1}(y)
      double dP = n * (y * b - a) / (y * y - 1.0);  // P_n'(y)
      double dy = b / dP;
      y -= dy;
      if (std::fabs(dy) < 1e-16) break;
    }
    double a, b, c;
    legendre_three<double>(n, y, a, b, c);
    double dP = n * (y * b - a) / (y * y - 1.0);
    g[q] = y; wg[q] = 2.0 / ((1.0 - y * y) * dP * dP);
  }
  std::vector<double> L(n * n), M(n * n, 0.0);   // L[q][j] = l_j(g_q)
  for (int q = 0; q < n; ++q) lagrange_row(n, x, g[q], &L[q * n]);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j)
      for (int q = 0; q < n; ++q) M[i * n + j] += wg[q] * L[q * n + i] * L[q * n + j];
  for (int m = 0; m < 2; ++m) {
    double *Pf = out + m * n * n, *Pr = out + (2 + m) * n * n;
    const double shift = m ? 1.0 : -1.0;
    for (int i = 0; i < n; ++i) lagrange_row(n, x, 0.5 * (x[i] + shift), &Pf[i * n]);
    // solve M X = 1/2 Pf^T M  (Gaussian elimination, partial pivoting)
    std::vector<double> A(M), B(n * n, 0.0);
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) {
        double s = 0.0;
        for (int k = 0; k < n; ++k) s += Pf[k * n + i] * M[k * n + j];
        B[i * n + j] = 0.5 * s;
      }
    for (int c = 0; c < n; ++c) {
      int piv = c;
      for (int r = c + 1; r < n; ++r) if (std::fabs(A[r * n + c]) > std::fabs(A[piv * n + c])) piv = r;
      if (A[piv * n + c] == 0.0) return false;
      if (piv != c)
        for (int k = 0; k < n; ++k) { std::swap(A[c * n + k], A[piv * n + k]); std::swap(B[c * n + k], B[piv * n + k]); }
      for (int r = c + 1; r < n; ++r) {
        double f = A[r * n + c] / A[c * n + c];
        for (int k = c; k < n; ++k) A[r * n + k] -= f * A[c * n + k];
        for (int k = 0; k < n; ++k) B[r * n + k] -= f * B[c * n + k];
      }
    }
    for (int c = n - 1; c >= 0; --c)
      for (int k = 0; k < n; ++k) {
        double s = B[c * n + k];
        for (int r = c + 1; r < n; ++r) s -= A[c * n + r] * Pr[r * n + k];
        Pr[c * n + k] = s / A[c * n + c];
      }
  }
  return true;
}

// ------------------------------------------------------------------------------------ metrics dispatch
template <int DIM>
static cudaError_t run_metrics(int np, const double *d_xyz, double *d_full, double *d_info, const double *d_D, long ne) {
#define MARUT_METRICS_CASE(NPV)                                                                            \
  case NPV: {                                                                                              \
    constexpr int NN = Geo<DIM, NPV>::NN;                                                                  \
    constexpr size_t smem = (size_t)((DIM + DIM * DIM) * NN + NPV * NPV + DIM * DIM + 2) * sizeof(double); \
    cudaError_t e1 = cudaFuncSetAttribute(metrics_kernel<DIM, NPV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
    if (e1 != cudaSuccess) return e1;                                                                      \
    metrics_kernel<DIM, NPV><<<(unsigned)ne, NN, smem>>>(d_xyz, d_full, d_info, d_D, ne);                  \
    return cudaGetLastError();                                                                             \
  }
  switch (np) {
    MARUT_METRICS_CASE(2) MARUT_METRICS_CASE(3) MARUT_METRICS_CASE(4) MARUT_METRICS_CASE(5)
    MARUT_METRICS_CASE(6) MARUT_METRICS_CASE(7) MARUT_METRICS_CASE(8)
  }
#undef MARUT_METRICS_CASE
  return cudaErrorNotSupported;
}
template <int DIM>
static cudaError_t run_compact(int np, const double *d_full, double *d_el, long ne) {
  const long total = ne * (DIM * DIM + 1);
  const unsigned grid = (unsigned)((total + 255) / 256);
  switch (np) {
    case 2: compact_metrics_kernel<DIM, 2><<<grid, 256>>>(d_full, d_el, ne); break;
    case 3: compact_metrics_kernel<DIM, 3><<<grid, 256>>>(d_full, d_el, ne); break;
    case 4: compact_metrics_kernel<DIM, 4><<<grid, 256>>>(d_full, d_el, ne); break;
    case 5: compact_metrics_kernel<DIM, 5><<<grid, 256>>>(d_full, d_el, ne); break;
    case 6: compact_metrics_kernel<DIM, 6><<<grid, 256>>>(d_full, d_el, ne); break;
    case 7: compact_metrics_kernel<DIM, 7><<<grid, 256>>>(d_full, d_el, ne); break;
    case 8: compact_metrics_kernel<DIM, 8><<<grid, 256>>>(d_full, d_el, ne); break;
    default: return cudaErrorNotSupported;
  }
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------ create / destroy
extern "C" void marut_mesh_destroy(marut_mesh *m) {
  if (!m) return;
  cudaDeviceSynchronize();
  cudaFree(m->d_metric); cudaFree(m->d_fnorm); cudaFree(m->d_conn); cudaFree(m->d_mortar_fine); cudaFree(m->d_mortar_info); cudaFree(m->d_mflux); cudaFree(m->d_mW); cudaFree(m->d_mortar_mat);
  cudaFree(m->d_Vinv); cudaFree(m->d_araw); cudaFree(m->d_subn); cudaFree(m->d_bc); cudaFree(m->d_S); cudaFree(m->d_T); cudaFree(m->d_mech); cudaFree(m->d_red);
  cudaFree(m->d_red_next); cudaFree(m->d_tiles_plain); cudaFree(m->d_tiles_mortar); cudaFree(m->d_tile_ctr);
  if (m->h_red) cudaFreeHost(m->h_red);
  delete m;
}

static marut_status create_impl(const marut_mesh_desc *d, marut_mesh *m) {
  if (d->dim != 2 && d->dim != 3) return fail(MARUT_EINVAL, "dim must be 2 or 3 (got %d)", d->dim);
  if (d->N < 1 || d->N > 7) return fail(MARUT_EINVAL, "N must be in 1..7 (got %d)", d->N);
  if (d->n_elem <= 0 || d->n_elem > 2000000000L) return fail(MARUT_EINVAL, "n_elem out of range");
  if (!d->node_xyz) return fail(MARUT_EINVAL, "node_xyz is NULL");
  if (d->n_iface < 0 || d->n_mortar < 0 || d->n_bface < 0 || d->n_bc < 0) return fail(MARUT_EINVAL, "negative count");
  if ((d->n_iface && !d->iface) || (d->n_mortar && !d->mortar) || (d->n_bface && !d->bface) || (d->n_bc && !d->bc_state))
    return fail(MARUT_EINVAL, "NULL connectivity array with non-zero count");
  if (d->physics < 0 || d->physics > 2) return fail(MARUT_EINVAL, "unknown physics %d", d->physics);
  if (d->physics == MARUT_REACTING_EULER && (d->n_mortar || d->n_bface))
    return fail(MARUT_EINVAL, "REACTING_EULER supports conforming interior faces only");
  if (d->physics != MARUT_REACTING_EULER && !(d->gamma > 1.0)) return fail(MARUT_EINVAL, "gamma must be > 1");
  if (d->physics == MARUT_NAVIER_STOKES && (!(d->mu >= 0.0) || !(d->Pr > 0.0))) return fail(MARUT_EINVAL, "need mu >= 0, Pr > 0");

  m->dim = d->dim; m->N = d->N; m->np = d->N + 1; m->ne = d->n_elem; m->physics = d->physics;
  m->nn = (d->dim == 2) ? m->np * m->np : m->np * m->np * m->np;
  m->gamma = d->gamma; m->mu = d->mu; m->Pr = d->Pr;
  if (d->physics == MARUT_NAVIER_STOKES) m->kappa = d->gamma * d->mu / (d->Pr * (d->gamma - 1.0));
  m->n_mortar = d->n_mortar;
  const int dim = m->dim, np = m->np, nn = m->nn, nf2 = 2 * dim;
  const long ne = m->ne;

  // mechanism
  if (d->physics == MARUT_REACTING_EULER) {
    const marut_mech *k = d->mech;
    if (!k) return fail(MARUT_EINVAL, "REACTING_EULER needs a mechanism");
    if (k->n_species < 1 || k->n_species > MAX_SPEC || k->n_reac < 0 || k->n_reac > MAX_REAC)
      return fail(MARUT_EINVAL, "mechanism size out of range");
    if (!k->W || !k->nasa || (k->n_reac && (!k->nu_r || !k->nu_p || !k->A || !k->b || !k->Ea)))
      return fail(MARUT_EINVAL, "NULL mechanism array");
    if (k->n_species != 5) return fail(MARUT_EINVAL, "this build instantiates the reacting kernels for 5 species only");
    MechDev h;
    memset(&h, 0, sizeof(h));
    h.ns = k->n_species; h.nr = k->n_reac; h.T_mid = k->T_mid;
    for (int s = 0; s < h.ns; ++s) {
      if (!(k->W[s] > 0.0)) return fail(MARUT_EINVAL, "molar mass must be positive");
      h.W[s] = k->W[s];
      h.Rs[s] = R_UNIVERSAL / k->W[s];
      for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 7; ++c) h.nasa[s][r][c] = k->nasa[(s * 2 + r) * 7 + c];
    }
    // reactions sorted (stably) by their net stoichiometric vector: reactions that differ only in the third body
    // share K_c, so the kernel evaluates exp(-dG) once per group
    std::vector<int> order(h.nr), grp(h.nr, -1);
    int ngrp = 0;
    for (int r = 0; r < h.nr; ++r) {
      for (int s = 0; s < h.ns; ++s) {
        int a = k->nu_r[r * h.ns + s], b = k->nu_p[r * h.ns + s];
        if (a < 0 || a > 3 || b < 0 || b > 3) return fail(MARUT_EINVAL, "stoichiometric coefficient out of 0..3");
      }
      for (int q = 0; q < r && grp[r] < 0; ++q) {
        bool same = true;
        for (int s = 0; s < h.ns; ++s)
          same = same && (k->nu_p[r * h.ns + s] - k->nu_r[r * h.ns + s] == k->nu_p[q * h.ns + s] - k->nu_r[q * h.ns + s]);
        if (same) grp[r] = grp[q];
      }
      if (grp[r] < 0) grp[r] = ngrp++;
    }
    for (int r = 0; r < h.nr; ++r) order[r] = r;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return grp[a] < grp[b]; });
    for (int i = 0; i < h.nr; ++i) {
      const int r = order[i];
      h.A[i] = k->A[r]; h.b[i] = k->b[r]; h.Ea[i] = k->Ea[r];
      h.new_group[i] = (i == 0 || grp[order[i - 1]] != grp[r]) ? 1 : 0;
      int nf = 0, nb = 0;
      for (int q = 0; q < 4; ++q) h.fr[i][q] = h.br[i][q] = -1;
      for (int s = 0; s < h.ns; ++s) {
        for (int q = 0; q < k->nu_r[r * h.ns + s]; ++q) { if (nf >= 3) return fail(MARUT_EINVAL, "reaction order above 3"); h.fr[i][nf++] = (signed char)s; }
        for (int q = 0; q < k->nu_p[r * h.ns + s]; ++q) { if (nb >= 3) return fail(MARUT_EINVAL, "reaction order above 3"); h.br[i][nb++] = (signed char)s; }
      }
      for (int s = 0; s < h.ns; ++s) {
        h.nu_r[i][s] = (signed char)k->nu_r[r * h.ns + s];
        h.nu_p[i][s] = (signed char)k->nu_p[r * h.ns + s];
      }
      h.dnu_sum[i] = 0.0;
      for (int s = 0; s < MAX_SPEC; ++s) {
        h.dnu[i][s] = (s < h.ns) ? (double)(k->nu_p[r * h.ns + s] - k->nu_r[r * h.ns + s]) : 0.0;
        h.dnu_sum[i] += h.dnu[i][s];
      }
    }
    m->nsp = h.ns;
    CUDA_TRY(cudaMalloc(&m->d_mech, sizeof(MechDev)));
    CUDA_TRY(cudaMemcpy(m->d_mech, &h, sizeof(MechDev), cudaMemcpyHostToDevice));
  }
  m->nvar = m->nsp + dim + 1;
  if (m->nvar > MAX_VAR) return fail(MARUT_EINVAL, "too many variables");
  if (d->n_bc && d->n_bface == 0) { /* unused states are fine */ }

  // ---- connectivity: element-face table, every face exactly once
  std::vector<int2> conn((size_t)ne * nf2, make_int2(-1, -1));
  auto claim = [&](long e, int f, int x, int info) -> bool {
    if (e < 0 || e >= ne || f < 0 || f >= nf2) return false;
    int2 &c = conn[(size_t)e * nf2 + f];
    if (c.y != -1) return false;
    c = make_int2(x, info);
    return true;
  };
  for (long i = 0; i < d->n_iface; ++i) {
    const int *I = d->iface + i * 5;
    if (I[4] < 0 || (dim == 3 && I[4] > 7) || (dim == 2 && I[4] > 1))
      return fail(MARUT_ETOPOLOGY, "iface %ld: unsupported orient %d", i, I[4]);
    if (dim == 3 && I[4] != 0) m->oriented = true;
    if (I[0] < 0 || I[0] >= ne || I[2] < 0 || I[2] >= ne || I[1] < 0 || I[1] >= nf2 || I[3] < 0 || I[3] >= nf2)
      return fail(MARUT_ETOPOLOGY, "iface %ld: index out of range", i);
    if (!claim(I[0], I[1], I[2], pack_info(FK_CONFORMING, I[3], I[4], 0)) ||
        !claim(I[2], I[3], I[0], pack_info(FK_CONFORMING, I[1], inverse_orientation(dim, I[4]), 0)))
      return fail(MARUT_ETOPOLOGY, "iface %ld: face listed twice", i);
  }
  // mortar rows: 2-D [6] = eC,fC,eF_lo,eF_up,fF,orient; 3-D [8] = eC,fC,eF_00,eF_10,eF_01,eF_11,fF,orient (R21)
  const int nfine = (dim == 2) ? 2 : 4, mstride = nfine + 4;
  if (dim == 3 && d->n_mortar > 0 && m->physics == MARUT_REACTING_EULER)
    return fail(MARUT_EINVAL, "3-D mortar faces are implemented for MARUT_EULER and MARUT_NAVIER_STOKES");
  std::vector<int> mfine((size_t)std::max<long>(1, d->n_mortar) * nfine, 0), minfo((size_t)std::max<long>(1, d->n_mortar) * 3, 0);
  for (long i = 0; i < d->n_mortar; ++i) {
    const int *M = d->mortar + i * mstride;
    const int fC = M[1], fF = M[2 + nfine];
    if (M[3 + nfine] != 0) return fail(MARUT_ETOPOLOGY, "mortar %ld: orient must be 0", i);
    if (M[0] < 0 || M[0] >= ne) return fail(MARUT_ETOPOLOGY, "mortar %ld: element out of range", i);
    for (int k = 0; k < nfine; ++k) if (M[2 + k] < 0 || M[2 + k] >= ne) return fail(MARUT_ETOPOLOGY, "mortar %ld: element out of range", i);
    if (fC < 0 || fC >= nf2 || fF < 0 || fF >= nf2) return fail(MARUT_ETOPOLOGY, "mortar %ld: face out of range", i);
    bool ok = claim(M[0], fC, (int)i, pack_info(FK_MORTAR_COARSE, fF, 0, 0));
    // fine side: conn.x = the coarse element (2-D; the mortar index rides in conn.y bits 10.. for the stored-flux path of the
    // line kernel) or the mortar index (3-D)
    if (dim == 2 && i >= (1L << 21)) return fail(MARUT_EINVAL, "more than 2^21 mortar faces");
    for (int k = 0; k < nfine && ok; ++k)
      ok = claim(M[2 + k], fF, (dim == 2) ? M[0] : (int)i, pack_info(FK_MORTAR_FINE, fC, 0, k) | ((dim == 2) ? (int)(i << 10) : 0));
    if (!ok) return fail(MARUT_ETOPOLOGY, "mortar %ld: face listed twice", i);
    for (int k = 0; k < nfine; ++k) mfine[i * nfine + k] = M[2 + k];
    minfo[i * 3] = M[0]; minfo[i * 3 + 1] = fC; minfo[i * 3 + 2] = fF;
  }
  for (long i = 0; i < d->n_bface; ++i) {
    const int *B = d->bface + i * 3;
    if (B[2] < 0 || B[2] >= d->n_bc) return fail(MARUT_ETOPOLOGY, "bface %ld: bc_id out of range", i);
    if (!claim(B[0], B[1], B[2], pack_info(FK_BOUNDARY, 0, 0, 0)))
      return fail(MARUT_ETOPOLOGY, "bface %ld: bad index or face listed twice", i);
  }
  for (size_t i = 0; i < conn.size(); ++i)
    if (conn[i].y == -1) return fail(MARUT_ETOPOLOGY, "element %ld face %d has no neighbour, mortar or boundary entry",
                                     (long)(i / nf2), (int)(i % nf2));

  // ---- operators
  double x[MAX_NP];
  build_operators(m->N, x, m->w, m->D);
  std::vector<double> mort((size_t)4 * np * np, 0.0);
  if (!build_mortar(m->N, x, mort.data())) return fail(MARUT_EINVAL, "singular mass matrix");

  // ---- uploads
  CUDA_TRY(cudaMalloc(&m->d_conn, conn.size() * sizeof(int2)));
  CUDA_TRY(cudaMemcpy(m->d_conn, conn.data(), conn.size() * sizeof(int2), cudaMemcpyHostToDevice));
  if (dim == 2 && d->n_mortar > 0) {
    // tiles of the persistent line kernel (128 / n consecutive elements, csrc/marut_pencil.cuh) with and without mortar
    // faces: the few with go to the kernel instantiation that carries the mortar path, the rest to the plain one
    const long et = 128 / np, nt = (ne + et - 1) / et;
    std::vector<int> plain, mort_t;
    for (long t = 0; t < nt; ++t) {
      bool has = false;
      for (long i = t * et * nf2; i < std::min<long>((t + 1) * et, ne) * nf2 && !has; ++i) has = (conn[i].y & 3) >= FK_MORTAR_FINE;
      (has ? mort_t : plain).push_back((int)t);
    }
    m->n_tiles_plain = (long)plain.size(); m->n_tiles_mortar = (long)mort_t.size();
    CUDA_TRY(cudaMalloc(&m->d_tiles_plain, std::max<size_t>(1, plain.size()) * sizeof(int)));
    CUDA_TRY(cudaMalloc(&m->d_tiles_mortar, std::max<size_t>(1, mort_t.size()) * sizeof(int)));
    if (!plain.empty()) CUDA_TRY(cudaMemcpy(m->d_tiles_plain, plain.data(), plain.size() * sizeof(int), cudaMemcpyHostToDevice));
    if (!mort_t.empty()) CUDA_TRY(cudaMemcpy(m->d_tiles_mortar, mort_t.data(), mort_t.size() * sizeof(int), cudaMemcpyHostToDevice));
  }
  CUDA_TRY(cudaMalloc(&m->d_mortar_fine, mfine.size() * sizeof(int)));
  CUDA_TRY(cudaMemcpy(m->d_mortar_fine, mfine.data(), mfine.size() * sizeof(int), cudaMemcpyHostToDevice));
  if (dim == 2 && d->n_mortar > 0 && m->physics == MARUT_EULER) {
    // the line kernel's mortar path: fluxes at the fine face nodes of every mortar, stored by mortar_flux2d_kernel
    CUDA_TRY(cudaMalloc(&m->d_mortar_info, minfo.size() * sizeof(int)));
    CUDA_TRY(cudaMemcpy(m->d_mortar_info, minfo.data(), minfo.size() * sizeof(int), cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMalloc(&m->d_mflux, (size_t)d->n_mortar * 2 * np * m->nvar * sizeof(double)));
  }
  if (dim == 3 && d->n_mortar > 0) {
    CUDA_TRY(cudaMalloc(&m->d_mortar_info, minfo.size() * sizeof(int)));
    CUDA_TRY(cudaMemcpy(m->d_mortar_info, minfo.data(), minfo.size() * sizeof(int), cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMalloc(&m->d_mflux, (size_t)d->n_mortar * 4 * np * np * m->nvar * sizeof(double)));
    if (m->physics == MARUT_NAVIER_STOKES) CUDA_TRY(cudaMalloc(&m->d_mW, (size_t)d->n_mortar * 4 * np * np * m->nvar * sizeof(double)));
  }
  CUDA_TRY(cudaMalloc(&m->d_mortar_mat, mort.size() * sizeof(double)));
  CUDA_TRY(cudaMemcpy(m->d_mortar_mat, mort.data(), mort.size() * sizeof(double), cudaMemcpyHostToDevice));
  m->n_bc = d->n_bc;
  m->n_bface = d->n_bface;
  const size_t nbc = (size_t)std::max(1, d->n_bc) * m->nvar;
  CUDA_TRY(cudaMalloc(&m->d_bc, nbc * sizeof(double)));
  if (d->n_bc) CUDA_TRY(cudaMemcpy(m->d_bc, d->bc_state, (size_t)d->n_bc * m->nvar * sizeof(double), cudaMemcpyHostToDevice));
  CUDA_TRY(cudaMalloc(&m->d_red, 5 * sizeof(unsigned long long)));   // [0..2] marut_max_dt, [3] marut_chem_implicit, [4] marut_positivity_floor
  CUDA_TRY(cudaMallocHost(&m->h_red, 5 * sizeof(unsigned long long)));
  CUDA_TRY(cudaMalloc(&m->d_red_next, 4 * sizeof(unsigned long long)));
  CUDA_TRY(cudaMalloc(&m->d_tile_ctr, 2 * sizeof(unsigned int)));
  CUDA_TRY(cudaMemset(m->d_tile_ctr, 0, 2 * sizeof(unsigned int)));
  CUDA_TRY(cudaMemset(m->d_red_next, 0, 4 * sizeof(unsigned long long)));

  // ---- metric terms on the device
  const int MD = dim * dim + 1;
  double *d_xyz = nullptr, *d_full = nullptr, *d_info = nullptr, *d_D = nullptr;
  auto cleanup = [&]() { cudaFree(d_xyz); cudaFree(d_full); cudaFree(d_info); cudaFree(d_D); };
  const size_t nxyz = (size_t)ne * dim * nn;
  cudaError_t ce;
  if ((ce = cudaMalloc(&d_xyz, nxyz * sizeof(double))) != cudaSuccess ||
      (ce = cudaMalloc(&d_full, (size_t)ne * MD * nn * sizeof(double))) != cudaSuccess ||
      (ce = cudaMalloc(&d_info, (size_t)ne * 2 * sizeof(double))) != cudaSuccess ||
      (ce = cudaMalloc(&d_D, np * np * sizeof(double))) != cudaSuccess) {
    cleanup();
    return fail(MARUT_ENOMEM, "device allocation for metrics failed: %s", cudaGetErrorString(ce));
  }
  std::vector<double> info((size_t)ne * 2);
  if ((ce = cudaMemcpy(d_xyz, d->node_xyz, nxyz * sizeof(double), cudaMemcpyHostToDevice)) != cudaSuccess ||
      (ce = cudaMemcpy(d_D, m->D, np * np * sizeof(double), cudaMemcpyHostToDevice)) != cudaSuccess ||
      (ce = (dim == 2 ? run_metrics<2>(np, d_xyz, d_full, d_info, d_D, ne) : run_metrics<3>(np, d_xyz, d_full, d_info, d_D, ne))) != cudaSuccess ||
      (ce = cudaMemcpy(info.data(), d_info, info.size() * sizeof(double), cudaMemcpyDeviceToHost)) != cudaSuccess) {
    cleanup();
    return fail(MARUT_ECUDA, "metric computation failed: %s", cudaGetErrorString(ce));
  }
  m->launches++;
  double dxm = 1e300, dev = 0.0;
  for (long e = 0; e < ne; ++e) {
    const double Jmin = info[e * 2];
    if (!(Jmin > 0.0) || !std::isfinite(Jmin)) { cleanup(); return fail(MARUT_ETOPOLOGY, "element %ld: Jacobian %g <= 0", e, Jmin); }
    dxm = std::min(dxm, 2.0 * std::pow(Jmin, 1.0 / dim));
    dev = std::max(dev, info[e * 2 + 1]);
  }
  m->dx_min = dxm;
  m->affine = dev < 1e-12;   // constant metrics to round-off -> keep one set per element
  if (m->affine) {
    if ((ce = cudaMalloc(&m->d_metric, (size_t)ne * MD * sizeof(double))) != cudaSuccess ||
        (ce = (dim == 2 ? run_compact<2>(np, d_full, m->d_metric, ne) : run_compact<3>(np, d_full, m->d_metric, ne))) != cudaSuccess ||
        (ce = cudaDeviceSynchronize()) != cudaSuccess) {
      cleanup();
      return fail(MARUT_ECUDA, "metric compaction failed: %s", cudaGetErrorString(ce));
    }
    m->launches++;
    if ((ce = cudaMalloc(&m->d_fnorm, (size_t)ne * dim * sizeof(double))) != cudaSuccess) { cleanup(); return fail(MARUT_ENOMEM, "fnorm allocation failed"); }
    const unsigned gfn = (unsigned)((ne * dim + 255) / 256);
    if (dim == 2) fnorm_kernel<2><<<gfn, 256>>>(m->d_metric, m->d_fnorm, ne);
    else fnorm_kernel<3><<<gfn, 256>>>(m->d_metric, m->d_fnorm, ne);
    if ((ce = cudaDeviceSynchronize()) != cudaSuccess) { cleanup(); return fail(MARUT_ECUDA, "fnorm kernel failed: %s", cudaGetErrorString(ce)); }
    m->launches++;
  } else {
    m->d_metric = d_full;
    d_full = nullptr;
  }
  cleanup();

  // ---- scratch
  if (m->physics == MARUT_NAVIER_STOKES) CUDA_TRY(cudaMalloc(&m->d_S, (size_t)ne * (dim * (dim + 1) / 2 + dim) * nn * sizeof(double)));
  if (m->physics == MARUT_REACTING_EULER) CUDA_TRY(cudaMalloc(&m->d_T, (size_t)ne * (2 + m->nsp) * nn * sizeof(double)));

  if (dim == 3 && d->n_mortar > 0 && !m->affine)
    return fail(MARUT_EINVAL, "3-D mortar faces need an affine mesh");
  return MARUT_OK;
}

extern "C" marut_status marut_mesh_create(const marut_mesh_desc *desc, marut_mesh **out) {
  if (!desc || !out) return fail(MARUT_EINVAL, "NULL argument");
  *out = nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(MARUT_ECUDA, "no CUDA device: this library has no CPU fallback");
  }
  marut_mesh *m = new (std::nothrow) marut_mesh;
  if (!m) return fail(MARUT_ENOMEM, "host allocation failed");
  if (cudaGetDevice(&m->device) != cudaSuccess ||
      cudaDeviceGetAttribute(&m->num_sms, cudaDevAttrMultiProcessorCount, m->device) != cudaSuccess || m->num_sms < 1) {
    delete m;
    cudaGetLastError();
    return fail(MARUT_ECUDA, "cannot query the current CUDA device");
  }
  marut_status st = create_impl(desc, m);
  if (st != MARUT_OK) {
    char keep[sizeof(g_err)];
    memcpy(keep, g_err, sizeof(keep));
    marut_mesh_destroy(m);
    cudaGetLastError();
    memcpy(g_err, keep, sizeof(keep));
    return st;
  }
  *out = m;
  return MARUT_OK;
}

// ------------------------------------------------------------------------------------ operator / stage
static bool misaligned(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

__global__ void dt_finalize_kernel(const unsigned long long *__restrict__ red, double cfl, double dx_min, double P2, double Pr,
                                   int ns, double *__restrict__ dt_out);

// fused CFL reduction of u_out in the stage kernel (marut_ssprk33_step_cfl): requested with cfl > 0 and dt_next; *done
// tells the caller whether the kernel that ran took it (else the caller runs marut_max_dt_async on u_out)
struct FuseCfl {
  double cfl = 0.0;
  double *dt_next = nullptr;
  bool done = false;
  // marut_ssprk33_step_dt, reacting mixture: the time step of THIS stage's input state, reduced inside eos_kernel and
  // finalized into dt_now before the stage kernel (which reads it as its device-resident dt) runs
  double *dt_now = nullptr;
};

static marut_status run_operator(marut_mesh *m, double ca, double cb, double cc, const double *u_n, const double *u_in,
                                 double *u_out, cudaStream_t st, const double *dt_dev = nullptr, FuseCfl *fuse = nullptr) {
  if (m->physics == MARUT_NAVIER_STOKES) {
    GradParams G;
    G.u = u_in; G.S = m->d_S; G.metric = m->d_metric; G.conn = m->d_conn;
    G.gamma = m->gamma; G.inv_wb = 1.0 / m->w[0]; G.mu = m->mu; G.kappa = m->kappa; G.ne = m->ne; G.oriented = m->oriented ? 1 : 0;
    G.bc_state = m->d_bc; G.boundary = (m->n_bface > 0 || m->n_mortar > 0) ? 1 : 0;
    G.mortar_fine = m->d_mortar_fine; G.mortar_mat = m->d_mortar_mat; G.mW = m->d_mW;
    if (m->dim == 3 && m->n_mortar > 0) {
      cudaError_t et = launch_mortar_trace3d(m->np, u_in, m->d_mortar_info, m->d_mortar_fine, m->d_mortar_mat, m->gamma, m->d_mW,
                                             m->n_mortar, st);
      if (et != cudaSuccess) return fail(MARUT_ECUDA, "mortar trace kernel: %s", cudaGetErrorString(et));
      m->launches++;
    }
    memcpy(G.D, m->D, sizeof(G.D));
    cudaError_t e = launch_gradient(m->dim, m->np, m->affine, G, st);
    if (e != cudaSuccess) return fail(e == cudaErrorNotSupported ? MARUT_EINVAL : MARUT_ECUDA, "gradient kernel: %s", cudaGetErrorString(e));
    m->launches++;
  }
  if (m->physics == MARUT_REACTING_EULER) {
    const long total = m->ne * m->nn;
    const unsigned grid = (unsigned)std::min<long>((total + 255) / 256, (long)m->num_sms * 16);
    const bool red = fuse && fuse->dt_now;
    if (red) CUDA_TRY(cudaMemsetAsync(m->d_red, 0, 3 * sizeof(unsigned long long), st));
    if (m->dim == 2) {
      if (red) eos_kernel<2, 5, true><<<grid, 256, 0, st>>>(u_in, m->d_T, m->d_mech, m->ne, m->nn, m->explicit_source, m->d_red);
      else eos_kernel<2, 5><<<grid, 256, 0, st>>>(u_in, m->d_T, m->d_mech, m->ne, m->nn, m->explicit_source);
    } else {
      if (red) eos_kernel<3, 5, true><<<grid, 256, 0, st>>>(u_in, m->d_T, m->d_mech, m->ne, m->nn, m->explicit_source, m->d_red);
      else eos_kernel<3, 5><<<grid, 256, 0, st>>>(u_in, m->d_T, m->d_mech, m->ne, m->nn, m->explicit_source);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(MARUT_ECUDA, "eos kernel: %s", cudaGetErrorString(e));
    m->launches++;
    if (red) {
      dt_finalize_kernel<<<1, 1, 0, st>>>(m->d_red, fuse->cfl, m->dx_min, 2.0 * m->N + 1.0, m->Pr, 0, fuse->dt_now);
      e = cudaGetLastError();
      if (e != cudaSuccess) return fail(MARUT_ECUDA, "dt kernel: %s", cudaGetErrorString(e));
      m->launches++;
    }
  }
  StageParams P;
  P.u_in = u_in; P.u_n = u_n; P.u_out = u_out;
  P.metric = m->d_metric; P.fnorm = m->d_fnorm; P.affine_flag = m->affine ? 1 : 0; P.explicit_source = m->explicit_source; P.conn = m->d_conn; P.mortar_fine = m->d_mortar_fine; P.mortar_mat = m->d_mortar_mat;
  P.bc_state = m->d_bc; P.S = m->d_S; P.Taux = m->d_T; P.mech = m->d_mech;
  P.ca = ca; P.cb = cb; P.cc = cc; P.dt_dev = dt_dev;
  P.gamma = m->gamma; P.mu = m->mu; P.kappa = m->kappa; P.inv_wb = 1.0 / m->w[0]; P.ne = m->ne; P.num_sms = m->num_sms;
  P.visc_only = 0; P.tile_list = nullptr; P.n_tile_list = 0; P.reverse = 0; P.zero = 0; P.tile_ctr = nullptr;
  P.red_next = nullptr; P.dt_next = nullptr; P.cfl = 0.0; P.dx_min = m->dx_min; P.P2 = 2.0 * m->N + 1.0;
  memcpy(P.D, m->D, sizeof(P.D));
  P.mflux = m->d_mflux;
  // Navier-Stokes with the strong form: the total flux F* - F_v* in one go; with the split form the hyperbolic flux for
  // stage_split_kernel here and -F_v* for the viscous-only launch further down
  const bool ns_total = m->physics == MARUT_NAVIER_STOKES && m->volume_form != MARUT_VOLUME_SPLIT_RANOCHA;
  if (m->dim == 3 && m->n_mortar > 0) {
    cudaError_t em = ns_total ? launch_mortar_flux3d_ns(m->np, true, u_in, m->d_S, m->d_metric, m->d_mortar_info, m->d_mortar_fine,
                                                        m->d_mortar_mat, m->gamma, m->d_mflux, m->n_mortar, st)
                              : launch_mortar_flux3d(m->np, u_in, m->d_metric, m->d_mortar_info, m->d_mortar_fine, m->d_mortar_mat, m->gamma,
                                          m->d_mflux, m->n_mortar, st);
    if (em != cudaSuccess) return fail(MARUT_ECUDA, "mortar flux kernel: %s", cudaGetErrorString(em));
    m->launches++;
  }
  P.alpha = nullptr; P.subn = m->d_subn;
  // Euler: outflow / slip-wall faces or 3-D mortars exist; Navier-Stokes: the mesh has boundary faces of any kind or mortars
  P.bc_kinds = (m->bc_kinds || (m->dim == 3 && m->n_mortar > 0) || (m->physics == MARUT_NAVIER_STOKES && (m->n_bface > 0 || m->n_mortar > 0))) ? 1 : 0;
  for (int i = 0; i < MAX_NP; ++i) P.inv_w[i] = (i < m->np) ? 1.0 / m->w[i] : 0.0;
  if (m->d_alpha) {
    if (m->physics == MARUT_REACTING_EULER || m->volume_form != MARUT_VOLUME_SPLIT_RANOCHA)
      return fail(MARUT_EINVAL, "a blending field is set: the DG/FV blend needs MARUT_VOLUME_SPLIT_RANOCHA (eq. 11)");
    P.alpha = m->d_alpha;
  }
  cudaError_t e;
  switch (m->physics) {
    case MARUT_EULER:
      if (m->volume_form == MARUT_VOLUME_SPLIT_RANOCHA) {
        // consecutive launches walk the element blocks in opposite directions, like the line kernel's tiles: a stage
        // starts on the end of the state its predecessor wrote last
        P.reverse = m->pencil_reverse;
        e = launch_stage_split(m->dim, m->np, m->affine, P, st);
        if (e == cudaSuccess) m->pencil_reverse ^= 1;
      }
      else {
        // affine meshes with conforming / prescribed-state / 2-D mortar faces: the persistent TMA-fed line kernel;
        // curved meshes, outflow / slip-wall faces and 3-D mortars: the thread-per-node kernel
        e = cudaErrorNotSupported;
        if (m->affine && !P.bc_kinds && m->stage_kernel_pref != 1) {
          if (fuse && fuse->dt_next) { P.red_next = m->d_red_next; P.dt_next = fuse->dt_next; P.cfl = fuse->cfl; }
          // consecutive launches walk the tiles in opposite directions (the start of one finds the end of the previous
          // one in L2); the result does not depend on the direction
          P.zero = 0;
          P.reverse = m->pencil_reverse;
          P.tile_ctr = (m->dim == 3) ? m->d_tile_ctr : nullptr;
          const bool force = m->stage_kernel_pref == 2;
          if (m->n_mortar > 0) {
            // two launches: the tiles without mortar faces through the plain instantiation (the one with the mortar
            // path runs every tile 63 % slower: 168 registers, a stack frame), then the few tiles with mortar faces.
            // The first contributes its maxima to the fused CFL reduction, the second finalizes it.
            const long nres = 3L * m->num_sms;
            if (m->n_tiles_plain + m->n_tiles_mortar < nres && !force) e = cudaErrorNotSupported;
            else {
              // the mortar fluxes, once per mortar, ahead of the stage
              e = launch_mortar_flux2d(m->np, u_in, m->d_metric, 1, m->d_mortar_info, m->d_mortar_fine, m->d_mortar_mat, m->gamma,
                                       m->d_mflux, m->n_mortar, st);
              if (e == cudaSuccess) m->launches++;
              else return fail(MARUT_ECUDA, "mortar flux kernel: %s", cudaGetErrorString(e));
              // (a mesh whose tiles mostly touch a mortar -- the c4 band mesh -- runs them all in the mortar instantiation:
              // one launch less)
              const bool split = m->n_tiles_plain > 0 && 4 * m->n_tiles_mortar < m->n_tiles_plain + m->n_tiles_mortar;
              if (split) {
                StageParams Pa = P;
                Pa.tile_list = m->d_tiles_plain; Pa.n_tile_list = m->n_tiles_plain; Pa.dt_next = nullptr;
                e = launch_stage_pencil(m->dim, m->np, false, true, Pa, st);
                if (e == cudaSuccess) m->launches++;
              }
              if (e == cudaSuccess) {
                if (split) { P.tile_list = m->d_tiles_mortar; P.n_tile_list = m->n_tiles_mortar; }
                e = launch_stage_pencil(m->dim, m->np, true, true, P, st);
                P.tile_list = nullptr; P.n_tile_list = 0;
              }
            }
          } else e = launch_stage_pencil(m->dim, m->np, false, force, P, st);
          if (e == cudaSuccess) m->pencil_reverse ^= 1;
          if (fuse) fuse->done = (e == cudaSuccess) && P.red_next != nullptr;
          P.red_next = nullptr;
        }
        if (e == cudaErrorNotSupported)
          e = (m->dim == 2) ? launch_stage_node2d(m->np, m->affine, P, st) : launch_stage_node3d(m->np, m->affine, P, st);
      }
      break;
    case MARUT_NAVIER_STOKES:
      P.reverse = 1;              // stage_phys_kernel walks against the gradient sweep (L2 reuse at both ends)
      if (m->volume_form == MARUT_VOLUME_SPLIT_RANOCHA) {
        // hyperbolic part with the split-form (and blended) volume integral, then the parabolic part added to u_out
        // (the two pipelines add their contributions into one residual)
        e = launch_stage_split(m->dim, m->np, m->affine, P, st);
        if (e != cudaSuccess) break;
        m->launches++;
        if (m->dim == 3 && m->n_mortar > 0) {
          e = launch_mortar_flux3d_ns(m->np, false, u_in, m->d_S, m->d_metric, m->d_mortar_info, m->d_mortar_fine, m->d_mortar_mat,
                                      m->gamma, m->d_mflux, m->n_mortar, st);
          if (e != cudaSuccess) break;
          m->launches++;
        }
        P.visc_only = 1;
        e = launch_stage_ns(m->dim, m->np, m->affine, P, st);
      } else e = launch_stage_ns(m->dim, m->np, m->affine, P, st);
      break;
    default:
      P.reverse = 1;              // against eos_kernel's sweep over the nodes
      e = launch_stage_react(m->dim, m->np, m->nsp, m->affine, P, st);
      break;
  }
  if (e == cudaErrorNotSupported) return fail(MARUT_EINVAL, "no kernel instantiated for dim=%d N=%d physics=%d", m->dim, m->N, m->physics);
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "stage kernel: %s", cudaGetErrorString(e));
  m->launches++;
  return MARUT_OK;
}

// sub-cell normals of a curved mesh (R16): nhat^l_{i+1/2} = Ja^l_0 + sum_{q<=i} w_q sum_r D_qr Ja^l_r along the
// line through the node in direction l; one thread per (element, l, c, node); stored at the node on the interface's
// lower side (the entry of the line's last node is Ja^l_N and unused)
struct SubnParams {
  const double *metric;
  double *subn;
  long ne;
  int dim, np, nn;
  double D[MAX_NP * MAX_NP], w[MAX_NP];
};
__global__ void subcell_normals_kernel(const __grid_constant__ SubnParams P) {
  const long total = P.ne * P.dim * P.dim * P.nn;
  const int md = P.dim * P.dim + 1;
  for (long g = blockIdx.x * (long)blockDim.x + threadIdx.x; g < total; g += (long)gridDim.x * blockDim.x) {
    const int p = (int)(g % P.nn);
    const long r1 = g / P.nn;
    const int c = (int)(r1 % P.dim), l = (int)((r1 / P.dim) % P.dim);
    const long e = r1 / (P.dim * P.dim);
    int st = 1;
    for (int k = 0; k < l; ++k) st *= P.np;
    const int il = (p / st) % P.np;
    const double *line = P.metric + (e * md + l * P.dim + c) * P.nn + (p - il * st);
    double nh = line[0];
    for (int q = 0; q <= il; ++q) {
      double s = 0.0;
      for (int r = 0; r < P.np; ++r) s += P.D[q * P.np + r] * line[r * st];
      nh += P.w[q] * s;
    }
    P.subn[g] = nh;
  }
}

extern "C" marut_status marut_set_blend(marut_mesh *m, const double *alpha) {
  if (!m) return fail(MARUT_EINVAL, "NULL argument");
  if (!alpha) { m->d_alpha = nullptr; return MARUT_OK; }
  if (m->physics == MARUT_REACTING_EULER) return fail(MARUT_EINVAL, "the DG/FV blend is implemented for MARUT_EULER and MARUT_NAVIER_STOKES");
  if (!m->affine && !m->d_subn) {
    const size_t n = (size_t)m->ne * m->dim * m->dim * m->nn;
    CUDA_TRY(cudaMalloc(&m->d_subn, n * sizeof(double)));
    SubnParams S;
    S.metric = m->d_metric; S.subn = m->d_subn; S.ne = m->ne; S.dim = m->dim; S.np = m->np; S.nn = m->nn;
    memcpy(S.D, m->D, sizeof(S.D)); memcpy(S.w, m->w, sizeof(S.w));
    subcell_normals_kernel<<<(unsigned)std::min<size_t>((n + 255) / 256, (size_t)m->num_sms * 16u), 256>>>(S);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaDeviceSynchronize());
  }
  m->d_alpha = alpha;
  return MARUT_OK;
}

extern "C" marut_status marut_set_volume_form(marut_mesh *m, int form) {
  if (!m) return fail(MARUT_EINVAL, "NULL argument");
  if (form != MARUT_VOLUME_STRONG && form != MARUT_VOLUME_SPLIT_RANOCHA) return fail(MARUT_EINVAL, "unknown volume form %d", form);
  if (form == MARUT_VOLUME_SPLIT_RANOCHA && m->physics == MARUT_REACTING_EULER)
    return fail(MARUT_EINVAL, "the split-form volume integral is implemented for MARUT_EULER and MARUT_NAVIER_STOKES");
  if (form == MARUT_VOLUME_SPLIT_RANOCHA && m->np > (m->dim == 2 ? 8 : 7)) return fail(MARUT_EINVAL, "split form: N <= 7 in 2-D, N <= 6 in 3-D");
  m->volume_form = form;
  return MARUT_OK;
}

extern "C" marut_status marut_rhs(marut_mesh *m, const double *u, double *du, double /*t*/, void *stream) {
  if (!m || !u || !du) return fail(MARUT_EINVAL, "NULL argument");
  if (u == du) return fail(MARUT_EINVAL, "du must not alias u");
  if (misaligned(u) || misaligned(du)) return fail(MARUT_EINVAL, "buffers must be 16-byte aligned");
  return run_operator(m, 0.0, 0.0, 1.0, nullptr, u, du, (cudaStream_t)stream);
}

extern "C" marut_status marut_ssprk_stage(marut_mesh *m, int stage, double dt, double /*t_n*/, const double *u_n,
                                          const double *u_in, double *u_out, void *stream) {
  if (!m || !u_in || !u_out) return fail(MARUT_EINVAL, "NULL argument");
  if (stage < 0 || stage > 2) return fail(MARUT_EINVAL, "stage must be 0, 1 or 2");
  if (stage > 0 && !u_n) return fail(MARUT_EINVAL, "u_n is NULL");
  if (u_out == u_in) return fail(MARUT_EINVAL, "u_out must not alias u_in");
  if (misaligned(u_in) || misaligned(u_out) || (stage > 0 && misaligned(u_n))) return fail(MARUT_EINVAL, "buffers must be 16-byte aligned");
  // Shu-Osher SSP-RK33: u_out = a u_n + b (u_in + dt L(u_in))
  static const double a[3] = {0.0, 0.75, 1.0 / 3.0}, b[3] = {1.0, 0.25, 2.0 / 3.0};
  return run_operator(m, a[stage], b[stage], b[stage] * dt, u_n, u_in, u_out, (cudaStream_t)stream);
}

// the same stage with the time step read from device memory (written by marut_max_dt_async on the same stream): no
// host synchronisation between the CFL reduction and the stages.  The kernel forms b * dt as the host does.
extern "C" marut_status marut_ssprk_stage_dev(marut_mesh *m, int stage, const double *dt_dev, double /*t_n*/, const double *u_n,
                                              const double *u_in, double *u_out, void *stream) {
  if (!m || !u_in || !u_out || !dt_dev) return fail(MARUT_EINVAL, "NULL argument");
  if (stage < 0 || stage > 2) return fail(MARUT_EINVAL, "stage must be 0, 1 or 2");
  if (stage > 0 && !u_n) return fail(MARUT_EINVAL, "u_n is NULL");
  if (u_out == u_in) return fail(MARUT_EINVAL, "u_out must not alias u_in");
  if (misaligned(u_in) || misaligned(u_out) || (stage > 0 && misaligned(u_n))) return fail(MARUT_EINVAL, "buffers must be 16-byte aligned");
  static const double a[3] = {0.0, 0.75, 1.0 / 3.0}, b[3] = {1.0, 0.25, 2.0 / 3.0};
  return run_operator(m, a[stage], b[stage], b[stage], u_n, u_in, u_out, (cudaStream_t)stream, dt_dev);
}

// ======================================================================================
// out = sum_k c_k u_k, k < n <= 4 (the stage combinations of eq. 45 that involve more than two earlier stages: last
// stage of SSP-RK54).  Elementwise, so out may alias any u_k.  HBM-bound: (n + 1) * 8 B per value.
// ======================================================================================
struct LincombParams {
  const double *u[4];
  double c[4];
  double *out;
  long len;
  int n;
};
__global__ void __launch_bounds__(256) lincomb_kernel(const __grid_constant__ LincombParams P) {
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < P.len; i += (long)gridDim.x * blockDim.x) {
    double acc = P.c[0] * P.u[0][i];
    for (int k = 1; k < P.n; ++k) acc += P.c[k] * P.u[k][i];
    P.out[i] = acc;
  }
}

// general stage of eq. 45 with two earlier stages: u_out = a u_a + b u_in + c_dt L(u_in)
extern "C" marut_status marut_rk_stage(marut_mesh *m, double a, double b, double c_dt, const double *u_a, const double *u_in,
                                       double *u_out, void *stream) {
  if (!m || !u_in || !u_out) return fail(MARUT_EINVAL, "NULL argument");
  if (a != 0.0 && !u_a) return fail(MARUT_EINVAL, "u_a is NULL");
  if (u_out == u_in) return fail(MARUT_EINVAL, "u_out must not alias u_in");
  if (misaligned(u_in) || misaligned(u_out) || (a != 0.0 && misaligned(u_a))) return fail(MARUT_EINVAL, "buffers must be 16-byte aligned");
  return run_operator(m, a, b, c_dt, u_a, u_in, u_out, (cudaStream_t)stream);
}

// marut_rk_stage with c_dt = c * dt formed in the kernel from the device-resident dt (marut_max_dt_async)
extern "C" marut_status marut_rk_stage_dev(marut_mesh *m, double a, double b, double c, const double *dt_dev, const double *u_a,
                                           const double *u_in, double *u_out, void *stream) {
  if (!m || !u_in || !u_out || !dt_dev) return fail(MARUT_EINVAL, "NULL argument");
  if (a != 0.0 && !u_a) return fail(MARUT_EINVAL, "u_a is NULL");
  if (u_out == u_in) return fail(MARUT_EINVAL, "u_out must not alias u_in");
  if (misaligned(u_in) || misaligned(u_out) || (a != 0.0 && misaligned(u_a))) return fail(MARUT_EINVAL, "buffers must be 16-byte aligned");
  return run_operator(m, a, b, c, u_a, u_in, u_out, (cudaStream_t)stream, dt_dev);
}

extern "C" marut_status marut_lincomb(marut_mesh *m, int n, const double *coef, const double *const *u, double *out, void *stream) {
  if (!m || !coef || !u || !out) return fail(MARUT_EINVAL, "NULL argument");
  if (n < 1 || n > 4) return fail(MARUT_EINVAL, "marut_lincomb: 1 <= n <= 4");
  LincombParams P;
  for (int k = 0; k < 4; ++k) { P.u[k] = (k < n) ? u[k] : nullptr; P.c[k] = (k < n) ? coef[k] : 0.0; }
  for (int k = 0; k < n; ++k) if (!u[k]) return fail(MARUT_EINVAL, "marut_lincomb: u[%d] is NULL", k);
  P.out = out; P.len = m->ne * m->nvar * m->nn; P.n = n;
  const unsigned grid = (unsigned)std::min<long>((P.len + 255) / 256, (long)m->num_sms * 32);
  lincomb_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(P);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "lincomb kernel: %s", cudaGetErrorString(e));
  m->launches++;
  return MARUT_OK;
}

extern "C" marut_status marut_chem_source(marut_mesh *m, const double *u, double *s, void *stream) {
  if (!m || !u || !s) return fail(MARUT_EINVAL, "NULL argument");
  if (m->physics != MARUT_REACTING_EULER) return fail(MARUT_EINVAL, "marut_chem_source needs a REACTING_EULER mesh");
  if (u == s) return fail(MARUT_EINVAL, "s must not alias u");
  const long total = m->ne * m->nn;
  const unsigned grid = (unsigned)std::min<long>((total + 255) / 256, (long)m->num_sms * 16);
  cudaStream_t st = (cudaStream_t)stream;
  if (m->dim == 2) chem_kernel<2, 5><<<grid, 256, 0, st>>>(u, s, m->d_mech, m->ne, m->nn);
  else chem_kernel<3, 5><<<grid, 256, 0, st>>>(u, s, m->d_mech, m->ne, m->nn);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "chem kernel: %s", cudaGetErrorString(e));
  m->launches++;
  return MARUT_OK;
}

extern "C" marut_status marut_set_explicit_source(marut_mesh *m, int on) {
  if (!m) return fail(MARUT_EINVAL, "NULL argument");
  if (m->physics != MARUT_REACTING_EULER) return fail(MARUT_EINVAL, "marut_set_explicit_source needs a REACTING_EULER mesh");
  m->explicit_source = on ? 1 : 0;
  return MARUT_OK;
}

extern "C" marut_status marut_chem_implicit(marut_mesh *m, double *u, double dt, int *sweeps_out, void *stream) {
  if (!m || !u) return fail(MARUT_EINVAL, "NULL argument");
  if (m->physics != MARUT_REACTING_EULER) return fail(MARUT_EINVAL, "marut_chem_implicit needs a REACTING_EULER mesh");
  if (!(dt >= 0.0)) return fail(MARUT_EINVAL, "dt must be >= 0");
  cudaStream_t st = (cudaStream_t)stream;
  int *d_sw = reinterpret_cast<int *>(m->d_red + 3);
  CUDA_TRY(cudaMemsetAsync(d_sw, 0, sizeof(unsigned long long), st));
  const long total = m->ne * m->nn;
  const unsigned grid = (unsigned)std::min<long>((total + 127) / 128, (long)m->num_sms * 8);
  if (m->dim == 2) chem_implicit_kernel<2, 5><<<grid, 128, 0, st>>>(u, m->d_mech, dt, m->ne, m->nn, d_sw);
  else chem_implicit_kernel<3, 5><<<grid, 128, 0, st>>>(u, m->d_mech, dt, m->ne, m->nn, d_sw);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "implicit chemistry kernel: %s", cudaGetErrorString(e));
  m->launches++;
  if (sweeps_out) {
    CUDA_TRY(cudaMemcpyAsync(m->h_red + 3, d_sw, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    *sweeps_out = (int)(m->h_red[3] & 0xffffffffu);
    if (*sweeps_out > 50) return fail(MARUT_ENOTFINITE, "implicit chemistry: Newton did not converge in 50 sweeps");
  }
  return MARUT_OK;
}

extern "C" marut_status marut_max_dt_async(marut_mesh *m, const double *u, double cfl, double *dt_dev, void *stream);

// ------------------------------------------------------------------------------------ whole time steps
// The step compositions of the paper's integrators, so that a C caller gets them without re-typing a coefficient
// table: SSP-RK33 (eq. 44-46, R10), SSP-RK54 (R19) and the Strang split of eq. 24.
// SSP-RK54 of Spiteri and Ruuth in the Shu-Osher form of eq. 45: rows (alpha_i0, alpha_i,i-1, beta_i,i-1) of stages
// 1-4, then (alpha_52, alpha_53, beta_53, alpha_54, beta_54) of the last stage (15 digits as published).
static const double RK54[4][3] = {{1.0, 0.0, 0.391752226571890},
                                  {0.444370493651235, 0.555629506348765, 0.368410593050371},
                                  {0.620101851488403, 0.379898148511597, 0.251891774271694},
                                  {0.178079954393132, 0.821920045606868, 0.544974750228521}};
static const double RK54_LAST[5] = {0.517231671970585, 0.096059710526147, 0.063692468666290, 0.386708617503269, 0.226007483236906};

static marut_status check_step_buffers(marut_mesh *m, const double *u, double *const *scratch, int ns) {
  if (!m || !u || !scratch) return fail(MARUT_EINVAL, "NULL argument");
  if (misaligned(u)) return fail(MARUT_EINVAL, "buffers must be 16-byte aligned");
  for (int i = 0; i < ns; ++i) {
    if (!scratch[i]) return fail(MARUT_EINVAL, "scratch[%d] is NULL", i);
    if (misaligned(scratch[i])) return fail(MARUT_EINVAL, "buffers must be 16-byte aligned");
    if (scratch[i] == u) return fail(MARUT_EINVAL, "scratch[%d] aliases u", i);
    for (int j = 0; j < i; ++j)
      if (scratch[i] == scratch[j]) return fail(MARUT_EINVAL, "scratch[%d] aliases scratch[%d]", i, j);
  }
  return MARUT_OK;
}

// c = b * dt on the host, or b with dt read from dt_dev inside the kernel (the same single rounded product)
static marut_status stage_any(marut_mesh *m, double a, double b, double c, double dt, const double *dt_dev, const double *u_a,
                              const double *u_in, double *u_out, cudaStream_t st) {
  return dt_dev ? run_operator(m, a, b, c, u_a, u_in, u_out, st, dt_dev) : run_operator(m, a, b, c * dt, u_a, u_in, u_out, st);
}

extern "C" marut_status marut_ssprk33_step(marut_mesh *m, double *u, double *const *scratch, double dt, const double *dt_dev,
                                           void *stream) {
  if (marut_status s = check_step_buffers(m, u, scratch, 2); s != MARUT_OK) return s;
  cudaStream_t st = (cudaStream_t)stream;
  double *ua = scratch[0], *ub = scratch[1];
  marut_status s;
  if ((s = stage_any(m, 0.0, 1.0, 1.0, dt, dt_dev, u, u, ua, st)) != MARUT_OK) return s;
  if ((s = stage_any(m, 0.75, 0.25, 0.25, dt, dt_dev, u, ua, ub, st)) != MARUT_OK) return s;
  return stage_any(m, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0, dt, dt_dev, u, ub, u, st);
}

extern "C" marut_status marut_ssprk33_step_cfl(marut_mesh *m, double *u, double *const *scratch, double cfl, const double *dt_in,
                                               double *dt_out, void *stream) {
  if (marut_status s = check_step_buffers(m, u, scratch, 2); s != MARUT_OK) return s;
  if (!dt_in || !dt_out) return fail(MARUT_EINVAL, "NULL argument");
  if (dt_in == dt_out) return fail(MARUT_EINVAL, "dt_out must not alias dt_in (CTAs of the last stage still read dt_in when the first ones finish)");
  if (!(cfl > 0.0)) return fail(MARUT_EINVAL, "cfl must be positive");
  cudaStream_t st = (cudaStream_t)stream;
  double *ua = scratch[0], *ub = scratch[1];
  marut_status s;
  if ((s = run_operator(m, 0.0, 1.0, 1.0, u, u, ua, st, dt_in)) != MARUT_OK) return s;
  if ((s = run_operator(m, 0.75, 0.25, 0.25, u, ua, ub, st, dt_in)) != MARUT_OK) return s;
  FuseCfl f;
  f.cfl = cfl;
  f.dt_next = dt_out;
  if ((s = run_operator(m, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0, u, ub, u, st, dt_in, &f)) != MARUT_OK) return s;
  if (!f.done) return marut_max_dt_async(m, u, cfl, dt_out, stream);   // stage kernels without the fused reduction
  return MARUT_OK;
}

extern "C" marut_status marut_ssprk33_step_dt(marut_mesh *m, double *u, double *const *scratch, double cfl, double *dt_out,
                                              void *stream) {
  if (marut_status s = check_step_buffers(m, u, scratch, 2); s != MARUT_OK) return s;
  if (!dt_out) return fail(MARUT_EINVAL, "NULL argument");
  if (!(cfl > 0.0)) return fail(MARUT_EINVAL, "cfl must be positive");
  cudaStream_t st = (cudaStream_t)stream;
  double *ua = scratch[0], *ub = scratch[1];
  marut_status s;
  if (m->physics == MARUT_REACTING_EULER) {
    // the first stage's thermochemistry pass has T and a of u: it reduces the wave speed on the way
    FuseCfl f;
    f.cfl = cfl;
    f.dt_now = dt_out;
    if ((s = run_operator(m, 0.0, 1.0, 1.0, u, u, ua, st, dt_out, &f)) != MARUT_OK) return s;
  } else {
    if ((s = marut_max_dt_async(m, u, cfl, dt_out, stream)) != MARUT_OK) return s;
    if ((s = run_operator(m, 0.0, 1.0, 1.0, u, u, ua, st, dt_out)) != MARUT_OK) return s;
  }
  if ((s = run_operator(m, 0.75, 0.25, 0.25, u, ua, ub, st, dt_out)) != MARUT_OK) return s;
  return run_operator(m, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0, u, ub, u, st, dt_out);
}

extern "C" marut_status marut_ssprk54_step(marut_mesh *m, double *u, double *const *scratch, double dt, const double *dt_dev,
                                           void *stream) {
  if (marut_status s = check_step_buffers(m, u, scratch, 3); s != MARUT_OK) return s;
  cudaStream_t st = (cudaStream_t)stream;
  double *ua = scratch[0], *ub = scratch[1], *uc = scratch[2];
  const double(*a)[3] = RK54;
  const double *b = RK54_LAST;
  marut_status s;
  if ((s = stage_any(m, 0.0, 1.0, a[0][2], dt, dt_dev, nullptr, u, ua, st)) != MARUT_OK) return s;      // U1 -> ua
  if ((s = stage_any(m, a[1][0], a[1][1], a[1][2], dt, dt_dev, u, ua, ub, st)) != MARUT_OK) return s;   // U2 -> ub
  if ((s = stage_any(m, a[2][0], a[2][1], a[2][2], dt, dt_dev, u, ub, ua, st)) != MARUT_OK) return s;   // U3 -> ua
  if ((s = stage_any(m, a[3][0], a[3][1], a[3][2], dt, dt_dev, u, ua, uc, st)) != MARUT_OK) return s;   // U4 -> uc
  // last stage: dt L(U3) = (U4 - a40 U0 - a43 U3)/b43 (reading R19), so
  // U5 = [a52 U2 + a53 U3 + a54 U4 + (b53/b43)(U4 - a40 U0 - a43 U3)] + b54 dt L(U4)
  const double r = b[2] / a[3][2];
  const double coef[4] = {-r * a[3][0], b[0], b[1] - r * a[3][1], b[3] + r};
  const double *us[4] = {u, ub, ua, uc};
  if ((s = marut_lincomb(m, 4, coef, us, ua, stream)) != MARUT_OK) return s;
  return stage_any(m, 1.0, 0.0, b[4], dt, dt_dev, ua, uc, u, st);                                        // U5 -> u
}

extern "C" marut_status marut_strang_step(marut_mesh *m, double *u, double *const *scratch, double dt, int *sweeps_out,
                                          void *stream) {
  if (marut_status s = check_step_buffers(m, u, scratch, 2); s != MARUT_OK) return s;
  if (m->physics != MARUT_REACTING_EULER) return fail(MARUT_EINVAL, "marut_strang_step needs a REACTING_EULER mesh");
  if (!(dt >= 0.0)) return fail(MARUT_EINVAL, "dt must be >= 0");
  const int keep = m->explicit_source;
  m->explicit_source = 0;                        // T = transport operator alone
  int sw1 = 0, sw2 = 0;
  marut_status s = marut_chem_implicit(m, u, 0.5 * dt, sweeps_out ? &sw1 : nullptr, stream);
  if (s == MARUT_OK) s = marut_ssprk33_step(m, u, scratch, dt, nullptr, stream);
  if (s == MARUT_OK) s = marut_chem_implicit(m, u, 0.5 * dt, sweeps_out ? &sw2 : nullptr, stream);
  m->explicit_source = keep;
  if (sweeps_out) *sweeps_out = std::max(sw1, sw2);
  return s;
}

// ------------------------------------------------------------------------------------ boundary kinds
__global__ void patch_boundary_kinds_kernel(int2 *conn, long n, const int *kinds) {
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
    int2 cn = conn[i];
    if ((cn.y & 3) == FK_BOUNDARY) {
      cn.y = FK_BOUNDARY | (kinds[cn.x] << 2);
      conn[i] = cn;
    }
  }
}

extern "C" marut_status marut_set_boundary_kinds(marut_mesh *m, const int *kinds, int n_bc) {
  if (!m || !kinds) return fail(MARUT_EINVAL, "NULL argument");
  if (n_bc != m->n_bc) return fail(MARUT_EINVAL, "n_bc = %d, the mesh has %d boundary ids", n_bc, m->n_bc);
  bool special = false;
  for (int i = 0; i < n_bc; ++i) {
    const int kmax = (m->physics == MARUT_NAVIER_STOKES) ? MARUT_BC_WALL_ISOTHERMAL : MARUT_BC_SLIP_WALL;
    if (kinds[i] < MARUT_BC_PRESCRIBED || kinds[i] > kmax)
      return fail(MARUT_EINVAL, "boundary kind %d is unknown or not available for this physics (no-slip walls: MARUT_NAVIER_STOKES)", kinds[i]);
    special = special || kinds[i] != MARUT_BC_PRESCRIBED;
  }
  if (special && m->physics == MARUT_REACTING_EULER)
    return fail(MARUT_EINVAL, "boundary kinds are implemented for MARUT_EULER and MARUT_NAVIER_STOKES");
  if (n_bc == 0) return MARUT_OK;
  int *d_k = nullptr;
  CUDA_TRY(cudaMalloc(&d_k, n_bc * sizeof(int)));
  cudaError_t e = cudaMemcpy(d_k, kinds, n_bc * sizeof(int), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    const long n = m->ne * 2 * m->dim;
    patch_boundary_kinds_kernel<<<(unsigned)std::min<long>((n + 255) / 256, (long)m->num_sms * 8), 256>>>(m->d_conn, n, d_k);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
  }
  cudaFree(d_k);
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "boundary kinds: %s", cudaGetErrorString(e));
  m->bc_kinds = special;
  return MARUT_OK;
}

// ------------------------------------------------------------------------------------ positivity floor
extern "C" marut_status marut_positivity_floor(marut_mesh *m, double *u, double rho_min, double p_min, long *changed_out,
                                               void *stream) {
  if (!m || !u) return fail(MARUT_EINVAL, "NULL argument");
  if (m->physics == MARUT_REACTING_EULER) return fail(MARUT_EINVAL, "marut_positivity_floor: ideal-gas meshes only");
  if (!(rho_min > 0.0) || !(p_min > 0.0)) return fail(MARUT_EINVAL, "the floors must be > 0");
  cudaStream_t st = (cudaStream_t)stream;
  unsigned long long *d_cnt = m->d_red + 4;
  if (changed_out) CUDA_TRY(cudaMemsetAsync(d_cnt, 0, sizeof(unsigned long long), st));
  const long total = m->ne * m->nn;
  const unsigned grid = (unsigned)std::min<long>((total + 255) / 256, (long)m->num_sms * 32);
  if (m->dim == 2) positivity_floor_kernel<2><<<grid, 256, 0, st>>>(u, m->gamma, rho_min, p_min, m->ne, m->nn, changed_out ? d_cnt : nullptr);
  else positivity_floor_kernel<3><<<grid, 256, 0, st>>>(u, m->gamma, rho_min, p_min, m->ne, m->nn, changed_out ? d_cnt : nullptr);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "positivity floor kernel: %s", cudaGetErrorString(e));
  m->launches++;
  if (changed_out) {
    CUDA_TRY(cudaMemcpyAsync(m->h_red + 4, d_cnt, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    *changed_out = (long)m->h_red[4];
  }
  return MARUT_OK;
}

// ------------------------------------------------------------------------------------ shock indicator
// V^-1 of the orthonormal Legendre basis on the LGL nodes: V_ik = sqrt((2k+1)/2) L_k(x_i), inverted by Gauss-Jordan
static bool build_modal_matrix(int N, const double *x, double *Vinv) {
  const int n = N + 1;
  std::vector<double> A((size_t)n * 2 * n, 0.0);
  for (int i = 0; i < n; ++i) {
    double Pm = 1.0, Pc = x[i];
    for (int k = 0; k < n; ++k) {
      double Pk = (k == 0) ? 1.0 : ((k == 1) ? x[i] : 0.0);
      if (k >= 2) { Pk = ((2.0 * k - 1.0) * x[i] * Pc - (k - 1.0) * Pm) / k; Pm = Pc; Pc = Pk; }
      A[(size_t)i * 2 * n + k] = std::sqrt((2.0 * k + 1.0) / 2.0) * Pk;
    }
    A[(size_t)i * 2 * n + n + i] = 1.0;
  }
  for (int c = 0; c < n; ++c) {
    int piv = c;
    for (int r = c + 1; r < n; ++r) if (std::fabs(A[(size_t)r * 2 * n + c]) > std::fabs(A[(size_t)piv * 2 * n + c])) piv = r;
    if (A[(size_t)piv * 2 * n + c] == 0.0) return false;
    if (piv != c) for (int q = 0; q < 2 * n; ++q) std::swap(A[(size_t)c * 2 * n + q], A[(size_t)piv * 2 * n + q]);
    const double inv = 1.0 / A[(size_t)c * 2 * n + c];
    for (int q = 0; q < 2 * n; ++q) A[(size_t)c * 2 * n + q] *= inv;
    for (int r = 0; r < n; ++r) if (r != c) {
      const double f = A[(size_t)r * 2 * n + c];
      for (int q = 0; q < 2 * n; ++q) A[(size_t)r * 2 * n + q] -= f * A[(size_t)c * 2 * n + q];
    }
  }
  for (int k = 0; k < n; ++k) for (int i = 0; i < n; ++i) Vinv[k * n + i] = A[(size_t)k * 2 * n + n + i];
  return true;
}

template <int DIM, int NP>
static cudaError_t run_indicator(marut_mesh *m, const double *u, double s_over_T, double T, double amin, double amax,
                                 double *out, cudaStream_t st) {
  constexpr int NN = Geo<DIM, NP>::NN, EB = (NN >= 96) ? 1 : 128 / NN, NT = ((EB * NN + 31) / 32) * 32;
  const unsigned grid = (unsigned)((m->ne + EB - 1) / EB);
  indicator_kernel<DIM, NP, EB><<<grid, NT, 0, st>>>(u, m->d_Vinv, m->gamma, s_over_T, T, amin, amax, m->ne, out);
  return cudaGetLastError();
}

extern "C" marut_status marut_shock_indicator(marut_mesh *m, const double *u, double s, double alpha_min, double alpha_max,
                                              int smooth, double *alpha, void *stream) {
  if (!m || !u || !alpha) return fail(MARUT_EINVAL, "NULL argument");
  if (m->physics == MARUT_REACTING_EULER) return fail(MARUT_EINVAL, "marut_shock_indicator: ideal-gas meshes only");
  if (!(s > 0.0) || !(alpha_min >= 0.0) || !(alpha_max >= alpha_min) || !(alpha_max <= 1.0))
    return fail(MARUT_EINVAL, "need s > 0 and 0 <= alpha_min <= alpha_max <= 1");
  cudaStream_t st = (cudaStream_t)stream;
  if (!m->d_Vinv) {
    double x[MAX_NP], w[MAX_NP], D[MAX_NP * MAX_NP], V[MAX_NP * MAX_NP];
    build_operators(m->N, x, w, D);
    if (!build_modal_matrix(m->N, x, V)) return fail(MARUT_EINVAL, "singular Vandermonde matrix");
    CUDA_TRY(cudaMalloc(&m->d_Vinv, m->np * m->np * sizeof(double)));
    CUDA_TRY(cudaMemcpy(m->d_Vinv, V, m->np * m->np * sizeof(double), cudaMemcpyHostToDevice));
  }
  if (smooth && !m->d_araw) CUDA_TRY(cudaMalloc(&m->d_araw, (size_t)m->ne * sizeof(double)));
  const double T = 0.5 * std::pow(10.0, -1.8 * std::pow((double)(m->N + 1), 0.25));
  double *raw = smooth ? m->d_araw : alpha;
  cudaError_t e = cudaErrorNotSupported;
#define MARUT_IND(D_, NP_) if (m->dim == D_ && m->np == NP_) e = run_indicator<D_, NP_>(m, u, s / T, T, alpha_min, alpha_max, raw, st);
  MARUT_IND(2, 2) MARUT_IND(2, 3) MARUT_IND(2, 4) MARUT_IND(2, 5) MARUT_IND(2, 6) MARUT_IND(2, 7) MARUT_IND(2, 8)
  MARUT_IND(3, 2) MARUT_IND(3, 3) MARUT_IND(3, 4) MARUT_IND(3, 5) MARUT_IND(3, 6) MARUT_IND(3, 7) MARUT_IND(3, 8)
#undef MARUT_IND
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "indicator kernel: %s", cudaGetErrorString(e));
  m->launches++;
  if (smooth) {
    const unsigned grid = (unsigned)((m->ne + 255) / 256);
    if (m->dim == 2) indicator_smooth_kernel<2><<<grid, 256, 0, st>>>(raw, m->d_conn, m->d_mortar_fine, m->d_mortar_info, m->ne, alpha);
    else indicator_smooth_kernel<3><<<grid, 256, 0, st>>>(raw, m->d_conn, m->d_mortar_fine, m->d_mortar_info, m->ne, alpha);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(MARUT_ECUDA, "indicator smoothing kernel: %s", cudaGetErrorString(e));
    m->launches++;
  }
  return MARUT_OK;
}

// ------------------------------------------------------------------------------------ shock indicator without allocations
// marut_shock_indicator allocates on its first call per handle (V^-1, and the unsmoothed alpha_e when smooth != 0).  Callers
// that must not allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc -- use
// marut_shock_indicator_noalloc: the same two kernels with their scratch in ONE file-scope device array of fixed size,
// [0, 64): V^-1 (n x n), [64, 64 + n_elem): the unsmoothed alpha_e.  8 MiB + 512 B per GPU that loads the library, held
// until exit.  The array is shared by every call on the device and keeps the last call's contents: each call rewrites
// all of what it reads (nothing has to start at zero), and two calls that overlap on the GPU (different streams) race.
constexpr long NOALLOC_MAX_ELEM = 1L << 20;
static __device__ __align__(256) double g_noalloc_scratch[64 + NOALLOC_MAX_ELEM];
struct VinvArg { double v[MAX_NP * MAX_NP]; };
__global__ void noalloc_set_vinv_kernel(VinvArg a, double *__restrict__ dst, int n) {
  if ((int)threadIdx.x < n) dst[threadIdx.x] = a.v[threadIdx.x];
}
// device address of the scratch array: in host code its name is a host-side stand-in, not a device address.  Queried
// once per device (with that device current), no allocation involved.
static cudaError_t noalloc_scratch_ptr(double **out) {
  static std::atomic<double *> ptr[64];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  double *p = (dev >= 0 && dev < 64) ? ptr[dev].load(std::memory_order_acquire) : nullptr;
  if (!p) {
    e = cudaGetSymbolAddress((void **)&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) ptr[dev].store(p, std::memory_order_release);
  }
  *out = p;
  return cudaSuccess;
}
template <int DIM, int NP>
static cudaError_t run_indicator_noalloc(const marut_mesh *m, const double *u, const double *Vinv, double s_over_T, double T,
                                         double amin, double amax, double *out, cudaStream_t st) {
  constexpr int NN = Geo<DIM, NP>::NN, EB = (NN >= 96) ? 1 : 128 / NN, NT = ((EB * NN + 31) / 32) * 32;
  const unsigned grid = (unsigned)((m->ne + EB - 1) / EB);
  indicator_kernel<DIM, NP, EB><<<grid, NT, 0, st>>>(u, Vinv, m->gamma, s_over_T, T, amin, amax, m->ne, out);
  return cudaGetLastError();
}
extern "C" long marut_noalloc_max_elements(void) { return NOALLOC_MAX_ELEM; }
extern "C" marut_status marut_shock_indicator_noalloc(marut_mesh *m, const double *u, double s, double alpha_min, double alpha_max,
                                                      int smooth, double *alpha, void *stream) {
  if (!m || !u || !alpha) return fail(MARUT_EINVAL, "NULL argument");
  if (m->physics == MARUT_REACTING_EULER) return fail(MARUT_EINVAL, "marut_shock_indicator_noalloc: ideal-gas meshes only");
  if (!(s > 0.0) || !(alpha_min >= 0.0) || !(alpha_max >= alpha_min) || !(alpha_max <= 1.0))
    return fail(MARUT_EINVAL, "need s > 0 and 0 <= alpha_min <= alpha_max <= 1");
  if (m->ne > NOALLOC_MAX_ELEM)
    return fail(MARUT_EINVAL, "marut_shock_indicator_noalloc: %ld elements exceed the fixed scratch of %ld elements "
                "(use marut_shock_indicator, which allocates)", m->ne, NOALLOC_MAX_ELEM);
  cudaStream_t st = (cudaStream_t)stream;
  double *scratch = nullptr;
  cudaError_t e = noalloc_scratch_ptr(&scratch);
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "cudaGetSymbolAddress(scratch): %s", cudaGetErrorString(e));
  VinvArg V;
  {
    double x[MAX_NP], w[MAX_NP], D[MAX_NP * MAX_NP];
    build_operators(m->N, x, w, D);
    for (int i = 0; i < MAX_NP * MAX_NP; ++i) V.v[i] = 0.0;
    if (!build_modal_matrix(m->N, x, V.v)) return fail(MARUT_EINVAL, "singular Vandermonde matrix");
  }
  noalloc_set_vinv_kernel<<<1, 64, 0, st>>>(V, scratch, m->np * m->np);    // the matrix travels as a kernel argument
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "scratch set-up kernel: %s", cudaGetErrorString(e));
  m->launches++;
  const double T = 0.5 * std::pow(10.0, -1.8 * std::pow((double)(m->N + 1), 0.25));
  double *raw = smooth ? scratch + 64 : alpha;
  e = cudaErrorNotSupported;
#define MARUT_IND(D_, NP_) if (m->dim == D_ && m->np == NP_) e = run_indicator_noalloc<D_, NP_>(m, u, scratch, s / T, T, alpha_min, alpha_max, raw, st);
  MARUT_IND(2, 2) MARUT_IND(2, 3) MARUT_IND(2, 4) MARUT_IND(2, 5) MARUT_IND(2, 6) MARUT_IND(2, 7) MARUT_IND(2, 8)
  MARUT_IND(3, 2) MARUT_IND(3, 3) MARUT_IND(3, 4) MARUT_IND(3, 5) MARUT_IND(3, 6) MARUT_IND(3, 7) MARUT_IND(3, 8)
#undef MARUT_IND
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "indicator kernel: %s", cudaGetErrorString(e));
  m->launches++;
  if (smooth) {
    const unsigned grid = (unsigned)((m->ne + 255) / 256);
    if (m->dim == 2) indicator_smooth_kernel<2><<<grid, 256, 0, st>>>(raw, m->d_conn, m->d_mortar_fine, m->d_mortar_info, m->ne, alpha);
    else indicator_smooth_kernel<3><<<grid, 256, 0, st>>>(raw, m->d_conn, m->d_mortar_fine, m->d_mortar_info, m->ne, alpha);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(MARUT_ECUDA, "indicator smoothing kernel: %s", cudaGetErrorString(e));
    m->launches++;
  }
  return MARUT_OK;
}

// ------------------------------------------------------------------------------------ time step
template <int DIM, int NSP, int PHYS>
static cudaError_t launch_wave_speed(marut_mesh *m, const double *u, const MechDev *mech, cudaStream_t st) {
  // one resident wave: grid = SMs x the CTAs per SM this instantiation's registers allow
  int &occ = m->ws_occ;   // per handle (= per device)
  if (occ == 0) {
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, wave_speed_kernel<DIM, NSP, PHYS>, 256, 0);
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
  }
  const long total = m->ne * m->nn;
  const unsigned grid = (unsigned)std::min<long>((total + 255) / 256, (long)m->num_sms * occ);
  wave_speed_kernel<DIM, NSP, PHYS><<<grid, 256, 0, st>>>(u, mech, m->gamma, m->mu, m->ne, m->nn, m->d_red);
  return cudaGetLastError();
}
template <int DIM>
static cudaError_t run_wave_speed(marut_mesh *m, const double *u, unsigned /*grid*/, cudaStream_t st) {
  switch (m->physics) {
    case MARUT_EULER: return launch_wave_speed<DIM, 1, PH_EULER>(m, u, nullptr, st);
    case MARUT_NAVIER_STOKES: return launch_wave_speed<DIM, 1, PH_NS>(m, u, nullptr, st);
    default: return launch_wave_speed<DIM, 5, PH_REACT>(m, u, m->d_mech, st);
  }
}

// eq. 17-18 from the reduced maxima, on the device: the expressions of marut_max_dt below, operation for operation
// (products and quotients only, so no contraction can change a rounding).  A non-finite or non-positive wave speed
// poisons dt with NaN.
__global__ void dt_finalize_kernel(const unsigned long long *__restrict__ red, double cfl, double dx_min, double P2, double Pr,
                                   int ns, double *__restrict__ dt_out) {
  const double lam = __longlong_as_double((long long)red[0]), nu = __longlong_as_double((long long)red[1]);
  double dt;
  if (red[2] != 0ULL || !(lam > 0.0) || !isfinite(lam)) dt = __longlong_as_double(0x7ff8000000000000LL);
  else {
    dt = __ddiv_rn(__dmul_rn(cfl, dx_min), __dmul_rn(P2, lam));
    if (ns && nu > 0.0) {
      const double numax = __dmul_rn(nu, fmax(1.0, __ddiv_rn(1.0, Pr)));
      dt = fmin(dt, __ddiv_rn(__dmul_rn(__dmul_rn(cfl, dx_min), dx_min), __dmul_rn(__dmul_rn(P2, P2), numax)));
    }
  }
  *dt_out = dt;
}

extern "C" marut_status marut_max_dt_async(marut_mesh *m, const double *u, double cfl, double *dt_dev, void *stream) {
  if (!m || !u || !dt_dev) return fail(MARUT_EINVAL, "NULL argument");
  if (!(cfl > 0.0)) return fail(MARUT_EINVAL, "cfl must be positive");
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(cudaMemsetAsync(m->d_red, 0, 3 * sizeof(unsigned long long), st));
  const long total = m->ne * m->nn;
  const unsigned grid = (unsigned)std::min<long>((total + 255) / 256, (long)m->num_sms * 8);
  cudaError_t e = (m->dim == 2) ? run_wave_speed<2>(m, u, grid, st) : run_wave_speed<3>(m, u, grid, st);
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "wave speed kernel: %s", cudaGetErrorString(e));
  dt_finalize_kernel<<<1, 1, 0, st>>>(m->d_red, cfl, m->dx_min, 2.0 * m->N + 1.0, m->Pr, m->physics == MARUT_NAVIER_STOKES ? 1 : 0, dt_dev);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "dt kernel: %s", cudaGetErrorString(e));
  m->launches += 2;
  return MARUT_OK;
}

extern "C" marut_status marut_max_dt(marut_mesh *m, const double *u, double cfl, double *dt_out, void *stream) {
  if (!m || !u || !dt_out) return fail(MARUT_EINVAL, "NULL argument");
  if (!(cfl > 0.0)) return fail(MARUT_EINVAL, "cfl must be positive");
  cudaStream_t st = (cudaStream_t)stream;
  CUDA_TRY(cudaMemsetAsync(m->d_red, 0, 4 * sizeof(unsigned long long), st));
  const long total = m->ne * m->nn;
  const unsigned grid = (unsigned)std::min<long>((total + 255) / 256, (long)m->num_sms * 8);
  cudaError_t e = (m->dim == 2) ? run_wave_speed<2>(m, u, grid, st) : run_wave_speed<3>(m, u, grid, st);
  if (e != cudaSuccess) return fail(MARUT_ECUDA, "wave speed kernel: %s", cudaGetErrorString(e));
  m->launches++;
  CUDA_TRY(cudaMemcpyAsync(m->h_red, m->d_red, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  double lam, nu;
  memcpy(&lam, &m->h_red[0], 8);
  memcpy(&nu, &m->h_red[1], 8);
  if (m->h_red[2] != 0 || !(lam > 0.0) || !std::isfinite(lam)) return fail(MARUT_ENOTFINITE, "non-finite or non-positive wave speed");
  const double P2 = 2.0 * m->N + 1.0;
  double dt = cfl * m->dx_min / (P2 * lam);                       // eq. 18
  if (m->physics == MARUT_NAVIER_STOKES && nu > 0.0) {
    const double numax = nu * std::max(1.0, 1.0 / m->Pr);
    dt = std::min(dt, cfl * m->dx_min * m->dx_min / (P2 * P2 * numax));  // eq. 17
  }
  *dt_out = dt;
  return MARUT_OK;
}

// ------------------------------------------------------------------------------------ introspection
extern "C" marut_status marut_get_metrics(marut_mesh *m, double *Ja, double *J) {
  if (!m || !Ja || !J) return fail(MARUT_EINVAL, "NULL argument");
  const int dim = m->dim, nn = m->nn, MD = dim * dim + 1;
  const size_t cnt = m->affine ? (size_t)m->ne * MD : (size_t)m->ne * MD * nn;
  std::vector<double> h(cnt);
  CUDA_TRY(cudaMemcpy(h.data(), m->d_metric, cnt * sizeof(double), cudaMemcpyDeviceToHost));
  for (long e = 0; e < m->ne; ++e)
    for (int p = 0; p < nn; ++p) {
      for (int k = 0; k < dim * dim; ++k)
        Ja[((size_t)e * nn + p) * dim * dim + k] = m->affine ? h[(size_t)e * MD + k] : h[((size_t)e * MD + k) * nn + p];
      const double iJ = m->affine ? h[(size_t)e * MD + dim * dim] : h[((size_t)e * MD + dim * dim) * nn + p];
      J[(size_t)e * nn + p] = 1.0 / iJ;
    }
  return MARUT_OK;
}
extern "C" int marut_is_affine(const marut_mesh *m) { return m && m->affine ? 1 : 0; }
extern "C" double marut_dx_min(const marut_mesh *m) { return m ? m->dx_min : 0.0; }
extern "C" long marut_launch_count(const marut_mesh *m) { return m ? m->launches.load() : 0; }
extern "C" marut_status marut_debug_stage_kernel(marut_mesh *m, int which) {
  if (!m || which < 0 || which > 2) return fail(MARUT_EINVAL, "bad argument");
  m->stage_kernel_pref = which;
  return MARUT_OK;
}
template <bool FAST>
__global__ void debug_rcp_sqrt_kernel(const double *__restrict__ x, double *__restrict__ r, double *__restrict__ s, long n) {
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
    r[i] = FAST ? rcp_pos_2ulp(x[i]) : rcp_pos(x[i]);
    s[i] = FAST ? sqrt_pos_2ulp(x[i]) : sqrt_pos(x[i]);
  }
}
extern "C" marut_status marut_debug_rcp_sqrt(const double *x, double *rcp, double *sq, long n, int variant, void *stream) {
  if (!x || !rcp || !sq || n < 0 || variant < 0 || variant > 1) return fail(MARUT_EINVAL, "bad argument");
  if (n == 0) return MARUT_OK;
  const unsigned grid = (unsigned)std::min<long>((n + 255) / 256, 148L * 8);
  if (variant) debug_rcp_sqrt_kernel<true><<<grid, 256, 0, (cudaStream_t)stream>>>(x, rcp, sq, n);
  else debug_rcp_sqrt_kernel<false><<<grid, 256, 0, (cudaStream_t)stream>>>(x, rcp, sq, n);
  CUDA_TRY(cudaGetLastError());
  return MARUT_OK;
}
extern "C" const char *marut_last_error(void) { return g_err; }
