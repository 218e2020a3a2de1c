// ============================================================================
// oracle/marut_oracle.cpp  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, fp64 CPU restatement of the hot path of MARUT (arxiv 2605.26388):
// the semi-discrete spectral-DG right-hand side for compressible Euler /
// Navier-Stokes (BR1) / reacting Euler with a finite-rate chemistry source, the
// SSP-RK33 stage update and the CFL time step.  It follows the paper step by
// step (citations are PAPER.md line numbers) and the readings listed in
// DESIGN.md section 3.  No blocking, no fusion, no reordering.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may build, load or call this file.  It shares no code, header,
// table or constant generator with paper_2605_26388_b200/ (the CUDA path).
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC  (see oracle/__init__.py)
// -ffp-contract=off: no FMA contraction, so every operation below is a single
// IEEE-754 double operation in the order written.
//
// Parity pins: every function below is pinned by tests/test_oracle_*.py to
// closed forms / invariants / paper-printed values;
// none is "parity unpinned".
//
// Layouts (all row-major, last index fastest):
//   node_xyz [e][c][node]     node = i + n*(j + n*k), n = N+1
//   u, du    [e][v][node]     v = rho_1..rho_ns, rho*u_1..rho*u_d, E
//   iface    [f][5] = eL,fL,eR,fR,orient      face f = 2*l + side
//   mortar   2-D: [m][6] = eC,fC,eF_lo,eF_up,fF,orient
//            3-D: [m][8] = eC,fC,eF_00,eF_10,eF_01,eF_11,fF,orient (eF_{s0 s1}: half s0 of the first, s1 of the
//            second face-local direction of the coarse face; orient must be 0)
//   bface    [b][3] = e,f,bc_id ;  bc_state [bc][nvar]
// ============================================================================
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

// Extended precision of the 1-D operator construction (O1).
typedef long double ExtReal;
// -DORACLE_LONG_DOUBLE: this same source with EVERY `double` an x87 80-bit long double (64-bit mantissa), interface
// arrays and scalars included.  Test infrastructure only (oracle.lib_ld()): the reference against which the round-off
// of the FP64 oracle and of the GPU path is measured at full size (reading T1).  Literals stay double
// constants; the few that are not exact (1/3, 2/3, ...) carry a relative error of 1e-16, far below what is measured.
#ifdef ORACLE_LONG_DOUBLE
#define double long double
#endif

namespace {

constexpr double R_UNIVERSAL = 8.31446261815324;   // J/(mol K)
constexpr double P_REF = 101325.0;                 // Pa, standard-state pressure of K_c
constexpr int MAXV = 16;                           // max variables per node
constexpr int MAXS = 8;                            // max species

enum Physics { EULER = 0, NAVIER_STOKES = 1, REACTING_EULER = 2 };

// ---------------------------------------------------------------------------
// O1. One-dimensional operators on Legendre-Gauss-Lobatto nodes.
// ---------------------------------------------------------------------------
// Legendre polynomial P_N(x) and its derivative by the three-term recurrence
//   (k+1) P_{k+1} = (2k+1) x P_k - k P_{k-1},   P'_{k+1} = P'_{k-1} + (2k+1) P_k.
template <typename T>
static void legendre(int N, T x, T &P, T &dP) {
  T Pm = 1, dPm = 0;                   // P_0
  if (N == 0) { P = Pm; dP = dPm; return; }
  T Pc = x, dPc = 1;                   // P_1
  for (int k = 1; k < N; ++k) {
    T Pn = ((2 * k + 1) * x * Pc - k * Pm) / (k + 1);
    T dPn = dPm + (2 * k + 1) * Pc;
    Pm = Pc; dPm = dPc; Pc = Pn; dPc = dPn;
  }
  P = Pc; dP = dPc;
}

struct Ops {
  int N = 0, n = 0;
  std::vector<double> x, w, D;         // D[i*n+j] = l_j'(x_i)
};

// LGL nodes: x_0=-1, x_N=+1 and the roots of P'_N; w_j = 2/(N(N+1) P_N(x_j)^2);
// D by barycentric weights, diagonal = -(sum of the off-diagonals of the row).
// Evaluated in extended precision (long double) and rounded once, so that x, w and D are the
// correctly rounded doubles of their exact values (independent of the formula used to get them).
static Ops make_ops(int N) {
  typedef ExtReal LD;
  Ops o; o.N = N; o.n = N + 1;
  const int n = o.n;
  std::vector<LD> x(n), w(n), D((size_t)n * n, 0);
  x[0] = -1; x[N] = 1;
  const LD PI = 3.141592653589793238462643383279502884L;
  for (int j = 1; j < N; ++j) {
    LD xj = -cosl(PI * j / N);                   // Chebyshev-Lobatto starting guess
    for (int it = 0; it < 100; ++it) {
      LD P, dP; legendre<LD>(N, xj, P, dP);
      // Legendre ODE: (1-x^2) P'' = 2 x P' - N(N+1) P
      LD d2P = (2 * xj * dP - N * (N + 1) * P) / (1 - xj * xj);
      LD dx = dP / d2P;
      xj -= dx;
      if (fabsl(dx) < 1e-20L) break;
    }
    x[j] = xj;
  }
  if (N % 2 == 0) x[N / 2] = 0;                  // the middle node is exactly 0 by symmetry
  for (int j = 0; j < n; ++j) {
    LD P, dP; legendre<LD>(N, x[j], P, dP);
    w[j] = 2 / (N * (N + 1) * P * P);
  }
  std::vector<LD> lam(n, 1);
  for (int j = 0; j < n; ++j) {
    LD prod = 1;
    for (int k = 0; k < n; ++k) if (k != j) prod *= (x[j] - x[k]);
    lam[j] = 1 / prod;
  }
  for (int i = 0; i < n; ++i) {
    LD sum = 0;
    for (int j = 0; j < n; ++j) if (j != i) {
      D[i * n + j] = (lam[j] / lam[i]) / (x[i] - x[j]);
      sum += D[i * n + j];
    }
    D[i * n + i] = -sum;
  }
  if (N % 2 == 0) D[(N / 2) * n + N / 2] = 0;    // antisymmetry of D about the centre: exact zero
  o.x.resize(n); o.w.resize(n); o.D.resize((size_t)n * n);
  for (int j = 0; j < n; ++j) { o.x[j] = (double)x[j]; o.w[j] = (double)w[j]; }
  for (int k = 0; k < n * n; ++k) o.D[k] = (double)D[k];
  return o;
}

// value of the j-th Lagrange polynomial on nodes x[] at point y (product form)
static double lagrange(const std::vector<double> &x, int j, double y) {
  double v = 1.0;
  for (size_t k = 0; k < x.size(); ++k) if ((int)k != j) v *= (y - x[k]) / (x[j] - x[k]);
  return v;
}

// Gauss-Legendre nodes/weights with m points: roots of P_m, w = 2/((1-x^2) P_m'(x)^2)
static void gauss_legendre(int m, std::vector<double> &g, std::vector<double> &wg) {
  g.assign(m, 0.0); wg.assign(m, 0.0);
  const double PI = 3.14159265358979323846;
  for (int q = 0; q < m; ++q) {
    double x = -std::cos(PI * (q + 0.75) / (m + 0.5));
    for (int it = 0; it < 100; ++it) {
      double P, dP; legendre<double>(m, x, P, dP);
      double dx = P / dP; x -= dx;
      if (std::fabs(dx) < 1e-16) break;
    }
    double P, dP; legendre<double>(m, x, P, dP);
    g[q] = x; wg[q] = 2.0 / ((1.0 - x * x) * dP * dP);
  }
}

// ---------------------------------------------------------------------------
// O7. 2:1 mortar projection matrices, reading R7.
// Coarse face parameter z in [-1,1]; "lo" mortar covers [-1,0], "up" covers [0,1].
//   P_fwd^lo[i][j] = l_j((x_i-1)/2),  P_fwd^up[i][j] = l_j((x_i+1)/2)
//   P_rev^m = exact L2 projection of the piecewise (lo,up) data onto degree-N
//   polynomials on the coarse face, via Legendre coefficients with (N+1)-point
//   Gauss quadrature, evaluated at the LGL nodes.
// ---------------------------------------------------------------------------
static void make_mortar(const Ops &o, std::vector<double> Pf[2], std::vector<double> Pr[2]) {
  const int n = o.n, N = o.N;
  std::vector<double> g, wg; gauss_legendre(n, g, wg);
  for (int m = 0; m < 2; ++m) {
    const double shift = (m == 0) ? -1.0 : 1.0;
    Pf[m].assign(n * n, 0.0); Pr[m].assign(n * n, 0.0);
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) Pf[m][i * n + j] = lagrange(o.x, j, (o.x[i] + shift) / 2.0);
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) {
        double acc = 0.0;
        for (int k = 0; k <= N; ++k) {
          // q_k = (2k+1)/2 * 1/2 * int_{-1}^{1} l_j(eta) L_k((eta+shift)/2) d eta
          double integ = 0.0;
          for (int q = 0; q < n; ++q) {
            double Lk, dLk; legendre<double>(k, (g[q] + shift) / 2.0, Lk, dLk);
            integ += wg[q] * lagrange(o.x, j, g[q]) * Lk;
          }
          double Lki, dLki; legendre<double>(k, o.x[i], Lki, dLki);
          acc += Lki * (2.0 * k + 1.0) / 2.0 * 0.5 * integ;
        }
        Pr[m][i * n + j] = acc;
      }
  }
}

// ---------------------------------------------------------------------------
// O12. Thermochemistry; single temperature.
// ---------------------------------------------------------------------------
struct Mech {
  int ns = 0, nr = 0;
  double T_mid = 1000.0;
  std::vector<double> W;        // [ns] kg/mol
  std::vector<double> nasa;     // [ns][2][7] (low range, then high range)
  std::vector<int> nu_r, nu_p;  // [nr][ns]  nu' (reactants), nu'' (products)
  std::vector<double> A, b, Ea; // [nr]   k_f = A T^b exp(-Ea/T); A in cm^3-mol-s units, Ea in K
};

static const double *nasa_range(const Mech &m, int s, double T) {
  return &m.nasa[(s * 2 + (T < m.T_mid ? 0 : 1)) * 7];
}
// NASA-7: cp/R = a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4
static double cp_over_R(const Mech &m, int s, double T) {
  const double *a = nasa_range(m, s, T);
  return a[0] + a[1] * T + a[2] * T * T + a[3] * T * T * T + a[4] * T * T * T * T;
}
// h/(RT) = a1 + a2 T/2 + a3 T^2/3 + a4 T^3/4 + a5 T^4/5 + a6/T
static double h_over_RT(const Mech &m, int s, double T) {
  const double *a = nasa_range(m, s, T);
  return a[0] + a[1] * T / 2.0 + a[2] * T * T / 3.0 + a[3] * T * T * T / 4.0 +
         a[4] * T * T * T * T / 5.0 + a[5] / T;
}
// s/R = a1 ln T + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7
static double s_over_R(const Mech &m, int s, double T) {
  const double *a = nasa_range(m, s, T);
  return a[0] * std::log(T) + a[1] * T + a[2] * T * T / 2.0 + a[3] * T * T * T / 3.0 +
         a[4] * T * T * T * T / 4.0 + a[6];
}
// specific internal energy e_s = h_s - R_s T (formation enthalpy inside h_s) [J/kg]
static double e_species(const Mech &m, int s, double T) {
  double Rs = R_UNIVERSAL / m.W[s];
  return Rs * T * (h_over_RT(m, s, T) - 1.0);
}
static double cv_species(const Mech &m, int s, double T) {
  double Rs = R_UNIVERSAL / m.W[s];
  return Rs * (cp_over_R(m, s, T) - 1.0);
}
// Newton on f(T) = sum_s rho_s e_s(T) - e_int = 0, f' = sum_s rho_s cv_s(T)
// (PAPER.md:288(i)); start 4000 K, stop |dT| <= 1e-13 T, cap 50 (R12).
static double temperature_from_energy(const Mech &m, const double *rho_s, double e_int) {
  double T = 4000.0;
  for (int it = 0; it < 50; ++it) {
    double f = -e_int, df = 0.0;
    for (int s = 0; s < m.ns; ++s) { f += rho_s[s] * e_species(m, s, T); df += rho_s[s] * cv_species(m, s, T); }
    double dT = f / df;
    T -= dT;
    if (std::fabs(dT) <= 1e-13 * T) break;
  }
  return T;
}
// forward rate constant, modified Arrhenius (eq. 6 with T_a = T)
static double k_forward(const Mech &m, int r, double T) {
  return m.A[r] * std::pow(T, m.b[r]) * std::exp(-m.Ea[r] / T);
}
// equilibrium constant in concentration units of mol/cm^3 (R12):
//   K_c = exp(-sum_s dnu_s g_s/(R_u T)) * (p_ref/(R_u T) * 1e-6)^(sum_s dnu_s),
//   g_s/(R_u T) = h_s/(R_u T) - s_s/R_u
static double k_equilibrium(const Mech &m, int r, double T) {
  double dG = 0.0; int dnu = 0;
  for (int s = 0; s < m.ns; ++s) {
    int d = m.nu_p[r * m.ns + s] - m.nu_r[r * m.ns + s];
    if (d != 0) { dG += d * (h_over_RT(m, s, T) - s_over_R(m, s, T)); dnu += d; }
  }
  double c0 = P_REF / (R_UNIVERSAL * T) * 1.0e-6;   // mol/cm^3
  double f = 1.0;
  for (int k = 0; k < std::abs(dnu); ++k) f *= c0;
  if (dnu < 0) f = 1.0 / f;
  return std::exp(-dG) * f;
}
// net molar rate of reaction r (eq. 21), concentrations [X_s] = rho_s/W_s in mol/cm^3
static double reaction_rate(const Mech &m, int r, double T, const double *X) {
  double kf = k_forward(m, r, T);
  double kb = kf / k_equilibrium(m, r, T);
  double pf = 1.0, pb = 1.0;
  for (int s = 0; s < m.ns; ++s) {
    for (int k = 0; k < m.nu_r[r * m.ns + s]; ++k) pf *= X[s];
    for (int k = 0; k < m.nu_p[r * m.ns + s]; ++k) pb *= X[s];
  }
  return kf * pf - kb * pb;
}
// species mass production rates (eq. 22), kg/(m^3 s)
static void production_rates(const Mech &m, double T, const double *rho_s, double *omega) {
  double X[MAXS];
  for (int s = 0; s < m.ns; ++s) { X[s] = rho_s[s] / m.W[s] * 1.0e-6; omega[s] = 0.0; }
  for (int r = 0; r < m.nr; ++r) {
    double Rr = reaction_rate(m, r, T, X);
    for (int s = 0; s < m.ns; ++s) omega[s] += (m.nu_p[r * m.ns + s] - m.nu_r[r * m.ns + s]) * Rr;
  }
  for (int s = 0; s < m.ns; ++s) omega[s] = m.W[s] * omega[s] * 1.0e6;
}

// ---------------------------------------------------------------------------
// Mesh + geometry
// ---------------------------------------------------------------------------
struct Mesh {
  int dim = 0, N = 0, n = 0, nn = 0, nvar = 0, ns = 1, physics = EULER;
  long ne = 0;
  Ops ops;
  std::vector<double> xyz;      // [e][c][node]
  std::vector<double> Ja;       // [e][node][l][c]  contravariant vectors J a^l
  std::vector<double> J;        // [e][node]
  std::vector<int> iface, mortar, bface;
  std::vector<double> bc_state;
  double gamma = 1.4, mu = 0.0, Pr = 0.72;
  Mech mech;
  std::vector<double> Pf[2], Pr_[2];
  double dx_min = 0.0;
  int explicit_source = 1;      // reacting: 1 = L includes the chemistry source S(U); 0 = transport operator only (Strang split)
  int volume_form = 0;          // 0: standard strong form (eq. 9); 1: entropy-stable split form (eq. 10)
  std::vector<double> alpha;    // per-element blending coefficient alpha_e of eq. 11 / 42; empty = no blending
  std::vector<int> bc_kind;     // per bc id: 0 prescribed exterior state, 1 outflow, 2 slip wall (O8b), 3 no-slip adiabatic
                                // wall, 4 no-slip isothermal wall (O9b, Navier-Stokes only); empty = all 0
};

static inline int node_index(const Mesh &m, const int *ijk) {
  int idx = 0;
  for (int c = m.dim - 1; c >= 0; --c) idx = idx * m.n + ijk[c];
  return idx;
}
static inline void node_ijk(const Mesh &m, int node, int *ijk) {
  for (int c = 0; c < m.dim; ++c) { ijk[c] = node % m.n; node /= m.n; }
}
// derivative along reference direction l of a nodal field f[node] at node `node`
static double dxi(const Mesh &m, const double *f, int node, int l) {
  int ijk[3]; node_ijk(m, node, ijk);
  const int il = ijk[l];
  double s = 0.0;
  for (int q = 0; q < m.n; ++q) {
    ijk[l] = q;
    s += m.ops.D[il * m.n + q] * f[node_index(m, ijk)];
  }
  return s;
}
// volume-node index of face node `a` (a = a0 + n*a1) of face f = 2*l + side:
// the index along l is 0 (side 0) or N (side 1); the remaining directions, in
// increasing order, take a0 (and a1).
static int face_node(const Mesh &m, int f, int a) {
  int l = f / 2, side = f % 2, ijk[3] = {0, 0, 0};
  int t = 0;
  for (int c = 0; c < m.dim; ++c) {
    if (c == l) ijk[c] = side ? m.N : 0;
    else { ijk[c] = (t == 0) ? (a % m.n) : (a / m.n); ++t; }
  }
  return node_index(m, ijk);
}
// partner face-node index under `orient` ("face-indexing tables, which encode the relative orientation of
// the two elements that share a face"; reading R20).  2-D: 1 = reversed.  3-D: a = a0 + n a1 -> b = b0 + n b1,
//   (c0, c1) = (a1, a0) if orient & 4 else (a0, a1);  b0 = N - c0 if orient & 1 else c0;  b1 = N - c1 if orient & 2 else c1
static int orient_map(const Mesh &m, int a, int orient) {
  if (orient == 0) return a;
  if (m.dim == 2) return m.N - a;
  int c0 = a % m.n, c1 = a / m.n;
  if (orient & 4) std::swap(c0, c1);
  if (orient & 1) c0 = m.N - c0;
  if (orient & 2) c1 = m.N - c1;
  return c0 + m.n * c1;
}

// O2. Metric terms.
//  2-D: Ja^1 = (y_eta, -x_eta), Ja^2 = (-y_xi, x_xi), J = x_xi y_eta - x_eta y_xi.
//  3-D: conservative curl form (R2):
//    (Ja^i)_n = d_{xi_k}[X_l d_{xi_j} X_m] - d_{xi_j}[X_l d_{xi_k} X_m],
//    (i,j,k) cyclic, (n,m,l) cyclic;  J = X_xi . (X_eta x X_zeta).
static void compute_metrics(Mesh &m) {
  const int nn = m.nn, d = m.dim;
  m.Ja.assign((size_t)m.ne * nn * d * d, 0.0);
  m.J.assign((size_t)m.ne * nn, 0.0);
#pragma omp parallel for schedule(static)
  for (long e = 0; e < m.ne; ++e) {
    // coordinates relative to the element's first node: derivatives and the curl form are
    // translation invariant (D 1 = 0, and the curl of const * grad X_m vanishes because the
    // tensor-product D's commute), so this is the same definition with round-off ~eps*h
    // instead of ~eps*|X| (R2)
    std::vector<double> Xs((size_t)d * nn);
    const double *X[3] = {nullptr, nullptr, nullptr};
    for (int c = 0; c < d; ++c) {
      const double *Xa = &m.xyz[((size_t)e * d + c) * nn];
      for (int p = 0; p < nn; ++p) Xs[(size_t)c * nn + p] = Xa[p] - Xa[0];
      X[c] = &Xs[(size_t)c * nn];
    }
    double *Ja = &m.Ja[(size_t)e * nn * d * d];
    double *J = &m.J[(size_t)e * nn];
    if (d == 2) {
      for (int p = 0; p < nn; ++p) {
        double x_xi = dxi(m, X[0], p, 0), x_eta = dxi(m, X[0], p, 1);
        double y_xi = dxi(m, X[1], p, 0), y_eta = dxi(m, X[1], p, 1);
        Ja[(p * 2 + 0) * 2 + 0] = y_eta;  Ja[(p * 2 + 0) * 2 + 1] = -x_eta;
        Ja[(p * 2 + 1) * 2 + 0] = -y_xi;  Ja[(p * 2 + 1) * 2 + 1] = x_xi;
        J[p] = x_xi * y_eta - x_eta * y_xi;
      }
    } else {
      std::vector<double> dX(9 * nn);            // dX[(c*3+l)*nn+p] = d X_c / d xi_l
      for (int c = 0; c < 3; ++c)
        for (int l = 0; l < 3; ++l)
          for (int p = 0; p < nn; ++p) dX[(c * 3 + l) * nn + p] = dxi(m, X[c], p, l);
      for (int p = 0; p < nn; ++p) {
        const double *g = &dX[0];
        auto G = [&](int c, int l) { return g[(c * 3 + l) * nn + p]; };
        J[p] = G(0, 0) * (G(1, 1) * G(2, 2) - G(1, 2) * G(2, 1)) -
               G(0, 1) * (G(1, 0) * G(2, 2) - G(1, 2) * G(2, 0)) +
               G(0, 2) * (G(1, 0) * G(2, 1) - G(1, 1) * G(2, 0));
      }
      std::vector<double> A(nn), B(nn);
      for (int i = 0; i < 3; ++i) {
        const int j = (i + 1) % 3, k = (i + 2) % 3;
        for (int c = 0; c < 3; ++c) {            // Cartesian component n = c
          const int mm = (c + 1) % 3, ll = (c + 2) % 3;
          for (int p = 0; p < nn; ++p) {
            A[p] = X[ll][p] * dX[(mm * 3 + j) * nn + p];   // X_l d_{xi_j} X_m
            B[p] = X[ll][p] * dX[(mm * 3 + k) * nn + p];   // X_l d_{xi_k} X_m
          }
          for (int p = 0; p < nn; ++p)
            Ja[(p * 3 + i) * 3 + c] = dxi(m, A.data(), p, k) - dxi(m, B.data(), p, j);
        }
      }
    }
  }
  // Affine elements (R2b; SURVEY 8(a) a0 "affine-element detection"): the mapping of an
  // affine element has constant metric terms; what varies from node to node is only the round-off
  // of the fp64 node coordinates (~eps*|X|/h).  An element whose metric terms all agree with their
  // node-0 values to 1e-12 (relative to max_k |Ja_k|, resp. |J|) uses the node-0 values at every node.
  for (long e = 0; e < m.ne; ++e) {
    double *Ja = &m.Ja[(size_t)e * nn * d * d];
    double *J = &m.J[(size_t)e * nn];
    double scale = 0.0, dev = 0.0;
    for (int k = 0; k < d * d; ++k) scale = std::max(scale, std::fabs(Ja[k]));
    for (int p = 0; p < nn; ++p) {
      dev = std::max(dev, std::fabs(J[p] - J[0]) / std::fabs(J[0]));
      for (int k = 0; k < d * d; ++k) dev = std::max(dev, std::fabs(Ja[p * d * d + k] - Ja[k]) / scale);
    }
    if (dev < 1e-12)
      for (int p = 1; p < nn; ++p) {
        J[p] = J[0];
        for (int k = 0; k < d * d; ++k) Ja[p * d * d + k] = Ja[k];
      }
  }
  // O11: characteristic element size dx_e = 2 (min_i J_i)^(1/d); dx_min = min_e
  double dxm = 1e300;
  for (long e = 0; e < m.ne; ++e) {
    double Jmin = 1e300;
    for (int p = 0; p < nn; ++p) Jmin = std::min(Jmin, m.J[(size_t)e * nn + p]);
    double dx = 2.0 * std::pow(Jmin, 1.0 / d);
    dxm = std::min(dxm, dx);
  }
  m.dx_min = dxm;
}

// ---------------------------------------------------------------------------
// O3. State -> primitives.
// ---------------------------------------------------------------------------
struct Prim {
  double rho, vel[3], p, a, T;
};
static Prim primitives(const Mesh &m, const double *U) {
  Prim q; q.vel[0] = q.vel[1] = q.vel[2] = 0.0;
  const int ns = m.ns, d = m.dim;
  double rho = 0.0;
  for (int s = 0; s < ns; ++s) rho += U[s];
  q.rho = rho;
  double ke = 0.0;
  for (int c = 0; c < d; ++c) { q.vel[c] = U[ns + c] / rho; ke += q.vel[c] * q.vel[c]; }
  ke = 0.5 * rho * ke;
  const double E = U[ns + d];
  if (m.physics == REACTING_EULER) {
    const Mech &k = m.mech;
    q.T = temperature_from_energy(k, U, E - ke);
    double R = 0.0, cp = 0.0;                       // mixture gas constant, frozen cp
    for (int s = 0; s < ns; ++s) {
      double Ys = U[s] / rho, Rs = R_UNIVERSAL / k.W[s];
      R += Ys * Rs; cp += Ys * Rs * cp_over_R(k, s, q.T);
    }
    q.p = rho * R * q.T;                            // p = rho R T
    double gf = cp / (cp - R);                      // frozen gamma (R12)
    q.a = std::sqrt(gf * R * q.T);
  } else {
    q.p = (m.gamma - 1.0) * (E - ke);
    q.a = std::sqrt(m.gamma * q.p / rho);
    q.T = q.p / rho;                                // R = 1
  }
  return q;
}
// inviscid flux contracted with a (scaled) vector nv: F_inv(U) . nv
static void flux_dot(const Mesh &m, const double *U, const Prim &q, const double *nv, double *F) {
  const int ns = m.ns, d = m.dim;
  double vn = 0.0;
  for (int c = 0; c < d; ++c) vn += q.vel[c] * nv[c];
  for (int s = 0; s < ns; ++s) F[s] = U[s] * vn;
  for (int c = 0; c < d; ++c) F[ns + c] = U[ns + c] * vn + q.p * nv[c];
  F[ns + d] = (U[ns + d] + q.p) * vn;
}
// O13. Logarithmic mean {{a}}^ln = (aL - aR)/(ln aL - ln aR).  The paper gives no evaluation that
// is stable near aL = aR; reading R13: Ismail & Roe's form, zeta = aL/aR, f = (zeta-1)/(zeta+1),
// u = f^2, F = 1 + u/3 + u^2/5 + u^3/7 for u < 1e-2, else ln(zeta)/(2 f); {{a}}^ln = (aL + aR)/(2 F).
static double logmean(double aL, double aR) {
  const double zeta = aL / aR, f = (zeta - 1.0) / (zeta + 1.0), u = f * f;
  const double F = (u < 1.0e-2) ? 1.0 + u / 3.0 + u * u / 5.0 + u * u * u / 7.0 : std::log(zeta) / (2.0 * f);
  return (aL + aR) / (2.0 * F);
}
// O14. Two-point volume flux of Ranocha contracted with a (scaled, averaged) vector nv (eq. 41):
//   F_rho = {{rho}}^ln {{v}}.n ;  F_rho v_c = {{rho}}^ln {{v}}.n {{v_c}} + {{p}} n_c ;
//   F_E = ( 1/((gamma-1) {{rho/p}}^ln) + 1/2 v_L.v_R ) {{rho}}^ln {{v}}.n + 1/2 (p_L v_R + p_R v_L).n ,  T = p/rho.
// Reading R13.  The paper prints the energy flux with 1/(2 (gamma-1) {{T^-1}}^ln), the kinetic term
// 1/2 sum_c {{v_c}}^2 and the pressure work {{p v}}.n.  The first contradicts the consistency F#(U,U) = F_inv(U) it
// states in eq. 40 (the 2 belongs to beta = rho/(2p) of the cited flux); the other two contradict the property it
// names on PAPER.md:611, "the kinetic energy preserving and entropy-conservative flux of Ranocha [19]": with them
// (w_R - w_L).F# != psi_R - psi_L at second order in the jump.  The stated properties fix the flux: 1/2 v_L.v_R and
// 1/2 (p_L v_R + p_R v_L) are the terms of the cited flux, and the only ones of this form that satisfy Tadmor's
// condition (pinned in tests/test_oracle_split.py).
static void ranocha_flux(const Mesh &m, const double *UL, const double *UR, const double *nv, double *F) {
  const int d = m.dim;
  const Prim L = primitives(m, UL), R = primitives(m, UR);
  const double rho_ln = logmean(L.rho, R.rho);
  const double tinv_ln = logmean(L.rho / L.p, R.rho / R.p);
  double vavg[3] = {0.0, 0.0, 0.0}, vn = 0.0, vLvR = 0.0, pvn = 0.0;
  for (int c = 0; c < d; ++c) {
    vavg[c] = 0.5 * (L.vel[c] + R.vel[c]);
    vn += vavg[c] * nv[c];
    vLvR += L.vel[c] * R.vel[c];
    pvn += 0.5 * (L.p * R.vel[c] + R.p * L.vel[c]) * nv[c];
  }
  const double pavg = 0.5 * (L.p + R.p);
  F[0] = rho_ln * vn;
  for (int c = 0; c < d; ++c) F[1 + c] = rho_ln * vn * vavg[c] + pavg * nv[c];
  F[1 + d] = (1.0 / ((m.gamma - 1.0) * tinv_ln) + 0.5 * vLvR) * rho_ln * vn + pvn;
}
// O5. Local Lax-Friedrichs / Rusanov flux with scaled outward normal nv:
//   F* = 1/2 (F(U-)+F(U+)).nv - 1/2 lambda |nv| (U+ - U-),
//   lambda = max(|v-.nhat| + a-, |v+.nhat| + a+),  nhat = nv/|nv|.
static void rusanov(const Mesh &m, const double *Um, const double *Up, const double *nv, double *Fs) {
  const int d = m.dim, nv_ = m.nvar;
  Prim qm = primitives(m, Um), qp = primitives(m, Up);
  double nrm = 0.0;
  for (int c = 0; c < d; ++c) nrm += nv[c] * nv[c];
  nrm = std::sqrt(nrm);
  double vnm = 0.0, vnp = 0.0;
  for (int c = 0; c < d; ++c) { vnm += qm.vel[c] * (nv[c] / nrm); vnp += qp.vel[c] * (nv[c] / nrm); }
  double lam = std::max(std::fabs(vnm) + qm.a, std::fabs(vnp) + qp.a);
  double Fm[MAXV], Fp[MAXV];
  flux_dot(m, Um, qm, nv, Fm); flux_dot(m, Up, qp, nv, Fp);
  for (int v = 0; v < nv_; ++v) Fs[v] = 0.5 * (Fm[v] + Fp[v]) - 0.5 * lam * nrm * (Up[v] - Um[v]);
}

static inline void gather(const Mesh &m, const double *u, long e, int node, double *U) {
  for (int v = 0; v < m.nvar; ++v) U[v] = u[((size_t)e * m.nvar + v) * m.nn + node];
}
// outward scaled normal of face f at volume node `node` of element e:  n_ref * Ja^{l_f}
static inline void face_normal(const Mesh &m, long e, int f, int node, double *nv) {
  const int l = f / 2; const double sgn = (f % 2) ? 1.0 : -1.0;
  const double *Ja = &m.Ja[((size_t)e * m.nn + node) * m.dim * m.dim + l * m.dim];
  for (int c = 0; c < m.dim; ++c) nv[c] = sgn * Ja[c];
}

// ---------------------------------------------------------------------------
// O17. First-order finite-volume residual on the LGL sub-cell grid (eq. 11, 42; the
// construction of the cited framework [15], reading R16 -- the paper names it without printing it).
// Along each reference direction l the N+1 nodes of a line own sub-cells of reference width w_0..w_N; the N interior
// sub-cell interfaces m+1/2 (between line indices m and m+1) carry the matching surface flux (Rusanov, O5)
//   fhat^l_{m+1/2} = F*(U_m, U_{m+1}; nhat^l_{m+1/2}),
// with the sub-cell normal  nhat^l_{m+1/2} = Ja^l_0 + sum_{q<=m} w_q sum_r D_qr Ja^l_r  (telescopes from Ja^l_0 to
// Ja^l_N by summation by parts; equals Ja^l on an affine element), and the two outermost interfaces carry the
// element's own flux fhat^l_{-1/2} = F(U_0).Ja^l_0, fhat^l_{N+1/2} = F(U_N).Ja^l_N -- exactly the term the surface
// lift of eq. 12, (F* - Ftilde)/(J w), which the DG and FV residuals share, replaces by the interface flux F*.
//   R^FV_i = -(1/J_i) sum_l ( fhat^l_{i_l+1/2} - fhat^l_{i_l-1/2} ) / w_{i_l}
// ---------------------------------------------------------------------------
static void subcell_normal(const Mesh &m, long e, int l, const int *ijk_line, int mi, double *nh) {
  const int d = m.dim, n = m.n, nn = m.nn;
  int q[3] = {ijk_line[0], ijk_line[1], ijk_line[2]};
  q[l] = 0;
  const double *Ja0 = &m.Ja[((size_t)e * nn + node_index(m, q)) * d * d + l * d];
  for (int c = 0; c < d; ++c) nh[c] = Ja0[c];
  for (int qq = 0; qq <= mi; ++qq)
    for (int r = 0; r < n; ++r) {
      q[l] = r;
      const double *Jar = &m.Ja[((size_t)e * nn + node_index(m, q)) * d * d + l * d];
      for (int c = 0; c < d; ++c) nh[c] += m.ops.w[qq] * m.ops.D[(size_t)qq * n + r] * Jar[c];
    }
}
static void fv_volume_residual(const Mesh &m, const double *u, long e, double *rfv /* [nvar][nn] */) {
  const int nn = m.nn, d = m.dim, nvar = m.nvar, N = m.N;
  for (int p = 0; p < nn; ++p) {
    int ijk[3] = {0, 0, 0}; node_ijk(m, p, ijk);
    double Ui[MAXV], acc[MAXV]; gather(m, u, e, p, Ui);
    for (int v = 0; v < nvar; ++v) acc[v] = 0.0;
    for (int l = 0; l < d; ++l) {
      const int il = ijk[l];
      const double *Jai = &m.Ja[((size_t)e * nn + p) * d * d + l * d];
      double fp[MAXV], fm[MAXV], nh[3], Uo[MAXV];
      int q[3] = {ijk[0], ijk[1], ijk[2]};
      if (il == N) flux_dot(m, Ui, primitives(m, Ui), Jai, fp);
      else {
        q[l] = il + 1; gather(m, u, e, node_index(m, q), Uo);
        subcell_normal(m, e, l, ijk, il, nh);
        rusanov(m, Ui, Uo, nh, fp);
      }
      if (il == 0) flux_dot(m, Ui, primitives(m, Ui), Jai, fm);
      else {
        q[l] = il - 1; gather(m, u, e, node_index(m, q), Uo);
        subcell_normal(m, e, l, ijk, il - 1, nh);
        rusanov(m, Uo, Ui, nh, fm);
      }
      for (int v = 0; v < nvar; ++v) acc[v] += (fp[v] - fm[v]) / m.ops.w[il];
    }
    for (int v = 0; v < nvar; ++v) rfv[(size_t)v * nn + p] = -acc[v] / m.J[(size_t)e * nn + p];
  }
}
// eq. 11 / 42: volume residual of element e <- (1 - alpha_e) R^DG + alpha_e R^FV (the surface lift is added afterwards)
static void blend_fv(const Mesh &m, const double *u, long e, double *du) {
  if (m.alpha.empty()) return;
  const double a = m.alpha[e];
  std::vector<double> rfv((size_t)m.nvar * m.nn);
  fv_volume_residual(m, u, e, rfv.data());
  for (int v = 0; v < m.nvar; ++v)
    for (int p = 0; p < m.nn; ++p) {
      double &x = du[((size_t)e * m.nvar + v) * m.nn + p];
      x = (1.0 - a) * x + a * rfv[(size_t)v * m.nn + p];
    }
}

// ---------------------------------------------------------------------------
// O18. Per-stage positivity floor ("a per-stage positivity floor enforces rho >= 1e-6 and
// p >= 5e-7"; how is not stated -- DESIGN.md reading R17): at every node, first rho <- max(rho, rho_min) with the
// momentum kept, then with p = (gamma-1)(E - |m|^2/(2 rho)) of the floored density, if p < p_min the total energy is
// raised to E = p_min/(gamma-1) + |m|^2/(2 rho).  Nodes already above both floors are not touched.  Returns the
// number of nodes changed.  Ideal gas (EULER / NAVIER_STOKES).
// ---------------------------------------------------------------------------
static long positivity_floor(const Mesh &m, double *u, double rho_min, double p_min) {
  const int nn = m.nn, d = m.dim, nvar = m.nvar;
  long changed = 0;
  for (long e = 0; e < m.ne; ++e)
    for (int p = 0; p < nn; ++p) {
      double *U = &u[(size_t)e * nvar * nn + p];     // variable v at U[v * nn]
      bool ch = false;
      double rho = U[0];
      if (rho < rho_min) { rho = rho_min; U[0] = rho; ch = true; }
      double m2 = 0.0;
      for (int c = 0; c < d; ++c) m2 += U[(size_t)(1 + c) * nn] * U[(size_t)(1 + c) * nn];
      const double ke = 0.5 * m2 / rho;
      const double pr = (m.gamma - 1.0) * (U[(size_t)(1 + d) * nn] - ke);
      if (pr < p_min) { U[(size_t)(1 + d) * nn] = p_min / (m.gamma - 1.0) + ke; ch = true; }
      changed += ch ? 1 : 0;
    }
  return changed;
}

// ---------------------------------------------------------------------------
// O4 + O6. Inviscid residual: volume term (eq. 9) and surface lift (eq. 12).
// ---------------------------------------------------------------------------
static void rhs_inviscid(const Mesh &m, const double *u, double *du) {
  const int nn = m.nn, d = m.dim, nvar = m.nvar, n = m.n;
  // --- volume: R_i = -(1/J_i) sum_l sum_m D_{i_l m} Ftilde^l_m,  Ftilde^l = Ja^l . F_inv
#pragma omp parallel for schedule(static)
  for (long e = 0; e < m.ne; ++e) {
    if (m.volume_form == 1) {
      // eq. 10: R_i = -(2/J_i) sum_l sum_m D_{i_l m} F#(U_i, U_m; 1/2 (Ja^l_i + Ja^l_m)),
      // m running over the nodes of the line through i along direction l
      for (int p = 0; p < nn; ++p) {
        int ijk[3] = {0, 0, 0}; node_ijk(m, p, ijk);
        double Ui[MAXV], acc[MAXV]; gather(m, u, e, p, Ui);
        for (int v = 0; v < nvar; ++v) acc[v] = 0.0;
        for (int l = 0; l < d; ++l) {
          const double *Jai = &m.Ja[((size_t)e * nn + p) * d * d + l * d];
          for (int mm = 0; mm < n; ++mm) {
            int q[3] = {ijk[0], ijk[1], ijk[2]}; q[l] = mm;
            const int pm = node_index(m, q);
            const double *Jam = &m.Ja[((size_t)e * nn + pm) * d * d + l * d];
            double Um[MAXV], nvv[3], F[MAXV]; gather(m, u, e, pm, Um);
            for (int c = 0; c < d; ++c) nvv[c] = 0.5 * (Jai[c] + Jam[c]);
            ranocha_flux(m, Ui, Um, nvv, F);
            const double dim_ = m.ops.D[(size_t)ijk[l] * n + mm];
            for (int v = 0; v < nvar; ++v) acc[v] += dim_ * F[v];
          }
        }
        for (int v = 0; v < nvar; ++v) du[((size_t)e * nvar + v) * nn + p] = -2.0 * acc[v] / m.J[(size_t)e * nn + p];
      }
      blend_fv(m, u, e, du);
      continue;
    }
    std::vector<double> Ft((size_t)d * nvar * nn);      // [l][v][node]
    for (int p = 0; p < nn; ++p) {
      double U[MAXV], F[MAXV]; gather(m, u, e, p, U);
      Prim q = primitives(m, U);
      for (int l = 0; l < d; ++l) {
        const double *Ja = &m.Ja[((size_t)e * nn + p) * d * d + l * d];
        flux_dot(m, U, q, Ja, F);
        for (int v = 0; v < nvar; ++v) Ft[((size_t)l * nvar + v) * nn + p] = F[v];
      }
    }
    for (int v = 0; v < nvar; ++v)
      for (int p = 0; p < nn; ++p) {
        double s = 0.0;
        for (int l = 0; l < d; ++l) s += dxi(m, &Ft[((size_t)l * nvar + v) * nn], p, l);
        du[((size_t)e * nvar + v) * nn + p] = -s / m.J[(size_t)e * nn + p];
      }
    blend_fv(m, u, e, du);
  }
  const int nf = (d == 2) ? n : n * n;                  // nodes per face
  const double wb = m.ops.w[0];                         // LGL weight of the boundary index (w_0 = w_N)
  auto lift = [&](long e, int node, const double *Fstar, const double *Fown) {
    const double Jn = m.J[(size_t)e * nn + node];
    for (int v = 0; v < nvar; ++v) du[((size_t)e * nvar + v) * nn + node] -= (Fstar[v] - Fown[v]) / (Jn * wb);
  };
  // --- conforming interfaces (O5/O6).  Eq. 12 is a per-node update in which F* takes
  // the element's OWN contravariant vector Ja^{l_f} as its normal argument, so each side of a face
  // evaluates F*(U-,U+; n_ref Ja^{l_f}) with its own metric terms (R5b).  In exact arithmetic
  // the two evaluations are equal and opposite; in floating point this keeps the bracket (F* - Ftilde)
  // free-stream preserving on each side even where the neighbours' normals differ by round-off.
  for (size_t f = 0; f < m.iface.size() / 5; ++f) {
    const int *I = &m.iface[f * 5];
    const long eL = I[0], eR = I[2]; const int fL = I[1], fR = I[3], orient = I[4];
    for (int a = 0; a < nf; ++a) {
      const int pL = face_node(m, fL, a), pR = face_node(m, fR, orient_map(m, a, orient));
      double Um[MAXV], Up[MAXV], nL[3], nR[3], Fs[MAXV], Fo[MAXV];
      gather(m, u, eL, pL, Um); gather(m, u, eR, pR, Up);
      face_normal(m, eL, fL, pL, nL); face_normal(m, eR, fR, pR, nR);
      rusanov(m, Um, Up, nL, Fs);
      flux_dot(m, Um, primitives(m, Um), nL, Fo);   lift(eL, pL, Fs, Fo);
      rusanov(m, Up, Um, nR, Fs);
      flux_dot(m, Up, primitives(m, Up), nR, Fo);   lift(eR, pR, Fs, Fo);
    }
  }
  // --- 4:1 mortars in 3-D (O7b; "factor 2 in 2D / 4 in 3D"; reading R21): the tensor product of the
  // 2-D construction.  The coarse trace is interpolated to each of the four sub-faces (Pf[s0] x Pf[s1]); the Riemann
  // problem is solved at the fine side's face nodes with the fine side's normal; the fine side lifts F*; the coarse
  // side receives the L2 projection (Pr[s0] x Pr[s1]) of the outward flux -F*, times the area ratio 4.
  for (size_t q = 0; d == 3 && q < m.mortar.size() / 8; ++q) {
    const int *M = &m.mortar[q * 8];
    const long eC = M[0]; const int fC = M[1], fF = M[6];
    std::vector<double> UC((size_t)nf * nvar), FC((size_t)nf * nvar, 0.0);
    for (int j = 0; j < nf; ++j) gather(m, u, eC, face_node(m, fC, j), &UC[(size_t)j * nvar]);
    for (int s = 0; s < 4; ++s) {
      const int s0 = s % 2, s1 = s / 2;
      const long eF = M[2 + s];
      for (int a = 0; a < nf; ++a) {
        const int a0 = a % n, a1 = a / n, pF = face_node(m, fF, a);
        double UF[MAXV], Ui[MAXV], nF[3], Fs[MAXV], Fo[MAXV];
        gather(m, u, eF, pF, UF);
        for (int v = 0; v < nvar; ++v) {
          double acc = 0.0;
          for (int j1 = 0; j1 < n; ++j1)
            for (int j0 = 0; j0 < n; ++j0) acc += m.Pf[s0][a0 * n + j0] * m.Pf[s1][a1 * n + j1] * UC[(size_t)(j0 + n * j1) * nvar + v];
          Ui[v] = acc;
        }
        face_normal(m, eF, fF, pF, nF);
        rusanov(m, UF, Ui, nF, Fs);
        flux_dot(m, UF, primitives(m, UF), nF, Fo);  lift(eF, pF, Fs, Fo);
        for (int i1 = 0; i1 < n; ++i1)
          for (int i0 = 0; i0 < n; ++i0)
            for (int v = 0; v < nvar; ++v)
              FC[(size_t)(i0 + n * i1) * nvar + v] += m.Pr_[s0][i0 * n + a0] * m.Pr_[s1][i1 * n + a1] * (4.0 * (-Fs[v]));
      }
    }
    for (int i = 0; i < nf; ++i) {
      const int pC = face_node(m, fC, i);
      double nC[3], Fo[MAXV];
      face_normal(m, eC, fC, pC, nC);
      flux_dot(m, &UC[(size_t)i * nvar], primitives(m, &UC[(size_t)i * nvar]), nC, Fo);
      lift(eC, pC, &FC[(size_t)i * nvar], Fo);
    }
  }
  // --- 2:1 mortars (O7), 2-D
  for (size_t q = 0; d == 2 && q < m.mortar.size() / 6; ++q) {
    const int *M = &m.mortar[q * 6];
    const long eC = M[0]; const int fC = M[1], fF = M[4];
    std::vector<double> UC((size_t)n * nvar), FC((size_t)n * nvar, 0.0);
    for (int j = 0; j < n; ++j) gather(m, u, eC, face_node(m, fC, j), &UC[(size_t)j * nvar]);
    for (int s = 0; s < 2; ++s) {
      const long eF = M[2 + s];
      for (int a = 0; a < n; ++a) {
        const int pF = face_node(m, fF, a);
        double UF[MAXV], Ui[MAXV], nF[3], Fs[MAXV], Fo[MAXV];
        gather(m, u, eF, pF, UF);
        for (int v = 0; v < nvar; ++v) {            // coarse trace interpolated to the mortar
          double acc = 0.0;
          for (int j = 0; j < n; ++j) acc += m.Pf[s][a * n + j] * UC[(size_t)j * nvar + v];
          Ui[v] = acc;
        }
        face_normal(m, eF, fF, pF, nF);
        rusanov(m, UF, Ui, nF, Fs);                 // fine-side normal, fine-side quadrature
        flux_dot(m, UF, primitives(m, UF), nF, Fo);  lift(eF, pF, Fs, Fo);
        // coarse side: outward flux on the mortar is -F*; area ratio 2
        for (int i = 0; i < n; ++i)
          for (int v = 0; v < nvar; ++v) FC[(size_t)i * nvar + v] += m.Pr_[s][i * n + a] * (2.0 * (-Fs[v]));
      }
    }
    for (int i = 0; i < n; ++i) {
      const int pC = face_node(m, fC, i);
      double nC[3], Fo[MAXV];
      face_normal(m, eC, fC, pC, nC);
      flux_dot(m, &UC[(size_t)i * nvar], primitives(m, &UC[(size_t)i * nvar]), nC, Fo);
      lift(eC, pC, &FC[(size_t)i * nvar], Fo);
    }
  }
  // --- boundary faces (O8): exterior state prescribed
  for (size_t b = 0; b < m.bface.size() / 3; ++b) {
    const long e = m.bface[b * 3]; const int f = m.bface[b * 3 + 1], bc = m.bface[b * 3 + 2];
    for (int a = 0; a < nf; ++a) {
      const int p = face_node(m, f, a);
      double Um[MAXV], nv[3], Fs[MAXV], Fo[MAXV];
      gather(m, u, e, p, Um); face_normal(m, e, f, p, nv);
      // O8b ("enforced weakly through the numerical surface flux"; reading R18): the exterior
      // state of an outflow face is the interior state, that of an inviscid slip wall the interior state with the
      // normal momentum reflected, m+ = m- - 2 (m- . nhat) nhat
      const int bk = m.bc_kind.empty() ? 0 : m.bc_kind[bc];
      double Ue[MAXV];
      for (int v = 0; v < nvar; ++v) Ue[v] = (bk == 0) ? m.bc_state[(size_t)bc * nvar + v] : Um[v];
      // viscous walls (kinds 3, 4; reading R22): the hyperbolic surface flux of a no-slip wall is the slip wall's
      if (bk >= 2) {
        double nrm = 0.0, mn = 0.0;
        for (int c = 0; c < d; ++c) nrm += nv[c] * nv[c];
        nrm = std::sqrt(nrm);
        for (int c = 0; c < d; ++c) mn += Um[m.ns + c] * (nv[c] / nrm);
        for (int c = 0; c < d; ++c) Ue[m.ns + c] = Um[m.ns + c] - 2.0 * mn * (nv[c] / nrm);
      }
      rusanov(m, Um, Ue, nv, Fs);
      flux_dot(m, Um, primitives(m, Um), nv, Fo);   lift(e, p, Fs, Fo);
    }
  }
}

// ---------------------------------------------------------------------------
// O9. BR1 viscous residual; conforming interfaces, boundary faces (O9b), 2-D mortars (O9c), 3-D mortars (O9d).
// W = (rho, u_1..u_d, T), T = p/rho.  S[e][node][w][c] = d W_w / d x_c.
// ---------------------------------------------------------------------------
static void prim_gradient_vars(const Mesh &m, const double *U, double *W) {
  Prim q = primitives(m, U);
  W[0] = q.rho;
  for (int c = 0; c < m.dim; ++c) W[1 + c] = q.vel[c];
  W[1 + m.dim] = q.T;
}
// viscous flux F_v(U,S) contracted with vector nv (eq. 15, q = -k grad T)
static void viscous_flux_dot(const Mesh &m, const double *U, const double *S, const double *nv, double *F) {
  const int d = m.dim;
  Prim q = primitives(m, U);
  const double mu = m.mu, k = m.gamma * mu / (m.Pr * (m.gamma - 1.0));
  // S[w*d + c]; velocity gradient dv[i][j] = d u_i / d x_j
  double divu = 0.0;
  for (int i = 0; i < d; ++i) divu += S[(1 + i) * d + i];
  double tau[3][3];
  for (int i = 0; i < d; ++i)
    for (int j = 0; j < d; ++j) {
      if (i == j) {
        double others = divu - S[(1 + i) * d + i];
        tau[i][j] = 4.0 / 3.0 * mu * S[(1 + i) * d + i] - 2.0 / 3.0 * mu * others;
      } else tau[i][j] = mu * (S[(1 + i) * d + j] + S[(1 + j) * d + i]);
    }
  F[0] = 0.0;
  double Fe = 0.0;
  for (int j = 0; j < d; ++j) {            // direction j of the flux, contracted with nv[j]
    double work = 0.0;
    for (int i = 0; i < d; ++i) work += q.vel[i] * tau[i][j];
    double qj = -k * S[(1 + d) * d + j];
    Fe += (work - qj) * nv[j];
  }
  for (int i = 0; i < d; ++i) {
    double s = 0.0;
    for (int j = 0; j < d; ++j) s += tau[i][j] * nv[j];
    F[1 + i] = s;
  }
  F[1 + d] = Fe;
}
static void br1_gradient(const Mesh &m, const double *u, std::vector<double> &S) {
  const int nn = m.nn, d = m.dim, nw = d + 2, n = m.n;
  S.assign((size_t)m.ne * nn * nw * d, 0.0);
#pragma omp parallel for schedule(static)
  for (long e = 0; e < m.ne; ++e) {
    std::vector<double> W((size_t)nw * nn), G(nn);
    for (int p = 0; p < nn; ++p) {
      double U[MAXV], Wp[MAXV]; gather(m, u, e, p, U); prim_gradient_vars(m, U, Wp);
      for (int w = 0; w < nw; ++w) W[(size_t)w * nn + p] = Wp[w];
    }
    for (int w = 0; w < nw; ++w)
      for (int c = 0; c < d; ++c) {
        // volume part: sum_l D_l( (Ja^l)_c W )
        std::vector<double> acc(nn, 0.0);
        for (int l = 0; l < d; ++l) {
          for (int p = 0; p < nn; ++p) G[p] = m.Ja[((size_t)e * nn + p) * d * d + l * d + c] * W[(size_t)w * nn + p];
          for (int p = 0; p < nn; ++p) acc[p] += dxi(m, G.data(), p, l);
        }
        for (int p = 0; p < nn; ++p) S[(((size_t)e * nn + p) * nw + w) * d + c] = acc[p];
      }
  }
  const int nf = (d == 2) ? n : n * n;
  const double wb = m.ops.w[0];
  // surface part: + (1/w_b) (What - W) n_c with What = 1/2 (W- + W+) (eq. 13)
  for (size_t f = 0; f < m.iface.size() / 5; ++f) {
    const int *I = &m.iface[f * 5];
    const long eL = I[0], eR = I[2]; const int fL = I[1], fR = I[3], orient = I[4];
    for (int a = 0; a < nf; ++a) {
      const int pL = face_node(m, fL, a), pR = face_node(m, fR, orient_map(m, a, orient));
      double Um[MAXV], Up[MAXV], Wm[MAXV], Wp[MAXV], nL[3], nR[3];
      gather(m, u, eL, pL, Um); gather(m, u, eR, pR, Up);
      prim_gradient_vars(m, Um, Wm); prim_gradient_vars(m, Up, Wp);
      face_normal(m, eL, fL, pL, nL); face_normal(m, eR, fR, pR, nR);
      for (int w = 0; w < nw; ++w) {
        double What = 0.5 * (Wm[w] + Wp[w]);
        for (int c = 0; c < d; ++c) {
          S[(((size_t)eL * nn + pL) * nw + w) * d + c] += (What - Wm[w]) * nL[c] / wb;
          S[(((size_t)eR * nn + pR) * nw + w) * d + c] += (What - Wp[w]) * nR[c] / wb;
        }
      }
    }
  }
  // O9c. 2:1 mortars, 2-D ("Non-conforming faces use the same forward and reverse projections as the
  // hyperbolic side"; reading R23): the coarse trace of W is interpolated to each mortar (P_fwd), the central
  // trace What is formed at the fine face nodes; the fine side lifts (What - W_F) n_F; the coarse side lifts the L2
  // projection (P_rev, area factor 2) of the mortar's outward What n, G*_C = sum_m P_rev^m (2 (-What_m n_F)), against
  // its own W_C n_C -- the hyperbolic mortar with the flux F.n replaced by W n.
  for (size_t q = 0; d == 2 && q < m.mortar.size() / 6; ++q) {
    const int *M = &m.mortar[q * 6];
    const long eC = M[0]; const int fC = M[1], fF = M[4];
    std::vector<double> WC((size_t)n * nw), GC((size_t)n * nw * d, 0.0);
    for (int j = 0; j < n; ++j) { double U[MAXV]; gather(m, u, eC, face_node(m, fC, j), U); prim_gradient_vars(m, U, &WC[(size_t)j * nw]); }
    for (int s = 0; s < 2; ++s) {
      const long eF = M[2 + s];
      for (int a = 0; a < n; ++a) {
        const int pF = face_node(m, fF, a);
        double UF[MAXV], WF[MAXV], nF[3];
        gather(m, u, eF, pF, UF); prim_gradient_vars(m, UF, WF); face_normal(m, eF, fF, pF, nF);
        for (int w = 0; w < nw; ++w) {
          double Wi = 0.0;
          for (int j = 0; j < n; ++j) Wi += m.Pf[s][a * n + j] * WC[(size_t)j * nw + w];
          const double What = 0.5 * (WF[w] + Wi);
          for (int c = 0; c < d; ++c) {
            S[(((size_t)eF * nn + pF) * nw + w) * d + c] += (What - WF[w]) * nF[c] / wb;
            for (int i = 0; i < n; ++i) GC[((size_t)i * nw + w) * d + c] += m.Pr_[s][i * n + a] * (2.0 * (-(What * nF[c])));
          }
        }
      }
    }
    for (int i = 0; i < n; ++i) {
      const int pC = face_node(m, fC, i);
      double nC[3]; face_normal(m, eC, fC, pC, nC);
      for (int w = 0; w < nw; ++w)
        for (int c = 0; c < d; ++c)
          S[(((size_t)eC * nn + pC) * nw + w) * d + c] += (GC[((size_t)i * nw + w) * d + c] - WC[(size_t)i * nw + w] * nC[c]) / wb;
    }
  }
  // O9d. 4:1 mortars, 3-D (same passage; readings R21 + R23): the tensor product of O9c -- the coarse trace of W goes
  // to each of the four sub-faces with Pf[s0] x Pf[s1], the coarse side lifts the projection Pr[s0] x Pr[s1] of the
  // mortars' outward What n with the area factor 4.
  for (size_t q = 0; d == 3 && q < m.mortar.size() / 8; ++q) {
    const int *M = &m.mortar[q * 8];
    const long eC = M[0]; const int fC = M[1], fF = M[6];
    std::vector<double> WC((size_t)nf * nw), GC((size_t)nf * nw * d, 0.0);
    for (int j = 0; j < nf; ++j) { double U[MAXV]; gather(m, u, eC, face_node(m, fC, j), U); prim_gradient_vars(m, U, &WC[(size_t)j * nw]); }
    for (int s = 0; s < 4; ++s) {
      const int s0 = s % 2, s1 = s / 2;
      const long eF = M[2 + s];
      for (int a = 0; a < nf; ++a) {
        const int a0 = a % n, a1 = a / n, pF = face_node(m, fF, a);
        double UF[MAXV], WF[MAXV], nF[3];
        gather(m, u, eF, pF, UF); prim_gradient_vars(m, UF, WF); face_normal(m, eF, fF, pF, nF);
        for (int w = 0; w < nw; ++w) {
          double Wt = 0.0;
          for (int j1 = 0; j1 < n; ++j1)
            for (int j0 = 0; j0 < n; ++j0) Wt += m.Pf[s0][a0 * n + j0] * m.Pf[s1][a1 * n + j1] * WC[(size_t)(j0 + n * j1) * nw + w];
          const double What = 0.5 * (WF[w] + Wt);
          for (int c = 0; c < d; ++c) {
            S[(((size_t)eF * nn + pF) * nw + w) * d + c] += (What - WF[w]) * nF[c] / wb;
            for (int i1 = 0; i1 < n; ++i1)
              for (int i0 = 0; i0 < n; ++i0)
                GC[((size_t)(i0 + n * i1) * nw + w) * d + c] += m.Pr_[s0][i0 * n + a0] * m.Pr_[s1][i1 * n + a1] * (4.0 * (-(What * nF[c])));
          }
        }
      }
    }
    for (int i = 0; i < nf; ++i) {
      const int pC = face_node(m, fC, i);
      double nC[3]; face_normal(m, eC, fC, pC, nC);
      for (int w = 0; w < nw; ++w)
        for (int c = 0; c < d; ++c)
          S[(((size_t)eC * nn + pC) * nw + w) * d + c] += (GC[((size_t)i * nw + w) * d + c] - WC[(size_t)i * nw + w] * nC[c]) / wb;
    }
  }
  // O9b. boundary faces (reading R22): the trace What is fixed by the boundary kind --
  //   prescribed state: the central trace with W(U_bc);  outflow: W- (no jump);  slip wall: "mirrors the velocity across
  //   the boundary normal", W+ = (rho-, v- - 2 (v-.nhat) nhat, T-), central trace;  no-slip adiabatic wall: "sets the wall
  //   velocity to zero and inherits interior (rho, T)", What = (rho-, 0, T-);  isothermal wall: "additionally fixes
  //   T = T_wall", What = (rho-, 0, T_wall), T_wall = the temperature of the boundary id's prescribed state.
  for (size_t b = 0; b < m.bface.size() / 3; ++b) {
    const long e = m.bface[b * 3]; const int f = m.bface[b * 3 + 1], bc = m.bface[b * 3 + 2];
    const int bk = m.bc_kind.empty() ? 0 : m.bc_kind[bc];
    for (int a = 0; a < nf; ++a) {
      const int p = face_node(m, f, a);
      double Um[MAXV], Wm[MAXV], What[MAXV], nv[3];
      gather(m, u, e, p, Um); prim_gradient_vars(m, Um, Wm); face_normal(m, e, f, p, nv);
      for (int w = 0; w < nw; ++w) What[w] = Wm[w];
      if (bk == 0) {
        double Wb[MAXV]; prim_gradient_vars(m, &m.bc_state[(size_t)bc * m.nvar], Wb);
        for (int w = 0; w < nw; ++w) What[w] = 0.5 * (Wm[w] + Wb[w]);
      } else if (bk == 2) {
        double nrm = 0.0, vn = 0.0;
        for (int c = 0; c < d; ++c) nrm += nv[c] * nv[c];
        nrm = std::sqrt(nrm);
        for (int c = 0; c < d; ++c) vn += Wm[1 + c] * (nv[c] / nrm);
        for (int c = 0; c < d; ++c) What[1 + c] = 0.5 * (Wm[1 + c] + (Wm[1 + c] - 2.0 * vn * (nv[c] / nrm)));
      } else if (bk == 3 || bk == 4) {
        for (int c = 0; c < d; ++c) What[1 + c] = 0.0;
        if (bk == 4) { double Wb[MAXV]; prim_gradient_vars(m, &m.bc_state[(size_t)bc * m.nvar], Wb); What[1 + d] = Wb[1 + d]; }
      }
      for (int w = 0; w < nw; ++w)
        for (int c = 0; c < d; ++c) S[(((size_t)e * nn + p) * nw + w) * d + c] += (What[w] - Wm[w]) * nv[c] / wb;
    }
  }
  // rescale by the inverse Jacobian
  for (long e = 0; e < m.ne; ++e)
    for (int p = 0; p < nn; ++p)
      for (int k = 0; k < nw * d; ++k) S[((size_t)e * nn + p) * nw * d + k] /= m.J[(size_t)e * nn + p];
}
static void rhs_viscous_add(const Mesh &m, const double *u, double *du) {
  const int nn = m.nn, d = m.dim, nvar = m.nvar, nw = d + 2, n = m.n;
  std::vector<double> S; br1_gradient(m, u, S);
  // volume: + (1/J) sum_l D_l (Ja^l . F_v)
#pragma omp parallel for schedule(static)
  for (long e = 0; e < m.ne; ++e) {
    std::vector<double> Ft((size_t)d * nvar * nn);
    for (int p = 0; p < nn; ++p) {
      double U[MAXV], F[MAXV]; gather(m, u, e, p, U);
      for (int l = 0; l < d; ++l) {
        const double *Ja = &m.Ja[((size_t)e * nn + p) * d * d + l * d];
        viscous_flux_dot(m, U, &S[((size_t)e * nn + p) * nw * d], Ja, F);
        for (int v = 0; v < nvar; ++v) Ft[((size_t)l * nvar + v) * nn + p] = F[v];
      }
    }
    for (int v = 0; v < nvar; ++v)
      for (int p = 0; p < nn; ++p) {
        double s = 0.0;
        for (int l = 0; l < d; ++l) s += dxi(m, &Ft[((size_t)l * nvar + v) * nn], p, l);
        du[((size_t)e * nvar + v) * nn + p] += s / m.J[(size_t)e * nn + p];
      }
  }
  // surface: + (1/(J w_b)) (F_v* - F_v) . n,  F_v* = 1/2 (F_v(U-,S-) + F_v(U+,S+)) (eq. 16)
  const int nf = (d == 2) ? n : n * n;
  const double wb = m.ops.w[0];
  for (size_t f = 0; f < m.iface.size() / 5; ++f) {
    const int *I = &m.iface[f * 5];
    const long eL = I[0], eR = I[2]; const int fL = I[1], fR = I[3], orient = I[4];
    for (int a = 0; a < nf; ++a) {
      const int pL = face_node(m, fL, a), pR = face_node(m, fR, orient_map(m, a, orient));
      double Um[MAXV], Up[MAXV], nL[3], nR[3], FmL[MAXV], FpL[MAXV], FmR[MAXV], FpR[MAXV];
      gather(m, u, eL, pL, Um); gather(m, u, eR, pR, Up);
      face_normal(m, eL, fL, pL, nL); face_normal(m, eR, fR, pR, nR);
      const double *Sm = &S[((size_t)eL * nn + pL) * nw * d], *Sp = &S[((size_t)eR * nn + pR) * nw * d];
      viscous_flux_dot(m, Um, Sm, nL, FmL); viscous_flux_dot(m, Up, Sp, nL, FpL);
      viscous_flux_dot(m, Um, Sm, nR, FmR); viscous_flux_dot(m, Up, Sp, nR, FpR);
      const double JL = m.J[(size_t)eL * nn + pL], JR = m.J[(size_t)eR * nn + pR];
      for (int v = 0; v < nvar; ++v) {
        // each side with its own outward normal (R5b)
        du[((size_t)eL * nvar + v) * nn + pL] += (0.5 * (FmL[v] + FpL[v]) - FmL[v]) / (JL * wb);
        du[((size_t)eR * nvar + v) * nn + pR] += (0.5 * (FpR[v] + FmR[v]) - FpR[v]) / (JR * wb);
      }
    }
  }
  // O9c. 2:1 mortars, 2-D ("a central surface pipeline (interface, mortar, and boundary kernels)"; reading
  // R23): state AND gradient of the coarse side are interpolated to the mortar (P_fwd), F_v* = mean of the two sides'
  // viscous fluxes with the fine-side normal; the fine side lifts F_v* - F_v,F; the coarse side lifts the projection
  // sum_m P_rev^m (2 (-F_v*_m)) against its own F_v(U_C, S_C).n_C.
  for (size_t q = 0; d == 2 && q < m.mortar.size() / 6; ++q) {
    const int *M = &m.mortar[q * 6];
    const long eC = M[0]; const int fC = M[1], fF = M[4];
    const int ng = nw * d;
    std::vector<double> UC((size_t)n * nvar), SC((size_t)n * ng), FC((size_t)n * nvar, 0.0);
    for (int j = 0; j < n; ++j) {
      const int pC = face_node(m, fC, j);
      gather(m, u, eC, pC, &UC[(size_t)j * nvar]);
      for (int k = 0; k < ng; ++k) SC[(size_t)j * ng + k] = S[((size_t)eC * nn + pC) * ng + k];
    }
    for (int s = 0; s < 2; ++s) {
      const long eF = M[2 + s];
      for (int a = 0; a < n; ++a) {
        const int pF = face_node(m, fF, a);
        double UF[MAXV], Ui[MAXV], Si[MAXV * 3], nF[3], FvF[MAXV], FvC[MAXV];
        gather(m, u, eF, pF, UF); face_normal(m, eF, fF, pF, nF);
        for (int v = 0; v < nvar; ++v) { double ui = 0.0; for (int j = 0; j < n; ++j) ui += m.Pf[s][a * n + j] * UC[(size_t)j * nvar + v]; Ui[v] = ui; }
        for (int k = 0; k < ng; ++k) { double si = 0.0; for (int j = 0; j < n; ++j) si += m.Pf[s][a * n + j] * SC[(size_t)j * ng + k]; Si[k] = si; }
        viscous_flux_dot(m, UF, &S[((size_t)eF * nn + pF) * ng], nF, FvF);
        viscous_flux_dot(m, Ui, Si, nF, FvC);
        const double JF = m.J[(size_t)eF * nn + pF];
        for (int v = 0; v < nvar; ++v) {
          const double Fs = 0.5 * (FvF[v] + FvC[v]);
          du[((size_t)eF * nvar + v) * nn + pF] += (Fs - FvF[v]) / (JF * wb);
          for (int i = 0; i < n; ++i) FC[(size_t)i * nvar + v] += m.Pr_[s][i * n + a] * (2.0 * (-Fs));
        }
      }
    }
    for (int i = 0; i < n; ++i) {
      const int pC = face_node(m, fC, i);
      double nC[3], Fo[MAXV];
      face_normal(m, eC, fC, pC, nC);
      viscous_flux_dot(m, &UC[(size_t)i * nvar], &SC[(size_t)i * ng], nC, Fo);
      const double JC = m.J[(size_t)eC * nn + pC];
      for (int v = 0; v < nvar; ++v) du[((size_t)eC * nvar + v) * nn + pC] += (FC[(size_t)i * nvar + v] - Fo[v]) / (JC * wb);
    }
  }
  // O9d. 4:1 mortars, 3-D: the tensor product of O9c (state and gradient of the coarse side to the four sub-faces with
  // Pf[s0] x Pf[s1]; the coarse side lifts Pr[s0] x Pr[s1] of the mortars' outward central flux with the area factor 4).
  for (size_t q = 0; d == 3 && q < m.mortar.size() / 8; ++q) {
    const int *M = &m.mortar[q * 8];
    const long eC = M[0]; const int fC = M[1], fF = M[6];
    const int ng = nw * d;
    std::vector<double> UC((size_t)nf * nvar), SC((size_t)nf * ng), FC((size_t)nf * nvar, 0.0);
    for (int j = 0; j < nf; ++j) {
      const int pC = face_node(m, fC, j);
      gather(m, u, eC, pC, &UC[(size_t)j * nvar]);
      for (int k = 0; k < ng; ++k) SC[(size_t)j * ng + k] = S[((size_t)eC * nn + pC) * ng + k];
    }
    for (int s = 0; s < 4; ++s) {
      const int s0 = s % 2, s1 = s / 2;
      const long eF = M[2 + s];
      for (int a = 0; a < nf; ++a) {
        const int a0 = a % n, a1 = a / n, pF = face_node(m, fF, a);
        double UF[MAXV], Ut[MAXV], St[MAXV * 3], nF[3], FvF[MAXV], FvC[MAXV];
        gather(m, u, eF, pF, UF); face_normal(m, eF, fF, pF, nF);
        for (int v = 0; v < nvar; ++v) Ut[v] = 0.0;
        for (int k = 0; k < ng; ++k) St[k] = 0.0;
        for (int j1 = 0; j1 < n; ++j1)
          for (int j0 = 0; j0 < n; ++j0) {
            const double pw = m.Pf[s0][a0 * n + j0] * m.Pf[s1][a1 * n + j1];
            for (int v = 0; v < nvar; ++v) Ut[v] += pw * UC[(size_t)(j0 + n * j1) * nvar + v];
            for (int k = 0; k < ng; ++k) St[k] += pw * SC[(size_t)(j0 + n * j1) * ng + k];
          }
        viscous_flux_dot(m, UF, &S[((size_t)eF * nn + pF) * ng], nF, FvF);
        viscous_flux_dot(m, Ut, St, nF, FvC);
        const double JF = m.J[(size_t)eF * nn + pF];
        for (int v = 0; v < nvar; ++v) {
          const double Fc = 0.5 * (FvF[v] + FvC[v]);
          du[((size_t)eF * nvar + v) * nn + pF] += (Fc - FvF[v]) / (JF * wb);
          for (int i1 = 0; i1 < n; ++i1)
            for (int i0 = 0; i0 < n; ++i0)
              FC[(size_t)(i0 + n * i1) * nvar + v] += m.Pr_[s0][i0 * n + a0] * m.Pr_[s1][i1 * n + a1] * (4.0 * (-Fc));
        }
      }
    }
    for (int i = 0; i < nf; ++i) {
      const int pC = face_node(m, fC, i);
      double nC[3], Fo[MAXV];
      face_normal(m, eC, fC, pC, nC);
      viscous_flux_dot(m, &UC[(size_t)i * nvar], &SC[(size_t)i * ng], nC, Fo);
      const double JC = m.J[(size_t)eC * nn + pC];
      for (int v = 0; v < nvar; ++v) du[((size_t)eC * nvar + v) * nn + pC] += (FC[(size_t)i * nvar + v] - Fo[v]) / (JC * wb);
    }
  }
  // O9b. boundary faces ("boundary kernels"; the wall flux is not printed: DESIGN.md reading R22).
  //   prescribed state, outflow, slip wall: F_v* = F_v(U-, S-), no viscous surface term;
  //   no-slip walls: F_v* is evaluated with the wall velocity (zero) and the interior gradient, F_v*(U_w, S-): the
  //   momentum rows carry the wall shear stress tau(S-).n (unchanged), the energy row loses the work of the stress
  //   (v_w = 0) and keeps the heat flux k grad T . n at an isothermal wall; at an adiabatic wall the heat flux through
  //   the wall vanishes as well: energy row of F_v* = 0.
  for (size_t b = 0; b < m.bface.size() / 3; ++b) {
    const long e = m.bface[b * 3]; const int f = m.bface[b * 3 + 1], bc = m.bface[b * 3 + 2];
    const int bk = m.bc_kind.empty() ? 0 : m.bc_kind[bc];
    if (bk != 3 && bk != 4) continue;
    for (int a = 0; a < nf; ++a) {
      const int p = face_node(m, f, a);
      double Um[MAXV], Uw[MAXV], nv[3], Fm[MAXV], Fw[MAXV];
      gather(m, u, e, p, Um); face_normal(m, e, f, p, nv);
      for (int v = 0; v < nvar; ++v) Uw[v] = Um[v];
      for (int c = 0; c < d; ++c) Uw[1 + c] = 0.0;          // wall velocity zero
      const double *Sm = &S[((size_t)e * nn + p) * nw * d];
      viscous_flux_dot(m, Um, Sm, nv, Fm); viscous_flux_dot(m, Uw, Sm, nv, Fw);
      if (bk == 3) Fw[1 + d] = 0.0;                          // adiabatic: no heat through the wall either
      const double Jp = m.J[(size_t)e * nn + p];
      for (int v = 0; v < nvar; ++v) du[((size_t)e * nvar + v) * nn + p] += (Fw[v] - Fm[v]) / (Jp * wb);
    }
  }
}
// K7/a9: chemistry source added per node (eq. 20 without the E_v row)
static void chem_source(const Mesh &m, const double *u, double *s, bool accumulate) {
  const int nn = m.nn, nvar = m.nvar, ns = m.ns;
#pragma omp parallel for schedule(static)
  for (long e = 0; e < m.ne; ++e)
    for (int p = 0; p < nn; ++p) {
      double U[MAXV], om[MAXS]; gather(m, u, e, p, U);
      Prim q = primitives(m, U);
      production_rates(m.mech, q.T, U, om);
      for (int v = 0; v < nvar; ++v) {
        double val = (v < ns) ? om[v] : 0.0;
        size_t idx = ((size_t)e * nvar + v) * nn + p;
        if (accumulate) s[idx] += val; else s[idx] = val;
      }
    }
}
// the semi-discrete operator L(U,t); t unused (no time-dependent BC/source)
// O15. Implicit source substep S_dt (eq. 24-25), single-temperature reading
// (R12): per node the reduced state Y = (rho_1..rho_Ns) is advanced by Newton iteration on the
// backward-Euler residual R(Y*) = Y* - Y^n - dt S_Y(Y*), S_Y = omega(T(Y*), Y*); total density, momentum and total
// energy are fixed parameters.  One sweep: (i) temperature from the caloric equation with the fixed
// momentum and energy, (ii) rates, (iii) Jacobian column by column from forward differences with
// eps_k = max(1e-7 |Y_k|, 1e-12), (iv) Y* <- Y* - J^-1 R by Gauss-Jordan elimination.
// Silent in the paper (R14): start Y* = Y^n; partial pivoting; stop when max_k |dY_k| <= 1e-13 rho,
// at most 50 sweeps.  Returns the number of sweeps.
static void implicit_residual(const Mech &k, const double *Y, const double *Yn, double dt, double e_kin_fixed_E,
                              double *R) {
  // e_kin_fixed_E = E - 1/2 rho |u|^2 with rho, momentum, E fixed (the internal energy available to the mixture)
  const double T = temperature_from_energy(k, Y, e_kin_fixed_E);
  double om[MAXV];
  production_rates(k, T, Y, om);
  for (int s = 0; s < k.ns; ++s) R[s] = Y[s] - Yn[s] - dt * om[s];
}
static int chem_implicit_node(const Mech &k, double *Y, double e_int, double dt) {
  const int ns = k.ns;
  double Yn[MAXV], rho = 0.0;
  for (int s = 0; s < ns; ++s) { Yn[s] = Y[s]; rho += Y[s]; }
  int it = 0;
  for (it = 1; it <= 50; ++it) {
    double R[MAXV], A[MAXV][MAXV + 1];
    implicit_residual(k, Y, Yn, dt, e_int, R);
    for (int c = 0; c < ns; ++c) {
      const double eps = std::max<double>(1e-7 * std::fabs(Y[c]), 1e-12);
      double Yp[MAXV], Rp[MAXV];
      for (int s = 0; s < ns; ++s) Yp[s] = Y[s];
      Yp[c] += eps;
      implicit_residual(k, Yp, Yn, dt, e_int, Rp);
      for (int s = 0; s < ns; ++s) A[s][c] = (Rp[s] - R[s]) / eps;
    }
    for (int s = 0; s < ns; ++s) A[s][ns] = R[s];
    // Gauss-Jordan with partial pivoting on [J | R]
    for (int c = 0; c < ns; ++c) {
      int piv = c;
      for (int r = c + 1; r < ns; ++r) if (std::fabs(A[r][c]) > std::fabs(A[piv][c])) piv = r;
      if (piv != c) for (int q = 0; q <= ns; ++q) std::swap(A[c][q], A[piv][q]);
      const double inv = 1.0 / A[c][c];
      for (int q = c; q <= ns; ++q) A[c][q] *= inv;
      for (int r = 0; r < ns; ++r) {
        if (r == c) continue;
        const double f = A[r][c];
        for (int q = c; q <= ns; ++q) A[r][q] -= f * A[c][q];
      }
    }
    double dmax = 0.0;
    for (int s = 0; s < ns; ++s) { Y[s] -= A[s][ns]; dmax = std::max(dmax, std::fabs(A[s][ns])); }
    if (dmax <= 1e-13 * rho) break;
  }
  return it;
}
static int chem_implicit(const Mesh &m, double *u, double dt) {
  const int nn = m.nn, ns = m.ns, d = m.dim, nvar = m.nvar;
  int worst = 0;
#pragma omp parallel for schedule(static) reduction(max : worst)
  for (long e = 0; e < m.ne; ++e)
    for (int p = 0; p < nn; ++p) {
      double U[MAXV]; gather(m, u, e, p, U);
      double rho = 0.0, m2 = 0.0;
      for (int s = 0; s < ns; ++s) rho += U[s];
      for (int c = 0; c < d; ++c) m2 += U[ns + c] * U[ns + c];
      const double e_int = U[ns + d] - 0.5 * m2 / rho;
      const int it = chem_implicit_node(m.mech, U, e_int, dt);
      worst = std::max(worst, it);
      for (int s = 0; s < ns; ++s) u[((size_t)e * nvar + s) * nn + p] = U[s];
    }
  return worst;
}
// O16. Hennemann-Gassner shock indicator with face-neighbour smoothing:
// indicator field q = rho p; modal coefficients of its degree-N interpolant in the orthonormal tensor-product Legendre
// basis (m = V^-1 q per direction, V_ik = sqrt((2k+1)/2) L_k(x_i)); E = max(E_high^N/E_tot^N, E_high^(N-1)/E_tot^(N-1));
// alpha = 1/(1 + exp(-(s/T)(E - T))), T = 0.5 * 10^(-1.8 (N+1)^(1/4)); alpha < alpha_min -> 0, alpha > alpha_max ->
// alpha_max (R15); then alpha_e <- max(alpha_e, alpha_e') over the elements e' sharing a face with e.
static void modal_matrix(const Ops &o, std::vector<double> &Vinv) {
  const int n = o.n;
  std::vector<double> V((size_t)n * n), A((size_t)n * 2 * n, 0.0);
  for (int i = 0; i < n; ++i)
    for (int k = 0; k < n; ++k) {
      double P, dP; legendre<double>(k, o.x[i], P, dP);
      V[(size_t)i * n + k] = std::sqrt((2.0 * k + 1.0) / 2.0) * P;
    }
  for (int i = 0; i < n; ++i) { for (int k = 0; k < n; ++k) A[(size_t)i * 2 * n + k] = V[(size_t)i * n + k]; A[(size_t)i * 2 * n + n + i] = 1.0; }
  for (int c = 0; c < n; ++c) {                      // Gauss-Jordan with partial pivoting on [V | I]
    int piv = c;
    for (int r = c + 1; r < n; ++r) if (std::fabs(A[(size_t)r * 2 * n + c]) > std::fabs(A[(size_t)piv * 2 * n + c])) piv = r;
    if (piv != c) for (int q = 0; q < 2 * n; ++q) std::swap(A[(size_t)c * 2 * n + q], A[(size_t)piv * 2 * n + q]);
    const double inv = 1.0 / A[(size_t)c * 2 * n + c];
    for (int q = 0; q < 2 * n; ++q) A[(size_t)c * 2 * n + q] *= inv;
    for (int r = 0; r < n; ++r) if (r != c) {
      const double f = A[(size_t)r * 2 * n + c];
      for (int q = 0; q < 2 * n; ++q) A[(size_t)r * 2 * n + q] -= f * A[(size_t)c * 2 * n + q];
    }
  }
  Vinv.assign((size_t)n * n, 0.0);
  for (int k = 0; k < n; ++k) for (int i = 0; i < n; ++i) Vinv[(size_t)k * n + i] = A[(size_t)k * 2 * n + n + i];
}
static void shock_indicator(const Mesh &m, const double *u, double s, double amin, double amax, double *alpha, bool smooth) {
  const int n = m.n, nn = m.nn, d = m.dim, N = m.N;
  std::vector<double> Vinv; modal_matrix(m.ops, Vinv);
  const double T = 0.5 * std::pow(10.0, -1.8 * std::pow((double)(N + 1), 0.25));
  std::vector<double> raw((size_t)m.ne);
  for (long e = 0; e < m.ne; ++e) {
    std::vector<double> q(nn), t(nn);
    for (int p = 0; p < nn; ++p) { double U[MAXV]; gather(m, u, e, p, U); Prim pr = primitives(m, U); q[p] = pr.rho * pr.p; }
    for (int l = 0; l < d; ++l) {                    // m = V^-1 q along every direction
      for (int p = 0; p < nn; ++p) {
        int ijk[3] = {0, 0, 0}; node_ijk(m, p, ijk);
        double acc = 0.0;
        for (int i = 0; i < n; ++i) { int r[3] = {ijk[0], ijk[1], ijk[2]}; r[l] = i; acc += Vinv[(size_t)ijk[l] * n + i] * q[node_index(m, r)]; }
        t[p] = acc;
      }
      q.swap(t);
    }
    double etot[2] = {0.0, 0.0}, ehigh[2] = {0.0, 0.0};      // [0]: K = N, [1]: K = N-1
    for (int p = 0; p < nn; ++p) {
      int ijk[3] = {0, 0, 0}; node_ijk(m, p, ijk);
      int mx = 0; for (int c = 0; c < d; ++c) mx = std::max(mx, ijk[c]);
      const double m2 = q[p] * q[p];
      etot[0] += m2; if (mx == N) ehigh[0] += m2;
      if (mx <= N - 1) { etot[1] += m2; if (mx == N - 1) ehigh[1] += m2; }
    }
    double E = ehigh[0] / etot[0];
    if (N >= 1 && etot[1] > 0.0) E = std::max(E, ehigh[1] / etot[1]);
    double a = 1.0 / (1.0 + std::exp(-(s / T) * (E - T)));
    if (a < amin) a = 0.0;
    if (a > amax) a = amax;
    raw[e] = a;
  }
  for (long e = 0; e < m.ne; ++e) alpha[e] = raw[e];
  if (!smooth) return;
  for (size_t f = 0; f < m.iface.size() / 5; ++f) {
    const long a = m.iface[f * 5], b = m.iface[f * 5 + 2];
    alpha[a] = std::max(alpha[a], raw[b]); alpha[b] = std::max(alpha[b], raw[a]);
  }
  const int mstride = (m.dim == 2) ? 6 : 8, mlast = (m.dim == 2) ? 3 : 5;
  for (size_t f = 0; f < m.mortar.size() / mstride; ++f) {
    const long c = m.mortar[f * mstride];
    for (int k = 2; k <= mlast; ++k) { const long b = m.mortar[f * mstride + k]; alpha[c] = std::max(alpha[c], raw[b]); alpha[b] = std::max(alpha[b], raw[c]); }
  }
}
static void rhs_full(const Mesh &m, const double *u, double *du) {
  rhs_inviscid(m, u, du);
  if (m.physics == NAVIER_STOKES) rhs_viscous_add(m, u, du);
  if (m.physics == REACTING_EULER && m.explicit_source) chem_source(m, u, du, true);
}
// O11. time step: dt = min(dt_C, dt_D)
static double max_dt(const Mesh &m, const double *u, double cfl, double *lam_out) {
  double lam = 0.0, nu = 0.0;
  for (long e = 0; e < m.ne; ++e)
    for (int p = 0; p < m.nn; ++p) {
      double U[MAXV]; gather(m, u, e, p, U);
      Prim q = primitives(m, U);
      double v2 = 0.0;
      for (int c = 0; c < m.dim; ++c) v2 += q.vel[c] * q.vel[c];
      lam = std::max(lam, std::sqrt(v2) + q.a);
      if (m.physics == NAVIER_STOKES) nu = std::max(nu, m.mu / q.rho);
    }
  if (lam_out) *lam_out = lam;
  const double P2 = 2.0 * m.N + 1.0;
  double dt = cfl * m.dx_min / (P2 * lam);
  if (m.physics == NAVIER_STOKES) {
    double numax = nu * std::max<double>(1.0, 1.0 / m.Pr);
    dt = std::min(dt, cfl * m.dx_min * m.dx_min / (P2 * P2 * numax));
  }
  return dt;
}

}  // namespace

// ============================================================================
// C interface for the Python tests (ctypes).  All pointers are host pointers.
// ============================================================================
extern "C" {

struct oracle_mech_desc {
  int n_species, n_reac;
  double T_mid;
  const double *W, *nasa;
  const int *nu_r, *nu_p;
  const double *A, *b, *Ea;
};
struct oracle_mesh_desc {
  int dim, N;
  long n_elem;
  const double *node_xyz;
  long n_iface; const int *iface;
  long n_mortar; const int *mortar;
  long n_bface; const int *bface;
  int n_bc; const double *bc_state;
  int physics;
  double gamma, mu, Pr;
  const oracle_mech_desc *mech;
};

static Mech to_mech(const oracle_mech_desc *d) {
  Mech k;
  if (!d) return k;
  k.ns = d->n_species; k.nr = d->n_reac; k.T_mid = d->T_mid;
  k.W.assign(d->W, d->W + k.ns);
  k.nasa.assign(d->nasa, d->nasa + (size_t)k.ns * 14);
  k.nu_r.assign(d->nu_r, d->nu_r + (size_t)k.nr * k.ns);
  k.nu_p.assign(d->nu_p, d->nu_p + (size_t)k.nr * k.ns);
  k.A.assign(d->A, d->A + k.nr); k.b.assign(d->b, d->b + k.nr); k.Ea.assign(d->Ea, d->Ea + k.nr);
  return k;
}

void oracle_operators(int N, double *x, double *w, double *D) {
  Ops o = make_ops(N);
  std::copy(o.x.begin(), o.x.end(), x); std::copy(o.w.begin(), o.w.end(), w);
  std::copy(o.D.begin(), o.D.end(), D);
}
void oracle_mortar_matrices(int N, double *Pf_lo, double *Pf_up, double *Pr_lo, double *Pr_up) {
  Ops o = make_ops(N); std::vector<double> Pf[2], Pr[2]; make_mortar(o, Pf, Pr);
  std::copy(Pf[0].begin(), Pf[0].end(), Pf_lo); std::copy(Pf[1].begin(), Pf[1].end(), Pf_up);
  std::copy(Pr[0].begin(), Pr[0].end(), Pr_lo); std::copy(Pr[1].begin(), Pr[1].end(), Pr_up);
}

void *oracle_mesh_create(const oracle_mesh_desc *d) {
  Mesh *m = new Mesh;
  m->dim = d->dim; m->N = d->N; m->n = d->N + 1; m->ne = d->n_elem;
  m->nn = (d->dim == 2) ? m->n * m->n : m->n * m->n * m->n;
  m->physics = d->physics; m->gamma = d->gamma; m->mu = d->mu; m->Pr = d->Pr;
  m->mech = to_mech(d->mech);
  m->ns = (m->physics == REACTING_EULER) ? m->mech.ns : 1;
  m->nvar = m->ns + m->dim + 1;
  m->ops = make_ops(m->N);
  make_mortar(m->ops, m->Pf, m->Pr_);
  m->xyz.assign(d->node_xyz, d->node_xyz + (size_t)m->ne * m->dim * m->nn);
  if (d->n_iface) m->iface.assign(d->iface, d->iface + d->n_iface * 5);
  if (d->n_mortar) m->mortar.assign(d->mortar, d->mortar + d->n_mortar * (m->dim == 2 ? 6 : 8));
  if (d->n_bface) m->bface.assign(d->bface, d->bface + d->n_bface * 3);
  if (d->n_bc) m->bc_state.assign(d->bc_state, d->bc_state + (size_t)d->n_bc * m->nvar);
  compute_metrics(*m);
  return m;
}
void oracle_mesh_destroy(void *h) { delete (Mesh *)h; }
int oracle_set_volume_form(void *h, int form) {
  Mesh *m = (Mesh *)h;
  if (form < 0 || form > 1 || (form == 1 && m->physics == REACTING_EULER)) return 1;
  m->volume_form = form;
  return 0;
}
// alpha: [n_elem] blending coefficients of eq. 11 (copied), or NULL to switch the blending off
int oracle_set_blend(void *h, const double *alpha) {
  Mesh *m = (Mesh *)h;
  if (alpha && m->physics == REACTING_EULER) return 1;   // eq. 11 blends the hyperbolic volume residual (Euler, Navier-Stokes)
  if (alpha) m->alpha.assign(alpha, alpha + m->ne); else m->alpha.clear();
  return 0;
}
// kinds: [n_bc] 0 prescribed state / 1 outflow / 2 slip wall (copied), or NULL for all prescribed
int oracle_set_boundary_kinds(void *h, const int *kinds, int n) {
  Mesh *m = (Mesh *)h;
  if (!kinds) { m->bc_kind.clear(); return 0; }
  if (m->physics == REACTING_EULER) return 1;
  for (int i = 0; i < n; ++i) if (kinds[i] < 0 || kinds[i] > (m->physics == NAVIER_STOKES ? 4 : 2)) return 2;
  m->bc_kind.assign(kinds, kinds + n);
  return 0;
}
long oracle_positivity_floor(void *h, double *u, double rho_min, double p_min) {
  Mesh &m = *(Mesh *)h;
  if (m.physics == REACTING_EULER) return -1;
  return positivity_floor(m, u, rho_min, p_min);
}
void oracle_fv_volume(void *h, const double *u, double *rfv) {
  Mesh &m = *(Mesh *)h;
#pragma omp parallel for schedule(static)
  for (long e = 0; e < m.ne; ++e) fv_volume_residual(m, u, e, rfv + (size_t)e * m.nvar * m.nn);
}
void oracle_subcell_normal(void *h, long e, int l, const int *ijk, int mi, double *nh) { subcell_normal(*(Mesh *)h, e, l, ijk, mi, nh); }
void oracle_shock_indicator(void *h, const double *u, double s, double amin, double amax, double *alpha, int smooth) {
  shock_indicator(*(Mesh *)h, u, s, amin, amax, alpha, smooth != 0);
}
void oracle_modal_matrix(int N, double *Vinv) {
  Ops o = make_ops(N); std::vector<double> V; modal_matrix(o, V); std::copy(V.begin(), V.end(), Vinv);
}
int oracle_set_explicit_source(void *h, int on) { ((Mesh *)h)->explicit_source = on ? 1 : 0; return 0; }
int oracle_chem_implicit(void *h, double *u, double dt) {
  Mesh *m = (Mesh *)h;
  if (m->physics != REACTING_EULER) return -1;
  return chem_implicit(*m, u, dt);
}
int oracle_chem_implicit_node(const oracle_mech_desc *d, double *rho_s, double e_int, double dt) {
  Mech k = to_mech(d);
  return chem_implicit_node(k, rho_s, e_int, dt);
}
double oracle_logmean(double aL, double aR) { return logmean(aL, aR); }
void oracle_ranocha(int dim, double gamma, const double *UL, const double *UR, const double *nv, double *F) {
  Mesh m; m.dim = dim; m.gamma = gamma; m.nvar = dim + 2; m.ns = 1; m.physics = EULER;
  ranocha_flux(m, UL, UR, nv, F);
}
int oracle_nvar(void *h) { return ((Mesh *)h)->nvar; }
double oracle_dx_min(void *h) { return ((Mesh *)h)->dx_min; }
// metrics out: Ja [e][node][l][c], J [e][node]
void oracle_metrics(void *h, double *Ja, double *J) {
  Mesh *m = (Mesh *)h;
  std::copy(m->Ja.begin(), m->Ja.end(), Ja); std::copy(m->J.begin(), m->J.end(), J);
}
void oracle_rhs(void *h, const double *u, double *du, double /*t*/) { rhs_full(*(Mesh *)h, u, du); }
void oracle_rhs_inviscid(void *h, const double *u, double *du) { rhs_inviscid(*(Mesh *)h, u, du); }
void oracle_rhs_viscous(void *h, const double *u, double *du) {
  Mesh *m = (Mesh *)h;
  std::fill(du, du + (size_t)m->ne * m->nvar * m->nn, 0.0);
  rhs_viscous_add(*m, u, du);
}
// S out: [e][node][w][c]
void oracle_br1_gradient(void *h, const double *u, double *S) {
  std::vector<double> s; br1_gradient(*(Mesh *)h, u, s); std::copy(s.begin(), s.end(), S);
}
void oracle_chem_source(void *h, const double *u, double *s) { chem_source(*(Mesh *)h, u, s, false); }
// O10. SSP-RK33 coefficients (Shu-Osher), shared by the two drivers below
static const double SSP_A[3] = {0.0, 3.0 / 4.0, 1.0 / 3.0}, SSP_B[3] = {1.0, 1.0 / 4.0, 2.0 / 3.0}, SSP_C[3] = {0.0, 1.0, 0.5};
// one SSP-RK33 stage:
//   u_out = a_s u_n + b_s (u_in + dt L(u_in, t_n + c_s dt)),
//   (a,b,c) = (0,1,0), (3/4,1/4,1), (1/3,2/3,1/2)
void oracle_ssprk_stage(void *h, int stage, double dt, double t_n, const double *u_n, const double *u_in,
                        double *u_out) {
  Mesh *m = (Mesh *)h;
  const double *a = SSP_A, *b = SSP_B, *c = SSP_C;
  const size_t len = (size_t)m->ne * m->nvar * m->nn;
  std::vector<double> L(len);
  (void)(t_n + c[stage] * dt);
  rhs_full(*m, u_in, L.data());
  for (size_t i = 0; i < len; ++i) u_out[i] = a[stage] * u_n[i] + b[stage] * (u_in[i] + dt * L[i]);
}
// O19. SSP-RK54 of Spiteri and Ruuth (five stages, fourth order, SSP coefficient ~1.508) in the
// Shu-Osher form of eq. 45, U^(i) = sum_k alpha_ik U^(k) + dt beta_ik L(U^(k)).  The paper does not
// print the coefficients; these are the published ones of the cited scheme (reading R19), pinned by the
// fourth-order conditions, the row sums of eq. 45 and the SSP coefficient the paper states.
static const double RK54_ALPHA[5][5] = {
    {1.0, 0, 0, 0, 0},
    {0.444370493651235, 0.555629506348765, 0, 0, 0},
    {0.620101851488403, 0, 0.379898148511597, 0, 0},
    {0.178079954393132, 0, 0, 0.821920045606868, 0},
    {0, 0, 0.517231671970585, 0.096059710526147, 0.386708617503269}};
static const double RK54_BETA[5][5] = {
    {0.391752226571890, 0, 0, 0, 0},
    {0, 0.368410593050371, 0, 0, 0},
    {0, 0, 0.251891774271694, 0, 0},
    {0, 0, 0, 0.544974750228521, 0},
    {0, 0, 0, 0.063692468666290, 0.226007483236906}};
void oracle_ssprk54_table(double *alpha, double *beta) {
  for (int i = 0; i < 5; ++i)
    for (int k = 0; k < 5; ++k) { alpha[i * 5 + k] = RK54_ALPHA[i][k]; beta[i * 5 + k] = RK54_BETA[i][k]; }
}
// one SSP-RK54 step of the semi-discrete system, u advanced in place (the operator is autonomous)
void oracle_ssprk54_step(void *h, double *u, double dt) {
  Mesh *m = (Mesh *)h;
  const size_t len = (size_t)m->ne * m->nvar * m->nn;
  std::vector<std::vector<double>> U(6, std::vector<double>(len)), L(5, std::vector<double>(len));
  U[0].assign(u, u + len);
  for (int i = 0; i < 5; ++i) {
    rhs_full(*m, U[i].data(), L[i].data());
    for (size_t q = 0; q < len; ++q) {
      double acc = 0.0;
      for (int k = 0; k <= i; ++k) acc += RK54_ALPHA[i][k] * U[k][q] + dt * RK54_BETA[i][k] * L[k][q];
      U[i + 1][q] = acc;
    }
  }
  std::copy(U[5].begin(), U[5].end(), u);
}
// the same table on the scalar ODE y' = lam*y + c2*t^2, stage times from the table (c_i = sum_k of the Butcher row)
double oracle_ssprk54_scalar(double y0, double lam, double c2, double t0, double dt) {
  double Y[6], Lv[5], c[6];
  Y[0] = y0; c[0] = 0.0;
  for (int i = 0; i < 5; ++i) {
    const double t = t0 + c[i] * dt;
    Lv[i] = lam * Y[i] + c2 * t * t;
    double acc = 0.0, ci = 0.0;
    for (int k = 0; k <= i; ++k) {
      acc += RK54_ALPHA[i][k] * Y[k] + dt * RK54_BETA[i][k] * Lv[k];
      ci += RK54_ALPHA[i][k] * c[k] + RK54_BETA[i][k];
    }
    Y[i + 1] = acc; c[i + 1] = ci;
  }
  return Y[5];
}
// generic SSPRK3 driver on a user ODE y' = lam*y + c2*t^2 (for the scalar pins of O10)
double oracle_ssprk3_scalar(double y0, double lam, double c2, double t0, double dt) {
  auto L = [&](double y, double t) { return lam * y + c2 * t * t; };
  double y = y0;
  for (int s = 0; s < 3; ++s) y = SSP_A[s] * y0 + SSP_B[s] * (y + dt * L(y, t0 + SSP_C[s] * dt));
  return y;
}
double oracle_max_dt(void *h, const double *u, double cfl, double *lam_max) { return max_dt(*(Mesh *)h, u, cfl, lam_max); }
// full SSPRK3 steps; if cfl > 0, dt is recomputed by max_dt each step, else fixed dt.
// returns the final time; u is advanced in place.  min_rho/min_p report positivity.
double oracle_run(void *h, double *u, int nsteps, double cfl, double dt_fixed, double t0, double *min_rho, double *min_p) {
  Mesh *m = (Mesh *)h;
  const size_t len = (size_t)m->ne * m->nvar * m->nn;
  std::vector<double> u1(len), u2(len);
  double t = t0, mr = 1e300, mp = 1e300;
  for (int s = 0; s < nsteps; ++s) {
    double dt = (cfl > 0.0) ? max_dt(*m, u, cfl, nullptr) : dt_fixed;
    oracle_ssprk_stage(h, 0, dt, t, u, u, u1.data());
    oracle_ssprk_stage(h, 1, dt, t, u, u1.data(), u2.data());
    oracle_ssprk_stage(h, 2, dt, t, u, u2.data(), u);
    t += dt;
    for (long e = 0; e < m->ne; ++e)
      for (int p = 0; p < m->nn; ++p) {
        double U[MAXV]; gather(*m, u, e, p, U);
        Prim q = primitives(*m, U);
        double rmin = q.rho;
        for (int k = 0; k < m->ns; ++k) rmin = std::min(rmin, U[k]);
        mr = std::min(mr, rmin); mp = std::min(mp, q.p);
      }
  }
  if (min_rho) *min_rho = mr;
  if (min_p) *min_p = mp;
  return t;
}
// --- pointwise pieces, exposed for the pins ---------------------------------
void oracle_rusanov(int dim, double gamma, const double *Um, const double *Up, const double *nv, double *Fs, double *lam) {
  Mesh m; m.dim = dim; m.ns = 1; m.nvar = dim + 2; m.gamma = gamma; m.physics = EULER;
  rusanov(m, Um, Up, nv, Fs);
  if (lam) {
    Prim qm = primitives(m, Um), qp = primitives(m, Up);
    double nrm = 0.0; for (int c = 0; c < dim; ++c) nrm += nv[c] * nv[c]; nrm = std::sqrt(nrm);
    double a = 0.0, b = 0.0;
    for (int c = 0; c < dim; ++c) { a += qm.vel[c] * (nv[c] / nrm); b += qp.vel[c] * (nv[c] / nrm); }
    *lam = std::max(std::fabs(a) + qm.a, std::fabs(b) + qp.a);
  }
}
void oracle_viscous_flux(int dim, double gamma, double mu, double Pr, const double *U, const double *S, const double *nv, double *F) {
  Mesh m; m.dim = dim; m.ns = 1; m.nvar = dim + 2; m.gamma = gamma; m.mu = mu; m.Pr = Pr; m.physics = NAVIER_STOKES;
  viscous_flux_dot(m, U, S, nv, F);
}
double oracle_k_forward(const oracle_mech_desc *d, int r, double T) { Mech k = to_mech(d); return k_forward(k, r, T); }
double oracle_k_equilibrium(const oracle_mech_desc *d, int r, double T) { Mech k = to_mech(d); return k_equilibrium(k, r, T); }
void oracle_production_rates(const oracle_mech_desc *d, double T, const double *rho_s, double *omega) {
  Mech k = to_mech(d); production_rates(k, T, rho_s, omega);
}
double oracle_temperature(const oracle_mech_desc *d, const double *rho_s, double e_int) {
  Mech k = to_mech(d); return temperature_from_energy(k, rho_s, e_int);
}
// thermo of one species: out = {cp/R, h/(RT), s/R, e [J/kg], cv [J/(kg K)]}
void oracle_species_thermo(const oracle_mech_desc *d, int s, double T, double *out) {
  Mech k = to_mech(d);
  out[0] = cp_over_R(k, s, T); out[1] = h_over_RT(k, s, T); out[2] = s_over_R(k, s, T);
  out[3] = e_species(k, s, T); out[4] = cv_species(k, s, T);
}
// primitives of a reacting/ideal state at one node: out = {rho, p, a, T, vel[0..2]}
void oracle_primitives(void *h, const double *U, double *out) {
  Prim q = primitives(*(Mesh *)h, U);
  out[0] = q.rho; out[1] = q.p; out[2] = q.a; out[3] = q.T; out[4] = q.vel[0]; out[5] = q.vel[1]; out[6] = q.vel[2];
}
int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
// number of OpenMP threads of the element loops from now on (bench.py's 1-core / all-core timings; no arithmetic)
void oracle_set_num_threads(int n) {
#ifdef _OPENMP
  if (n >= 1) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

}  // extern "C"
