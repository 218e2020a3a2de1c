/* ============================================================================
 * marut.h -- C ABI of the B200-native DG right-hand side + SSP-RK33 hot path
 *            of MARUT (arxiv 2605.26388).  Implemented in hand-written CUDA for
 *            sm_100a (paper_2605_26388_b200/csrc).  No CPU fallback exists.
 *
 * Citations are "PAPER.md:<line>" (text of the paper) and DESIGN.md readings.
 *
 * Conventions
 *  - n = N+1 LGL nodes per direction; a volume node is node = i + n*(j + n*k).
 *  - Solution / residual arrays (u, du, s, u_n, u_in, u_out) are DEVICE pointers
 *    owned by the caller, FP64, layout [n_elem][n_var][n^dim] (element-contiguous,
 *    variable-planar), base pointer 16-byte aligned.
 *    Variables: rho_1..rho_ns, rho*u_1..rho*u_dim, E  (ns = 1 unless REACTING_EULER).
 *  - Faces: f = 2*l + side (l = reference direction, side 0: xi_l = -1, 1: xi_l = +1).
 *    Face nodes are indexed by the remaining directions in increasing order
 *    (a = a0 + n*a1).  orient = 0: face node a of L meets face node a of R;
 *    2-D: orient = 1: a meets N - a.  3-D: orient in 0..7 ("relative orientation"; R20): node
 *    (a0, a1) of L meets node (b0, b1) of R, (c0, c1) = (a1, a0) if orient & 4 else (a0, a1),
 *    b0 = N - c0 if orient & 1 else c0,  b1 = N - c1 if orient & 2 else c1; any face of L may meet any face of R.
 *  - Descriptor arrays are HOST pointers, copied at create; the handle owns all
 *    device geometry, connectivity and scratch.
 *  - Every call returns a status; no exceptions, no abort, nothing on stdout.
 *    marut_last_error() gives a thread-local message for the last failure.
 *  - Calls are asynchronous on `cuda_stream` (a cudaStream_t, NULL = default
 *    stream) except marut_mesh_create, marut_mesh_destroy and marut_max_dt.
 * ========================================================================== */
#ifndef MARUT_H
#define MARUT_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct marut_mesh marut_mesh; /* opaque */

typedef enum {
  MARUT_OK = 0,
  MARUT_EINVAL = 1,     /* bad argument: NULL pointer, N or dim out of range, misaligned buffer, aliasing */
  MARUT_ENOMEM = 2,     /* host or device allocation failed */
  MARUT_ECUDA = 3,      /* CUDA runtime error (no device, launch failure) */
  MARUT_ETOPOLOGY = 4,  /* index out of range, face listed twice or never, unsupported orient, J <= 0 */
  MARUT_ENOTFINITE = 5  /* marut_max_dt met a non-finite or non-positive wave speed */
} marut_status;

enum { MARUT_EULER = 0, MARUT_NAVIER_STOKES = 1, MARUT_REACTING_EULER = 2 };

/* Finite-rate mechanism (R12).  Host struct, caller-owned.
 * Species thermodynamics in NASA-7 form: nasa[s][range][7], range 0: T < T_mid, range 1: T >= T_mid.
 * Reaction r: sum_s nu_r[r][s] X_s <-> sum_s nu_p[r][s] X_s (third bodies appear on both sides),
 * k_f = A T^b exp(-Ea/T) with A in cm^3-mol-s units and Ea in kelvin; k_b = k_f / K_c(T).      */
typedef struct {
  int n_species;        /* 1..8  */
  int n_reac;           /* 0..32 */
  double T_mid;
  const double *W;      /* [n_species] molar mass, kg/mol */
  const double *nasa;   /* [n_species][2][7] */
  const int *nu_r;      /* [n_reac][n_species] reactant coefficients nu'  (0..3) */
  const int *nu_p;      /* [n_reac][n_species] product  coefficients nu'' (0..3) */
  const double *A, *b, *Ea; /* [n_reac] */
} marut_mech;

/* Mesh + physics descriptor: the paper's statement of the problem. */
typedef struct {
  int dim;                /* 2 | 3 */
  int N;                  /* polynomial degree, 1..7 (the paper's P) */
  long n_elem;
  const double *node_xyz; /* [n_elem][dim][n^dim] isoparametric LGL node coordinates */
  long n_iface;
  const int *iface;       /* [n_iface][5]  = eL,fL,eR,fR,orient : conforming interior faces */
  long n_mortar;
  const int *mortar;      /* 2-D: [n_mortar][6] = eC,fC,eF_lo,eF_up,fF,orient : 2:1 hanging faces;
                             eF_lo covers the coarse face parameter [-1,0], eF_up covers [0,1]; orient must be 0.
                             EULER and NAVIER_STOKES (BR1 across the mortar: PAPER.md:223, R23).
                             3-D: [n_mortar][8] = eC,fC,eF_00,eF_10,eF_01,eF_11,fF,orient : 4:1 hanging faces (DESIGN.md
                             R21); eF_{s0 s1} covers half s0 / s1 of the coarse face's first / second face-local direction
                             (the remaining reference directions in increasing order); orient must be 0; EULER and
                             NAVIER_STOKES (BR1 across the mortar: DESIGN.md R23), affine meshes only (else EINVAL) */
  long n_bface;
  const int *bface;       /* [n_bface][3]  = e,f,bc_id : boundary faces with a prescribed exterior state */
  int n_bc;
  const double *bc_state; /* [n_bc][n_var] conserved exterior states */
  int physics;            /* MARUT_EULER | MARUT_NAVIER_STOKES | MARUT_REACTING_EULER */
  double gamma;           /* ratio of specific heats (EULER, NAVIER_STOKES) */
  double mu, Pr;          /* constant dynamic viscosity and Prandtl number (NAVIER_STOKES) */
  const marut_mech *mech; /* REACTING_EULER only, else NULL */
} marut_mesh_desc;

/* Setup: LGL nodes/weights/D, GCL-preserving metric terms
 * Ja^l and 1/J on the device, affine-element detection, mortar projection matrices, element-face
 * connectivity tables, scratch buffers.  Synchronous.  Every face of every element must appear exactly
 * once in iface/mortar/bface.  Errors: EINVAL, ENOMEM, ECUDA, ETOPOLOGY (reported here, never later). */
marut_status marut_mesh_create(const marut_mesh_desc *desc, marut_mesh **out);

/* NULL-safe; synchronises the device. */
void marut_mesh_destroy(marut_mesh *mesh);

/* du = L(u, t): the semi-discrete DG operator (eq. 9, 12; 707), including the BR1
 * viscous part (eq. 13-16) for NAVIER_STOKES and the chemistry source (PAPER.md:204,
 * eq. 20-22) for REACTING_EULER.  u, du: device, [n_elem][n_var][n^dim]; du must not alias u. */
marut_status marut_rhs(marut_mesh *mesh, const double *u, double *du, double t, void *cuda_stream);

/* One SSP-RK33 stage (Shu-Osher; eq. 45), fused with the operator:
 *   u_out = a_s*u_n + b_s*(u_in + dt*L(u_in, t_n + c_s*dt)),  (a,b,c) = (0,1,0), (3/4,1/4,1), (1/3,2/3,1/2)
 * stage in {0,1,2}.  u_out must not alias u_in (neighbours read u_in); u_out may alias u_n.
 * u_n is not read for stage 0. */
marut_status marut_ssprk_stage(marut_mesh *mesh, int stage, double dt, double t_n, const double *u_n,
                               const double *u_in, double *u_out, void *cuda_stream);

/* General stage of the Shu-Osher form, eq. 45, with two earlier stages, fused with the operator:
 *   u_out = a*u_a + b*u_in + c_dt*L(u_in)
 * (marut_ssprk_stage is this call with the SSP-RK33 table).  u_out must not alias u_in; it may alias u_a; u_a is not
 * read when a == 0.  With marut_lincomb it composes SSP-RK54 (SURVEY 8(f) NEXT-2b; R19):
 *   U1 = U0 + b10 dt L(U0); U2 = a20 U0 + a21 U1 + b21 dt L(U1); U3 = a30 U0 + a32 U2 + b32 dt L(U2);
 *   U4 = a40 U0 + a43 U3 + b43 dt L(U3);
 *   U5 = [a52 U2 + a53 U3 + a54 U4 + (b53/b43)(U4 - a40 U0 - a43 U3)] + b54 dt L(U4)   (bracket: marut_lincomb). */
marut_status marut_rk_stage(marut_mesh *mesh, double a, double b, double c_dt, const double *u_a, const double *u_in,
                            double *u_out, void *cuda_stream);

/* out = sum_{k<n} coef[k]*u[k], 1 <= n <= 4.  coef: HOST [n]; u: HOST array of n DEVICE pointers, each
 * [n_elem][n_var][n^dim]; out: DEVICE, may alias any u[k] (elementwise). */
marut_status marut_lincomb(marut_mesh *mesh, int n, const double *coef, const double *const *u, double *out,
                           void *cuda_stream);

/* dt = min(dt_C, dt_D) (eq. 17-18; R11):
 *   dt_C = cfl*dx_min/((2N+1)*max_i(|u_i|_2 + a_i)),  dt_D = cfl*dx_min^2/((2N+1)^2*nu_max) (NAVIER_STOKES),
 *   dx_min = min_e 2*(min_i J_i)^(1/dim),  nu_max = max_i(mu/rho_i)*max(1, 1/Pr).
 * Warp-shuffle max reduction on the device; dt_out is a HOST pointer; synchronises the stream. */
marut_status marut_max_dt(marut_mesh *mesh, const double *u, double cfl, double *dt_out, void *cuda_stream);

/* The same dt (bit for bit: the same reduction, eq. 17-18 evaluated on the device with the host's operation order),
 * written to DEVICE memory dt_dev (one double, caller-owned) without synchronising: the step's stages are queued
 * behind it on the same stream by marut_ssprk_stage_dev.  A non-finite
 * or non-positive wave speed cannot be reported here: dt_dev is then NaN and poisons the solution; marut_max_dt is
 * the checked call.  Uses the handle's reduction scratch: one stream per handle at a time. */
marut_status marut_max_dt_async(marut_mesh *mesh, const double *u, double cfl, double *dt_dev, void *cuda_stream);

/* marut_ssprk_stage with dt read from DEVICE memory (dt_dev, written earlier on the same stream); the kernel forms
 * b_s*dt with the rounding of the host product, so results equal marut_ssprk_stage's bit for bit (eq. 45). */
marut_status marut_ssprk_stage_dev(marut_mesh *mesh, int stage, const double *dt_dev, double t_n, const double *u_n,
                                   const double *u_in, double *u_out, void *cuda_stream);

/* marut_rk_stage with c_dt = c*dt formed in the kernel from dt_dev (DEVICE, one double): u_out = a*u_a + b*u_in +
 * (c*dt)*L(u_in) (eq. 45); equal to marut_rk_stage(a, b, c*dt, ...) bit for bit.  With
 * marut_lincomb (which needs no dt) it composes an SSP-RK54 step without a host synchronisation. */
marut_status marut_rk_stage_dev(marut_mesh *mesh, double a, double b, double c, const double *dt_dev, const double *u_a,
                                const double *u_in, double *u_out, void *cuda_stream);

/* s = S(u): per-node finite-rate chemistry source (eq. 21-22); species rows omega_s,
 * momentum and energy rows 0.  REACTING_EULER meshes only (else EINVAL). */
marut_status marut_chem_source(marut_mesh *mesh, const double *u, double *s, void *cuda_stream);

/* Implicit source substep S_dt of the Strang split (eq. 24-25; R14):
 * per node, Newton on the backward-Euler residual Y* - Y^n - dt*omega(T(Y*), Y*) of the partial densities with a
 * forward-difference Jacobian (eps_k = max(1e-7|Y_k|, 1e-12)) and Gauss-Jordan elimination; total density, momentum
 * and total energy are fixed.  u (DEVICE, layout as above) is advanced IN PLACE: only its species rows change.
 * sweeps_out (HOST, may be NULL): largest number of Newton sweeps any node needed; when given, the call synchronises
 * the stream and returns ENOTFINITE if a node did not converge within 50 sweeps.  REACTING_EULER meshes only. */
marut_status marut_chem_implicit(marut_mesh *mesh, double *u, double dt, int *sweeps_out, void *cuda_stream);

/* Hennemann-Gassner shock indicator with face-neighbour smoothing (first part of 8(f) NEXT-3; PAPER.md:177,
 * 629-653; R15): per element, the modal energy of rho*p in the two highest Legendre shells,
 *   E = max(E_high^N/E_tot^N, E_high^(N-1)/E_tot^(N-1)),  alpha = 1/(1 + exp(-(s/T)(E - T))),
 *   T = 0.5*10^(-1.8 (N+1)^(1/4)),  alpha < alpha_min -> 0,  alpha > alpha_max -> alpha_max,
 * then, if smooth != 0, alpha_e <- max(alpha_e, alpha_e') over the elements e' sharing a face (conforming or mortar).
 * alpha: DEVICE, [n_elem].  EULER / NAVIER_STOKES meshes.  Feed it to marut_set_blend for the blended residual. */
marut_status marut_shock_indicator(marut_mesh *mesh, const double *u, double s, double alpha_min, double alpha_max,
                                   int smooth, double *alpha, void *cuda_stream);

/* marut_shock_indicator for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc).  marut_shock_indicator allocates on its first call per handle (V^-1; the unsmoothed alpha_e
 * when smooth != 0); this variant runs the same kernels with that scratch in ONE fixed device array inside the library
 * (8 MiB + 512 B per GPU that loads the library, held until exit) and calls no cudaMalloc / cudaFree / allocating
 * routine.  Same arguments, same result (bit for bit).  Limit: n_elem <= marut_noalloc_max_elements() = 2^20, else
 * EINVAL.  Every call on a device shares the array, which keeps the last call's contents; each call rewrites all it
 * reads, so nothing needs clearing -- but two calls that OVERLAP on the GPU (different streams, same device) race: keep
 * them on one stream or order them with events.  The first call per device looks up the array's device address
 * (cudaGetSymbolAddress, no allocation); make that call outside a graph capture. */
marut_status marut_shock_indicator_noalloc(marut_mesh *mesh, const double *u, double s, double alpha_min, double alpha_max,
                                           int smooth, double *alpha, void *cuda_stream);
long marut_noalloc_max_elements(void);

/* Blended DG / sub-cell finite-volume volume residual (eq. 11, 655-672 eq. 42; DESIGN.md
 * reading R16):  R_i = (1 - alpha_e) R_i^(split) + alpha_e R_i^(FV), with the first-order finite-volume residual on the
 * LGL sub-cell grid
 *   R_i^FV = -(1/J_i) sum_l ( fhat^l_{i_l+1/2} - fhat^l_{i_l-1/2} ) / w_{i_l},
 * interior sub-cell interfaces carrying the Rusanov flux F*(U_m, U_m+1; nhat^l_{m+1/2}) with the sub-cell normals
 * nhat^l_{m+1/2} = Ja^l_0 + sum_{q<=m} w_q sum_r D_qr Ja^l_r, the two outermost ones the element's own flux (completed by
 * the surface lift of eq. 12, which both residuals share).
 * alpha: DEVICE, [n_elem], values in [0,1] -- normally the output of marut_shock_indicator for the same state.  The
 * pointer is KEPT, not copied: the caller owns the buffer, may rewrite it between stages (the paper recomputes it once
 * per Runge-Kutta substage), and must keep it alive until marut_set_blend(mesh, NULL) or marut_mesh_destroy.
 * NULL switches the blending off (default).  MARUT_EULER and MARUT_NAVIER_STOKES meshes (the blend acts on the hyperbolic
 * volume residual); marut_rhs / marut_ssprk_stage return EINVAL while a
 * blending field is set unless the volume form is MARUT_VOLUME_SPLIT_RANOCHA (eq. 11 blends the split form).  On a
 * curved mesh the first call allocates and fills the sub-cell normals ([n_elem][dim][dim][n^dim] doubles). */
marut_status marut_set_blend(marut_mesh *mesh, const double *alpha);

/* Boundary kinds ("wall/slip/outflow"; "enforced weakly through the numerical surface
 * flux", PAPER.md:223 the wall traces of the BR1 gradient; readings R18, R22).  kinds: HOST, [n_bc], one per
 * boundary id of the mesh description:
 *   MARUT_BC_PRESCRIBED       exterior state = bc_state[id] (default); Navier-Stokes: BR1 trace = mean of W- and W(bc_state),
 *                             no viscous surface term,
 *   MARUT_BC_OUTFLOW          exterior state = interior state (F* = F(U-).n, no lift; no BR1 jump),
 *   MARUT_BC_SLIP_WALL        exterior state = interior state with the normal momentum reflected, m+ = m- - 2 (m-.nhat) nhat;
 *                             Navier-Stokes: the BR1 trace mirrors the velocity across the normal,
 *   MARUT_BC_WALL_ADIABATIC   (MARUT_NAVIER_STOKES only) no-slip adiabatic wall: hyperbolic flux of the slip wall, BR1 trace
 *                             (rho-, 0, T-), viscous wall flux with v_w = 0 and no heat flux through the wall,
 *   MARUT_BC_WALL_ISOTHERMAL  (MARUT_NAVIER_STOKES only) as above with T_wall = temperature p/rho of bc_state[id] in the
 *                             trace and the heat flux k grad T . n kept in the wall flux.
 * Rewrites the connectivity table on the device (synchronises); takes effect from the next call.  MARUT_EULER and
 * MARUT_NAVIER_STOKES meshes (REACTING_EULER: PRESCRIBED only, else EINVAL); n_bc must equal the description's. */
enum { MARUT_BC_PRESCRIBED = 0, MARUT_BC_OUTFLOW = 1, MARUT_BC_SLIP_WALL = 2, MARUT_BC_WALL_ADIABATIC = 3, MARUT_BC_WALL_ISOTHERMAL = 4 };
marut_status marut_set_boundary_kinds(marut_mesh *mesh, const int *kinds, int n_bc);

/* Per-stage positivity floor ("a per-stage positivity floor enforces rho >= 1e-6 and
 * p >= 5e-7"; reading R17), in place on u (DEVICE, [n_elem][nvar][n^dim]): at every node
 *   rho <- max(rho, rho_min), momentum kept;  if (gamma-1)(E - |m|^2/(2 rho)) < p_min:  E <- p_min/(gamma-1) + |m|^2/(2 rho).
 * Nodes above both floors are not written.  changed_out (HOST, may be NULL): number of nodes changed; asking for it
 * synchronises the stream.  EULER / NAVIER_STOKES meshes; rho_min, p_min > 0 (else EINVAL). */
marut_status marut_positivity_floor(marut_mesh *mesh, double *u, double rho_min, double p_min, long *changed_out,
                                    void *cuda_stream);

/* Whole time steps (SURVEY 8(f) NEXT-2 / NEXT-2b), composed inside the library from the stage calls above, so that no
 * caller has to carry a coefficient table.  u (DEVICE) is advanced in place; scratch[k] are state-sized DEVICE buffers
 * owned by the caller, 16-byte aligned, distinct from u and from one another.  dt_dev != NULL: the time step is read
 * from that DEVICE double inside the kernels (marut_max_dt_async; `dt` is ignored and nothing waits for the GPU), else
 * the HOST value `dt` is used.  Asynchronous on the stream.
 *   marut_ssprk33_step: eq. 44-46 (R10), three marut_ssprk_stage calls; 2 scratch buffers.
 *   marut_ssprk54_step: the five-stage fourth-order scheme PAPER.md:725 names (table: DESIGN.md R19), five stage
 *                       kernels and one four-term combination; 3 scratch buffers.
 *   marut_strang_step : eq. 24, u <- S_{dt/2} T_dt S_{dt/2} u with S = marut_chem_implicit and
 *                       T_dt = one SSP-RK33 step of the transport operator without the explicit source (the handle's
 *                       marut_set_explicit_source setting is restored); REACTING_EULER meshes, HOST dt; 2 scratch
 *                       buffers.  sweeps_out (HOST, may be NULL): the larger Newton sweep count of the two substeps;
 *                       asking for it synchronises, and > 50 returns MARUT_ENOTFINITE.  Whether or not it is asked
 *                       for, a node whose Newton iteration does not converge gets NaN species densities. */
marut_status marut_ssprk33_step(marut_mesh *mesh, double *u, double *const *scratch, double dt, const double *dt_dev,
                                void *cuda_stream);
/* One SSP-RK33 step with the time step read from dt_in (DEVICE double) that also leaves the CFL step of the NEW state
 * in dt_out (DEVICE double, != dt_in): dt_out = marut_max_dt_async(u^{n+1}, cfl), bit for bit.  Where the stage kernel
 * supports it (MARUT_EULER, strong form, affine meshes large enough for the line kernel) the maximum wave speed of
 * u^{n+1} (eq. 18) is reduced inside the last stage's kernel from the values it writes -- no
 * separate pass over u (8 B/DOF saved per step) -- and the CTA that finishes last evaluates eq. 18;
 * elsewhere the call runs the separate reduction after the last stage.  A step loop alternates two DEVICE doubles:
 *   marut_max_dt_async(u, cfl, dt[0]); for k = 0, 1, ...: marut_ssprk33_step_cfl(u, scratch, cfl, dt[k&1], dt[(k+1)&1]).
 * A non-finite or non-positive wave speed poisons dt_out with NaN (as marut_max_dt_async).  Asynchronous. */
marut_status marut_ssprk33_step_cfl(marut_mesh *mesh, double *u, double *const *scratch, double cfl, const double *dt_in,
                                    double *dt_out, void *cuda_stream);
/* One SSP-RK33 step that takes its own time step: dt = cfl dx_min / ((2N+1) max(|v| + a)) of the state u it starts from
 * (eq. 17-18; = marut_max_dt(u, cfl), bit for bit) is formed on the device, left in dt_out (DEVICE
 * double) and used by the three stages -- the composition marut_max_dt_async + marut_ssprk33_step(dt_dev) in one call.
 * REACTING_EULER: the reduction rides on the first stage's thermochemistry pass (eos_kernel has T and the frozen sound
 * speed of every node of u), so no separate wave-speed pass (a Newton solve per node) runs.  Other physics: the
 * separate reduction, then the stages.  A non-finite or non-positive wave speed poisons dt_out -- and through it the new
 * state -- with NaN.  scratch: 2 DEVICE buffers like u.  Asynchronous. */
marut_status marut_ssprk33_step_dt(marut_mesh *mesh, double *u, double *const *scratch, double cfl, double *dt_out,
                                   void *cuda_stream);
marut_status marut_ssprk54_step(marut_mesh *mesh, double *u, double *const *scratch, double dt, const double *dt_dev,
                                void *cuda_stream);
marut_status marut_strang_step(marut_mesh *mesh, double *u, double *const *scratch, double dt, int *sweeps_out,
                               void *cuda_stream);

/* REACTING_EULER meshes: whether L(u) of marut_rhs / marut_ssprk_stage includes the explicit chemistry source S(u)
 * (on != 0, the default) or is the transport operator T alone (on == 0), as the Strang split of eq. 24 needs:
 *   u^{n+1} = S_{dt/2} o T_dt o S_{dt/2} (u^n) = marut_chem_implicit(dt/2), SSP-RK steps of T, marut_chem_implicit(dt/2). */
marut_status marut_set_explicit_source(marut_mesh *mesh, int on);

/* Volume-integral form of L.  MARUT_VOLUME_STRONG (default): eq. 9, the standard strong form.
 * MARUT_VOLUME_SPLIT_RANOCHA: the entropy-stable split form, eq. 10,
 *   R_i = -(2/J_i) sum_l sum_m D_{i_l m} F#(U_i, U_m; 1/2 (Ja^l_i + Ja^l_m)),
 * with the two-point flux of Ranocha (eq. 41) and logarithmic means (R13); the surface
 * terms are unchanged.  MARUT_EULER and MARUT_NAVIER_STOKES meshes with N <= 7 (2-D) / N <= 6 (3-D) (else EINVAL).  The
 * form replaces the HYPERBOLIC volume integral only: on a Navier-Stokes mesh the parabolic RHS (eq. 13-16) is added
 * unchanged by a second kernel launch of the stage.  Takes effect from the next call. */
enum { MARUT_VOLUME_STRONG = 0, MARUT_VOLUME_SPLIT_RANOCHA = 1 };
marut_status marut_set_volume_form(marut_mesh *mesh, int form);

/* --- introspection (used by the tests to check setup row a0; no compute path depends on them) --- */
/* copy the device metric terms to HOST arrays: Ja [n_elem][n^dim][dim][dim] (Ja^l_c), J [n_elem][n^dim]. */
marut_status marut_get_metrics(marut_mesh *mesh, double *Ja_host, double *J_host);
/* 1 if every element was detected affine (metrics stored per element), else 0; dx_min as used by marut_max_dt */
int marut_is_affine(const marut_mesh *mesh);
double marut_dx_min(const marut_mesh *mesh);
/* number of kernel launches issued through this handle so far (bench.py's gpu_launches) */
long marut_launch_count(const marut_mesh *mesh);

/* Euler strong-form stage on affine meshes: which of the two stage kernels runs.  0 (default): the line kernel
 * (csrc/marut_pencil.cuh) when the mesh has enough elements to fill the device with its tiles, else the thread-per-node
 * kernel (csrc/marut_node.cuh); 1: always the thread-per-node kernel; 2: the line kernel whenever the mesh kind allows
 * it, whatever its size.  Both kernels compute the same operator; the parity tests use 1 / 2 to cover both on small
 * meshes.  No effect on other physics / volume forms. */
marut_status marut_debug_stage_kernel(marut_mesh *mesh, int which);

/* the kernels' branch-free 1/x and sqrt(x) for positive normal-range operands (csrc/marut_common.cuh) evaluated on n
 * DEVICE doubles x -> rcp, sq (DEVICE, n doubles each).  variant 0: rcp_pos / sqrt_pos (the CFL reduction's: equal to
 * IEEE division and square root bit for bit, the tests check it); variant 1: rcp_pos_2ulp / sqrt_pos_2ulp (the line
 * kernel's: the same sequences without the final correction step, at most 2 ulp from the exact value).  Asynchronous on
 * the stream.  EINVAL for another variant. */
marut_status marut_debug_rcp_sqrt(const double *x, double *rcp, double *sq, long n, int variant, void *cuda_stream);

const char *marut_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MARUT_H */
