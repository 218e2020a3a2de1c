"""ctypes wrapper around oracle/marut_oracle.cpp -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_2605_26388_b200 and shares no
code with it; inputs come from the neutral `workloads` module.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "marut_oracle.cpp")
_LIB = os.path.join(_HERE, "libmarut_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c++17", "-shared", "-fPIC", _SRC, "-o", _LIB]
        subprocess.run(cmd, check=True)
    return _LIB


class _MechDesc(C.Structure):
    _fields_ = [("n_species", C.c_int), ("n_reac", C.c_int), ("T_mid", C.c_double),
                ("W", C.c_void_p), ("nasa", C.c_void_p), ("nu_r", C.c_void_p), ("nu_p", C.c_void_p),
                ("A", C.c_void_p), ("b", C.c_void_p), ("Ea", C.c_void_p)]


class _MeshDesc(C.Structure):
    _fields_ = [("dim", C.c_int), ("N", C.c_int), ("n_elem", C.c_long), ("node_xyz", C.c_void_p),
                ("n_iface", C.c_long), ("iface", C.c_void_p), ("n_mortar", C.c_long), ("mortar", C.c_void_p),
                ("n_bface", C.c_long), ("bface", C.c_void_p), ("n_bc", C.c_int), ("bc_state", C.c_void_p),
                ("physics", C.c_int), ("gamma", C.c_double), ("mu", C.c_double), ("Pr", C.c_double),
                ("mech", C.c_void_p)]


def _setup(L):
    if True:
        dp, vp = C.POINTER(C.c_double), C.c_void_p
        L.oracle_mesh_create.restype = vp
        L.oracle_mesh_create.argtypes = [vp]
        L.oracle_mesh_destroy.argtypes = [vp]
        L.oracle_nvar.argtypes = [vp]
        L.oracle_dx_min.restype = C.c_double
        L.oracle_dx_min.argtypes = [vp]
        L.oracle_max_dt.restype = C.c_double
        L.oracle_max_dt.argtypes = [vp, vp, C.c_double, vp]
        L.oracle_run.restype = C.c_double
        L.oracle_run.argtypes = [vp, vp, C.c_int, C.c_double, C.c_double, C.c_double, vp, vp]
        L.oracle_rhs.argtypes = [vp, vp, vp, C.c_double]
        L.oracle_rhs_inviscid.argtypes = [vp, vp, vp]
        L.oracle_rhs_viscous.argtypes = [vp, vp, vp]
        L.oracle_br1_gradient.argtypes = [vp, vp, vp]
        L.oracle_chem_source.argtypes = [vp, vp, vp]
        L.oracle_metrics.argtypes = [vp, vp, vp]
        L.oracle_primitives.argtypes = [vp, vp, vp]
        L.oracle_ssprk_stage.argtypes = [vp, C.c_int, C.c_double, C.c_double, vp, vp, vp]
        L.oracle_ssprk3_scalar.restype = C.c_double
        L.oracle_ssprk3_scalar.argtypes = [C.c_double] * 5
        L.oracle_operators.argtypes = [C.c_int, vp, vp, vp]
        L.oracle_mortar_matrices.argtypes = [C.c_int, vp, vp, vp, vp]
        L.oracle_rusanov.argtypes = [C.c_int, C.c_double, vp, vp, vp, vp, vp]
        L.oracle_viscous_flux.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, vp, vp, vp, vp]
        L.oracle_k_forward.restype = C.c_double
        L.oracle_k_forward.argtypes = [vp, C.c_int, C.c_double]
        L.oracle_k_equilibrium.restype = C.c_double
        L.oracle_k_equilibrium.argtypes = [vp, C.c_int, C.c_double]
        L.oracle_production_rates.argtypes = [vp, C.c_double, vp, vp]
        L.oracle_temperature.restype = C.c_double
        L.oracle_temperature.argtypes = [vp, vp, C.c_double]
        L.oracle_species_thermo.argtypes = [vp, C.c_int, C.c_double, vp]
        L.oracle_num_threads.restype = C.c_int
        L.oracle_set_explicit_source.argtypes = [vp, C.c_int]
        L.oracle_shock_indicator.argtypes = [vp, vp, C.c_double, C.c_double, C.c_double, vp, C.c_int]
        L.oracle_modal_matrix.argtypes = [C.c_int, vp]
        L.oracle_chem_implicit.restype = C.c_int
        L.oracle_chem_implicit.argtypes = [vp, vp, C.c_double]
        L.oracle_chem_implicit_node.restype = C.c_int
        L.oracle_chem_implicit_node.argtypes = [vp, vp, C.c_double, C.c_double]
        L.oracle_set_volume_form.restype = C.c_int
        L.oracle_set_volume_form.argtypes = [vp, C.c_int]
        L.oracle_ssprk54_table.argtypes = [vp, vp]
        L.oracle_ssprk54_step.argtypes = [vp, vp, C.c_double]
        L.oracle_ssprk54_scalar.restype = C.c_double
        L.oracle_ssprk54_scalar.argtypes = [C.c_double] * 5
        L.oracle_set_boundary_kinds.restype = C.c_int
        L.oracle_set_boundary_kinds.argtypes = [vp, vp, C.c_int]
        L.oracle_positivity_floor.restype = C.c_long
        L.oracle_positivity_floor.argtypes = [vp, vp, C.c_double, C.c_double]
        L.oracle_set_blend.restype = C.c_int
        L.oracle_set_blend.argtypes = [vp, vp]
        L.oracle_fv_volume.argtypes = [vp, vp, vp]
        L.oracle_subcell_normal.argtypes = [vp, C.c_long, C.c_int, vp, C.c_int, vp]
        L.oracle_logmean.restype = C.c_double
        L.oracle_logmean.argtypes = [C.c_double, C.c_double]
        L.oracle_ranocha.argtypes = [C.c_int, C.c_double, vp, vp, vp, vp]
    return L


def lib():
    global _lib
    if _lib is None:
        _lib = _setup(C.CDLL(build()))
    return _lib


_LIB_LD = os.path.join(_HERE, "libmarut_oracle_ld.so")
_lib_ld = None


class _MeshDescLD(C.Structure):
    _fields_ = [("dim", C.c_int), ("N", C.c_int), ("n_elem", C.c_long), ("node_xyz", C.c_void_p),
                ("n_iface", C.c_long), ("iface", C.c_void_p), ("n_mortar", C.c_long), ("mortar", C.c_void_p),
                ("n_bface", C.c_long), ("bface", C.c_void_p), ("n_bc", C.c_int), ("bc_state", C.c_void_p),
                ("physics", C.c_int), ("gamma", C.c_longdouble), ("mu", C.c_longdouble), ("Pr", C.c_longdouble),
                ("mech", C.c_void_p)]


def lib_ld():
    """The SAME source compiled with -DORACLE_LONG_DOUBLE: every `double` of the oracle, interface included, becomes an
    x87 80-bit long double (64-bit mantissa, unit round-off 5.4e-20).  Only oracle_mesh_create / oracle_rhs /
    oracle_mesh_destroy are bound (rhs_ld below).  It is the reference against which the round-off of the FP64 oracle and
    of the GPU path is measured at full size (reading T1): |fp64 - ld| is a side's own rounding error.  None
    when numpy's longdouble is not the 80-bit type (non-x86 hosts)."""
    global _lib_ld
    if _lib_ld is None:
        if np.finfo(np.longdouble).nmant != 63 or C.sizeof(C.c_longdouble) != np.dtype(np.longdouble).itemsize:
            return None
        if not os.path.exists(_LIB_LD) or os.path.getmtime(_LIB_LD) < os.path.getmtime(_SRC):
            cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c++17", "-shared", "-fPIC", "-DORACLE_LONG_DOUBLE", _SRC, "-o", _LIB_LD]
            subprocess.run(cmd, check=True)
        L = C.CDLL(_LIB_LD)
        L.oracle_mesh_create.restype = C.c_void_p
        L.oracle_mesh_create.argtypes = [C.c_void_p]
        L.oracle_mesh_destroy.argtypes = [C.c_void_p]
        L.oracle_rhs.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longdouble]
        _lib_ld = L
    return _lib_ld


def rhs_ld(mesh, u):
    """L(u) of the long-double build for a non-reacting mesh with the strong form, returned as float64 (the rounding
    of the long-double result to double is 1.1e-16 relative to each entry: exact for the purpose)"""
    L = lib_ld()
    assert L is not None and mesh.mech is None and not getattr(mesh, "volume_form", 0)
    ld = np.longdouble
    keep = [np.ascontiguousarray(mesh.node_xyz, dtype=ld), _i32(mesh.iface), _i32(mesh.mortar), _i32(mesh.bface),
            np.ascontiguousarray(mesh.bc_state, dtype=ld)]
    d = _MeshDescLD(mesh.dim, mesh.N, mesh.n_elem, _p(keep[0]), len(keep[1]), _p(keep[1]), len(keep[2]), _p(keep[2]),
                    len(keep[3]), _p(keep[3]), len(keep[4]), _p(keep[4]), mesh.physics, mesh.gamma, mesh.mu, mesh.Pr, None)
    h = L.oracle_mesh_create(C.addressof(d))
    try:
        ul = np.ascontiguousarray(u, dtype=ld)
        out = np.zeros_like(ul)
        L.oracle_rhs(h, _p(ul), _p(out), 0.0)
        return out.astype(np.float64)
    finally:
        L.oracle_mesh_destroy(h)


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None and a.size else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


class MechHandle:
    """keeps the numpy arrays behind an oracle_mech_desc alive"""

    def __init__(self, mech):
        self.keep = [_f64(mech.W), _f64(mech.nasa), _i32(mech.nu_r), _i32(mech.nu_p), _f64(mech.A), _f64(mech.b), _f64(mech.Ea)]
        k = self.keep
        self.desc = _MechDesc(len(k[0]), len(k[4]), float(mech.T_mid), _p(k[0]), _p(k[1]), _p(k[2]), _p(k[3]), _p(k[4]), _p(k[5]), _p(k[6]))
        self.ns = len(k[0])

    @property
    def ptr(self):
        return C.addressof(self.desc)

    def k_forward(self, r, T):
        return lib().oracle_k_forward(self.ptr, r, T)

    def k_equilibrium(self, r, T):
        return lib().oracle_k_equilibrium(self.ptr, r, T)

    def production_rates(self, T, rho_s):
        rho_s = _f64(rho_s)
        om = np.zeros(self.ns)
        lib().oracle_production_rates(self.ptr, T, _p(rho_s), _p(om))
        return om

    def temperature(self, rho_s, e_int):
        rho_s = _f64(rho_s)
        return lib().oracle_temperature(self.ptr, _p(rho_s), e_int)

    def implicit_step(self, rho_s, e_int, dt):
        """backward-Euler Newton source step of one node: returns (rho_s after dt, sweeps)"""
        y = _f64(rho_s).copy()
        it = lib().oracle_chem_implicit_node(self.ptr, _p(y), float(e_int), float(dt))
        return y, it

    def species_thermo(self, s, T):
        out = np.zeros(5)
        lib().oracle_species_thermo(self.ptr, s, T, _p(out))
        return dict(cp_R=out[0], h_RT=out[1], s_R=out[2], e=out[3], cv=out[4])


class OracleMesh:
    def __init__(self, mesh, L=None):
        L = L or lib()
        self.L = L
        self.mesh = mesh
        self._keep = [_f64(mesh.node_xyz), _i32(mesh.iface), _i32(mesh.mortar), _i32(mesh.bface), _f64(mesh.bc_state)]
        k = self._keep
        self._mech = MechHandle(mesh.mech) if mesh.mech is not None else None
        d = _MeshDesc(mesh.dim, mesh.N, mesh.n_elem, _p(k[0]), len(k[1]), _p(k[1]), len(k[2]), _p(k[2]),
                      len(k[3]), _p(k[3]), len(k[4]), _p(k[4]), mesh.physics, mesh.gamma, mesh.mu, mesh.Pr,
                      self._mech.ptr if self._mech else None)
        self.h = L.oracle_mesh_create(C.addressof(d))
        self.nvar = L.oracle_nvar(self.h)
        self.shape = (mesh.n_elem, self.nvar, mesh.nn)
        if getattr(mesh, "volume_form", 0):
            if L.oracle_set_volume_form(self.h, int(mesh.volume_form)) != 0:
                raise ValueError("unsupported volume_form for this physics")

    def __del__(self):
        if getattr(self, "h", None) and getattr(self, "L", None) is not None:
            self.L.oracle_mesh_destroy(self.h)
            self.h = None

    @property
    def dx_min(self):
        return self.L.oracle_dx_min(self.h)

    def metrics(self):
        m = self.mesh
        Ja = np.zeros((m.n_elem, m.nn, m.dim, m.dim))
        J = np.zeros((m.n_elem, m.nn))
        self.L.oracle_metrics(self.h, _p(Ja), _p(J))
        return Ja, J

    def _call(self, fn, u, *extra):
        u = _f64(u)
        out = np.zeros(self.shape)
        fn(self.h, _p(u), _p(out), *extra)
        return out

    def rhs(self, u, t=0.0):
        return self._call(self.L.oracle_rhs, u, t)

    def rhs_inviscid(self, u):
        return self._call(self.L.oracle_rhs_inviscid, u)

    def rhs_viscous(self, u):
        return self._call(self.L.oracle_rhs_viscous, u)

    def chem_source(self, u):
        return self._call(self.L.oracle_chem_source, u)

    def shock_indicator(self, u, s=9.21024, alpha_min=0.001, alpha_max=0.5, smooth=True):
        """Hennemann-Gassner blending coefficient alpha_e per element (with face-neighbour maximum if smooth)"""
        u = _f64(u)
        a = np.zeros(self.mesh.n_elem)
        self.L.oracle_shock_indicator(self.h, _p(u), s, alpha_min, alpha_max, _p(a), int(smooth))
        return a

    def ssprk54_step(self, u, dt):
        """O19: one SSP-RK54 step (eq. 45 with the Spiteri-Ruuth table); returns the new state"""
        v = _f64(u).copy()
        self.L.oracle_ssprk54_step(self.h, _p(v), float(dt))
        return v

    def set_boundary_kinds(self, kinds):
        """O8b: per bc id 0 = prescribed exterior state, 1 = outflow (interior state), 2 = inviscid slip wall"""
        if kinds is None:
            self.L.oracle_set_boundary_kinds(self.h, None, 0)
            return
        k = np.ascontiguousarray(kinds, dtype=np.int32)
        assert k.shape == (self.mesh.bc_state.shape[0],)
        if self.L.oracle_set_boundary_kinds(self.h, k.ctypes.data_as(C.c_void_p), len(k)) != 0:
            raise ValueError("boundary kinds: Euler meshes, values 0..2")

    def positivity_floor(self, u, rho_min=1e-6, p_min=5e-7):
        """O18 (reading R17): returns (floored copy of u, number of nodes changed)"""
        v = _f64(u).copy()
        n = self.L.oracle_positivity_floor(self.h, _p(v), rho_min, p_min)
        if n < 0:
            raise ValueError("the positivity floor is defined for the ideal-gas systems only")
        return v, int(n)

    def set_blend(self, alpha):
        """eq. 11 / 42: per-element blending coefficients alpha_e (copied) of the DG / sub-cell FV volume residual;
        None switches the blending off"""
        if alpha is None:
            self.L.oracle_set_blend(self.h, None)
            return
        a = _f64(alpha)
        assert a.shape == (self.mesh.n_elem,)
        if self.L.oracle_set_blend(self.h, _p(a)) != 0:
            raise ValueError("blending is defined for the Euler equations only")

    def fv_volume(self, u):
        """O17: the first-order sub-cell finite-volume VOLUME residual R^FV (no surface lift), [e][v][node]"""
        u = _f64(u)
        r = np.empty_like(u)
        self.L.oracle_fv_volume(self.h, _p(u), _p(r))
        return r

    def subcell_normal(self, e, l, ijk, mi):
        """O17: sub-cell normal nhat^l_{mi+1/2} on the line through node ijk along direction l"""
        q = np.ascontiguousarray(list(ijk) + [0] * (3 - len(ijk)), dtype=np.int32)
        nh = np.zeros(3)
        self.L.oracle_subcell_normal(self.h, int(e), int(l), q.ctypes.data_as(C.c_void_p), int(mi), _p(nh))
        return nh[: self.mesh.dim]

    def set_explicit_source(self, on):
        """reacting meshes: whether L(U) includes the chemistry source (default) or is the transport operator only"""
        self.L.oracle_set_explicit_source(self.h, int(bool(on)))

    def strang_step(self, u, dt):
        """eq. 24: S_{dt/2} o T_dt o S_{dt/2} with T = one SSP-RK33 step of the transport operator"""
        self.set_explicit_source(False)
        try:
            u, _ = self.chem_implicit(u, 0.5 * dt)
            u = self.run(u, 1, cfl=0.0, dt=dt)[0]   # cfl = 0: fixed dt
            u, _ = self.chem_implicit(u, 0.5 * dt)
        finally:
            self.set_explicit_source(True)
        return u

    def chem_implicit(self, u, dt):
        """implicit source substep on every node (a copy of u is advanced); returns (u, worst sweep count)"""
        u = _f64(u).copy()
        it = self.L.oracle_chem_implicit(self.h, _p(u), float(dt))
        if it < 0:
            raise ValueError("chem_implicit needs a REACTING_EULER mesh")
        return u, it

    def br1_gradient(self, u):
        m = self.mesh
        u = _f64(u)
        S = np.zeros((m.n_elem, m.nn, m.dim + 2, m.dim))
        self.L.oracle_br1_gradient(self.h, _p(u), _p(S))
        return S

    def primitives(self, U):
        U = _f64(U)
        out = np.zeros(7)
        self.L.oracle_primitives(self.h, _p(U), _p(out))
        return dict(rho=out[0], p=out[1], a=out[2], T=out[3], vel=out[4:7].copy())

    def ssprk_stage(self, stage, dt, t_n, u_n, u_in):
        u_n, u_in = _f64(u_n), _f64(u_in)
        out = np.zeros(self.shape)
        self.L.oracle_ssprk_stage(self.h, stage, dt, t_n, _p(u_n), _p(u_in), _p(out))
        return out

    def max_dt(self, u, cfl, return_lambda=False):
        u = _f64(u)
        lam = C.c_double(0.0)
        dt = self.L.oracle_max_dt(self.h, _p(u), cfl, C.addressof(lam))
        return (dt, lam.value) if return_lambda else dt

    def run(self, u, nsteps, cfl=0.5, dt=0.0, t0=0.0):
        """advance a copy of u by nsteps SSPRK3 steps, dt from the CFL reduction each step if cfl > 0, else the fixed dt;
        returns (u, t_end, min_rho, min_p)"""
        u = _f64(u).copy()
        mr, mp = C.c_double(0.0), C.c_double(0.0)
        t = self.L.oracle_run(self.h, _p(u), nsteps, cfl, dt, t0, C.addressof(mr), C.addressof(mp))
        return u, t, mr.value, mp.value


def operators(N):
    n = N + 1
    x, w, D = np.zeros(n), np.zeros(n), np.zeros((n, n))
    lib().oracle_operators(N, _p(x), _p(w), _p(D))
    return x, w, D


def mortar_matrices(N):
    n = N + 1
    M = [np.zeros((n, n)) for _ in range(4)]
    lib().oracle_mortar_matrices(N, *[_p(a) for a in M])
    return M  # Pf_lo, Pf_up, Pr_lo, Pr_up


def ssprk54_table():
    a, b = np.zeros((5, 5)), np.zeros((5, 5))
    lib().oracle_ssprk54_table(_p(a), _p(b))
    return a, b


def ssprk54_scalar(y0, lam, c2, t0, dt):
    return lib().oracle_ssprk54_scalar(y0, lam, c2, t0, dt)


def rusanov(dim, gamma, Um, Up, nv):
    Um, Up, nv = _f64(Um), _f64(Up), _f64(nv)
    Fs = np.zeros(dim + 2)
    lam = C.c_double(0.0)
    lib().oracle_rusanov(dim, gamma, _p(Um), _p(Up), _p(nv), _p(Fs), C.addressof(lam))
    return Fs, lam.value


def viscous_flux(dim, gamma, mu, Pr, U, S, nv):
    U, S, nv = _f64(U), _f64(S), _f64(nv)
    F = np.zeros(dim + 2)
    lib().oracle_viscous_flux(dim, gamma, mu, Pr, _p(U), _p(S), _p(nv), _p(F))
    return F


def modal_matrix(N):
    """V^-1 of the orthonormal Legendre basis on the LGL nodes: nodal values -> modal coefficients"""
    V = np.zeros((N + 1, N + 1))
    lib().oracle_modal_matrix(N, _p(V))
    return V


def logmean(aL, aR):
    return lib().oracle_logmean(float(aL), float(aR))


def ranocha(dim, gamma, UL, UR, nv):
    UL, UR, nv = _f64(UL), _f64(UR), _f64(nv)
    F = np.zeros(dim + 2)
    lib().oracle_ranocha(dim, gamma, _p(UL), _p(UR), _p(nv), _p(F))
    return F


def ssprk3_scalar(y0, lam, c2, t0, dt):
    return lib().oracle_ssprk3_scalar(y0, lam, c2, t0, dt)


def num_threads():
    return lib().oracle_num_threads()


def set_num_threads(n):
    lib().oracle_set_num_threads(int(n))
