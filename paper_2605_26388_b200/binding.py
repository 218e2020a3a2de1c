"""ctypes binding of include/marut.h.  Same names as the C entry points; marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

EULER, NAVIER_STOKES, REACTING_EULER = 0, 1, 2
_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libmarut.so")
_lib = None

_STATUS = {0: "MARUT_OK", 1: "MARUT_EINVAL", 2: "MARUT_ENOMEM", 3: "MARUT_ECUDA", 4: "MARUT_ETOPOLOGY", 5: "MARUT_ENOTFINITE"}

# every symbol include/marut.h declares
SYMBOLS = ["marut_mesh_create", "marut_mesh_destroy", "marut_rhs", "marut_ssprk_stage", "marut_max_dt", "marut_max_dt_async", "marut_ssprk_stage_dev", "marut_rk_stage_dev",
           "marut_chem_source", "marut_chem_implicit", "marut_shock_indicator", "marut_rk_stage", "marut_lincomb", "marut_set_blend", "marut_set_boundary_kinds", "marut_positivity_floor", "marut_set_explicit_source", "marut_set_volume_form", "marut_get_metrics", "marut_is_affine", "marut_dx_min", "marut_launch_count", "marut_debug_rcp_sqrt", "marut_debug_stage_kernel", "marut_ssprk33_step", "marut_ssprk33_step_cfl", "marut_ssprk54_step", "marut_strang_step",
           "marut_shock_indicator_noalloc", "marut_noalloc_max_elements", "marut_ssprk33_step_dt", "marut_last_error"]


class MarutError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class _Mech(C.Structure):
    _fields_ = [("n_species", C.c_int), ("n_reac", C.c_int), ("T_mid", C.c_double), ("W", C.c_void_p),
                ("nasa", C.c_void_p), ("nu_r", C.c_void_p), ("nu_p", C.c_void_p), ("A", C.c_void_p),
                ("b", C.c_void_p), ("Ea", C.c_void_p)]


class _Desc(C.Structure):
    _fields_ = [("dim", C.c_int), ("N", C.c_int), ("n_elem", C.c_long), ("node_xyz", C.c_void_p),
                ("n_iface", C.c_long), ("iface", C.c_void_p), ("n_mortar", C.c_long), ("mortar", C.c_void_p),
                ("n_bface", C.c_long), ("bface", C.c_void_p), ("n_bc", C.c_int), ("bc_state", C.c_void_p),
                ("physics", C.c_int), ("gamma", C.c_double), ("mu", C.c_double), ("Pr", C.c_double),
                ("mech", C.c_void_p)]


def lib_path() -> str:
    return _LIB_PATH


def lib():
    """load libmarut.so; fails loudly when it has not been built (no fallback of any kind)"""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2605_26388_b200.build` (needs nvcc); "
                              "this package has no CPU or PyTorch fallback")
        L = C.CDLL(_LIB_PATH)
        vp, dbl = C.c_void_p, C.c_double
        L.marut_mesh_create.restype = C.c_int
        L.marut_mesh_create.argtypes = [vp, C.POINTER(vp)]
        L.marut_mesh_destroy.restype = None
        L.marut_mesh_destroy.argtypes = [vp]
        L.marut_rhs.restype = C.c_int
        L.marut_rhs.argtypes = [vp, vp, vp, dbl, vp]
        L.marut_ssprk_stage.restype = C.c_int
        L.marut_ssprk_stage.argtypes = [vp, C.c_int, dbl, dbl, vp, vp, vp, vp]
        L.marut_max_dt.restype = C.c_int
        L.marut_max_dt.argtypes = [vp, vp, dbl, C.POINTER(dbl), vp]
        L.marut_max_dt_async.restype = C.c_int
        L.marut_max_dt_async.argtypes = [vp, vp, dbl, vp, vp]
        L.marut_ssprk_stage_dev.restype = C.c_int
        L.marut_ssprk_stage_dev.argtypes = [vp, C.c_int, vp, dbl, vp, vp, vp, vp]
        L.marut_chem_source.restype = C.c_int
        L.marut_chem_source.argtypes = [vp, vp, vp, vp]
        L.marut_chem_implicit.restype = C.c_int
        L.marut_chem_implicit.argtypes = [vp, vp, dbl, C.POINTER(C.c_int), vp]
        L.marut_shock_indicator.restype = C.c_int
        L.marut_shock_indicator.argtypes = [vp, vp, dbl, dbl, dbl, C.c_int, vp, vp]
        L.marut_shock_indicator_noalloc.restype = C.c_int
        L.marut_shock_indicator_noalloc.argtypes = [vp, vp, dbl, dbl, dbl, C.c_int, vp, vp]
        L.marut_noalloc_max_elements.restype = C.c_long
        L.marut_noalloc_max_elements.argtypes = []
        L.marut_rk_stage_dev.restype = C.c_int
        L.marut_rk_stage_dev.argtypes = [vp, dbl, dbl, dbl, vp, vp, vp, vp, vp]
        L.marut_rk_stage.restype = C.c_int
        L.marut_rk_stage.argtypes = [vp, dbl, dbl, dbl, vp, vp, vp, vp]
        L.marut_lincomb.restype = C.c_int
        L.marut_lincomb.argtypes = [vp, C.c_int, vp, vp, vp, vp]
        L.marut_set_boundary_kinds.restype = C.c_int
        L.marut_set_boundary_kinds.argtypes = [vp, vp, C.c_int]
        L.marut_positivity_floor.restype = C.c_int
        L.marut_positivity_floor.argtypes = [vp, vp, dbl, dbl, vp, vp]
        L.marut_set_blend.restype = C.c_int
        L.marut_set_blend.argtypes = [vp, vp]
        L.marut_set_explicit_source.restype = C.c_int
        L.marut_set_explicit_source.argtypes = [vp, C.c_int]
        L.marut_set_volume_form.restype = C.c_int
        L.marut_set_volume_form.argtypes = [vp, C.c_int]
        L.marut_get_metrics.restype = C.c_int
        L.marut_get_metrics.argtypes = [vp, vp, vp]
        L.marut_is_affine.restype = C.c_int
        L.marut_is_affine.argtypes = [vp]
        L.marut_dx_min.restype = dbl
        L.marut_dx_min.argtypes = [vp]
        L.marut_launch_count.restype = C.c_long
        L.marut_launch_count.argtypes = [vp]
        L.marut_ssprk33_step.restype = C.c_int
        L.marut_ssprk33_step.argtypes = [vp, vp, vp, dbl, vp, vp]
        L.marut_ssprk33_step_cfl.restype = C.c_int
        L.marut_ssprk33_step_cfl.argtypes = [vp, vp, vp, dbl, vp, vp, vp]
        L.marut_ssprk33_step_dt.restype = C.c_int
        L.marut_ssprk33_step_dt.argtypes = [vp, vp, vp, dbl, vp, vp]
        L.marut_ssprk54_step.restype = C.c_int
        L.marut_ssprk54_step.argtypes = [vp, vp, vp, dbl, vp, vp]
        L.marut_strang_step.restype = C.c_int
        L.marut_strang_step.argtypes = [vp, vp, vp, dbl, vp, vp]
        L.marut_debug_stage_kernel.restype = C.c_int
        L.marut_debug_stage_kernel.argtypes = [vp, C.c_int]
        L.marut_debug_rcp_sqrt.restype = C.c_int
        L.marut_debug_rcp_sqrt.argtypes = [vp, vp, vp, C.c_long, C.c_int, vp]
        L.marut_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(status):
    if status != 0:
        raise MarutError(status, lib().marut_last_error().decode())


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None and a.size else None


def _dev(t):
    """device pointer of a CUDA float64 torch tensor (contiguous)"""
    if t is None:
        return None
    if not (t.is_cuda and t.is_contiguous() and t.dtype.is_floating_point and t.element_size() == 8):
        raise TypeError("expected a contiguous float64 CUDA tensor")
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        import torch

        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(stream if isinstance(stream, int) else stream.cuda_stream)


# ------------------------------------------------------------------ the C entry points, same names
def marut_mesh_create(mesh):
    """mesh: any object with the fields of marut_mesh_desc as numpy arrays (e.g. workloads.Mesh). Returns a handle."""
    keep = [_np(mesh.node_xyz, np.float64), _np(mesh.iface, np.int32), _np(mesh.mortar, np.int32),
            _np(mesh.bface, np.int32), _np(mesh.bc_state, np.float64)]
    mech_ptr = None
    if getattr(mesh, "mech", None) is not None:
        k = mesh.mech
        mk = [_np(k.W, np.float64), _np(k.nasa, np.float64), _np(k.nu_r, np.int32), _np(k.nu_p, np.int32),
              _np(k.A, np.float64), _np(k.b, np.float64), _np(k.Ea, np.float64)]
        md = _Mech(len(mk[0]), len(mk[4]), float(k.T_mid), *[_ptr(a) for a in mk])
        keep += mk + [md]
        mech_ptr = C.addressof(md)
    n_bc = keep[4].shape[0] if keep[4].ndim == 2 else 0
    d = _Desc(mesh.dim, mesh.N, keep[0].shape[0], _ptr(keep[0]), len(keep[1]), _ptr(keep[1]), len(keep[2]), _ptr(keep[2]),
              len(keep[3]), _ptr(keep[3]), n_bc, _ptr(keep[4]), mesh.physics, mesh.gamma, mesh.mu, mesh.Pr, mech_ptr)
    h = C.c_void_p()
    _check(lib().marut_mesh_create(C.addressof(d), C.byref(h)))
    return h


def marut_mesh_destroy(h):
    lib().marut_mesh_destroy(h)


def marut_rhs(h, u, du, t=0.0, stream=None):
    _check(lib().marut_rhs(h, _dev(u), _dev(du), t, _stream(stream)))


def marut_ssprk_stage(h, stage, dt, t_n, u_n, u_in, u_out, stream=None):
    _check(lib().marut_ssprk_stage(h, stage, dt, t_n, _dev(u_n), _dev(u_in), _dev(u_out), _stream(stream)))


def marut_max_dt(h, u, cfl, stream=None):
    dt = C.c_double(0.0)
    _check(lib().marut_max_dt(h, _dev(u), cfl, C.byref(dt), _stream(stream)))
    return dt.value


def marut_max_dt_async(h, u, cfl, dt_dev, stream=None):
    _check(lib().marut_max_dt_async(h, _dev(u), cfl, _dev(dt_dev), _stream(stream)))


def marut_ssprk_stage_dev(h, stage, dt_dev, t_n, u_n, u_in, u_out, stream=None):
    _check(lib().marut_ssprk_stage_dev(h, stage, _dev(dt_dev), t_n, _dev(u_n), _dev(u_in), _dev(u_out), _stream(stream)))


def marut_chem_source(h, u, s, stream=None):
    _check(lib().marut_chem_source(h, _dev(u), _dev(s), _stream(stream)))


def marut_chem_implicit(h, u, dt, stream=None, want_sweeps=True):
    sw = C.c_int(0)
    _check(lib().marut_chem_implicit(h, _dev(u), dt, C.byref(sw) if want_sweeps else None, _stream(stream)))
    return sw.value


def marut_set_volume_form(h, form):
    _check(lib().marut_set_volume_form(h, int(form)))


def ssprk3_step(h, u, ua, ub, dt, t=0.0, stream=None):
    """one SSP-RK33 step = three marut_ssprk_stage calls; u is overwritten with u^{n+1}. ua, ub: scratch."""
    marut_ssprk_stage(h, 0, dt, t, u, u, ua, stream)
    marut_ssprk_stage(h, 1, dt, t, u, ua, ub, stream)
    marut_ssprk_stage(h, 2, dt, t, u, ub, u, stream)


def marut_rk_stage(h, a, b, c_dt, u_a, u_in, u_out, stream=None):
    _check(lib().marut_rk_stage(h, a, b, c_dt, _dev(u_a), _dev(u_in), _dev(u_out), _stream(stream)))


def marut_rk_stage_dev(h, a, b, c, dt_dev, u_a, u_in, u_out, stream=None):
    _check(lib().marut_rk_stage_dev(h, a, b, c, _dev(dt_dev), _dev(u_a), _dev(u_in), _dev(u_out), _stream(stream)))


def marut_lincomb(h, coef, us, out, stream=None):
    n = len(us)
    cf = (C.c_double * n)(*[float(x) for x in coef])
    ptrs = (C.c_void_p * n)(*[_dev(t).value for t in us])
    _check(lib().marut_lincomb(h, n, cf, ptrs, _dev(out), _stream(stream)))


def _bufs(ts):
    return (C.c_void_p * len(ts))(*[_dev(t).value for t in ts])


def ssprk54_step(h, u, ua, ub, uc, dt, stream=None):
    """one SSP-RK54 step (marut_ssprk54_step), u advanced in place; ua, ub, uc: scratch"""
    _check(lib().marut_ssprk54_step(h, _dev(u), _bufs((ua, ub, uc)), float(dt), None, _stream(stream)))


def ssprk54_step_dev(h, u, ua, ub, uc, dt_dev, stream=None):
    """ssprk54_step with the time step in device memory (marut_max_dt_async): nothing here waits for the GPU"""
    _check(lib().marut_ssprk54_step(h, _dev(u), _bufs((ua, ub, uc)), 0.0, _dev(dt_dev), _stream(stream)))


def marut_ssprk33_step_cfl(h, u, ua, ub, cfl, dt_in, dt_out, stream=None):
    _check(lib().marut_ssprk33_step_cfl(h, _dev(u), _bufs((ua, ub)), float(cfl), _dev(dt_in), _dev(dt_out), _stream(stream)))


def marut_ssprk33_step_dt(h, u, ua, ub, cfl, dt_out, stream=None):
    """one SSP-RK33 step with its own CFL time step (formed on the device from u, left in dt_out) = marut_ssprk33_step_dt"""
    _check(lib().marut_ssprk33_step_dt(h, _dev(u), _bufs((ua, ub)), float(cfl), _dev(dt_out), _stream(stream)))


def marut_ssprk33_step(h, u, ua, ub, dt=0.0, dt_dev=None, stream=None):
    _check(lib().marut_ssprk33_step(h, _dev(u), _bufs((ua, ub)), float(dt), None if dt_dev is None else _dev(dt_dev), _stream(stream)))


def marut_shock_indicator(h, u, alpha, s=9.21024, alpha_min=0.001, alpha_max=0.5, smooth=True, stream=None):
    _check(lib().marut_shock_indicator(h, _dev(u), s, alpha_min, alpha_max, int(bool(smooth)), _dev(alpha), _stream(stream)))


def marut_shock_indicator_noalloc(h, u, alpha, s=9.21024, alpha_min=0.001, alpha_max=0.5, smooth=True, stream=None):
    """marut_shock_indicator with its scratch in a fixed device array of the library: no allocation, n_elem <= 2^20"""
    _check(lib().marut_shock_indicator_noalloc(h, _dev(u), s, alpha_min, alpha_max, int(bool(smooth)), _dev(alpha), _stream(stream)))


def marut_noalloc_max_elements():
    return int(lib().marut_noalloc_max_elements())


def marut_set_boundary_kinds(h, kinds):
    """kinds: one of 0 (prescribed state) / 1 (outflow) / 2 (slip wall) per boundary id (host integers)"""
    k = np.ascontiguousarray(kinds, dtype=np.int32)
    _check(lib().marut_set_boundary_kinds(h, k.ctypes.data_as(C.c_void_p), int(k.size)))


def marut_positivity_floor(h, u, rho_min=1e-6, p_min=5e-7, stream=None, want_count=False):
    """in place on u; returns the number of nodes changed if want_count (synchronises), else None"""
    n = C.c_long(0)
    _check(lib().marut_positivity_floor(h, _dev(u), rho_min, p_min, C.byref(n) if want_count else None, _stream(stream)))
    return n.value if want_count else None


def marut_set_blend(h, alpha):
    """alpha: CUDA tensor [n_elem] (kept by the library, not copied -- keep it alive) or None"""
    _check(lib().marut_set_blend(h, None if alpha is None else _dev(alpha)))


def marut_debug_rcp_sqrt(x, rcp, sq, variant=0, stream=None):
    _check(lib().marut_debug_rcp_sqrt(_dev(x), _dev(rcp), _dev(sq), x.numel(), int(variant), _stream(stream)))


def marut_set_explicit_source(h, on):
    _check(lib().marut_set_explicit_source(h, int(bool(on))))


def strang_step(h, u, ua, ub, dt, t=0.0, stream=None, want_sweeps=False):
    """U^{n+1} = S_{dt/2} o T_dt o S_{dt/2} (U^n) (eq. 24) = marut_strang_step; u is overwritten; ua, ub:
    scratch.  Returns the larger Newton sweep count of the two implicit substeps if want_sweeps (synchronises)."""
    n = C.c_int(0)
    _check(lib().marut_strang_step(h, _dev(u), _bufs((ua, ub)), float(dt), C.byref(n) if want_sweeps else None, _stream(stream)))
    return n.value if want_sweeps else None


class MarutMesh:
    """RAII wrapper around the opaque marut_mesh handle."""

    def __init__(self, mesh):
        self.h = marut_mesh_create(mesh)
        self.mesh = mesh
        ns = mesh.mech.ns if mesh.physics == REACTING_EULER else 1
        self.shape = (mesh.node_xyz.shape[0], ns + mesh.dim + 1, (mesh.N + 1) ** mesh.dim)
        if getattr(mesh, "volume_form", 0):
            marut_set_volume_form(self.h, mesh.volume_form)

    def close(self):
        if getattr(self, "h", None):
            marut_mesh_destroy(self.h)
            self.h = None

    __del__ = close

    def rhs(self, u, du, t=0.0, stream=None):
        marut_rhs(self.h, u, du, t, stream)

    def stage(self, stage, dt, t_n, u_n, u_in, u_out, stream=None):
        marut_ssprk_stage(self.h, stage, dt, t_n, u_n, u_in, u_out, stream)

    def max_dt(self, u, cfl, stream=None):
        return marut_max_dt(self.h, u, cfl, stream)

    def max_dt_async(self, u, cfl, dt_dev, stream=None):
        marut_max_dt_async(self.h, u, cfl, dt_dev, stream)

    def stage_dev(self, stage, dt_dev, t_n, u_n, u_in, u_out, stream=None):
        marut_ssprk_stage_dev(self.h, stage, dt_dev, t_n, u_n, u_in, u_out, stream)

    def chem_source(self, u, s, stream=None):
        marut_chem_source(self.h, u, s, stream)

    def chem_implicit(self, u, dt, stream=None, want_sweeps=True):
        return marut_chem_implicit(self.h, u, dt, stream, want_sweeps)

    def shock_indicator(self, u, alpha, **kw):
        marut_shock_indicator(self.h, u, alpha, **kw)

    def positivity_floor(self, u, rho_min=1e-6, p_min=5e-7, stream=None, want_count=False):
        return marut_positivity_floor(self.h, u, rho_min, p_min, stream, want_count)

    def set_boundary_kinds(self, kinds):
        marut_set_boundary_kinds(self.h, kinds)

    def rk_stage(self, a, b, c_dt, u_a, u_in, u_out, stream=None):
        marut_rk_stage(self.h, a, b, c_dt, u_a, u_in, u_out, stream)

    def lincomb(self, coef, us, out, stream=None):
        marut_lincomb(self.h, coef, us, out, stream)

    def ssprk54_step(self, u, ua, ub, uc, dt, stream=None):
        ssprk54_step(self.h, u, ua, ub, uc, dt, stream)

    def rk_stage_dev(self, a, b, c, dt_dev, u_a, u_in, u_out, stream=None):
        marut_rk_stage_dev(self.h, a, b, c, dt_dev, u_a, u_in, u_out, stream)

    def ssprk54_step_dev(self, u, ua, ub, uc, dt_dev, stream=None):
        ssprk54_step_dev(self.h, u, ua, ub, uc, dt_dev, stream)

    def set_blend(self, alpha):
        self._alpha = alpha          # the library keeps the pointer: hold the tensor
        marut_set_blend(self.h, alpha)

    def strang_step(self, u, ua, ub, dt, t=0.0, stream=None, want_sweeps=False):
        return strang_step(self.h, u, ua, ub, dt, t, stream, want_sweeps)

    def ssprk33_step_cfl(self, u, ua, ub, cfl, dt_in, dt_out, stream=None):
        marut_ssprk33_step_cfl(self.h, u, ua, ub, cfl, dt_in, dt_out, stream)

    def ssprk33_step_dt(self, u, ua, ub, cfl, dt_out, stream=None):
        marut_ssprk33_step_dt(self.h, u, ua, ub, cfl, dt_out, stream)

    def ssprk33_step(self, u, ua, ub, dt=0.0, dt_dev=None, stream=None):
        marut_ssprk33_step(self.h, u, ua, ub, dt, dt_dev, stream)

    def step(self, u, ua, ub, dt, t=0.0, stream=None):
        ssprk3_step(self.h, u, ua, ub, dt, t, stream)

    def metrics(self):
        m = self.mesh
        ne, nn, d = self.shape[0], self.shape[2], m.dim
        Ja, J = np.zeros((ne, nn, d, d)), np.zeros((ne, nn))
        _check(lib().marut_get_metrics(self.h, _ptr(Ja), _ptr(J)))
        return Ja, J

    @property
    def is_affine(self):
        return bool(lib().marut_is_affine(self.h))

    @property
    def dx_min(self):
        return lib().marut_dx_min(self.h)

    def debug_stage_kernel(self, which):
        _check(lib().marut_debug_stage_kernel(self.h, which))

    @property
    def launch_count(self):
        return lib().marut_launch_count(self.h)
