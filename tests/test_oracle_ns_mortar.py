"""Pins of the BR1 viscous terms across 2-D 2:1 mortars and 3-D 4:1 mortars (oracle O9c, O9d; "Non-conforming faces use the same
forward and reverse projections as the hyperbolic side", "interface, mortar, and boundary kernels"; DESIGN.md
reading R23).  Pinned against what the mathematics fixes: the closed-form gradient and viscous residual of a smooth
field (spectral accuracy kept at the elements that touch a mortar), free-stream preservation, and conservation of the
viscous residual to round-off.  Each check also runs on the mutant of tests/mutation_util.py that makes the mistake it is
meant to catch and must fail there."""
import math

import numpy as np
import pytest

import oracle
import workloads as wl
from mutation_util import mutant

G, MU, PR = 1.4, 0.05, 0.72


def _ns(m):
    m.physics, m.mu, m.Pr = wl.NAVIER_STOKES, MU, PR
    return m


def _wave(m):
    """W = (rho, v1, v2, T) = W0 + amp sin(phi), phi = g.x, on [0,4] x [0,1] (periodic in y).  Returns U, the closed-form
    viscous residual div F_v (eq. 15 with q = -k grad T, k = gamma mu / (Pr (gamma-1)), R = 1) and grad W [e][node][w][c]."""
    x, y = m.node_xyz[:, 0, :], m.node_xyz[:, 1, :]
    g = np.array([2 * math.pi / 4.0, 2 * math.pi])
    A, c, C, D = np.array([0.3, -0.2]), np.array([0.5, 0.4]), 0.15, 0.2
    ph = g[0] * x + g[1] * y
    s, co = np.sin(ph), np.cos(ph)
    rho, T = 1.0 + D * s, 1.2 + C * s
    v = [c[i] + A[i] * s for i in range(2)]
    E = rho * T / (G - 1) + 0.5 * rho * (v[0] ** 2 + v[1] ** 2)
    u = np.stack([rho, rho * v[0], rho * v[1], E], axis=1)
    # tau = mu M cos(phi), M = A g^T + g A^T - 2/3 (A.g) I;  div tau = -mu M g sin(phi)
    M = np.outer(A, g) + np.outer(g, A) - (2.0 / 3.0) * np.eye(2) * (A @ g)
    Mg = M @ g
    k = G * MU / (PR * (G - 1))
    du = np.zeros_like(u)
    for i in range(2):
        du[:, 1 + i] = -MU * Mg[i] * s
    # div(tau v + k grad T) = grad v : tau + v . div tau + k lap T
    du[:, 3] = MU * (np.outer(A, g) * M).sum() * co ** 2 - MU * (v[0] * Mg[0] + v[1] * Mg[1]) * s - k * C * (g @ g) * s
    amp = np.array([D, A[0], A[1], C])
    S = amp[None, None, :, None] * g[None, None, None, :] * co[:, :, None, None]
    return np.ascontiguousarray(u), du, S


def _quadtree(N):
    m = _ns(wl.quadtree_mesh(N, base=(32, 8), band=0.15, jitter=0.3))
    m.bc_state = np.stack([np.array([1.0, 0.5, 0.4, 3.2])] * 2)
    return m


def mortar_errors(L, N):
    """relative nodal errors (gradient, viscous residual) at the elements that touch a mortar, and the same two on the
    conforming mesh of the coarsest element size.  x boundaries: outflow (one-sided trace, no jump), their elements are
    kept out of the measurement."""
    m = _quadtree(N)
    om = oracle.OracleMesh(m, L)
    om.set_boundary_kinds([1, 1])
    u, du, Sx = _wave(m)
    touch = np.setdiff1d(np.unique(np.asarray(m.mortar)[:, [0, 2, 3]]), np.asarray(m.bface)[:, 0])
    assert len(touch) > 400
    eS = np.abs(om.br1_gradient(u)[touch] - Sx[touch]).max() / np.abs(Sx).max()
    eR = np.abs(om.rhs_viscous(u)[touch] - du[touch]).max() / np.abs(du).max()
    mc = _ns(wl.cartesian_mesh(2, N, (32, 8), (0.0, 0.0), (4.0, 1.0)))
    uc, duc, Sc = _wave(mc)
    oc = oracle.OracleMesh(mc, L)
    cS = np.abs(oc.br1_gradient(uc) - Sc).max() / np.abs(Sc).max()
    cR = np.abs(oc.rhs_viscous(uc) - duc).max() / np.abs(duc).max()
    return eS, eR, cS, cR


def test_br1_across_mortars_keeps_the_accuracy_of_the_conforming_mesh():
    err = {}
    for N in (2, 3, 5):
        eS, eR, cS, cR = err[N] = mortar_errors(None, N)
        assert eS < 1.5 * cS, (N, eS, cS)                 # 1.0x: the coarse elements carry the largest error
        assert eR < 10.0 * cR, (N, eR, cR)                # 1.3x, 4.3x, 4.3x
    # spectral: gradient 5.1e-2, 4.0e-3, 9.8e-6; residual 0.42, 6.8e-2, 5.4e-4
    assert err[3][0] < err[2][0] / 8 and err[5][0] < err[3][0] / 200
    assert err[3][1] < err[2][1] / 4 and err[5][1] < err[3][1] / 50
    # wrong half of the coarse face in the gradient's trace: O(1) off in the gradient (and so in the residual)
    eS, eR, cS, cR = mortar_errors(mutant("br1_mortar_wrong_half"), 3)
    assert eS > 20 * err[3][0] and eR > 20 * err[3][1]
    # wrong half for the interpolated coarse GRADIENT in the flux: the gradient is untouched, the residual is off
    eS, eR, cS, cR = mortar_errors(mutant("viscous_mortar_gradient_wrong_half"), 3)
    assert eS == err[3][0] and eR > 20 * err[3][1]


def _free_stream_defect(L):
    m = _quadtree(3)
    om = oracle.OracleMesh(m, L)
    om.set_boundary_kinds([1, 1])
    U = np.array([1.3, 0.4, -0.7, 2.9])
    u = np.broadcast_to(U[None, :, None], om.shape).copy()
    return np.abs(om.br1_gradient(u)).max(), np.abs(om.rhs_viscous(u)).max()


def test_free_stream_across_mortars():
    gS, gR = _free_stream_defect(None)
    # round-off of terms of size W / (w_0 h) = 1e3 (gradient) and mu W / (w_0 h)^2 = 1e5 (residual), h = 1/64
    assert gS < 1e-10 and gR < 1e-8
    # without the area factor the projected coarse trace is half of W n_C: an O(W / (w_0 h)) spurious gradient
    gS, gR = _free_stream_defect(mutant("br1_mortar_no_area_factor"))
    assert gS > 10.0


def _bump_state(m):
    """perturbation with compact support 0.2 < x < 2.6 (the refined band x_s(y) = 1 + 0.2 sin(2 pi y) lies inside):
    the state is exactly uniform at the x boundaries, so no viscous flux crosses them"""
    x, y = m.node_xyz[:, 0, :], m.node_xyz[:, 1, :]
    t = (x - 1.4) / 1.2
    b = np.where(np.abs(t) < 1.0, np.exp(1.0 - 1.0 / np.maximum(1.0 - t * t, 1e-300)), 0.0)
    rho = 1.0 + 0.3 * b * np.cos(2 * math.pi * y)
    v1 = 0.5 + 0.4 * b * np.sin(2 * math.pi * y + 0.3)
    v2 = -0.2 + 0.3 * b * np.cos(4 * math.pi * y)
    T = 1.1 + 0.2 * b * np.sin(2 * math.pi * y - 1.0)
    E = rho * T / (G - 1) + 0.5 * rho * (v1 * v1 + v2 * v2)
    return np.ascontiguousarray(np.stack([rho, rho * v1, rho * v2, E], axis=1))


def _conservation_defect(L):
    m = _quadtree(3)
    om = oracle.OracleMesh(m, L)
    om.set_boundary_kinds([1, 1])
    u = _bump_state(m)
    # the boundary elements see a uniform state
    be = np.asarray(m.bface)[:, 0]
    assert np.abs(u[be] - u[be][:, :, :1]).max() == 0.0
    _, J = om.metrics()
    _, w, _ = oracle.operators(m.N)
    w2 = np.outer(w, w).reshape(-1)
    r = om.rhs_viscous(u)
    total = (r * (J * w2[None, :])[:, None, :]).sum(axis=(0, 2))
    scale = (np.abs(r) * (J * w2[None, :])[:, None, :]).sum(axis=(0, 2))
    assert scale[1:].min() > 1e-2                         # the momentum and energy rows are not trivially zero
    return np.abs(total[1:] / scale[1:]).max()


def test_viscous_residual_is_conservative_across_mortars():
    assert _conservation_defect(None) < 1e-13
    assert _conservation_defect(mutant("viscous_mortar_no_area_factor")) > 1e-4


# ------------------------------------------------------------------ 3-D 4:1 mortars (O9d; readings R21 + R23)
def _wave3(m):
    """the 3-D analogue of _wave on the periodic unit box: W = W0 + amp sin(2 pi (x + y + z))"""
    X = m.node_xyz
    g = 2 * math.pi * np.ones(3)
    A, c, C, D = np.array([0.3, -0.2, 0.15]), np.array([0.5, 0.4, -0.3]), 0.15, 0.2
    ph = g[0] * X[:, 0] + g[1] * X[:, 1] + g[2] * X[:, 2]
    s, co = np.sin(ph), np.cos(ph)
    rho, T = 1.0 + D * s, 1.2 + C * s
    v = [c[i] + A[i] * s for i in range(3)]
    E = rho * T / (G - 1) + 0.5 * rho * sum(vi * vi for vi in v)
    u = np.stack([rho, rho * v[0], rho * v[1], rho * v[2], E], axis=1)
    M = np.outer(A, g) + np.outer(g, A) - (2.0 / 3.0) * np.eye(3) * (A @ g)
    Mg = M @ g
    k = G * MU / (PR * (G - 1))
    du = np.zeros_like(u)
    for i in range(3):
        du[:, 1 + i] = -MU * Mg[i] * s
    du[:, 4] = MU * (np.outer(A, g) * M).sum() * co ** 2 - MU * sum(v[i] * Mg[i] for i in range(3)) * s - k * C * (g @ g) * s
    amp = np.array([D, A[0], A[1], A[2], C])
    S = amp[None, None, :, None] * g[None, None, None, :] * co[:, :, None, None]
    return np.ascontiguousarray(u), du, S


def _refine(axis):
    return lambda ix, iy, iz: (ix, iy, iz)[axis] < 2


def mortar3d_errors(L, N, axis=0):
    m = _ns(wl.octree_box_mesh(N, K=4, refine=_refine(axis)))
    om = oracle.OracleMesh(m, L)
    u, du, Sx = _wave3(m)
    mo = np.asarray(m.mortar)
    touch = np.unique(mo[:, [0, 2, 3, 4, 5]])
    eS = np.abs(om.br1_gradient(u)[touch] - Sx[touch]).max() / np.abs(Sx).max()
    eR = np.abs(om.rhs_viscous(u)[touch] - du[touch]).max() / np.abs(du).max()
    mc = _ns(wl.cartesian_mesh(3, N, (4, 4, 4), (0.0,) * 3, (1.0,) * 3))
    uc, duc, Sc = _wave3(mc)
    oc = oracle.OracleMesh(mc, L)
    cS = np.abs(oc.br1_gradient(uc) - Sc).max() / np.abs(Sc).max()
    cR = np.abs(oc.rhs_viscous(uc) - duc).max() / np.abs(duc).max()
    return eS, eR, cS, cR


def test_br1_across_3d_mortars_keeps_the_accuracy_of_the_conforming_mesh():
    err = {}
    for N in (2, 4):
        eS, eR, cS, cR = err[N] = mortar3d_errors(None, N)
        assert eS < 2.0 * cS and eR < 10.0 * cR, (N, err[N])
    assert err[4][0] < err[2][0] / 30 and err[4][1] < err[2][1] / 10
    for axis in (1, 2):                                   # the other face numberings and face-local direction pairs
        eS, eR, cS, cR = mortar3d_errors(None, 3, axis)
        assert eS < 2.0 * cS and eR < 10.0 * cR, (axis, eS, eR, cS, cR)
    eS, eR, cS, cR = mortar3d_errors(mutant("br1_mortar3d_wrong_subface"), 4)
    assert eS > 20 * err[4][0] and eR > 20 * err[4][1]
    eS, eR, cS, cR = mortar3d_errors(mutant("viscous_mortar3d_wrong_subface"), 4)
    assert eS == err[4][0] and eR > 20 * err[4][1]


def _defects3d(L, axis):
    """free-stream defect of the gradient, and the relative conservation defect of the viscous residual of a general
    periodic field"""
    m = _ns(wl.octree_box_mesh(3, K=4, refine=_refine(axis)))
    om = oracle.OracleMesh(m, L)
    U = np.array([1.3, 0.4, -0.7, 0.2, 3.1])
    const = np.broadcast_to(U[None, :, None], om.shape).copy()
    gS = np.abs(om.br1_gradient(const)).max()
    gR = np.abs(om.rhs_viscous(const)).max()
    u, _, _ = _wave3(m)
    u[:, 2] *= 1.0 + 0.2 * np.cos(2 * math.pi * m.node_xyz[:, 0])
    r = om.rhs_viscous(u)
    _, J = om.metrics()
    _, w, _ = oracle.operators(m.N)
    W = np.einsum("k,j,i->kji", w, w, w).reshape(-1)
    total = np.einsum("evn,en,n->v", r, J, W)
    scale = np.einsum("evn,en,n->v", np.abs(r), J, W)
    return gS, gR, np.abs(total[1:] / scale[1:]).max()


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_free_stream_and_conservation_across_3d_mortars(axis):
    gS, gR, cons = _defects3d(None, axis)
    assert gS < 1e-11 and gR < 1e-9 and cons < 1e-13


def test_3d_area_factor_mutants_fail():
    gS, gR, cons = _defects3d(mutant("br1_mortar3d_area_factor_2"), 0)
    assert gS > 1.0
    gS, gR, cons = _defects3d(mutant("viscous_mortar3d_area_factor_2"), 0)
    assert gS < 1e-11 and cons > 1e-6          # 8.3e-5 (the real oracle: < 1e-13)
