"""Pins of the three oracle parts that round 1 left without an effective pin: the lo / up
assignment of the 2-D mortar (O7), the prescribed exterior state of boundary faces (O8) and the central trace of the BR1
gradient (O9, eq. 13).  Each check is a function of the oracle library, run on the real oracle (must hold) and on the
mutant of tests/mutation_util.py that makes the named mistake (must fail)."""
import math

import numpy as np
import pytest

import oracle
import workloads as wl
from mutation_util import mutant

G = 1.4


# ------------------------------------------------------------------ O7: 2-D 2:1 mortar
def _advected_2d(m, kx=1, ky=1, amp=0.2, vel=(0.7, -0.4), p=1.5):
    """density wave rho = 1 + amp sin(2 pi (kx x / 4 + ky y)) carried by a constant velocity at constant pressure on
    [0,4] x [0,1]: an exact Euler solution, dU/dt = -(v.grad rho) (1, v, |v|^2/2) in closed form"""
    x, y = m.node_xyz[:, 0, :], m.node_xyz[:, 1, :]
    ph = 2 * math.pi * (kx * x / 4.0 + ky * y)
    rho = 1.0 + amp * np.sin(ph)
    drho = -amp * np.cos(ph) * 2 * math.pi * (vel[0] * kx / 4.0 + vel[1] * ky)
    v2 = vel[0] ** 2 + vel[1] ** 2
    u = np.stack([rho, rho * vel[0], rho * vel[1], p / (G - 1) + 0.5 * rho * v2], axis=1)
    du = np.stack([drho, drho * vel[0], drho * vel[1], 0.5 * v2 * drho], axis=1)
    return np.ascontiguousarray(u), du


def mortar_error(L, N):
    """relative nodal error of the RHS at the elements that touch a mortar, and the same on the conforming mesh of the
    coarsest element size"""
    m = wl.quadtree_mesh(N, base=(32, 8), band=0.15, jitter=0.3)
    u, exact = _advected_2d(m)
    # the Dirichlet faces do not carry the wave (mean state outside): the elements that own a boundary face are kept
    # out of the measurement (the 2:1 balance refines a few of them, so some do touch a mortar)
    m.bc_state = np.stack([np.array([1.0, 0.7, -0.4, 1.5 / (G - 1) + 0.5 * 0.65])] * 2)
    r = oracle.OracleMesh(m, L).rhs(u)
    touch = np.setdiff1d(np.unique(np.asarray(m.mortar)[:, [0, 2, 3]]), np.asarray(m.bface)[:, 0])
    assert len(touch) > 400
    err = np.abs(r[touch] - exact[touch]).max() / np.abs(exact).max()
    mc = wl.cartesian_mesh(2, N, (32, 8), (0.0, 0.0), (4.0, 1.0))
    uc, exc = _advected_2d(mc)
    conf = np.abs(oracle.OracleMesh(mc, L).rhs(uc) - exc).max() / np.abs(exc).max()
    return err, conf


def test_mortar2d_keeps_the_accuracy_of_the_conforming_mesh():
    errs = {}
    for N in (2, 3, 5):
        errs[N], conf = mortar_error(None, N)
        assert errs[N] < 10.0 * conf, (N, errs[N], conf)          # 4.1x, 5.3x, 6.5x the conforming mesh's error
    assert errs[3] < errs[2] / 5 and errs[5] < errs[3] / 100     # spectral: 0.38, 3.8e-2, 1.1e-4
    # the mutant that interpolates the coarse trace to the wrong half is O(1) off at those elements (84 here)
    e_mut, conf = mortar_error(mutant("mortar2d_lo_up_swapped"), 3)
    assert e_mut > 100 * errs[3] and e_mut > 10.0 * conf


# ------------------------------------------------------------------ O8: prescribed exterior state
def boundary_residual_mismatch(L):
    """uniform interior state U, prescribed states U_bc != U: the RHS vanishes except at the nodes of the boundary
    faces, where it is -(F*(U, U_bc; n) - F(U).n)/(J w_0) with the separately pinned Rusanov flux.  Returns the largest
    deviation from that closed form relative to the largest expected value."""
    m = wl.quadtree_mesh(3, base=(16, 4), band=0.15, jitter=0.3)
    U = np.array([1.3, 0.4, -0.7, 2.9])
    Ubc = np.array([[0.9, 0.6, 0.2, 3.4], [1.7, -0.3, -0.5, 2.2]])
    m.bc_state = Ubc.copy()
    om = oracle.OracleMesh(m, L)
    n = m.N + 1
    _, w, _ = oracle.operators(m.N)
    u = np.broadcast_to(U[None, :, None], om.shape).copy()
    du = om.rhs(u)
    expect = np.zeros_like(du)
    X = m.node_xyz
    for e, f, bc in np.asarray(m.bface):
        assert f in (0, 1)                                  # the x boundaries
        hx = X[e, 0].max() - X[e, 0].min()
        hy = X[e, 1].max() - X[e, 1].min()
        nv = np.array([(1.0 if f == 1 else -1.0) * hy / 2, 0.0])     # scaled outward normal n_ref Ja^1
        J = hx * hy / 4
        Fs, _ = oracle.rusanov(2, G, U, Ubc[bc], nv)
        Fown, _ = oracle.rusanov(2, G, U, U, nv)             # consistency (pinned): F*(U,U;n) = F(U).n
        s = 0 if f == 0 else n - 1
        for a in range(n):
            expect[e, :, s + n * a] = -(Fs - Fown) / (J * w[0])
    assert np.abs(expect).max() > 1.0                        # the closed form is not trivially small
    return np.abs(du - expect).max() / np.abs(expect).max()


def test_boundary_faces_use_the_prescribed_exterior_state():
    assert boundary_residual_mismatch(None) < 1e-12
    assert boundary_residual_mismatch(mutant("boundary_state_ignored")) > 0.5


# ------------------------------------------------------------------ O9: BR1 trace What = (W- + W+)/2, eq. 13
def br1_jump_mismatch(L, dim):
    """W = (rho, v, T) constant per element with seeded jumps on a Cartesian periodic mesh: the BR1 gradient is the
    lifted jump alone, S_c = (W+ - W-)/2 n_c / (w_0 h/2) at the nodes of the faces normal to c (one term per face the
    node lies on) and 0 at the other nodes.  Returns the largest deviation relative to the largest expected entry."""
    N, K = 3, 3
    hi = (3.0,) * dim
    m = wl.cartesian_mesh(dim, N, (K,) * dim, (0.0,) * dim, hi, order="lex")
    m.physics, m.mu, m.Pr = wl.NAVIER_STOKES, 0.01, 0.72
    om = oracle.OracleMesh(m, L)
    n, h = N + 1, 1.0
    _, w, _ = oracle.operators(N)
    rng = np.random.default_rng(5)
    Wel = np.concatenate([rng.uniform(0.5, 2.0, (m.n_elem, 1)), rng.uniform(-1, 1, (m.n_elem, dim)), rng.uniform(0.5, 2.0, (m.n_elem, 1))], axis=1)
    rho, v, T = Wel[:, 0], Wel[:, 1:1 + dim], Wel[:, -1]
    E = rho * T / (G - 1) + 0.5 * rho * (v * v).sum(axis=1)            # p = rho T (R = 1)
    Uel = np.concatenate([rho[:, None], rho[:, None] * v, E[:, None]], axis=1)
    u = np.ascontiguousarray(np.broadcast_to(Uel[:, :, None], om.shape))
    S = om.br1_gradient(u)                                             # [e][node][w][c]
    expect = np.zeros_like(S)
    idx = np.indices((n,) * dim).reshape(dim, -1)[::-1]                # idx[c][node] = index along direction c (i fastest)
    for eL, fL, eR, fR, _ in np.asarray(m.iface):
        c = fL >> 1
        assert fR >> 1 == c and (fL & 1) == 1 and (fR & 1) == 0        # the generator's faces: L's + face meets R's - face
        jump = 0.5 * (Wel[eR] - Wel[eL]) / (w[0] * h / 2)
        expect[eL, idx[c] == N, :, c] += jump                          # outward normal +e_c, What - W- = +(W+ - W-)/2
        expect[eR, idx[c] == 0, :, c] += jump                          # outward normal -e_c, What - W+ = -(W+ - W-)/2
    assert np.abs(expect).max() > 1.0
    return np.abs(S - expect).max() / np.abs(expect).max()


@pytest.mark.parametrize("dim", [2, 3])
def test_br1_gradient_of_a_piecewise_constant_field_is_the_lifted_central_jump(dim):
    assert br1_jump_mismatch(None, dim) < 1e-13
    assert br1_jump_mismatch(mutant("br1_trace_not_central"), dim) > 0.2


# ------------------------------------------------------------------ the split-form flux pin against its mutant
def test_the_entropy_pin_rejects_the_printed_energy_flux():
    """tests/test_oracle_split.py pins Tadmor's condition on the real oracle; here the same quantity on the mutant that
    carries the pressure work as PAPER.md:621 prints it"""
    from test_oracle_split import _cons, _entropy_vars

    def worst(L):
        rng = np.random.default_rng(11)
        out = 0.0
        for _ in range(20):
            UL = _cons(rng.uniform(0.2, 3), rng.uniform(-2, 2, 2), rng.uniform(0.2, 5))
            UR = _cons(rng.uniform(0.2, 3), rng.uniform(-2, 2, 2), rng.uniform(0.2, 5))
            nv = rng.uniform(-1, 1, 2)
            F = np.zeros(4)
            (L or oracle.lib()).oracle_ranocha(2, G, oracle._p(oracle._f64(UL)), oracle._p(oracle._f64(UR)), oracle._p(oracle._f64(nv)), oracle._p(F))
            (wL, mL), (wR, mR) = _entropy_vars(UL), _entropy_vars(UR)
            out = max(out, abs((wR - wL) @ F - (mR - mL) @ nv) / (np.abs(wR - wL) @ np.abs(F) + 1e-300))
        return out

    assert worst(None) < 1e-8 and worst(mutant("ranocha_printed_energy_flux")) > 1e-3
