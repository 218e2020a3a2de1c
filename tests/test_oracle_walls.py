"""Pins of the oracle's Navier-Stokes boundary faces (wall kinds; "At a no-slip adiabatic
wall the boundary kernel sets the wall velocity to zero and inherits interior (rho, T); at an isothermal wall it
additionally fixes T = T_wall; at a slip wall it mirrors the velocity across the boundary normal"; reading R22):
closed forms of the BR1 wall traces, conservation of mass and energy between adiabatic walls, the steady heat-conduction
state between isothermal walls, the wall heat flux.  Channel meshes: periodic in x (and z), walls at y = lo, hi."""
import math

import numpy as np
import pytest

import oracle
import workloads as wl
from mutation_util import mutant

G, MU, PR = 1.4, 0.02, 0.72
KAPPA = G * MU / (PR * (G - 1))


def channel(dim, N=3, cells=4, kinds=(3, 3), Twall=(1.0, 1.0), L=None, warp=False):
    lo, hi = (0.0,) * dim, (1.0,) * dim
    w = wl.sine_warp((cells,) * dim, lo, hi, k=1) if warp else None
    m = wl.open_direction(wl.cartesian_mesh(dim, N, (cells,) * dim, lo, hi, warp=w, order="lex"), axis=1)
    m.physics, m.mu, m.Pr = wl.NAVIER_STOKES, MU, PR
    # prescribed states of the two boundary ids: their temperature T = p / rho is the wall temperature of kind 4
    st = []
    for T in Twall:
        rho, p = 1.0, T
        st.append([rho] + [0.0] * dim + [p / (G - 1)])
    m.bc_state = np.array(st)
    om = oracle.OracleMesh(m, L)
    om.set_boundary_kinds(kinds)
    return m, om


def cons(rho, vel, p):
    vel = [np.asarray(v, float) for v in vel]
    return np.ascontiguousarray(np.stack([rho] + [rho * v for v in vel] + [p / (G - 1) + 0.5 * rho * sum(v * v for v in vel)], axis=1))


def quad(m, om):
    _, J = om.metrics()
    _, w, _ = oracle.operators(m.N)
    w = np.asarray(w)
    W = np.einsum("j,i->ji", w, w).reshape(-1) if m.dim == 2 else np.einsum("k,j,i->kji", w, w, w).reshape(-1)
    return J, W, w


def rough(m, seed=4):
    rng = np.random.default_rng(seed)
    X = m.node_xyz
    s = lambda k: np.sin(2 * math.pi * (X[:, 0] * k + 0.3 * X[:, 1] ** 2 + 0.1 * k))
    rho = 1.0 + 0.2 * s(1) * np.cos(3 * X[:, 1])
    vel = [0.3 * s(2) + 0.1, 0.2 * np.cos(2 * math.pi * X[:, 0]) * (0.5 + X[:, 1])] + ([0.15 * s(1)] if m.dim == 3 else [])
    p = 1.0 + 0.1 * s(1) * X[:, 1]
    return cons(rho, vel, p)


# ------------------------------------------------------------------ BR1 traces at boundary faces
@pytest.mark.parametrize("dim", [2, 3])
def test_br1_wall_traces_closed_form(dim):
    """uniform interior state with velocity v: S = (What - W) n / (w_0 h/2) at the boundary nodes of the faces normal
    to y and 0 elsewhere; What per kind as PAPER.md:223 states"""
    h = 0.25
    vel = [0.4, -0.3, 0.2][:dim]
    rho, p = 1.3, 2.0
    T = p / rho
    nhat = np.zeros(dim); nhat[1] = 1.0
    expect_jump = {
        0: lambda s, Tb: np.array([0.5 * (1.0 - rho)] + [0.5 * (0.0 - v) for v in vel] + [0.5 * (Tb - T)]),      # central with W(U_bc)
        1: lambda s, Tb: np.zeros(dim + 2),                                                                      # outflow
        2: lambda s, Tb: np.array([0.0] + [-(vel[1]) * nhat[c] for c in range(dim)] + [0.0]),                    # mirrored normal velocity
        3: lambda s, Tb: np.array([0.0] + [-v for v in vel] + [0.0]),                                            # v_wall = 0, (rho, T) inherited
        4: lambda s, Tb: np.array([0.0] + [-v for v in vel] + [Tb - T]),                                         # ... and T = T_wall
    }
    for kind in (0, 1, 2, 3, 4):
        m, om = channel(dim, kinds=(kind, kind), Twall=(0.8, 1.7))
        u = np.broadcast_to(cons(np.array([rho]), [np.array([v]) for v in vel], np.array([p]))[0][None, :, None], om.shape).copy()
        S = om.br1_gradient(u)                                  # [e][node][w][c]
        n = m.N + 1
        _, w, _ = oracle.operators(m.N)
        expect = np.zeros_like(S)
        j_of = (np.arange(m.nn) // n) % n                       # index along y of every node
        for e, f, bc in np.asarray(m.bface):
            sgn = 1.0 if f == 3 else -1.0
            nodes = j_of == (n - 1 if f == 3 else 0)
            jump = expect_jump[kind](sgn, (0.8, 1.7)[bc])
            expect[e, nodes, :, 1] += jump * sgn / (w[0] * h / 2)
        assert np.abs(expect).max() > 0.5 or kind == 1
        assert np.abs(S - expect).max() <= 1e-12 * max(1.0, np.abs(expect).max()), kind
    # mutants: wall velocity not set to zero / wall temperature not applied
    m, om = channel(dim, kinds=(4, 4), Twall=(0.8, 1.7), L=mutant("wall_trace_keeps_velocity"))
    u = np.broadcast_to(cons(np.array([rho]), [np.array([v]) for v in vel], np.array([p]))[0][None, :, None], om.shape).copy()
    assert np.abs(om.br1_gradient(u)[:, :, 1:1 + dim, :]).max() < 1e-12           # the mutant sees no velocity jump


# ------------------------------------------------------------------ adiabatic no-slip walls: closed system
@pytest.mark.parametrize("dim,warp", [(2, False), (2, True), (3, False)])
def test_adiabatic_walls_conserve_mass_and_energy(dim, warp):
    """v_wall = 0 and no heat through the wall: neither mass nor total energy crosses an adiabatic no-slip wall, for any
    interior field: sum J W dU/dt = 0 for rho and E; the walls do exert a force (momentum changes)"""
    m, om = channel(dim, kinds=(3, 3), warp=warp)
    u = rough(m)
    r = om.rhs(u)
    J, W, _ = quad(m, om)
    total = np.einsum("evn,en,n->v", r, J, W)
    scale = np.einsum("evn,en,n->v", np.abs(r), J, W)
    assert abs(total[0]) <= 1e-12 * scale[0] and abs(total[-1]) <= 1e-12 * scale[-1], (total, scale)
    assert abs(total[1]) > 1e-4 * scale[1]                      # wall shear acts on the x momentum
    # the mutant that keeps the stress work / heat flux in the wall's energy flux does not conserve energy
    mm, omm = channel(dim, kinds=(3, 3), warp=warp, L=mutant("adiabatic_wall_energy_flux_kept"))
    rm = omm.rhs(u)
    tm = np.einsum("evn,en,n->v", rm, J, W)
    assert abs(tm[-1]) > 1e-6 * scale[-1]


# ------------------------------------------------------------------ isothermal walls: heat conduction
def test_isothermal_walls_steady_conduction_and_wall_heat_flux():
    """fluid at rest, uniform pressure, T linear between two isothermal walls at T(0) and T(1): a steady solution of
    the compressible Navier-Stokes equations (constant mu, k); every term of the discretisation is exact for it, so
    the RHS vanishes to round-off.  With the upper wall hotter than the profile by dT the energy enters at the rate
    the wall heat flux k grad T . n gives (grad T from the separately pinned BR1 gradient)."""
    T0, T1, p = 1.0, 1.6, 2.0
    m, om = channel(2, kinds=(4, 4), Twall=(T0, T1))
    y = m.node_xyz[:, 1, :]
    T = T0 + (T1 - T0) * y
    u = cons(p / T, [np.zeros_like(T), np.zeros_like(T)], p * np.ones_like(T))
    r = om.rhs(u)
    assert np.abs(r).max() <= 1e-10 * KAPPA * (T1 - T0) / 0.25 ** 2
    # hotter upper wall: total energy rate = wall heat flux integrated over the walls
    dT = 0.3
    m2, om2 = channel(2, kinds=(4, 4), Twall=(T0, T1 + dT))
    r2 = om2.rhs(u)
    J, W, w = quad(m2, om2)
    rate = np.einsum("en,en,n->", r2[:, -1, :], J, W)
    S = om2.br1_gradient(u)
    n, h = m2.N + 1, 0.25
    j_of = (np.arange(m2.nn) // n) % n
    heat = 0.0
    for e, f, bc in np.asarray(m2.bface):
        sgn = 1.0 if f == 3 else -1.0
        nodes = np.nonzero(j_of == (n - 1 if f == 3 else 0))[0]
        for a, nd in enumerate(nodes):
            heat += w[a] * (h / 2) * KAPPA * S[e, nd, 3, 1] * sgn           # k dT/dy n_y, face quadrature
    assert heat > 0.0
    assert abs(rate - heat) <= 1e-11 * abs(heat)
    assert np.abs(np.einsum("en,en,n->", r2[:, 0, :], J, W)) <= 1e-12 * np.abs(r2[:, 0, :]).max()   # no mass through the wall
