"""Pins of the oracle's outflow and slip-wall boundary faces (boundary kinds; "enforced
weakly through the numerical surface flux"; reading R18), on the quadtree mesh of config 4 (boundaries at
x = 0 and x = 4, y periodic, 2:1 mortars inside)."""
import numpy as np
import pytest

import oracle
import workloads as wl

G = 1.4


def _setup(kinds):
    c = wl.make_case("c4", cells=16)
    om = oracle.OracleMesh(c.mesh)
    om.set_boundary_kinds(kinds)
    Ja, J = om.metrics()
    _, w, _ = oracle.operators(c.mesh.N)
    W = np.einsum("j,i->ji", w, w).reshape(-1)
    return c, om, Ja, J, w, W


def _smooth(mesh):
    x, y = mesh.node_xyz[:, 0, :], mesh.node_xyz[:, 1, :]
    rho = 1.0 + 0.2 * np.sin(1.3 * x) * np.cos(2 * np.pi * y)
    vx, vy = 0.4 * np.cos(0.7 * x + 0.3), 0.3 * np.sin(2 * np.pi * y) + 0.1
    p = 1.0 + 0.1 * np.cos(x) * np.sin(2 * np.pi * y)
    return np.ascontiguousarray(np.stack([rho, rho * vx, rho * vy, p / (G - 1) + 0.5 * rho * (vx ** 2 + vy ** 2)], axis=1))


def _uniform(mesh, rho, vx, vy, p):
    U = np.array([rho, rho * vx, rho * vy, p / (G - 1) + 0.5 * rho * (vx * vx + vy * vy)])
    return np.broadcast_to(U[None, :, None], (mesh.n_elem, 4, mesh.nn)).copy()


def test_prescribed_kinds_change_nothing():
    c, om, *_ = _setup([0, 0])
    r = om.rhs(c.u0)
    om.set_boundary_kinds(None)
    assert np.array_equal(om.rhs(c.u0), r)


def test_slip_walls_keep_tangential_flow_and_fluid_at_rest():
    c, om, *_ = _setup([2, 2])
    for vy in (0.0, 0.8):
        r = om.rhs(_uniform(c.mesh, 1.3, 0.0, vy, 2.0))
        assert np.abs(r).max() < 1e-10


def test_slip_walls_conserve_mass_and_energy_but_not_momentum():
    c, om, Ja, J, w, W = _setup([2, 2])
    r = om.rhs(_smooth(c.mesh))
    total = np.einsum("evn,en,n->v", r, J, W)
    scale = np.einsum("evn,en,n->v", np.abs(r), J, W)
    assert abs(total[0]) <= 1e-12 * scale[0] and abs(total[3]) <= 1e-12 * scale[3]      # F*_rho = F*_E = 0 at a wall
    assert abs(total[2]) <= 1e-12 * scale[2]                                              # walls normal to x: no y force
    assert abs(total[1]) > 1e-3 * scale[1]                                                # the wall pressure acts on x momentum


def test_slip_wall_flux_of_a_normal_flow_is_the_rusanov_flux_with_the_mirror_state():
    """uniform flow into the wall at x = 4: volume and interior terms vanish, so at the wall's nodes
    du = -(F*(U, mirror U; n) - F(U).n)/(J w_0), with F* from the separately pinned oracle.rusanov and the mirror state
    written out here; the opposite wall sees the flow leave"""
    c, om, Ja, J, w, W = _setup([2, 2])
    m = c.mesh
    u = _uniform(m, 1.1, 0.6, 0.0, 1.5)
    r = om.rhs(u)
    n = m.N + 1
    U, Umir = u[0, :, 0], u[0, :, 0] * np.array([1, -1, 1, 1])
    seen = 0
    for e, f, bc in m.bface:
        side = f % 2
        for a in range(n):
            node = a * n + (m.N if side else 0)                      # faces 0 / 1: xi = -1 / +1, face index along eta
            nv = (1.0 if side else -1.0) * Ja[e, node, 0]
            Fs, _ = oracle.rusanov(2, G, U, Umir, nv)
            vn = (U[1] * nv[0] + U[2] * nv[1]) / U[0]
            p = (G - 1) * (U[3] - 0.5 * (U[1] ** 2 + U[2] ** 2) / U[0])
            Fown = np.array([U[0] * vn, U[1] * vn + p * nv[0], U[2] * vn + p * nv[1], (U[3] + p) * vn])
            expect = -(Fs - Fown) / (J[e, node] * w[0])
            assert np.allclose(r[e, :, node], expect, rtol=1e-11, atol=1e-11)
            assert abs(Fs[0]) < 1e-14 and abs(Fs[3]) < 1e-13 and Fs[1] * nv[0] > 0     # no mass / energy flux; pressure pushes outwards
            seen += 1
    assert seen == len(m.bface) * n > 0
    interior = np.ones((m.n_elem, m.nn), bool)
    for e, f, bc in m.bface:
        for a in range(n):
            interior[e, a * n + (m.N if f % 2 else 0)] = False
    assert np.abs(r.transpose(0, 2, 1)[interior]).max() < 1e-10


def test_outflow_faces_carry_the_interior_flux():
    """F*(U, U; n) = F(U).n: the lift vanishes, and the total mass change is minus the boundary integral of rho v.n,
    evaluated here from the face nodes with the LGL face quadrature"""
    c, om, Ja, J, w, W = _setup([1, 1])
    m = c.mesh
    u = _smooth(m)
    r = om.rhs(u)
    n = m.N + 1
    out = 0.0
    for e, f, bc in m.bface:
        side = f % 2
        for a in range(n):
            node = a * n + (m.N if side else 0)
            nv = (1.0 if side else -1.0) * Ja[e, node, 0]
            out += w[a] * (u[e, 1, node] * nv[0] + u[e, 2, node] * nv[1])
    total = np.einsum("en,en,n->", r[:, 0, :], J, W)
    assert total == pytest.approx(-out, rel=1e-11)
    # and a uniform state leaves through outflow faces undisturbed
    assert np.abs(om.rhs(_uniform(m, 1.1, 0.6, 0.2, 1.5))).max() < 1e-10


def test_kinds_are_validated():
    c, om, *_ = _setup(None)
    with pytest.raises(ValueError):
        om.set_boundary_kinds([0, 3])
    ns = wl.make_case("c3", cells=2)
    with pytest.raises((ValueError, AssertionError)):
        oracle.OracleMesh(ns.mesh).set_boundary_kinds([1])
