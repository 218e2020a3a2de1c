"""Pins of the oracle's 3-D 4:1 mortar ("factor 2 in 2D / 4 in 3D"; DESIGN.md reading
R21) on periodic boxes whose cells are split once in half of the domain (workloads.octree_box_mesh)."""
import numpy as np
import pytest

import oracle
import workloads as wl

G = 1.4
V = np.array([1.0, 0.5, -0.3])


def _advected(mesh, amp=0.1):
    """rho = 1 + amp sin(2 pi (x+y+z)), constant velocity and pressure: an exact solution of the Euler equations that
    is advected, so dU/dt is known in closed form"""
    X = mesh.node_xyz
    ph = 2 * np.pi * (X[:, 0] + X[:, 1] + X[:, 2])
    rho = 1.0 + amp * np.sin(ph)
    drho_dt = -amp * 2 * np.pi * np.cos(ph) * V.sum()
    u = np.stack([rho, rho * V[0], rho * V[1], rho * V[2], 1.0 / (G - 1) + 0.5 * rho * (V @ V)], axis=1)
    dudt = np.stack([drho_dt, drho_dt * V[0], drho_dt * V[1], drho_dt * V[2], 0.5 * (V @ V) * drho_dt], axis=1)
    return np.ascontiguousarray(u), dudt


def _quad(mesh, om):
    _, J = om.metrics()
    _, w, _ = oracle.operators(mesh.N)
    return J, np.einsum("k,j,i->kji", w, w, w).reshape(-1)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_free_stream_and_conservation_across_mortars(axis):
    refine = lambda ix, iy, iz: (ix, iy, iz)[axis] < 2
    m = wl.octree_box_mesh(3, K=4, refine=refine)
    assert len(m.mortar) == 32 and m.n_elem == 32 + 32 * 8
    om = oracle.OracleMesh(m)
    const = np.broadcast_to(np.array([1.3, 0.4, -0.2, 0.7, 3.0])[None, :, None], (m.n_elem, 5, m.nn)).copy()
    assert np.abs(om.rhs(const)).max() < 1e-12
    u, _ = _advected(m, amp=0.3)
    u[:, 1] *= 1.0 + 0.2 * np.cos(2 * np.pi * m.node_xyz[:, 1])      # a general field: no exact solution needed here
    r = om.rhs(u)
    J, W = _quad(m, om)
    total = np.einsum("evn,en,n->v", r, J, W)
    scale = np.einsum("evn,en,n->v", np.abs(r), J, W)
    assert np.all(np.abs(total) <= 1e-12 * scale)


def test_mortar_faces_keep_spectral_accuracy():
    """nodal error of the RHS against the closed-form dU/dt of an advected density wave, at the nodes of the elements that
    touch a mortar: as small as on the conforming mesh of the coarse size, and falling fast with N.  A wrong sub-face,
    node or direction pairing anywhere in the mortar leaves an O(1) error here."""
    errs = {}
    for N in (2, 4, 6):
        m = wl.octree_box_mesh(N, K=4)
        om = oracle.OracleMesh(m)
        u, exact = _advected(m)
        r = om.rhs(u)
        touch = np.unique(m.mortar[:, :6].ravel()[np.isin(np.arange(m.mortar[:, :6].size) % 6, (0, 2, 3, 4, 5))])
        errs[N] = np.abs(r[touch] - exact[touch]).max() / np.abs(exact).max()
        mc = wl.cartesian_mesh(3, N, (4, 4, 4), (0.0,) * 3, (1.0,) * 3)
        uc, exc = _advected(mc)
        conf = np.abs(oracle.OracleMesh(mc).rhs(uc) - exc).max() / np.abs(exc).max()
        assert errs[N] < 5.0 * conf + 1e-12, (N, errs[N], conf)
    print(errs)
    assert errs[4] < errs[2] / 10 and errs[6] < errs[4] / 10 and errs[6] < 3e-4


def test_relabelling_the_axes_gives_the_same_field():
    """the box refined in x < 1/2 with a field f(x, y, z), and the box refined in y < 1/2 with f(z, x, y) (the same
    configuration with the coordinates cycled: other face numbers, other face-local directions, other sub-face order)
    give the same RHS at corresponding points, velocity components cycled"""
    N = 3
    ma = wl.octree_box_mesh(N, K=4, refine=lambda ix, iy, iz: ix < 2)
    mb = wl.octree_box_mesh(N, K=4, refine=lambda ix, iy, iz: iy < 2)

    def field(x, y, z, vel):
        rho = 1.0 + 0.2 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y) + 0.1 * np.sin(2 * np.pi * z)
        v = [0.3 + 0.1 * np.cos(2 * np.pi * y), -0.2 + 0.1 * np.sin(2 * np.pi * (x + z)), 0.25 * np.cos(2 * np.pi * x)]
        p = 1.0 + 0.1 * np.cos(2 * np.pi * (x - z))
        v = [v[k] for k in vel]
        return np.ascontiguousarray(np.stack([rho, rho * v[0], rho * v[1], rho * v[2], p / (G - 1) + 0.5 * rho * sum(c * c for c in v)], axis=1))

    Xa, Xb = ma.node_xyz, mb.node_xyz
    ua = field(Xa[:, 0], Xa[:, 1], Xa[:, 2], (0, 1, 2))
    # mesh b: physical point (x', y', z') = (z, x, y) of mesh a, velocity (vz, vx, vy)
    ub = field(Xb[:, 1], Xb[:, 2], Xb[:, 0], (2, 0, 1))
    ra, rb = oracle.OracleMesh(ma).rhs(ua), oracle.OracleMesh(mb).rhs(ub)
    key = lambda x, y, z: (round(float(x) * 4096), round(float(y) * 4096), round(float(z) * 4096))
    # interior nodes only (a face node belongs to several elements with different one-sided values)
    n = N + 1
    idx = np.indices((n, n, n)).reshape(3, -1)
    inner = np.all((idx > 0) & (idx < N), axis=0)
    table = {}
    for e in range(ma.n_elem):
        for p in np.nonzero(inner)[0]:
            table[key(Xa[e, 0, p], Xa[e, 1, p], Xa[e, 2, p])] = ra[e, :, p]
    worst = 0.0
    for e in range(mb.n_elem):
        for p in np.nonzero(inner)[0]:
            a = table[key(Xb[e, 1, p], Xb[e, 2, p], Xb[e, 0, p])]
            b = rb[e, :, p]
            worst = max(worst, np.abs(b - np.array([a[0], a[3], a[1], a[2], a[4]])).max())
    assert worst < 1e-10 * np.abs(ra).max()
