"""GPU parity of the outflow and slip-wall boundary faces (marut_set_boundary_kinds, boundary kinds;
PAPER.md:325; R18) on the quadtree mortar mesh of config 4, strong and split-form stage kernels."""
import numpy as np
import pytest

import workloads as wl
from parity_util import RHS_TOL, RUN_TOL, parity_error

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kinds", [(1, 2), (2, 2), (0, 1), (2, 0)])
@pytest.mark.parametrize("split", [0, 1])
def test_boundary_kinds_rhs_and_run(kinds, split):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    c = wl.make_case("c4", cells=32)
    c.mesh.volume_form = split
    m = c.mesh
    # mild prescribed states (the Mach-10 states of config 4 next to this smooth field would be a shock at the boundary)
    m.bc_state = np.array([[1.0, 0.3, 0.1, 1.0 / 0.4 + 0.05], [1.1, 0.2, 0.0, 1.1 / 0.4 + 0.02]])
    x, y = m.node_xyz[:, 0, :], m.node_xyz[:, 1, :]
    rho = 1.0 + 0.2 * np.sin(1.3 * x) * np.cos(2 * np.pi * y)
    vx, vy = 0.4 * np.cos(0.7 * x + 0.3), 0.3 * np.sin(2 * np.pi * y) + 0.1
    p = 1.0 + 0.1 * np.cos(x) * np.sin(2 * np.pi * y)
    u0 = np.ascontiguousarray(np.stack([rho, rho * vx, rho * vy, p / 0.4 + 0.5 * rho * (vx ** 2 + vy ** 2)], axis=1))
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    before = du.cpu().numpy()
    om.set_boundary_kinds(kinds)
    gm.set_boundary_kinds(kinds)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    ref = om.rhs(u0)
    g = du.cpu().numpy()
    assert parity_error(g, ref).max() <= RHS_TOL
    assert np.abs(g - before).max() > 1e-6 * np.abs(ref).max()           # the kinds took effect
    # a few steps with the new faces
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    uh = u0
    for _ in range(5):
        dt = om.max_dt(uh, 0.5)
        uh = om.run(uh, 1, cfl=0.0, dt=dt)[0]
        gm.step(u, ua, ub, dt)
    torch.cuda.synchronize()
    assert parity_error(u.cpu().numpy(), uh).max() <= RUN_TOL
    # back to prescribed states: the first result again, bit for bit
    gm.set_boundary_kinds((0, 0))
    gm.rhs(torch.from_numpy(u0).cuda(), du)
    torch.cuda.synchronize()
    assert np.array_equal(du.cpu().numpy(), before)
    gm.close()


def test_boundary_kinds_are_validated():
    import paper_2605_26388_b200 as mb

    c = wl.make_case("c4", cells=16)
    gm = mb.MarutMesh(c.mesh)
    with pytest.raises(mb.MarutError):
        gm.set_boundary_kinds((0, 3))
    with pytest.raises(mb.MarutError):
        gm.set_boundary_kinds((1,))
    gm.close()
    ns = wl.make_case("c4", cells=16)
    ns.mesh.physics, ns.mesh.mu = wl.NAVIER_STOKES, 0.01
    gn = mb.MarutMesh(ns.mesh)                  # Navier-Stokes on the mortar mesh (reading R23): kinds 0..4 (R22)
    with pytest.raises(mb.MarutError):
        gn.set_boundary_kinds((5, 0))
    gn.set_boundary_kinds((1, 2))
    gn.set_boundary_kinds((3, 4))
    gn.set_boundary_kinds((0, 0))
    gn.close()


def _open_x(mesh):
    """turn the periodic wrap-around interfaces in x of a Cartesian mesh into boundary faces (bc 0 at x = lo, 1 at x = hi)"""
    xc = mesh.node_xyz[:, 0, :].mean(axis=1)
    first, last = np.isclose(xc, xc.min()), np.isclose(xc, xc.max())
    wrap = (mesh.iface[:, 1] == 1) & last[mesh.iface[:, 0]] & first[mesh.iface[:, 2]]
    assert wrap.sum() == last.sum() > 0
    w = mesh.iface[wrap]
    mesh.bface = np.ascontiguousarray(np.concatenate([np.stack([w[:, 0], w[:, 1], np.ones(len(w), np.int32)], axis=1),
                                                      np.stack([w[:, 2], w[:, 3], np.zeros(len(w), np.int32)], axis=1)]).astype(np.int32))
    mesh.iface = np.ascontiguousarray(mesh.iface[~wrap])
    return mesh


@pytest.mark.parametrize("dim,N,curved,split", [(3, 2, False, 0), (3, 4, False, 1), (3, 3, True, 0), (3, 3, True, 1), (2, 5, True, 0)])
def test_boundary_kinds_on_opened_box_meshes(dim, N, curved, split):
    import math

    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    cells = 3 if dim == 3 else 5
    lo, hi = (0.0,) * dim, (2 * math.pi,) * dim
    warp = wl.sine_warp((cells,) * dim, lo, hi, k=1) if curved else None
    m = _open_x(wl.cartesian_mesh(dim, N, (cells,) * dim, lo, hi, warp=warp))
    m.volume_form = split
    u0 = wl.taylor_green(m, noise=1e-2) if dim == 3 else wl.isentropic_vortex(m)
    m.bc_state = np.ascontiguousarray(np.stack([u0[0, :, 0], u0[-1, :, -1]]))
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    for kinds in ((0, 0), (2, 1), (1, 2)):
        om.set_boundary_kinds(kinds)
        gm.set_boundary_kinds(kinds)
        gm.rhs(u, du)
        torch.cuda.synchronize()
        assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL, kinds
    gm.close()
