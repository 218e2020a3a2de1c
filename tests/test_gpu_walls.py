"""GPU parity of the Navier-Stokes boundary faces (wall kinds; reading R22):
gradient_kernel / stage_phys_kernel instantiations with boundary faces against the oracle, for every boundary kind
(prescribed state, outflow, slip wall, no-slip adiabatic wall, isothermal wall), 2-D and 3-D, affine and curved channel
meshes (periodic in x and z, boundary faces at y = lo, hi), N = 2..4: one marut_rhs, marut_max_dt, a stage, five steps."""
import math

import numpy as np
import pytest

import workloads as wl
from parity_util import RHS_TOL, RUN_TOL, gpu_run, parity_error

pytestmark = pytest.mark.gpu

G = 1.4


def _channel(dim, N, cells, curved):
    lo, hi = (0.0,) * dim, (2 * math.pi,) * dim
    warp = wl.sine_warp((cells,) * dim, lo, hi, k=1) if curved else None
    m = wl.open_direction(wl.cartesian_mesh(dim, N, (cells,) * dim, lo, hi, warp=warp), axis=1)
    m.physics, m.mu, m.Pr = wl.NAVIER_STOKES, 0.02, 0.72
    u0 = wl.taylor_green(m, noise=1e-2) if dim == 3 else wl.isentropic_vortex(m, center=(math.pi, math.pi), L=2 * math.pi)
    # prescribed states: a sample of the field, and a colder / hotter variant of it (their p / rho is T_wall of kind 4)
    a, b = u0[0, :, 0].copy(), u0[-1, :, -1].copy()
    b[-1] *= 1.2
    m.bc_state = np.ascontiguousarray(np.stack([a, b]))
    return m, u0


@pytest.mark.parametrize("dim,N,cells,curved", [(2, 3, 5, False), (2, 4, 4, True), (3, 2, 3, True), (3, 3, 3, False), (3, 3, 3, True)])
def test_navier_stokes_boundary_kinds(dim, N, cells, curved):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m, u0 = _channel(dim, N, cells, curved)
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    for kinds in ((0, 0), (3, 4), (4, 3), (2, 1), (1, 2), (3, 3)):
        om.set_boundary_kinds(kinds)
        gm.set_boundary_kinds(kinds)
        gm.rhs(u, du)
        torch.cuda.synchronize()
        ref = om.rhs(u0)
        assert parity_error(du.cpu().numpy(), ref).max() <= RHS_TOL, kinds
        dt = om.max_dt(u0, 0.3)
        assert abs(gm.max_dt(u, 0.3) - dt) <= 1e-13 * dt
    # walls: a stage and five steps
    om.set_boundary_kinds((3, 4))
    gm.set_boundary_kinds((3, 4))
    un_h = u0 * (1.0 + 1e-3)
    out = torch.empty_like(u)
    gm.stage(1, dt, 0.0, torch.from_numpy(un_h).cuda(), u, out)
    torch.cuda.synchronize()
    assert parity_error(out.cpu().numpy(), om.ssprk_stage(1, dt, 0.0, un_h, u0)).max() <= RHS_TOL
    ug, tg = gpu_run(gm, u0, 5, 0.3, torch)
    uc, tc, min_rho, min_p = om.run(u0, 5, cfl=0.3)
    assert min_rho > 0 and min_p > 0 and abs(tg - tc) <= 1e-12 * tc
    assert parity_error(ug, uc).max() <= RUN_TOL
    with pytest.raises(mb.MarutError):
        gm.set_boundary_kinds((5, 0))
    gm.close()


def test_wall_kinds_need_navier_stokes():
    import paper_2605_26388_b200 as mb

    m, _ = _channel(2, 3, 4, False)
    m.physics, m.mu = wl.EULER, 0.0
    gm = mb.MarutMesh(m)
    with pytest.raises(mb.MarutError):
        gm.set_boundary_kinds((3, 3))
    gm.close()
