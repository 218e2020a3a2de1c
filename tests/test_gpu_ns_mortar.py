"""GPU parity of the BR1 viscous terms across 2-D 2:1 mortars and 3-D 4:1 mortars (
DESIGN.md readings R23, R21): the mortar branches of gradient_kernel (`br1_mortar_jump_2d`) and of stage_phys_kernel (`node_mortar_flux_2d` for
the hyperbolic flux + `ns_mortar_viscous_2d`) against the oracle on the c4 band mesh run as a Navier-Stokes problem:
N = 1..5, strong and split form, blended, all boundary kinds at the x boundaries; marut_rhs, marut_max_dt, a stage, steps,
the shock-capturing composition; and the full c4 mesh size.  3-D: the half-refined periodic box (refinement along x, y,
z), N = 1..5: the pre-kernels mortar_trace3d_kernel / mortar_flux3d_ns_kernel and the 3-D mortar branches."""
import math

import numpy as np
import pytest

import workloads as wl
from parity_util import RHS_TOL, RUN_TOL, gpu_run, parity_error

pytestmark = pytest.mark.gpu

G = 1.4
CFL = 0.1      # the seeded node-level noise makes the viscous operator stiff at N = 5: 0.3 loses positivity there


def _band(N, base, mu=0.02):
    """the c4 band mesh (3 levels, 2:1 balanced, y periodic, x bounded) with a smooth viscous flow + seeded noise"""
    m = wl.quadtree_mesh(N, base=base, band=0.15, jitter=0.3)
    m.physics, m.mu, m.Pr = wl.NAVIER_STOKES, mu, 0.72
    x, y = m.node_xyz[:, 0, :], m.node_xyz[:, 1, :]
    ph = 2 * math.pi * (x / 4.0 + y)
    idx = np.arange(x.size).reshape(x.shape)
    nz = [1.0 + 1e-2 * (2.0 * wl.uniform(wl.SEED, 70 + k, idx) - 1.0) for k in range(4)]
    rho = (1.0 + 0.2 * np.sin(ph)) * nz[0]
    v1 = (0.5 + 0.3 * np.sin(ph + 0.4)) * nz[1]
    v2 = (-0.3 + 0.2 * np.cos(2 * ph)) * nz[2]
    T = (1.2 + 0.15 * np.sin(ph - 1.0)) * nz[3]
    E = rho * T / (G - 1) + 0.5 * rho * (v1 * v1 + v2 * v2)
    u0 = np.ascontiguousarray(np.stack([rho, rho * v1, rho * v2, E], axis=1))
    m.bc_state = np.ascontiguousarray(np.stack([[1.0, 0.5, -0.1, 3.2], [1.1, 0.4, -0.3, 3.6]]))
    return m, u0


@pytest.mark.parametrize("N,base", [(1, (16, 4)), (2, (16, 4)), (3, (16, 4)), (4, (8, 4)), (5, (8, 4))])
def test_navier_stokes_across_2d_mortars(N, base):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m, u0 = _band(N, base)
    assert len(m.mortar) > 20
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    for kinds in ((0, 0), (1, 1), (3, 4), (2, 0)):
        om.set_boundary_kinds(kinds)
        gm.set_boundary_kinds(kinds)
        gm.rhs(u, du)
        torch.cuda.synchronize()
        assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL, kinds
    dt = om.max_dt(u0, 0.3)
    assert abs(gm.max_dt(u, 0.3) - dt) <= 1e-13 * dt
    un_h = u0 * (1.0 + 1e-3)
    out = torch.empty_like(u)
    gm.stage(1, dt, 0.0, torch.from_numpy(un_h).cuda(), u, out)
    torch.cuda.synchronize()
    assert parity_error(out.cpu().numpy(), om.ssprk_stage(1, dt, 0.0, un_h, u0)).max() <= RHS_TOL
    ug, tg = gpu_run(gm, u0, 5, CFL, torch)
    uc, tc, min_rho, min_p = om.run(u0, 5, cfl=CFL)
    assert min_rho > 0 and min_p > 0 and abs(tg - tc) <= 1e-12 * tc
    assert parity_error(ug, uc).max() <= RUN_TOL
    gm.close()


@pytest.mark.parametrize("N,base", [(2, (16, 4)), (3, (16, 4)), (4, (8, 4))])
def test_split_form_blend_and_shock_capturing_across_mortars(N, base):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m, u0 = _band(N, base)
    m.volume_form = 1
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    om.set_boundary_kinds((0, 1))
    gm.set_boundary_kinds((0, 1))
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    alpha = np.random.default_rng(3).uniform(0, 1, m.n_elem)
    alpha[::5] = 0.0
    ad = torch.from_numpy(alpha).cuda()
    for a in (None, alpha):
        om.set_blend(a)
        gm.set_blend(None if a is None else ad)
        gm.rhs(u, du)
        torch.cuda.synchronize()
        assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL, a is not None
    # three steps of the shock-capturing composition: indicator -> blend -> stage -> floor, every stage
    sc = dict(s=9.21024, alpha_min=1e-3, alpha_max=0.5, smooth=True)
    al = torch.zeros(m.n_elem, dtype=torch.float64, device="cuda")
    gm.set_blend(al)
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    uh = u0
    for _ in range(3):
        dt = om.max_dt(uh, CFL)
        assert abs(gm.max_dt(u, CFL) - dt) <= 1e-12 * dt
        hn, hin = uh, uh
        for s_, (gn, gin, gout) in enumerate(((u, u, ua), (u, ua, ub), (u, ub, u))):
            ah = om.shock_indicator(hin, **sc)
            om.set_blend(ah)
            hin = om.positivity_floor(om.ssprk_stage(s_, dt, 0.0, hn, hin))[0]
            gm.shock_indicator(gin, al, **sc)
            gm.stage(s_, dt, 0.0, gn, gin, gout)
            gm.positivity_floor(gout)
        uh = hin
    torch.cuda.synchronize()
    assert parity_error(u.cpu().numpy(), uh).max() <= RUN_TOL
    gm.close()


def test_full_c4_mesh_as_a_navier_stokes_problem():
    """the c4 mesh of BASELINE.json (base 128 x 32, N = 3, ~24.5 K elements, mortar-dense), every element: RHS, 3 steps"""
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m, u0 = _band(3, (128, 32), mu=2e-3)
    assert m.n_elem > 20000
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL
    ug, tg = gpu_run(gm, u0, 3, CFL, torch)
    uc, tc, min_rho, min_p = om.run(u0, 3, cfl=CFL)
    assert min_rho > 0 and min_p > 0 and abs(tg - tc) <= 1e-12 * tc
    assert parity_error(ug, uc).max() <= RUN_TOL
    gm.close()


def _box3(N, axis, mu=0.02):
    m = wl.octree_box_mesh(N, K=4, lo=(0.0,) * 3, hi=(2 * math.pi,) * 3, refine=lambda ix, iy, iz: (ix, iy, iz)[axis] < 2)
    m.physics, m.mu, m.Pr = wl.NAVIER_STOKES, mu, 0.72
    return m, wl.taylor_green(m, noise=1e-2)


@pytest.mark.parametrize("N,axis", [(1, 0), (2, 1), (3, 2), (4, 0), (5, 1)])
def test_navier_stokes_across_3d_mortars(N, axis):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m, u0 = _box3(N, axis)
    assert len(m.mortar) == 32
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL
    dt = om.max_dt(u0, 0.3)
    assert abs(gm.max_dt(u, 0.3) - dt) <= 1e-13 * dt
    un_h = u0 * (1.0 + 1e-3)
    un = torch.from_numpy(un_h).cuda()
    gm.stage(2, dt, 0.0, un, u, un)
    torch.cuda.synchronize()
    assert parity_error(un.cpu().numpy(), om.ssprk_stage(2, dt, 0.0, un_h, u0)).max() <= RHS_TOL
    ug, tg = gpu_run(gm, u0, 3, 0.3, torch)
    uc, tc, min_rho, min_p = om.run(u0, 3, cfl=0.3)
    assert min_rho > 0 and min_p > 0 and abs(tg - tc) <= 1e-12 * tc
    assert parity_error(ug, uc).max() <= RUN_TOL
    gm.close()


@pytest.mark.parametrize("N,axis", [(2, 2), (3, 0), (4, 1)])
def test_split_form_and_blend_across_3d_mortars(N, axis):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m, u0 = _box3(N, axis)
    m.volume_form = 1
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    alpha = np.random.default_rng(3).uniform(0, 1, m.n_elem)
    alpha[::5] = 0.0
    ad = torch.from_numpy(alpha).cuda()
    for a in (None, alpha):
        om.set_blend(a)
        gm.set_blend(None if a is None else ad)
        gm.rhs(u, du)
        torch.cuda.synchronize()
        assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL, a is not None
    dt = om.max_dt(u0, 0.3)
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    uh = u0
    for _ in range(3):
        uh = om.run(uh, 1, cfl=0.0, dt=dt)[0]
        gm.step(u, ua, ub, dt)
    torch.cuda.synchronize()
    assert parity_error(u.cpu().numpy(), uh).max() <= RUN_TOL
    gm.close()
