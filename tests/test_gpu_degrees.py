"""GPU parity for polynomial degrees and mesh kinds beyond the five configs: every kernel instantiation the library
dispatches (2-D / 3-D, N = 1..7, affine / curved, Euler / Navier-Stokes / reacting) against the oracle on one
marut_rhs and one marut_ssprk_stage, on small periodic meshes with a ragged last CTA."""
import math

import numpy as np
import pytest

import workloads as wl
from parity_util import RHS_TOL, parity_error

pytestmark = pytest.mark.gpu


def _mesh(dim, N, cells, curved):
    lo, hi = (0.0,) * dim, ((10.0,) * 2 if dim == 2 else (2 * math.pi,) * 3)
    counts = (cells,) * dim
    warp = wl.sine_warp(counts, lo, hi, k=1) if curved else None
    return wl.cartesian_mesh(dim, N, counts, lo, hi, warp=warp)


CASES = [(2, N, 5, curved, "euler") for N in (1, 2, 3, 4, 5, 7) for curved in (False, True)] + \
        [(3, N, 3, curved, "euler") for N in (1, 2, 3, 4, 5, 6) for curved in (False, True)] + \
        [(3, 7, 2, False, "euler"), (3, 7, 2, True, "euler"), (2, 6, 4, True, "euler")] + \
        [(3, 2, 3, True, "ns"), (3, 4, 3, False, "ns"), (2, 3, 5, True, "ns"), (3, 2, 3, False, "react"), (3, 4, 3, False, "react")]


@pytest.mark.parametrize("dim,N,cells,curved,phys", CASES)
def test_rhs_and_stage(dim, N, cells, curved, phys):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m = _mesh(dim, N, cells, curved and phys != "react")
    if phys == "react":
        L = wl.C5_LENGTH * cells / 32.0
        m = wl.cartesian_mesh(3, N, (cells,) * 3, (0.0,) * 3, (L,) * 3)
        m.physics, m.mech = wl.REACTING_EULER, wl.air5_mechanism()
        u0 = wl.reacting_field(m, L)
    else:
        if phys == "ns":
            m.physics, m.mu, m.Pr = wl.NAVIER_STOKES, 1.0 / 100.0, 0.72
        u0 = wl.isentropic_vortex(m) if dim == 2 else wl.taylor_green(m, noise=1e-3)
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    assert gm.is_affine == (not (curved and phys != "react"))
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL
    dt = om.max_dt(u0, 0.5)
    assert abs(gm.max_dt(u, 0.5) - dt) <= 1e-13 * dt
    un_h = u0 * (1.0 + 1e-3)
    out = torch.empty_like(u)
    gm.stage(2, dt, 0.0, torch.from_numpy(un_h).cuda(), u, out)
    torch.cuda.synchronize()
    assert parity_error(out.cpu().numpy(), om.ssprk_stage(2, dt, 0.0, un_h, u0)).max() <= RHS_TOL
    gm.close()


SPLIT = [(2, 3, 6, False), (2, 4, 5, True), (3, 4, 3, False), (3, 3, 3, True), (3, 1, 3, False), (3, 5, 2, False),
         (3, 6, 2, False), (3, 6, 2, True), (2, 6, 4, True), (2, 7, 3, False)]      # N = 6: the degree of the paper's TGV runs


@pytest.mark.parametrize("dim,N,cells,curved", SPLIT)
def test_split_form_rhs_stage_and_run(dim, N, cells, curved):
    """entropy-stable split-form volume integral (marut_set_volume_form) against the oracle"""
    import torch

    import oracle
    import paper_2605_26388_b200 as mb
    from parity_util import RUN_TOL, gpu_run

    m = _mesh(dim, N, cells, curved)
    m.volume_form = 1
    u0 = wl.isentropic_vortex(m) if dim == 2 else wl.taylor_green(m, noise=1e-3)
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL
    dt = om.max_dt(u0, 0.4)
    un_h = u0 * (1.0 + 1e-3)
    out = torch.empty_like(u)
    gm.stage(1, dt, 0.0, torch.from_numpy(un_h).cuda(), u, out)
    torch.cuda.synchronize()
    assert parity_error(out.cpu().numpy(), om.ssprk_stage(1, dt, 0.0, un_h, u0)).max() <= RHS_TOL
    ug, tg = gpu_run(gm, u0, 5, 0.4, torch)
    uc, tc, _, _ = om.run(u0, 5, cfl=0.4)
    assert abs(tg - tc) <= 1e-12 * tc and parity_error(ug, uc).max() <= RUN_TOL
    gm.close()


@pytest.mark.parametrize("dim,N,cells", [(2, 3, 6), (3, 4, 3)])
def test_split_form_rough_states_take_the_logarithm_branch(dim, N, cells):
    """node-to-node jumps of a factor up to 15 in density and pressure: most pairs leave the series branch of the
    logarithmic mean (u = ((aL-aR)/(aL+aR))^2 >= 1e-2); one RHS against the oracle"""
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m = _mesh(dim, N, cells, False)
    m.volume_form = 1
    shape = (m.n_elem, dim + 2, (N + 1) ** dim)
    idx = np.arange(np.prod(shape), dtype=np.uint64).reshape(shape)
    r = wl.uniform(wl.SEED, 77, idx)
    rho, p = 0.2 + 2.8 * r[:, 0], 0.2 + 4.8 * r[:, -1]
    vel = 2.0 * r[:, 1:1 + dim] - 1.0
    u0 = np.empty(shape)
    u0[:, 0] = rho
    u0[:, 1:1 + dim] = rho[:, None] * vel
    u0[:, -1] = p / 0.4 + 0.5 * rho * (vel ** 2).sum(axis=1)
    ratio = rho[:, 1:] / rho[:, :-1]
    assert (np.abs((ratio - 1) / (ratio + 1)) > 0.1).mean() > 0.5      # the logarithm branch is exercised
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL
    gm.close()


@pytest.mark.parametrize("N,split", [(1, False), (2, False), (4, False), (5, False), (3, True), (4, True)])
def test_quadtree_mortars_and_boundaries_other_degrees(N, split):
    """2:1 mortar faces and prescribed-state boundary faces (a3, a4) at degrees other than config 4's N = 3, with the
    strong and the split-form volume integral: RHS, dt and five steps against the oracle"""
    import torch

    import oracle
    import paper_2605_26388_b200 as mb
    from parity_util import RUN_TOL, gpu_run

    m = wl.quadtree_mesh(N, base=(16, 4), band=0.15, jitter=0.3)
    m.bc_state = wl.shock_states(m.gamma)
    if split:
        m.volume_form = 1
    assert len(m.mortar) > 0 and len(m.bface) > 0
    u0 = wl.mach10_shock(m, half_width=6.0 * m.info["h_fine"])
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL
    dt = om.max_dt(u0, 0.3)
    assert abs(gm.max_dt(u, 0.3) - dt) <= 1e-13 * dt
    ug, tg = gpu_run(gm, u0, 5, 0.3, torch)
    uc, tc, _, _ = om.run(u0, 5, cfl=0.3)
    assert abs(tg - tc) <= 1e-12 * tc and parity_error(ug, uc).max() <= RUN_TOL
    gm.close()


@pytest.mark.parametrize("kind,N", [("c4", 3), ("c4", 5), ("tgv3", 4), ("tgv3", 2), ("vortex", 7)])
def test_shock_indicator_parity(kind, N):
    """Hennemann-Gassner blending coefficient (marut_shock_indicator) against the oracle: raw and smoothed,
    on the Mach-10 front of the quadtree mesh (mortar neighbours, alpha from 0 to alpha_max) and on smooth fields"""
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    if kind == "c4":
        m = wl.quadtree_mesh(N, base=(32, 8), band=0.15, jitter=0.3)
        m.bc_state = wl.shock_states(m.gamma)
        u0 = wl.mach10_shock(m, half_width=1.0 * m.info["h_fine"])      # a front sharper than the bench recipe's
    elif kind == "tgv3":
        m = _mesh(3, N, 3, True)
        u0 = wl.taylor_green(m, noise=5e-2)
    else:
        m = _mesh(2, N, 4, False)
        u0 = wl.isentropic_vortex(m)
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    a = torch.empty(m.n_elem, dtype=torch.float64, device="cuda")
    for smooth in (False, True):
        for amin, amax in ((0.0, 1.0), (1e-3, 0.5)):
            gm.shock_indicator(u, a, alpha_min=amin, alpha_max=amax, smooth=smooth)
            ref = om.shock_indicator(u0, alpha_min=amin, alpha_max=amax, smooth=smooth)
            g = a.cpu().numpy()
            assert np.abs(g - ref).max() <= 1e-11 * max(ref.max(), 1e-300), (kind, N, smooth, amin)
    if kind == "c4" and N == 3:
        assert ref.max() == 0.5 and (ref == 0).sum() > 0          # the front saturates, the far field stays pure DG
    gm.close()
