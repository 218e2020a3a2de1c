"""GPU parity on 3-D meshes with 4:1 mortar faces (R21): boxes split in
half of the domain along each axis (workloads.octree_box_mesh), strong and split-form Euler stage, blended residual,
indicator smoothing across mortars."""
import numpy as np
import pytest

import workloads as wl
from parity_util import RHS_TOL, RUN_TOL, gpu_run, parity_error

pytestmark = pytest.mark.gpu


def _field(m):
    x, y, z = m.node_xyz[:, 0], m.node_xyz[:, 1], m.node_xyz[:, 2]
    rho = 1.0 + 0.2 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y) + 0.1 * np.sin(2 * np.pi * z)
    v = [0.3 + 0.1 * np.cos(2 * np.pi * y), -0.2 + 0.1 * np.sin(2 * np.pi * (x + z)), 0.25 * np.cos(2 * np.pi * x)]
    p = 1.0 + 0.1 * np.cos(2 * np.pi * (x - z))
    return np.ascontiguousarray(np.stack([rho, rho * v[0], rho * v[1], rho * v[2], p / 0.4 + 0.5 * rho * sum(c * c for c in v)], axis=1))


@pytest.mark.parametrize("N,axis,split", [(1, 0, 0), (2, 1, 0), (3, 2, 0), (3, 0, 1), (4, 1, 0), (4, 2, 1), (5, 0, 0)])
def test_mortar3d_parity(N, axis, split):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m = wl.octree_box_mesh(N, K=4, refine=lambda ix, iy, iz: (ix, iy, iz)[axis] < 2)
    m.volume_form = split
    u0 = _field(m)
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    assert gm.is_affine
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL
    dt = om.max_dt(u0, 0.4)
    assert abs(gm.max_dt(u, 0.4) - dt) <= 1e-13 * dt
    if split:
        a = np.random.default_rng(4).uniform(0, 1, m.n_elem)
        om.set_blend(a)
        ad = torch.from_numpy(a).cuda()
        gm.set_blend(ad)
        gm.rhs(u, du)
        torch.cuda.synchronize()
        assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL
        om.set_blend(None)
        gm.set_blend(None)
    al = torch.empty(m.n_elem, dtype=torch.float64, device="cuda")
    gm.shock_indicator(u, al, alpha_min=1e-9)
    torch.cuda.synchronize()
    ref = om.shock_indicator(u0, alpha_min=1e-9)
    assert ref.max() > 0 and np.abs(al.cpu().numpy() - ref).max() <= 1e-9          # neighbour maximum over the four fine elements
    ug, tg = gpu_run(gm, u0, 3, 0.4, torch)
    uc, tc, _, _ = om.run(u0, 3, cfl=0.4)
    assert abs(tg - tc) <= 1e-12 * tc and parity_error(ug, uc).max() <= RUN_TOL
    gm.close()


def test_mortar3d_is_rejected_where_it_is_not_built():
    import paper_2605_26388_b200 as mb

    c = wl.make_case("c5", cells=2)                      # a reacting case: its mechanism on the half-refined box
    m = wl.octree_box_mesh(2, K=4)
    m.physics, m.mech = wl.REACTING_EULER, c.mesh.mech
    with pytest.raises(mb.MarutError):
        mb.MarutMesh(m)


def test_mortar3d_full_size_c2m():
    """the instance bench.py times as workload c2m (62,208 elements, 1,152 mortars), every element of one RHS and one
    stage against the oracle"""
    import math

    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m = wl.octree_box_mesh(4, K=24, lo=(0.0,) * 3, hi=(2 * math.pi,) * 3)
    u0 = wl.taylor_green(m, noise=1e-3)
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    ref = om.rhs(u0)
    err = parity_error(du.cpu().numpy(), ref).max()
    print(f"c2m: {m.n_elem} elements, {len(m.mortar)} mortars, rhs err {err:.2e}")
    tol = RHS_TOL
    assert err <= tol
    dt = om.max_dt(u0, 0.4)
    assert abs(gm.max_dt(u, 0.4) - dt) <= 1e-13 * dt
    un_h = u0 * (1.0 + 1e-3)
    out = torch.empty_like(u)
    gm.stage(2, dt, 0.0, torch.from_numpy(un_h).cuda(), u, out)
    torch.cuda.synchronize()
    assert parity_error(out.cpu().numpy(), om.ssprk_stage(2, dt, 0.0, un_h, u0)).max() <= tol
    gm.close()
