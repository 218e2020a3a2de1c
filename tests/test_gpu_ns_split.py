"""GPU parity of the split-form / blended hyperbolic volume integral on Navier-Stokes meshes (
PAPER.md:183-191 'Three operators are available and selected once at solver setup', 331-394: the 3-D Navier-Stokes
Taylor-Green runs use the split form): stage_split_kernel for the hyperbolic part, then the viscous-only
instantiation of stage_phys_kernel adds the parabolic part.  RHS, a stage, steps; with a blending field, with the
per-stage shock-capturing composition, and on a channel with no-slip walls."""
import math

import numpy as np
import pytest

import workloads as wl
from parity_util import RHS_TOL, RUN_TOL, parity_error

pytestmark = pytest.mark.gpu


def _case(kind):
    if kind == "c3":                                   # 3-D curved periodic, N = 3
        c = wl.make_case("c3", cells=3)
        return c.mesh, wl.taylor_green(c.mesh, noise=1e-2), None
    if kind == "3d_affine_n4":
        m = wl.cartesian_mesh(3, 4, (3,) * 3, (0.0,) * 3, (2 * math.pi,) * 3)
        m.physics, m.mu, m.Pr = wl.NAVIER_STOKES, 0.01, 0.72
        return m, wl.taylor_green(m, noise=1e-2), None
    if kind == "2d_curved":
        lo, hi = (0.0, 0.0), (10.0, 10.0)
        m = wl.cartesian_mesh(2, 3, (6, 6), lo, hi, warp=wl.sine_warp((6, 6), lo, hi, k=1))
        m.physics, m.mu, m.Pr = wl.NAVIER_STOKES, 0.02, 0.72
        return m, wl.isentropic_vortex(m), None
    if kind == "channel":                              # walls at y = lo, hi
        lo, hi = (0.0,) * 3, (2 * math.pi,) * 3
        m = wl.open_direction(wl.cartesian_mesh(3, 3, (3,) * 3, lo, hi, warp=wl.sine_warp((3,) * 3, lo, hi, k=1)), axis=1)
        m.physics, m.mu, m.Pr = wl.NAVIER_STOKES, 0.02, 0.72
        u0 = wl.taylor_green(m, noise=1e-2)
        m.bc_state = np.ascontiguousarray(np.stack([u0[0, :, 0], u0[-1, :, -1]]))
        return m, u0, (3, 4)
    raise ValueError(kind)


@pytest.mark.parametrize("kind", ["c3", "3d_affine_n4", "2d_curved", "channel"])
def test_split_form_and_blend_navier_stokes(kind):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m, u0, kinds = _case(kind)
    m.volume_form = 1
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    if kinds:
        om.set_boundary_kinds(kinds)
        gm.set_boundary_kinds(kinds)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    rng = np.random.default_rng(3)
    alpha = rng.uniform(0, 1, m.n_elem)
    alpha[::5] = 0.0
    ad = torch.from_numpy(alpha).cuda()
    for a in (None, alpha):
        om.set_blend(a)
        gm.set_blend(None if a is None else ad)
        gm.rhs(u, du)
        torch.cuda.synchronize()
        assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL, (kind, a is not None)
    dt = om.max_dt(u0, 0.3)
    un_h = u0 * (1.0 + 1e-3)
    un = torch.from_numpy(un_h).cuda()
    gm.stage(2, dt, 0.0, un, u, un)                                   # last stage writes over u_n, blend on
    torch.cuda.synchronize()
    assert parity_error(un.cpu().numpy(), om.ssprk_stage(2, dt, 0.0, un_h, u0)).max() <= RHS_TOL
    # three steps of the shock-capturing composition: indicator -> blend -> stage -> floor, every stage
    sc = dict(s=9.21024, alpha_min=1e-3, alpha_max=0.5, smooth=True)
    al = torch.zeros(m.n_elem, dtype=torch.float64, device="cuda")
    gm.set_blend(al)
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    uh = u0
    for _ in range(3):
        dt = om.max_dt(uh, 0.3)
        assert abs(gm.max_dt(u, 0.3) - dt) <= 1e-12 * dt
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
    gm.set_blend(None)
    gm.close()
