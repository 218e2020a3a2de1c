"""GPU parity of SSP-RK54 (SURVEY 8(f) NEXT-2b; eq. 45; R19): marut_rk_stage + marut_lincomb
composed by the binding's ssprk54_step against the oracle's step, for every physics and mesh kind."""
import numpy as np
import pytest

import workloads as wl
from parity_util import RHS_TOL, RUN_TOL, parity_error

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,cells,split", [("c1", 8, 0), ("c1", 8, 1), ("c2", 3, 0), ("c3", 3, 0), ("c4", 32, 0), ("c4", 16, 1), ("c5", 4, 0)])
def test_ssprk54_steps(name, cells, split):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    c = wl.make_case(name, cells=cells)
    c.mesh.volume_form = split
    om, gm = oracle.OracleMesh(c.mesh), mb.MarutMesh(c.mesh)
    u = torch.from_numpy(c.u0).cuda()
    ua, ub, uc = torch.empty_like(u), torch.empty_like(u), torch.empty_like(u)
    uh = c.u0
    for step in range(3):
        f = 1.0 if name == "c5" else 1.5                    # the larger step the scheme's SSP coefficient admits (not the chemistry)
        dt = f * om.max_dt(uh, c.cfl)
        assert abs(f * gm.max_dt(u, c.cfl) - dt) <= 1e-12 * dt
        uh = om.ssprk54_step(uh, dt)
        gm.ssprk54_step(u, ua, ub, uc, dt)
        torch.cuda.synchronize()
        err = parity_error(u.cpu().numpy(), uh).max()
        assert err <= (RHS_TOL if step == 0 else RUN_TOL), (step, err)
    assert np.isfinite(uh).all()
    gm.close()


def test_rk_stage_and_lincomb_arguments():
    import torch

    import paper_2605_26388_b200 as mb

    c = wl.make_case("c1", cells=4)
    gm = mb.MarutMesh(c.mesh)
    u = torch.from_numpy(c.u0).cuda()
    a, b = torch.empty_like(u), torch.empty_like(u)
    # the SSP-RK33 stage is the general stage with its table
    dt = gm.max_dt(u, 0.5)
    gm.stage(1, dt, 0.0, u, u * 1.01, a)
    gm.rk_stage(0.75, 0.25, 0.25 * dt, u, u * 1.01, b)
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    with pytest.raises(mb.MarutError):
        gm.rk_stage(1.0, 1.0, dt, u, a, a)                   # u_out aliases u_in
    with pytest.raises(mb.MarutError):
        gm.rk_stage(1.0, 1.0, dt, None, u, a)                # a != 0 needs u_a
    # lincomb, in place on one of its inputs
    x, y, z = torch.rand_like(u), torch.rand_like(u), torch.rand_like(u)
    ref = 0.3 * x - 1.7 * y + 0.25 * z
    gm.lincomb((0.3, -1.7, 0.25), (x, y, z), y)
    torch.cuda.synchronize()
    assert torch.allclose(y, ref, rtol=1e-14, atol=1e-15)
    with pytest.raises(mb.MarutError):
        gm.lincomb((1.0,) * 5, (x,) * 5, y)
    gm.close()


def test_library_steps_equal_their_stage_compositions():
    """marut_ssprk33_step / marut_ssprk54_step (host dt and device dt) against the stage-by-stage calls they are
    composed of, bit for bit; argument checks of the step calls"""
    import torch

    import paper_2605_26388_b200 as mb
    from paper_2605_26388_b200 import binding as B

    c = wl.make_case("c2", cells=3)
    gm = mb.MarutMesh(c.mesh)
    u0 = torch.from_numpy(c.u0).cuda()
    dt = gm.max_dt(u0, c.cfl)
    dt_dev = torch.tensor([dt], dtype=torch.float64, device="cuda")
    # SSP-RK33: three marut_ssprk_stage calls
    u, ua, ub, uc = u0.clone(), torch.empty_like(u0), torch.empty_like(u0), torch.empty_like(u0)
    gm.step(u, ua, ub, dt)
    v = u0.clone()
    gm.ssprk33_step(v, ua, ub, dt)
    w = u0.clone()
    gm.ssprk33_step(w, ua, ub, dt_dev=dt_dev)
    torch.cuda.synchronize()
    assert torch.equal(u, v) and torch.equal(u, w)
    # SSP-RK54: host dt against device dt, and against marut_rk_stage / marut_lincomb called one by one with the
    # published table (typed here once more, independently of the library's copy)
    a = ((1.0, 0.0, 0.391752226571890), (0.444370493651235, 0.555629506348765, 0.368410593050371),
         (0.620101851488403, 0.379898148511597, 0.251891774271694), (0.178079954393132, 0.821920045606868, 0.544974750228521))
    b = (0.517231671970585, 0.096059710526147, 0.063692468666290, 0.386708617503269, 0.226007483236906)
    x = u0.clone()
    gm.rk_stage(0.0, 1.0, a[0][2] * dt, None, x, ua)
    gm.rk_stage(a[1][0], a[1][1], a[1][2] * dt, x, ua, ub)
    gm.rk_stage(a[2][0], a[2][1], a[2][2] * dt, x, ub, ua)
    gm.rk_stage(a[3][0], a[3][1], a[3][2] * dt, x, ua, uc)
    r = b[2] / a[3][2]
    gm.lincomb((-r * a[3][0], b[0], b[1] - r * a[3][1], b[3] + r), (x, ub, ua, uc), ua)
    gm.rk_stage(1.0, 0.0, b[4] * dt, ua, uc, x)
    y, z = u0.clone(), u0.clone()
    gm.ssprk54_step(y, ua, ub, uc, dt)
    gm.ssprk54_step_dev(z, ua, ub, uc, dt_dev)
    torch.cuda.synchronize()
    assert torch.equal(x, y) and torch.equal(x, z)
    with pytest.raises(mb.MarutError):
        gm.ssprk54_step(y, ua, ua, uc, dt)                   # scratch buffers alias one another
    with pytest.raises(mb.MarutError):
        gm.ssprk33_step(y, y, ub, dt)                        # scratch aliases u
    with pytest.raises(mb.MarutError):
        B.strang_step(gm.h, y, ua, ub, dt)                   # not a reacting mesh
    gm.close()


def test_strang_step_reports_sweeps_and_poisons_unconverged_nodes():
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    c = wl.make_case("c5", cells=4)
    om, gm = oracle.OracleMesh(c.mesh), mb.MarutMesh(c.mesh)
    dt = om.max_dt(c.u0, c.cfl)
    u = torch.from_numpy(c.u0).cuda()
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    sweeps = gm.strang_step(u, ua, ub, dt, want_sweeps=True)
    assert 1 <= sweeps <= 50
    assert parity_error(u.cpu().numpy(), om.strang_step(c.u0, dt)).max() <= RHS_TOL * 100
    # a state the Newton iteration cannot handle (negative species densities at a few nodes): the unchecked call
    # leaves NaN there instead of an unconverged value, and the checked calls report it
    bad = c.u0.copy()
    bad[0, :5, :3] = -1.0
    ub_ = torch.from_numpy(bad).cuda()
    gm.strang_step(ub_, ua, ub, dt)
    torch.cuda.synchronize()
    assert torch.isnan(ub_[0, :5, :3]).all()
    with pytest.raises(mb.MarutError):
        gm.max_dt(ub_, 0.5)
    gm.close()
