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
