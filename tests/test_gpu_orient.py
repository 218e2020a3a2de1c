"""GPU parity on 3-D meshes whose elements' local axes are rotated at random (workloads.rotate_elements): every face
pairing and every orientation code of reading R20 (orientation tables), for
the Euler (strong / split / blended), Navier-Stokes and reacting stage kernels."""
import math

import numpy as np
import pytest

import workloads as wl
from parity_util import RHS_TOL, RUN_TOL, gpu_run, parity_error

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("N,curved,phys,split", [(1, False, "euler", 0), (2, True, "euler", 0), (3, False, "euler", 1),
                                                 (4, False, "euler", 0), (4, True, "euler", 1), (5, True, "euler", 0),
                                                 (2, True, "ns", 0), (3, False, "ns", 0), (3, False, "react", 0)])
def test_rotated_mesh_parity(N, curved, phys, split):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    cells = 4 if phys == "react" else 3       # the 3^3 reacting instance leaves its well-posed window at once
    if phys == "react":
        L = wl.C5_LENGTH * cells / 32.0
        base = wl.cartesian_mesh(3, N, (cells,) * 3, (0.0,) * 3, (L,) * 3)
        base.physics, base.mech = wl.REACTING_EULER, wl.air5_mechanism()
    else:
        lo, hi = (0.0,) * 3, (2 * math.pi,) * 3
        warp = wl.sine_warp((cells,) * 3, lo, hi, k=1) if curved else None
        base = wl.cartesian_mesh(3, N, (cells,) * 3, lo, hi, warp=warp)
        if phys == "ns":
            base.physics, base.mu, base.Pr = wl.NAVIER_STOKES, 0.02, 0.72
    base.volume_form = split
    m, node_map = wl.rotate_elements(base)
    assert len(set(m.iface[:, 4])) == 8
    u_base = wl.reacting_field(base, L) if phys == "react" else wl.taylor_green(base, noise=1e-2)
    u0 = np.ascontiguousarray(np.stack([u_base[e][:, node_map[e]] for e in range(m.n_elem)]))
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL
    if split:
        a = np.random.default_rng(2).uniform(0, 1, m.n_elem)
        om.set_blend(a)
        ad = torch.from_numpy(a).cuda()
        gm.set_blend(ad)
        gm.rhs(u, du)
        torch.cuda.synchronize()
        assert parity_error(du.cpu().numpy(), om.rhs(u0)).max() <= RHS_TOL
        om.set_blend(None)
        gm.set_blend(None)
    if phys != "react":
        al = torch.empty(m.n_elem, dtype=torch.float64, device="cuda")
        gm.shock_indicator(u, al)
        torch.cuda.synchronize()
        assert np.abs(al.cpu().numpy() - om.shock_indicator(u0)).max() <= 1e-9     # neighbour maximum over rotated faces
    ug, tg = gpu_run(gm, u0, 3, 0.4, torch)
    uc, tc, _, _ = om.run(u0, 3, cfl=0.4)
    assert abs(tg - tc) <= 1e-12 * tc
    assert parity_error(ug, uc).max() <= RUN_TOL
    gm.close()
