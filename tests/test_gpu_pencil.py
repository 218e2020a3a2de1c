"""GPU parity of the persistent line kernel (csrc/marut_pencil.cuh: TMA-fed tiles, one thread per line) that runs the
strong-form Euler stage on affine meshes.  The library picks it by itself only for meshes that fill
the device, so the small cases select it through marut_debug_stage_kernel; every case is also run with the
thread-per-node kernel, and both are compared with the oracle (RHS, the three SSP-RK33 stage kinds with u_out aliasing
u_n in the last one, a few steps).  Mesh sizes are chosen to hit the kernel's paths: several tiles per CTA (the ring
wraps), a ragged last tile, an odd-sized state array (last tile copied by the threads instead of TMA), neighbours
inside and outside the tile, boundary faces, 2-D mortars, rotated 3-D orientations."""
import math

import numpy as np
import pytest

import workloads as wl
from parity_util import RHS_TOL, RUN_TOL, gpu_run, parity_error

pytestmark = pytest.mark.gpu


def _compare(m, u0, steps=2, cfl=0.4):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    om = oracle.OracleMesh(m)
    du_c = om.rhs(u0)
    dt = om.max_dt(u0, cfl)
    un_h = u0 * (1.0 + 1e-3)
    stages_c = [om.ssprk_stage(s, dt, 0.0, un_h, u0) for s in range(3)]
    uc, tc, _, _ = om.run(u0, steps, cfl=cfl)
    for which in (2, 1):
        gm = mb.MarutMesh(m)
        gm.debug_stage_kernel(which)
        u = torch.from_numpy(u0).cuda()
        du = torch.empty_like(u)
        gm.rhs(u, du)
        torch.cuda.synchronize()
        assert parity_error(du.cpu().numpy(), du_c).max() <= RHS_TOL, which
        for s in range(3):
            un = torch.from_numpy(un_h).cuda()
            out = un if s == 2 else torch.empty_like(u)      # the last stage writes over u_n (own-node dependence only)
            gm.stage(s, dt, 0.0, un, u, out)
            torch.cuda.synchronize()
            assert parity_error(out.cpu().numpy(), stages_c[s]).max() <= RHS_TOL, (which, s)
        ug, tg = gpu_run(gm, u0, steps, cfl, torch)
        assert abs(tg - tc) <= 1e-12 * tc
        assert parity_error(ug, uc).max() <= RUN_TOL, which
        gm.close()


@pytest.mark.parametrize("dim,N,cells", [(2, 1, 9), (2, 2, 7), (2, 3, 13), (2, 4, 7), (2, 5, 6), (2, 6, 5), (2, 7, 5),
                                         (3, 1, 5), (3, 2, 5), (3, 3, 5), (3, 4, 3), (3, 5, 3)])
def test_small_periodic_meshes_every_degree(dim, N, cells):
    lo, hi = (0.0,) * dim, ((10.0,) * 2 if dim == 2 else (2 * math.pi,) * 3)
    m = wl.cartesian_mesh(dim, N, (cells,) * dim, lo, hi)
    u0 = wl.isentropic_vortex(m) if dim == 2 else wl.taylor_green(m, noise=1e-2)
    _compare(m, u0)


def test_ring_wraps_and_ragged_tail_3d_n4():
    # 14^3 = 2744 elements = 549 tiles of 5 (last one ragged) on 444 resident CTAs: the two-slot ring wraps, and
    # 2744 * 625 doubles is even, so every tile comes in by TMA
    m = wl.cartesian_mesh(3, 4, (14,) * 3, (0.0,) * 3, (2 * math.pi,) * 3)
    _compare(m, wl.taylor_green(m, noise=1e-3), steps=2)


@pytest.mark.parametrize("N,cells", [(4, 19), (2, 27)])
def test_tiles_drawn_from_the_device_counter_3d(N, cells):
    # more than three tiles per resident CTA (444 CTAs): beyond its first three tiles a CTA draws the rest from the
    # device-wide counter, which the last CTA to finish resets (N = 4: 19^3 = 6859 elements = 1372 tiles, odd-sized
    # array: the last tile without TMA; N = 2: 27^3 = 19683 elements = 1406 tiles of 14); RHS, the three stage kinds and
    # two steps run back to back on one handle, so every launch relies on the reset of the one before
    m = wl.cartesian_mesh(3, N, (cells,) * 3, (0.0,) * 3, (2 * math.pi,) * 3)
    _compare(m, wl.taylor_green(m, noise=1e-3), steps=2)


def test_odd_sized_array_last_tile_without_tma_3d_n4():
    # 11^3 = 1331 elements: 1331 * 625 doubles is odd: the last tile's 16-byte window would leave the array
    m = wl.cartesian_mesh(3, 4, (11,) * 3, (0.0,) * 3, (2 * math.pi,) * 3)
    _compare(m, wl.taylor_green(m, noise=1e-3), steps=2)


def test_mortars_and_boundary_faces_2d():
    c = wl.make_case("c4", cells=32, steps=3)
    assert len(c.mesh.mortar) > 0 and len(c.mesh.bface) > 0
    _compare(c.mesh, c.u0, steps=3, cfl=c.cfl)


@pytest.mark.parametrize("N", [2, 4])
def test_rotated_orientations_3d(N):
    base = wl.cartesian_mesh(3, N, (4,) * 3, (0.0,) * 3, (2 * math.pi,) * 3)
    m, node_map = wl.rotate_elements(base)
    u_base = wl.taylor_green(base, noise=1e-2)
    u0 = np.ascontiguousarray(np.stack([u_base[e][:, node_map[e]] for e in range(m.n_elem)]))
    _compare(m, u0)
