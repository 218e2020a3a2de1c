"""GPU parity of the blended DG / sub-cell finite-volume volume residual (PAPER.md:187-191
eq. 11, 655-672 eq. 42; R16): marut_set_blend + marut_rhs / marut_ssprk_stage against the oracle, element by
element, on affine and curved meshes in 2-D and 3-D, the quadtree mortar mesh, and the shock-capturing composition
indicator -> blend -> stage on the Mach-10 shock."""
import math

import numpy as np
import pytest

import workloads as wl
from parity_util import RHS_TOL, RUN_TOL, gpu_run, parity_error

pytestmark = pytest.mark.gpu


def _mesh(dim, N, cells, curved):
    lo, hi = (0.0,) * dim, ((10.0,) * 2 if dim == 2 else (2 * math.pi,) * 3)
    counts = (cells,) * dim
    warp = wl.sine_warp(counts, lo, hi, k=1) if curved else None
    return wl.cartesian_mesh(dim, N, counts, lo, hi, warp=warp)


def _alpha(ne, seed=3):
    a = np.random.default_rng(seed).uniform(0.0, 1.0, ne)
    a[0], a[1], a[ne - 1] = 0.0, 1.0, 1.0          # pure DG, pure FV, and the (ragged) last CTA
    return a


CASES = [(2, N, 5, curved) for N in (1, 2, 3, 4, 5) for curved in (False, True)] + \
        [(3, N, 3, curved) for N in (1, 2, 3, 4, 5) for curved in (False, True)] + [(3, 6, 2, True), (2, 7, 3, True)]


@pytest.mark.parametrize("dim,N,cells,curved", CASES)
def test_blended_rhs_and_stage(dim, N, cells, curved):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m = _mesh(dim, N, cells, curved)
    m.volume_form = 1
    u0 = wl.isentropic_vortex(m) if dim == 2 else wl.taylor_green(m, noise=1e-2)
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    a = _alpha(m.n_elem)
    om.set_blend(a)
    ad = torch.from_numpy(a).cuda()
    gm.set_blend(ad)
    u = torch.from_numpy(u0).cuda()
    du = torch.empty_like(u)
    gm.rhs(u, du)
    torch.cuda.synchronize()
    ref = om.rhs(u0)
    assert parity_error(du.cpu().numpy(), ref).max() <= RHS_TOL
    om.set_blend(None)
    assert np.abs(ref - om.rhs(u0)).max() > 1e-3 * np.abs(ref).max()       # the blend is not a no-op on this input
    om.set_blend(a)
    dt = om.max_dt(u0, 0.5)
    un_h = u0 * (1.0 + 1e-3)
    out = torch.empty_like(u)
    gm.stage(2, dt, 0.0, torch.from_numpy(un_h).cuda(), u, out)
    torch.cuda.synchronize()
    assert parity_error(out.cpu().numpy(), om.ssprk_stage(2, dt, 0.0, un_h, u0)).max() <= RHS_TOL
    # the pointer is kept: rewriting the field takes effect at the next call; alpha = 0 is the split form bit for bit
    ad.zero_()
    gm.rhs(u, du)
    gm.set_blend(None)
    du0 = torch.empty_like(u)
    gm.rhs(u, du0)
    torch.cuda.synchronize()
    assert torch.equal(du, du0)
    gm.close()


def test_blend_needs_the_split_form():
    import torch

    import paper_2605_26388_b200 as mb

    m = _mesh(2, 3, 4, False)
    gm = mb.MarutMesh(m)
    u = torch.from_numpy(wl.isentropic_vortex(m)).cuda()
    gm.set_blend(torch.zeros(m.n_elem, dtype=torch.float64, device="cuda"))
    with pytest.raises(mb.MarutError):
        gm.rhs(u, torch.empty_like(u))
    gm.set_blend(None)
    gm.rhs(u, torch.empty_like(u))
    gm.close()
    rc = wl.make_case("c5", cells=3)                 # reacting meshes have no blend (Navier-Stokes ones do: test_gpu_ns_split.py)
    gn = mb.MarutMesh(rc.mesh)
    with pytest.raises(mb.MarutError):
        gn.set_blend(torch.zeros(rc.mesh.n_elem, dtype=torch.float64, device="cuda"))
    gn.close()


@pytest.mark.parametrize("name,cells,width", [("c4", 16, 6.0), ("c4", 32, 6.0), ("c4w", None, 1.0)])
def test_shock_capturing_composition_on_the_mortar_mesh(name, cells, width):
    """Mach-10 shock on the quadtree mesh (2:1 mortars, boundary states): per stage alpha = indicator(u), then the blended
    stage -- the order the paper states -- for a few SSP-RK33 steps on both sides.  ("c4w", None, 1.0) is
    the full-size instance bench.py times as workload c4b (~250K elements; shock profile one fine element wide, which the
    indicator flags where the 6-element profile of c4 / c4w is resolved and gives alpha = 0), every element compared."""
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    c = wl.make_case(name, cells=cells)
    c.mesh.volume_form = 1
    c.u0 = wl.mach10_shock(c.mesh, half_width=width * c.mesh.info["h_fine"])
    om, gm = oracle.OracleMesh(c.mesh), mb.MarutMesh(c.mesh)
    ne = c.mesh.n_elem
    kw = dict(s=9.21024, alpha_min=1e-3, alpha_max=0.5, smooth=True)
    u = torch.from_numpy(c.u0).cuda()
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    alpha = torch.zeros(ne, dtype=torch.float64, device="cuda")
    gm.set_blend(alpha)
    uh = c.u0.copy()
    seen = 0.0
    for _ in range(3):
        dt = om.max_dt(uh, c.cfl)
        assert abs(gm.max_dt(u, c.cfl) - dt) <= 1e-12 * dt
        # oracle: three stages, each with its own indicator field
        stage_in, un = uh, uh
        gin = u
        for k, gout in zip(range(3), (ua, ub, u)):
            a_h = om.shock_indicator(stage_in, **kw)
            om.set_blend(a_h)
            gm.shock_indicator(gin, alpha, **kw)
            torch.cuda.synchronize()
            assert np.abs(alpha.cpu().numpy() - a_h).max() <= 1e-9
            seen = max(seen, a_h.max())
            stage_in, n_h = om.positivity_floor(om.ssprk_stage(k, dt, 0.0, un, stage_in))
            gm.stage(k, dt, 0.0, u, gin, gout)
            assert gm.positivity_floor(gout, want_count=True) == n_h           # per-stage floor
            gin = gout
        uh = stage_in
    torch.cuda.synchronize()
    assert seen == 0.5                                                     # the shock saturates the indicator at alpha_max
    assert parity_error(u.cpu().numpy(), uh).max() <= RUN_TOL
    assert uh[:, 0, :].min() > 0
    gm.close()


@pytest.mark.parametrize("dim,N,cells,ns", [(2, 3, 9, False), (3, 4, 3, False), (3, 2, 4, True)])
def test_positivity_floor(dim, N, cells, ns):
    """marut_positivity_floor against the oracle (reading R17): a smooth field with seeded nodes pushed below the density
    floor, below the pressure floor, and into vacuum; untouched nodes bit for bit, the count exactly"""
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    m = _mesh(dim, N, cells, False)
    if ns:
        m.physics, m.mu = wl.NAVIER_STOKES, 0.01
    u0 = (wl.isentropic_vortex(m) if dim == 2 else wl.taylor_green(m, noise=1e-2)).copy()
    rng = np.random.default_rng(17)
    ne, nn = m.n_elem, m.nn
    pick = rng.random((ne, nn))
    low_rho, low_p, vac = pick < 0.05, (pick >= 0.05) & (pick < 0.12), (pick >= 0.12) & (pick < 0.15)
    u0[:, 0, :][low_rho] = 1e-6 * rng.uniform(0.01, 0.99, low_rho.sum())
    u0[:, dim + 1, :][low_p] *= rng.uniform(-0.5, -0.01, low_p.sum())
    for v in range(dim + 2):
        u0[:, v, :][vac] = 1e-9 * rng.uniform(-1, 1, vac.sum())
    u0[:, 0, :][vac] = 1e-9
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    ref, n_ref = om.positivity_floor(u0)
    assert n_ref >= (low_rho | low_p | vac).sum() > 10
    u = torch.from_numpy(u0).cuda()
    n = gm.positivity_floor(u, want_count=True)
    g = u.cpu().numpy()
    assert n == n_ref
    same = ref == u0
    assert np.array_equal(g[same], u0[same])
    assert np.allclose(g, ref, rtol=1e-14, atol=0)
    gm.positivity_floor(u)                                                # without the count: no synchronisation, same result
    torch.cuda.synchronize()
    assert np.allclose(u.cpu().numpy(), ref, rtol=1e-14, atol=0)
    with pytest.raises(mb.MarutError):
        gm.positivity_floor(u, rho_min=0.0)
    gm.close()


def test_shock_capturing_step_solves_the_sod_problem_on_the_gpu():
    """property at a size the oracle is not run at: 256 x 4 elements, the whole shock-capturing step through the C ABI to
    t = 0.2 against the exact Riemann solution (tests/sod_util.py); the first steps element by element against the
    oracle"""
    import torch

    import oracle
    import paper_2605_26388_b200 as mb
    from sod_util import SHOCK_CAPTURE, pressure, sod_exact_on, sod_strip

    def gpu_step(gm, u, ua, ub, alpha, dt):
        for k, (uin, uout) in enumerate(((u, ua), (ua, ub), (ub, u))):
            gm.shock_indicator(uin, alpha, **SHOCK_CAPTURE)
            gm.stage(k, dt, 0.0, u, uin, uout)
            gm.positivity_floor(uout)

    # parity of the first steps (small strip)
    m, u0 = sod_strip(32, rows=2)
    om, gm = oracle.OracleMesh(m), mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    alpha = torch.zeros(m.n_elem, dtype=torch.float64, device="cuda")
    gm.set_blend(alpha)
    uh = u0
    for _ in range(5):
        dt = om.max_dt(uh, 0.5)
        un, uin = uh, uh
        for k in range(3):
            om.set_blend(om.shock_indicator(uin, **SHOCK_CAPTURE))
            uin, _ = om.positivity_floor(om.ssprk_stage(k, dt, 0.0, un, uin))
        uh = uin
        gpu_step(gm, u, ua, ub, alpha, dt)
    torch.cuda.synchronize()
    g = u.cpu().numpy()
    assert np.abs(uh[:, 2]).max() < 1e-14 and np.abs(g[:, 2]).max() < 1e-14      # rho*v is round-off on both sides:
    g[:, 2], uh[:, 2] = 0.0, 0.0                                                   # no scale of its own to compare against
    assert parity_error(g, uh).max() <= RUN_TOL
    gm.close()

    # the full run against the exact solution
    ne, T = 256, 0.2
    m, u0 = sod_strip(ne, rows=4)
    gm = mb.MarutMesh(m)
    u = torch.from_numpy(u0).cuda()
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    alpha = torch.zeros(m.n_elem, dtype=torch.float64, device="cuda")
    gm.set_blend(alpha)
    t = 0.0
    while t < T - 1e-14:
        dt = min(gm.max_dt(u, 0.5), T - t)
        gpu_step(gm, u, ua, ub, alpha, dt)
        t += dt
    g = u.cpu().numpy()
    _, J = gm.metrics()
    _, w, _ = oracle.operators(m.N)
    W = np.einsum("j,i->ji", w, w).reshape(-1)
    l1 = np.einsum("en,en,n->", np.abs(g[:, 0, :] - sod_exact_on(m, T)), J, W) / (2.0 * 4 * 2.0 / ne)
    print(f"Sod, {ne} x 4 elements: L1 density error {l1:.3e}")
    assert l1 < 4.0e-3                                    # first order from 1.13e-2 at 64 elements: ~2.8e-3
    assert g[:, 0].min() > 0.125 - 1e-4 and g[:, 0].max() < 1.0 + 1e-4 and pressure(g).min() > 0.1 - 1e-4
    assert np.abs(g[:, 2]).max() < 1e-10                  # the strip stays one-dimensional
    gm.close()
