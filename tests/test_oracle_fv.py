"""Pins of the oracle's sub-cell finite-volume residual and the DG / FV blend (PAPER.md:187-191
eq. 11, 655-672 eq. 42; reading R16).  The interface flux itself (oracle.rusanov) is pinned in
test_oracle_pins.py; here: the sub-cell normals, the telescoping structure of R^FV with its weights and signs, free
stream on curved meshes, conservation under an arbitrary per-element blend, and the blend's linearity in alpha_e."""
import numpy as np
import pytest

import oracle
import workloads as wl


def _cons(rho, v, p, g=1.4):
    v = np.asarray(v, float)
    return np.concatenate([[rho], rho * v, [p / (g - 1) + 0.5 * rho * v @ v]])


def _flux(U, nv, g=1.4):
    d = len(nv)
    rho, m, E = U[0], U[1:1 + d], U[1 + d]
    v = m / rho
    p = (g - 1) * (E - 0.5 * rho * v @ v)
    vn = v @ nv
    return np.concatenate([[rho * vn], m * vn + p * np.asarray(nv), [(E + p) * vn]])


def _curved(dim, N, k):
    lo, hi = (0.0,) * dim, (2 * np.pi,) * dim
    return wl.cartesian_mesh(dim, N, (k,) * dim, lo, hi, warp=wl.sine_warp((k,) * dim, lo, hi, k=2))


def test_subcell_normals_telescope_and_are_constant_on_affine_elements():
    m = _curved(3, 3, 3)
    om = oracle.OracleMesh(m)
    Ja, _ = om.metrics()                      # [e][node][l][c]
    n = m.N + 1
    for e in (0, 7, 20):
        for l in range(3):
            for (a, b) in [(0, 0), (1, 2), (3, 1)]:
                ijk = [a, b]
                ijk.insert(l, 0)
                # summation by parts: sum_q w_q D_qr = delta_rN - delta_r0, so nhat_{N+1/2} = Ja^l at the line's last node
                ijk_last = list(ijk)
                ijk_last[l] = m.N
                last = ijk_last[0] + n * (ijk_last[1] + n * ijk_last[2])
                assert np.allclose(om.subcell_normal(e, l, ijk, m.N), Ja[e, last, l], rtol=0, atol=1e-13)
    ma = wl.cartesian_mesh(2, 4, (3, 2), (0.0, 0.0), (3.0, 1.0))
    oa = oracle.OracleMesh(ma)
    Jaa, _ = oa.metrics()
    for l in range(2):
        for mi in range(4):
            assert np.allclose(oa.subcell_normal(1, l, [2, 3], mi), Jaa[1, 0, l], rtol=0, atol=1e-15)


@pytest.mark.parametrize("dim,N", [(2, 3), (2, 5), (3, 3)])
def test_fv_residual_preserves_the_free_stream_on_curved_meshes(dim, N):
    m = _curved(dim, N, 3)
    om = oracle.OracleMesh(m)
    U = _cons(1.3, [0.4, -0.2, 0.7][:dim], 2.1)
    const = np.broadcast_to(U[None, :, None], (m.n_elem, dim + 2, m.nn)).copy()
    assert np.abs(om.fv_volume(const)).max() < 2e-11


@pytest.mark.parametrize("direction", [0, 1])
def test_fv_residual_telescopes_to_the_interface_fluxes(direction):
    """data varying along one reference direction only, on a Cartesian mesh with hx != hy: the other direction's sub-cell
    fluxes cancel (F*(U,U) = F(U).n), and  sum_{q<=m} w_q J R^FV_q = -( F*(U_m, U_m+1; Ja^l) - F(U_0).Ja^l )
    with F* from the separately pinned oracle.rusanov and F written out here"""
    N, n = 4, 5
    m = wl.cartesian_mesh(2, N, (3, 2), (0.0, 0.0), (3.0, 0.5))
    om = oracle.OracleMesh(m)
    Ja, J = om.metrics()
    _, w, _ = oracle.operators(N)
    rng = np.random.default_rng(11 + direction)
    line = np.array([[_cons(rng.uniform(0.5, 2), rng.uniform(-1, 1, 2), rng.uniform(0.5, 3)) for _ in range(n)]
                     for _ in range(m.n_elem)])                       # [e][q][v]
    u = np.empty((m.n_elem, 4, n, n))                                   # [e][v][j][i]
    for q in range(n):
        if direction == 0:
            u[:, :, :, q] = line[:, q, :, None]
        else:
            u[:, :, q, :] = line[:, q, :, None]
    r = om.fv_volume(u.reshape(m.n_elem, 4, n * n)).reshape(m.n_elem, 4, n, n)
    for e in range(m.n_elem):
        nv = Ja[e, 0, direction]
        assert nv[direction] > 0 and nv[1 - direction] == 0 and J[e, 0] > 0
        for other in range(n):
            acc = np.zeros(4)
            for q in range(n):
                rq = r[e, :, other, q] if direction == 0 else r[e, :, q, other]
                acc += w[q] * J[e, 0] * rq
                if q < N:
                    Fs, _ = oracle.rusanov(2, 1.4, line[e, q], line[e, q + 1], nv)
                    expect = -(Fs - _flux(line[e, 0], nv))
                else:
                    expect = -(_flux(line[e, N], nv) - _flux(line[e, 0], nv))
                assert np.allclose(acc, expect, rtol=1e-12, atol=1e-12), (e, other, q)


def test_blend_is_conservative_for_any_alpha_and_linear_in_alpha():
    m = _curved(2, 4, 4)
    m.volume_form = 1
    om = oracle.OracleMesh(m)
    _, J = om.metrics()
    _, w, _ = oracle.operators(m.N)
    W = np.einsum("j,i->ji", w, w).reshape(-1)
    X = m.node_xyz                                                        # [e][c][node]
    rho = 1.0 + 0.3 * np.sin(X[:, 0]) * np.cos(2 * X[:, 1])
    vx, vy = 0.5 + 0.2 * np.cos(X[:, 1]), -0.3 + 0.1 * np.sin(X[:, 0] + X[:, 1])
    p = 1.5 + 0.4 * np.cos(X[:, 0])
    u = np.stack([rho, rho * vx, rho * vy, p / 0.4 + 0.5 * rho * (vx ** 2 + vy ** 2)], axis=1)
    r0 = om.rhs(u)
    alpha = np.random.default_rng(5).uniform(0, 1, m.n_elem)
    alpha[:3] = [0.0, 1.0, 0.5]
    om.set_blend(alpha)
    ra = om.rhs(u)
    total = np.einsum("evn,en,n->v", ra, J, W)
    scale = np.einsum("evn,en,n->v", np.abs(ra), J, W)
    assert np.all(np.abs(total) <= 1e-12 * scale)                       # both residuals telescope to the same element-boundary fluxes
    om.set_blend(np.ones(m.n_elem))
    r1 = om.rhs(u)
    om.set_blend(np.zeros(m.n_elem))
    assert np.array_equal(om.rhs(u), r0)                                # alpha = 0 is the split form
    om.set_blend(None)
    assert np.array_equal(om.rhs(u), r0)
    a = alpha[:, None, None]
    assert np.allclose(ra, (1 - a) * r0 + a * r1, rtol=0, atol=1e-12 * np.abs(r1).max())   # eq. 11, shared surface lift
    # the field is continuous across faces, so F* = F.n there and the lift vanishes: alpha = 1 leaves R^FV alone
    assert np.allclose(r1, om.fv_volume(u), rtol=0, atol=1e-11 * np.abs(r1).max())
    assert np.abs(r1 - r0).max() > 1e-2 * np.abs(r0).max()             # and R^FV is not the DG residual


def test_pure_fv_run_converges_to_the_vortex_at_first_order():
    """alpha_e = 1 everywhere is a first-order finite-volume scheme on the sub-cell grid: to t = 1 the L1 density error of
    the isentropic vortex falls by ~1.5 - 2 per halving of h (measured 1.33e-2, 8.8e-3, 5.1e-3), far above the DG error"""
    errs, errs_dg = [], []
    _, w, _ = oracle.operators(3)
    W = np.einsum("j,i->ji", w, w).reshape(-1)
    for k in (8, 16, 32):
        c = wl.make_case("c1", cells=k)
        om = oracle.OracleMesh(c.mesh)
        _, J = om.metrics()
        steps = int(np.ceil(1.0 / om.max_dt(c.u0, 0.5)))
        dt = 1.0 / steps
        udg, t, _, _ = om.run(c.u0, steps, cfl=0.0, dt=dt)
        om.set_blend(np.ones(c.mesh.n_elem))
        ufv, t2, _, _ = om.run(c.u0, steps, cfl=0.0, dt=dt)
        assert t == t2
        exact = wl.isentropic_vortex(c.mesh, t=t)
        errs.append(np.einsum("en,en,n->", np.abs(ufv - exact)[:, 0, :], J, W) / 100.0)
        errs_dg.append(np.einsum("en,en,n->", np.abs(udg - exact)[:, 0, :], J, W) / 100.0)
    assert all(f > 3 * d for f, d in zip(errs, errs_dg)) and errs[2] > 100 * errs_dg[2]
    assert 1.3 < errs[0] / errs[1] < 2.2 and 1.5 < errs[1] / errs[2] < 2.2


def test_positivity_floor_closed_forms():
    """O18 (reading R17): hand-built nodes below / above the floors"""
    m = wl.cartesian_mesh(2, 1, (2, 1), (0.0, 0.0), (2.0, 1.0))
    om = oracle.OracleMesh(m)
    g, rmin, pmin = 1.4, 1e-6, 5e-7
    u = np.empty((2, 4, 4))
    good = _cons(1.2, [0.3, -0.4], 0.9)
    u[:] = good[None, :, None]
    u[0, :, 1] = [1e-9, 2e-7, -1e-7, 3.0]                      # density below the floor, pressure fine afterwards
    u[0, :, 2] = _cons(0.8, [2.0, 1.0], 1.0) - [0, 0, 0, 2.6]   # negative pressure (p = 1 - 0.4*2.6 < 0)
    u[1, :, 3] = [1e-8, 0.0, 0.0, 0.0]                          # both: vacuum
    u[1, :, 0] = _cons(2.0, [0.0, 0.0], pmin)                   # exactly at the pressure floor: untouched
    v, n = om.positivity_floor(u, rmin, pmin)
    assert n == 3
    untouched = np.ones((2, 4), bool)
    untouched[0, 1] = untouched[0, 2] = untouched[1, 3] = False
    assert np.array_equal(v.transpose(0, 2, 1)[untouched], u.transpose(0, 2, 1)[untouched])   # bit for bit
    a = v[0, :, 1]
    assert a[0] == rmin and np.array_equal(a[1:], u[0, 1:, 1])
    b = v[0, :, 2]
    assert np.array_equal(b[:3], u[0, :3, 2])
    assert (g - 1) * (b[3] - 0.5 * (b[1] ** 2 + b[2] ** 2) / b[0]) == pytest.approx(pmin, rel=1e-9)
    c = v[1, :, 3]
    assert c[0] == rmin and c[1] == 0 and c[2] == 0 and c[3] == pytest.approx(pmin / (g - 1), rel=1e-15)
    w, n2 = om.positivity_floor(v, rmin, pmin)                  # idempotent up to the rounding of p at the floor
    assert np.allclose(w, v, rtol=1e-15, atol=0)


def _oracle_sod(ne, capture, T=0.2):
    from sod_util import SHOCK_CAPTURE, sod_exact_on, sod_strip

    m, u = sod_strip(ne)
    om = oracle.OracleMesh(m)
    t = 0.0
    while t < T - 1e-14:
        dt = min(om.max_dt(u, 0.5), T - t)
        un, uin = u, u
        for k in range(3):
            if capture:
                om.set_blend(om.shock_indicator(uin, **SHOCK_CAPTURE))
            uin, _ = om.positivity_floor(om.ssprk_stage(k, dt, 0.0, un, uin))
        u, t = uin, t + dt
    _, J = om.metrics()
    _, w, _ = oracle.operators(m.N)
    W = np.einsum("j,i->ji", w, w).reshape(-1)
    l1 = np.einsum("en,en,n->", np.abs(u[:, 0, :] - sod_exact_on(m, T)), J, W) / (2.0 * 2.0 / ne)
    return l1, u


def test_shock_capturing_step_solves_the_sod_problem():
    """the whole shock-capturing step (indicator -> blended DG/FV stage -> floor) against the exact Riemann solution:
    first-order L1 convergence (the best a discontinuous solution allows; measured 2.15e-2, 1.13e-2), and the density /
    pressure stay within the initial bounds, where the unblended split-form DG run undershoots by 23 %"""
    from sod_util import pressure

    e32, u32 = _oracle_sod(32, True)
    e64, u64 = _oracle_sod(64, True)
    assert e32 < 0.025 and 1.6 < e32 / e64 < 2.3
    for u in (u32, u64):
        assert u[:, 0].min() > 0.125 - 1e-4 and u[:, 0].max() < 1.0 + 1e-4
        assert pressure(u).min() > 0.1 - 1e-4
    _, udg = _oracle_sod(32, False)
    assert udg[:, 0].min() < 0.11 and pressure(udg).min() < 0.08
