"""Pins of the oracle's entropy-stable split-form volume integral (eq. 10,
594-627 eq. 39-41): logarithmic mean, Ranocha two-point flux, and the split operator's structural properties."""
import math

import numpy as np
import pytest

import oracle
import workloads as wl


def test_logmean_closed_forms_and_bounds():
    assert oracle.logmean(3.7, 3.7) == pytest.approx(3.7, rel=1e-15)
    assert oracle.logmean(1.0, math.e) == pytest.approx(math.e - 1.0, rel=1e-14)            # (e - 1)/(1 - 0)
    assert oracle.logmean(2.0, 8.0) == pytest.approx(6.0 / math.log(4.0), rel=1e-14)
    for a, b in [(1.0, 1.0 + 1e-9), (0.3, 0.31), (5.0, 0.01), (1e-3, 2e-3)]:
        m = oracle.logmean(a, b)
        assert m == pytest.approx(oracle.logmean(b, a), rel=1e-14)                             # symmetric
        assert min(a, b) <= m <= 0.5 * (a + b) * (1 + 1e-15)                                   # <= arithmetic mean
        assert m >= math.sqrt(a * b) * (1 - 1e-15)                                             # >= geometric mean
    # the series and the logarithm branch agree where they meet (u = f^2 = 1e-2  <->  zeta = 11/9)
    z = 11.0 / 9.0
    lo, hi = oracle.logmean(z * (1 - 1e-9), 1.0), oracle.logmean(z * (1 + 1e-9), 1.0)
    exact = (z - 1.0) / math.log(z)
    assert lo == pytest.approx(exact, rel=1e-8) and hi == pytest.approx(exact, rel=1e-8)
    assert abs(oracle.logmean(z * (1 - 1e-13), 1.0) / exact - 1) < 2e-9                        # series truncation error at the switch


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


@pytest.mark.parametrize("dim", [2, 3])
def test_ranocha_consistency_symmetry_and_worked_value(dim):
    rng = np.random.default_rng(7)
    for _ in range(20):
        U = _cons(rng.uniform(0.2, 3), rng.uniform(-2, 2, dim), rng.uniform(0.2, 5))
        V = _cons(rng.uniform(0.2, 3), rng.uniform(-2, 2, dim), rng.uniform(0.2, 5))
        nv = rng.uniform(-1, 1, dim)
        # eq. 40: F#(U,U) = F_inv(U) -- this pins the factor in the energy term (reading R13)
        assert np.allclose(oracle.ranocha(dim, 1.4, U, U, nv), _flux(U, nv), rtol=1e-13, atol=1e-14)
        assert np.allclose(oracle.ranocha(dim, 1.4, U, V, nv), oracle.ranocha(dim, 1.4, V, U, nv), rtol=1e-14, atol=1e-15)
        # linear in the (averaged metric) vector
        assert np.allclose(oracle.ranocha(dim, 1.4, U, V, 2.5 * nv), 2.5 * oracle.ranocha(dim, 1.4, U, V, nv), rtol=1e-13)
    # worked value, the flux of reading R13 written out by hand: rho 1|2, u 1|0, v 0, p 1|2 (rho/p = 1|1), n = e_x:
    # f_rho = {{rho}}^ln {{u}}, F_m = f_rho {{u}} + {{p}}, F_E = f_rho (1/(gamma-1) + 1/2 u_L u_R) + 1/2 (p_L u_R + p_R u_L)
    UL, UR = _cons(1.0, [1.0] + [0.0] * (dim - 1), 1.0), _cons(2.0, [0.0] * dim, 2.0)
    rl = 1.0 / math.log(2.0)
    F = oracle.ranocha(dim, 1.4, UL, UR, [1.0] + [0.0] * (dim - 1))
    assert F[0] == pytest.approx(rl * 0.5, rel=1e-14)
    assert F[1] == pytest.approx(rl * 0.25 + 1.5, rel=1e-14)
    assert F[-1] == pytest.approx((1.0 / 0.4 + 0.0) * rl * 0.5 + 1.0, rel=1e-14)


def _split(case):
    case.mesh.volume_form = 1
    return oracle.OracleMesh(case.mesh)


def test_split_form_free_stream_and_conservation():
    c = wl.make_case("c3", cells=3)
    c.mesh.physics, c.mesh.mu = wl.EULER, 0.0
    om = _split(c)
    _, J = om.metrics()
    _, w, _ = oracle.operators(c.mesh.N)
    W = np.einsum("k,j,i->kji", w, w, w).reshape(-1)
    const = np.broadcast_to(_cons(1.3, [0.4, -0.2, 0.7], 2.1)[None, :, None], c.u0.shape).copy()
    assert np.abs(om.rhs(const)).max() < 2e-11                       # free stream on the curved mesh (discrete GCL)
    du = om.rhs(c.u0)
    total = np.einsum("evn,en,n->v", du, J, W)
    scale = np.einsum("evn,en,n->v", np.abs(du), J, W)
    assert np.all(np.abs(total) <= 1e-12 * scale)                    # conservation (SBP + symmetric two-point flux)


def test_split_form_converges_to_the_strong_form_and_to_the_vortex():
    errs, errs_strong, diffs = [], [], []
    for k in (8, 16):
        c = wl.make_case("c1", cells=k)
        strong_mesh = oracle.OracleMesh(c.mesh)
        strong = strong_mesh.rhs(c.u0)
        om = _split(c)
        diffs.append(np.abs(om.rhs(c.u0) - strong).max())
        dt = 0.2 * om.max_dt(c.u0, 0.5)
        u, t, _, _ = om.run(c.u0, 10, cfl=0.0, dt=dt)
        u2, _, _, _ = strong_mesh.run(c.u0, 10, cfl=0.0, dt=dt)
        exact = wl.isentropic_vortex(c.mesh, t=t)
        errs.append(np.abs(u - exact)[:, 0, :].max())
        errs_strong.append(np.abs(u2 - exact)[:, 0, :].max())
    assert diffs[1] < diffs[0] / 4            # the two volume forms differ by truncation error only (0.243 -> 0.054)
    assert errs[1] < errs[0] / 5              # the split form keeps the high order (8.5e-3 -> 1.2e-3)
    assert all(abs(a / b - 1) < 0.3 for a, b in zip(errs, errs_strong))   # and the accuracy of the strong form


def _entropy_vars(U, g=1.4):
    """entropy variables w = dS/dU of S = -rho s/(gamma-1), s = ln p - gamma ln rho, and the entropy potential
    psi = rho v (textbook: Tadmor's condition [[w]].F# = [[psi]].n characterises entropy-conservative fluxes)"""
    d = len(U) - 2
    rho, m, E = U[0], U[1:1 + d], U[1 + d]
    v = m / rho
    p = (g - 1) * (E - 0.5 * rho * v @ v)
    s = math.log(p) - g * math.log(rho)
    w = np.concatenate([[(g - s) / (g - 1) - 0.5 * rho * (v @ v) / p], rho * v / p, [-rho / p]])
    return w, m


@pytest.mark.parametrize("dim", [2, 3])
def test_ranocha_flux_is_entropy_conservative_and_kinetic_energy_preserving(dim):
    """PAPER.md:611 names 'the kinetic energy preserving and entropy-conservative flux of Ranocha [19]'.  Entropy
    conservation is Tadmor's condition (w_R - w_L).F#(U_L, U_R; n) = (psi_R - psi_L).n; kinetic-energy preservation in
    Ranocha's sense is F_m = {{v}} F_rho + {{p}} n.  The energy flux as PAPER.md:621 prints it ({{v}}^2 kinetic term,
    {{p v}} pressure work) violates the first by O(jump^2): reading R13 takes the stated property."""
    rng = np.random.default_rng(11)
    for _ in range(50):
        UL = _cons(rng.uniform(0.2, 3), rng.uniform(-2, 2, dim), rng.uniform(0.2, 5))
        UR = _cons(rng.uniform(0.2, 3), rng.uniform(-2, 2, dim), rng.uniform(0.2, 5))
        nv = rng.uniform(-1, 1, dim)
        F = oracle.ranocha(dim, 1.4, UL, UR, nv)
        wL, mL = _entropy_vars(UL)
        wR, mR = _entropy_vars(UR)
        lhs, rhs = (wR - wL) @ F, (mR - mL) @ nv
        scale = np.abs(wR - wL) @ np.abs(F) + abs(rhs) + 1e-300
        # to the accuracy of the logarithmic mean's series branch (truncation <= 2e-9, test_logmean_...), round-off
        # on the logarithm branch; the printed energy flux misses by O(jump^2) ~ 0.1
        assert abs(lhs - rhs) <= 1e-8 * scale
        vavg = 0.5 * (UL[1:1 + dim] / UL[0] + UR[1:1 + dim] / UR[0])
        pavg = 0.5 * (0.4 * (UL[-1] - 0.5 * UL[1:1 + dim] @ UL[1:1 + dim] / UL[0]) + 0.4 * (UR[-1] - 0.5 * UR[1:1 + dim] @ UR[1:1 + dim] / UR[0]))
        assert np.allclose(F[1:1 + dim], vavg * F[0] + pavg * nv, rtol=1e-13, atol=1e-14)
    # worked value with a velocity AND a pressure jump (the terms the printed formula gets wrong):
    # rho 1|1, u 1|0, p 1|2, n = e_x:  F_E = f_rho (1/((g-1) {{rho/p}}^ln) + 1/2 uL uR) + 1/2 (pL uR + pR uL)
    UL, UR = _cons(1.0, [1.0] + [0.0] * (dim - 1), 1.0), _cons(1.0, [0.0] * dim, 2.0)
    F = oracle.ranocha(dim, 1.4, UL, UR, [1.0] + [0.0] * (dim - 1))
    beta_ln = (1.0 - 0.5) / math.log(2.0)                # {{rho/p}}^ln of 1 and 1/2
    assert F[0] == pytest.approx(0.5, rel=1e-14)
    assert F[-1] == pytest.approx(0.5 * (1.0 / (0.4 * beta_ln) + 0.0) + 0.5 * (1.0 * 0.0 + 2.0 * 1.0), rel=1e-14)


def test_split_form_semi_discrete_entropy_rate_is_the_interface_dissipation():
    """With an entropy-conservative volume flux and the SBP operator the entropy rate of the semi-discretisation,
    sum_e sum_i J_i W_i w(U_i).dU_i/dt, comes from the interfaces alone (PAPER.md:627 'globally nonlinearly
    entropy-stable'): it equals  sum_faces sum_j omega_j ( [[w]].F* - [[psi]].n )  with F* from the separately pinned
    Rusanov routine, [[a]] = a+ - a-, n the scaled normal from - to +, and it is <= 0.  A rough (element-wise random)
    field makes every volume term large; a volume flux that is not entropy conservative breaks the identity at O(1)."""
    c = wl.make_case("c1", cells=5)
    m = c.mesh
    om = _split(c)
    _, J = om.metrics()
    n = m.N + 1
    _, w, _ = oracle.operators(m.N)
    w = np.asarray(w)
    W = np.einsum("j,i->ji", w, w).reshape(-1)
    rng = np.random.default_rng(3)
    u = c.u0.copy()
    u[:, 0, :] *= 1.0 + 0.2 * rng.uniform(-1, 1, u[:, 0, :].shape)
    u[:, 1, :] += 0.3 * rng.uniform(-1, 1, u[:, 1, :].shape)
    u[:, 3, :] *= 1.0 + 0.2 * rng.uniform(-1, 1, u[:, 3, :].shape)
    du = om.rhs(u)
    rate = sum(J[e, i] * W[i] * (_entropy_vars(u[e, :, i])[0] @ du[e, :, i]) for e in range(u.shape[0]) for i in range(n * n))
    h = 10.0 / 5

    def face_nodes(f):
        l, s = f >> 1, (n - 1 if f & 1 else 0)
        return [s + n * a for a in range(n)] if l == 0 else [a + n * s for a in range(n)]

    prod = 0.0
    for eL, fL, eR, fR, orient in np.asarray(m.iface):
        nL, nR = face_nodes(fL), face_nodes(fR)
        if orient:
            nR = nR[::-1]
        nv = np.zeros(2)
        nv[fL >> 1] = (1.0 if fL & 1 else -1.0) * h / 2      # scaled outward normal of the left element (affine: Ja^l)
        for j in range(n):
            Um, Up = u[eL, :, nL[j]], u[eR, :, nR[j]]
            Fs, _ = oracle.rusanov(2, 1.4, Um, Up, nv)
            wm, mm = _entropy_vars(Um)
            wp, mp = _entropy_vars(Up)
            prod += w[j] * ((wp - wm) @ Fs - (mp - mm) @ nv)
    assert prod < 0.0
    assert abs(rate - prod) <= 1e-9 * abs(prod)      # the series branch of the logarithmic mean again (1.2e-11 here)


def test_split_form_and_blend_with_the_viscous_terms():
    """'Three operators are available and selected once at solver setup' -- the split form and the
    DG/FV blend replace the HYPERBOLIC volume integral; the parabolic RHS (Table 2) is added unchanged.
    On the curved periodic Navier-Stokes mesh of config 3: free stream, conservation of mass, momentum and energy with a
    random blending field, and the viscous contribution (difference to the Euler operator on the same mesh) equal for
    the three volume operators."""
    c = wl.make_case("c3", cells=3)
    rng = np.random.default_rng(9)
    alpha = rng.uniform(0, 1, c.mesh.n_elem)
    u = wl.taylor_green(c.mesh, noise=1e-2)

    def operators(physics, mu):
        out = []
        for form, a in ((0, None), (1, None), (1, alpha)):
            c.mesh.physics, c.mesh.mu, c.mesh.volume_form = physics, mu, form
            om = oracle.OracleMesh(c.mesh)
            om.set_blend(a)
            out.append(om)
        return out

    ns = operators(wl.NAVIER_STOKES, 1.0 / 100.0)
    eu = operators(wl.EULER, 0.0)
    _, J = ns[0].metrics()
    _, w, _ = oracle.operators(c.mesh.N)
    W = np.einsum("k,j,i->kji", w, w, w).reshape(-1)
    const = np.broadcast_to(_cons(1.3, [0.4, -0.2, 0.7], 2.1)[None, :, None], u.shape).copy()
    visc = []
    for om_ns, om_eu in zip(ns, eu):
        assert np.abs(om_ns.rhs(const)).max() < 2e-11
        r = om_ns.rhs(u)
        total = np.einsum("evn,en,n->v", r, J, W)
        scale = np.einsum("evn,en,n->v", np.abs(r), J, W)
        assert np.all(np.abs(total) <= 1e-12 * scale)
        visc.append(r - om_eu.rhs(u))
    assert np.abs(visc[0]).max() > 1e-3
    assert np.abs(visc[1] - visc[0]).max() <= 1e-12 * np.abs(ns[0].rhs(u)).max()
    assert np.abs(visc[2] - visc[0]).max() <= 1e-12 * np.abs(ns[0].rhs(u)).max()
    c.mesh.volume_form = 0
