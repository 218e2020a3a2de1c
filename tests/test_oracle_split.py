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
    # worked value, eq. 41 written out by hand: rho 1|2, u 1|0, v 0, p 1|2 (T^-1 = 1|1), n = e_x
    UL, UR = _cons(1.0, [1.0] + [0.0] * (dim - 1), 1.0), _cons(2.0, [0.0] * dim, 2.0)
    rl = 1.0 / math.log(2.0)
    F = oracle.ranocha(dim, 1.4, UL, UR, [1.0] + [0.0] * (dim - 1))
    assert F[0] == pytest.approx(rl * 0.5, rel=1e-14)
    assert F[1] == pytest.approx(rl * 0.25 + 1.5, rel=1e-14)
    assert F[-1] == pytest.approx((1.0 / 0.4 + 0.125) * rl * 0.5 + 0.5, rel=1e-14)


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
    assert diffs[1] < diffs[0] / 5            # the two volume forms differ by truncation error only (0.236 -> 0.040)
    assert errs[1] < errs[0] / 5              # the split form keeps the high order (8.5e-3 -> 1.2e-3)
    assert all(abs(a / b - 1) < 0.3 for a, b in zip(errs, errs_strong))   # and the accuracy of the strong form
