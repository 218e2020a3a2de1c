"""Pins of the oracle's SSP-RK54 (SURVEY 8(f) NEXT-2b; eq. 45; reading R19): the paper gives
the scheme's properties (five stages, fourth order, Shu-Osher form with non-negative coefficients and unit row sums,
SSP coefficient ~1.508), not its coefficients -- the table is checked against exactly those properties."""
import math

import numpy as np

import oracle
import workloads as wl


def _butcher(alpha, beta):
    A = np.zeros((6, 5))                      # U^(i) = U^(0) + dt sum_j A[i][j] L(U^(j))
    for i in range(5):
        for k in range(i + 1):
            A[i + 1] += alpha[i, k] * A[k]
            A[i + 1, k] += beta[i, k]
    return A[:5], A[5]


def test_table_satisfies_eq45_constraints_fourth_order_conditions_and_the_ssp_coefficient():
    alpha, beta = oracle.ssprk54_table()
    assert (alpha >= 0).all() and (beta >= 0).all()
    assert np.allclose(alpha.sum(axis=1), 1.0, rtol=0, atol=1e-15)
    assert np.array_equal(alpha, np.tril(alpha)) and np.array_equal(beta, np.tril(beta))   # explicit
    A, b = _butcher(alpha, beta)
    c = A.sum(axis=1)
    conds = [b.sum() - 1, b @ c - 1 / 2, b @ c ** 2 - 1 / 3, b @ A @ c - 1 / 6, b @ c ** 3 - 1 / 4,
             (b * c) @ A @ c - 1 / 8, b @ A @ c ** 2 - 1 / 12, b @ A @ A @ c - 1 / 24]
    assert np.abs(conds).max() < 5e-15                                       # all eight conditions of order four
    assert abs(b @ c ** 4 - 1 / 5) > 1e-3                                    # and not of order five
    ratios = [alpha[i, k] / beta[i, k] for i in range(5) for k in range(5) if beta[i, k] > 0]
    assert abs(min(ratios) - 1.508) < 5e-4                                   # PAPER.md:725 "c ~ 1.508"


def test_scalar_ode_fourth_order_and_exact_quadrature():
    # y' = t^2 (lam = 0): a fourth-order method integrates a cubic exactly -- pins the stage abscissae
    y = oracle.ssprk54_scalar(0.3, 0.0, 2.0, 0.5, 0.7)
    assert abs(y - (0.3 + 2.0 * ((1.2 ** 3 - 0.5 ** 3) / 3.0))) < 1e-14
    errs = []
    for n in (10, 20, 40):
        dt, yv, t = 1.0 / n, 1.0, 0.0
        for _ in range(n):
            yv = oracle.ssprk54_scalar(yv, -1.5, 0.0, t, dt)
            t += dt
        errs.append(abs(yv - math.exp(-1.5)))
    assert 14 < errs[0] / errs[1] < 18 and 14 < errs[1] / errs[2] < 18
    # linear stability polynomial: exp(z) through z^4, the z^5 coefficient is not 1/120
    z = 0.1
    R = oracle.ssprk54_scalar(1.0, z, 0.0, 0.0, 1.0)
    assert abs(R - sum(z ** k / math.factorial(k) for k in range(5))) < 2e-7
    assert abs(R - math.exp(z)) > 1e-9


def test_pde_step_is_fifth_order_locally_against_a_finely_stepped_rk33():
    c = wl.make_case("c1", cells=4)
    om = oracle.OracleMesh(c.mesh)
    dt = om.max_dt(c.u0, 0.5)
    ref, _, _, _ = om.run(c.u0, 200, cfl=0.0, dt=dt / 200)
    e1 = np.abs(om.ssprk54_step(c.u0, dt) - ref).max()
    half = om.ssprk54_step(om.ssprk54_step(c.u0, dt / 2), dt / 2)
    e2 = np.abs(half - ref).max()
    e33 = np.abs(om.run(c.u0, 1, cfl=0.0, dt=dt)[0] - ref).max()
    assert e1 < e33 / 5                      # more accurate than one SSP-RK33 step of the same size
    assert 10 < e1 / e2 < 24                 # two half steps: local error 2 (dt/2)^5 -> ratio 16
