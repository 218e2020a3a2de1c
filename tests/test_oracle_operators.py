"""Pins for the oracle's 1-D operators, mortar matrices, pointwise fluxes and SSPRK3
(O1, O5, O7, O10).  CPU only."""
import math
import os

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    rows = {}
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        rows[k] = np.array([float(t) for t in v])
    return rows


def test_lgl_closed_forms():
    x, w, D = oracle.operators(3)
    assert np.allclose(x, [-1, -1 / math.sqrt(5), 1 / math.sqrt(5), 1], atol=1e-15)
    assert np.allclose(w, [1 / 6, 5 / 6, 5 / 6, 1 / 6], atol=1e-15)
    x, w, D = oracle.operators(4)
    assert np.allclose(x, [-1, -math.sqrt(3 / 7), 0, math.sqrt(3 / 7), 1], atol=1e-15)
    assert np.allclose(w, [1 / 10, 49 / 90, 32 / 45, 49 / 90, 1 / 10], atol=1e-15)


def test_D_golden_rows():
    g = _gold("operators_N3_N4.txt")
    _, _, D3 = oracle.operators(3)
    _, _, D4 = oracle.operators(4)
    assert np.allclose(D3[0], g["N3_D0"], atol=1e-11)
    assert np.allclose(D3[1], g["N3_D1"], atol=1e-11)
    assert abs(D4[0, 0] - g["N4_D00"][0]) < 1e-12
    assert np.allclose(D4[2], g["N4_D2"], atol=1e-11)


@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6, 7])
def test_D_properties(N):
    x, w, D = oracle.operators(N)
    n = N + 1
    assert abs(w.sum() - 2.0) < 1e-14
    assert np.abs(D @ np.ones(n)).max() < 1e-13  # D 1 = 0
    for k in range(1, N + 1):  # exact on polynomials of degree <= N
        assert np.abs(D @ x ** k - k * x ** (k - 1)).max() < 1e-11
    Q = np.diag(w) @ D  # SBP: Q + Q^T = diag(-1,0,..,0,1)
    B = np.zeros((n, n))
    B[0, 0], B[-1, -1] = -1.0, 1.0
    assert np.abs(Q + Q.T - B).max() < 1e-13
    # quadrature exact to degree 2N-1
    for k in range(0, 2 * N):
        exact = 0.0 if k % 2 else 2.0 / (k + 1)
        assert abs(w @ x ** k - exact) < 1e-13


def test_mortar_golden_and_identities():
    g = _gold("mortar_N3.txt")
    Pf_lo, Pf_up, Pr_lo, Pr_up = oracle.mortar_matrices(3)
    assert np.allclose(Pf_lo[1], g["Pfwd_lo_1"], atol=1e-11)
    assert np.allclose(Pf_lo[3], g["Pfwd_lo_3"], atol=1e-11)
    assert np.allclose(Pr_lo[0], g["Prev_lo_0"], atol=1e-11)
    assert np.allclose(Pr_lo[3], g["Prev_lo_3"], atol=1e-11)


@pytest.mark.parametrize("N", [1, 2, 3, 4, 5])
def test_mortar_identities(N):
    x, w, _ = oracle.operators(N)
    n = N + 1
    Pf_lo, Pf_up, Pr_lo, Pr_up = oracle.mortar_matrices(N)
    one = np.ones(n)
    assert np.abs(Pr_lo @ Pf_lo + Pr_up @ Pf_up - np.eye(n)).max() < 1e-13  # (i) project(interp) = id
    assert np.abs(w @ Pr_lo - 0.5 * w).max() < 1e-14  # (ii) conservation
    assert np.abs(w @ Pr_up - 0.5 * w).max() < 1e-14
    assert np.abs((Pr_lo + Pr_up) @ one - one).max() < 1e-13  # (iii)
    assert np.abs(Pf_lo @ one - one).max() < 1e-13 and np.abs(Pf_up @ one - one).max() < 1e-13
    # interpolation is exact for polynomials of degree <= N
    for k in range(N + 1):
        assert np.abs(Pf_lo @ x ** k - ((x - 1) / 2) ** k).max() < 1e-13
        assert np.abs(Pf_up @ x ** k - ((x + 1) / 2) ** k).max() < 1e-13
    # mirror symmetry lo <-> up
    assert np.abs(Pf_up - Pf_lo[::-1, ::-1]).max() < 1e-13
    assert np.abs(Pr_up - Pr_lo[::-1, ::-1]).max() < 1e-13


def _cons(rho, u, v, p, g=1.4):
    return np.array([rho, rho * u, rho * v, p / (g - 1) + 0.5 * rho * (u * u + v * v)])


def test_rusanov_worked_values():
    rows = [l.split() for l in open(os.path.join(GOLD, "rusanov_worked.txt")) if not l.startswith("#") and l.strip()]
    for r in rows:
        v = np.array([float(t) for t in r[1:]])
        Um, Up = (v[0:4], v[4:8]) if r[0] == "cons" else (_cons(*v[0:4]), _cons(*v[4:8]))
        Fs, lam = oracle.rusanov(2, 1.4, Um, Up, [1.0, 0.0])
        assert abs(lam - v[8]) < 1e-14
        assert np.allclose(Fs, v[9:13], atol=2e-8)  # fixture printed to 8 decimals


def test_rusanov_consistency_and_symmetry():
    rng = np.random.default_rng(1)
    for dim in (2, 3):
        for _ in range(20):
            rho, p = rng.uniform(0.5, 2.0, 2)
            vel = rng.uniform(-1, 1, dim)
            U = np.concatenate([[rho], rho * vel, [p / 0.4 + 0.5 * rho * vel @ vel]])
            rho2, p2 = rng.uniform(0.5, 2.0, 2)
            vel2 = rng.uniform(-1, 1, dim)
            U2 = np.concatenate([[rho2], rho2 * vel2, [p2 / 0.4 + 0.5 * rho2 * vel2 @ vel2]])
            nv = rng.uniform(-1, 1, dim) * 0.3
            Fs, _ = oracle.rusanov(dim, 1.4, U, U, nv)
            vn = vel @ nv  # F*(U,U;n) = F(U).n, written out from PAPER.md:50
            F = np.concatenate([[rho * vn], rho * vel * vn + p * nv, [(U[-1] + p) * vn]])
            assert np.allclose(Fs, F, rtol=1e-14, atol=1e-15)
            A, _ = oracle.rusanov(dim, 1.4, U, U2, nv)
            B, _ = oracle.rusanov(dim, 1.4, U2, U, -nv)
            assert np.allclose(A, -B, rtol=1e-14, atol=1e-15)  # F*(U-,U+;n) = -F*(U+,U-;-n)
            # scaling the normal scales the flux (area absorbed)
            C, _ = oracle.rusanov(dim, 1.4, U, U2, 2.0 * nv)
            assert np.allclose(C, 2.0 * A, rtol=1e-14, atol=1e-15)


def test_viscous_flux_closed_forms():
    g, mu, Pr = 1.4, 0.01, 0.72
    k = g * mu / (Pr * (g - 1))
    rho, vel, p = 1.2, np.array([0.3, -0.2, 0.5]), 0.9
    U = np.concatenate([[rho], rho * vel, [p / (g - 1) + 0.5 * rho * vel @ vel]])
    S = np.zeros((5, 3))
    S[1, 1] = 2.0  # du/dy : pure shear
    F = oracle.viscous_flux(3, g, mu, Pr, U, S, [0, 1, 0])  # G_v
    assert np.allclose(F, [0, mu * 2.0, 0, 0, vel[0] * mu * 2.0], atol=1e-15)
    F = oracle.viscous_flux(3, g, mu, Pr, U, S, [1, 0, 0])  # F_v: tau_xy symmetric
    assert np.allclose(F, [0, 0, mu * 2.0, 0, vel[1] * mu * 2.0], atol=1e-15)
    S = np.zeros((5, 3))
    S[1, 0] = 3.0  # du/dx : compression -> tau_xx = 4/3 mu, tau_yy = tau_zz = -2/3 mu  (eq. 15)
    F = oracle.viscous_flux(3, g, mu, Pr, U, S, [1, 0, 0])
    assert np.allclose(F, [0, 4 / 3 * mu * 3, 0, 0, vel[0] * 4 / 3 * mu * 3], atol=1e-15)
    F = oracle.viscous_flux(3, g, mu, Pr, U, S, [0, 0, 1])
    assert np.allclose(F, [0, 0, 0, -2 / 3 * mu * 3, vel[2] * (-2 / 3) * mu * 3], atol=1e-15)
    S = np.zeros((5, 3))
    S[4, 2] = 5.0  # dT/dz : q_z = -k dT/dz, energy flux = -q_z
    F = oracle.viscous_flux(3, g, mu, Pr, U, S, [0, 0, 1])
    assert np.allclose(F, [0, 0, 0, 0, k * 5.0], atol=1e-15)
    # trace-free stress (Stokes hypothesis)
    S = np.random.default_rng(0).uniform(-1, 1, (5, 3))
    tr = sum(oracle.viscous_flux(3, g, mu, Pr, U, S, np.eye(3)[c])[1 + c] for c in range(3))
    assert abs(tr) < 1e-16


def test_ssprk3_scalar_pins():
    # y' = lam y  ->  amplification 1 + z + z^2/2 + z^3/6 exactly
    for z in (-0.5, 0.1, -1.3):
        y = oracle.ssprk3_scalar(1.0, z, 0.0, 0.0, 1.0)
        assert abs(y - (1 + z + z * z / 2 + z ** 3 / 6)) < 1e-15
    # y' = t^2 from 0 -> dt^3/3 exactly (stage times c = 0, 1, 1/2)
    for dt in (0.3, 1.7):
        assert abs(oracle.ssprk3_scalar(0.0, 0.0, 1.0, 0.0, dt) - dt ** 3 / 3) < 1e-15
