"""Pins of the oracle's Hennemann-Gassner shock indicator (first part):
modal transform against numpy's Legendre class, the blending coefficient against closed forms on fields whose
rho*p is a known Legendre expansion, the threshold value, clipping and the face-neighbour maximum."""
import math

import numpy as np
import pytest
from numpy.polynomial import legendre as npl

import oracle
import workloads as wl

S_HG = math.log((1 - 1e-4) / 1e-4)     # steepness: alpha(E = 0) = 1e-4 (the indicator paper's choice; R15)


def _ortho(k, x):
    return math.sqrt((2 * k + 1) / 2.0) * npl.legval(x, [0] * k + [1])


@pytest.mark.parametrize("N", [2, 3, 4, 6])
def test_modal_matrix_against_numpy_legendre(N):
    x = wl.lgl_points(N)
    Vinv = oracle.modal_matrix(N)
    for k in range(N + 1):
        m = Vinv @ _ortho(k, x)                       # nodal values of the k-th orthonormal Legendre polynomial
        assert np.allclose(m, np.eye(N + 1)[k], atol=1e-12)
    # Parseval: sum of squared modes = integral of q^2 over [-1,1] for a polynomial q of degree <= N
    c = np.arange(1, N + 2, dtype=float)
    q = npl.legval(x, c)
    integral = sum(c[k] ** 2 * 2.0 / (2 * k + 1) for k in range(N + 1))
    assert (Vinv @ q) @ (Vinv @ q) == pytest.approx(integral, rel=1e-12)


def _field(mesh, q_ref):
    """state with rho = 1, velocity 0 and p = q_ref(xi, eta[, zeta]) in EVERY element (rho*p = q_ref)"""
    N, d = mesh.N, mesh.dim
    x = wl.lgl_points(N)
    grids = np.meshgrid(*([x] * d), indexing="ij")     # index order (xi, eta, zeta) -> node index i fastest
    q = q_ref(*grids)
    q = np.transpose(q, tuple(range(d - 1, -1, -1))).reshape(-1)
    u = np.zeros((mesh.n_elem, d + 2, (N + 1) ** d))
    u[:, 0, :] = 1.0
    u[:, -1, :] = q[None, :] / (mesh.gamma - 1.0)
    return u


@pytest.mark.parametrize("dim,N", [(2, 3), (3, 4), (2, 5)])
def test_alpha_closed_forms(dim, N):
    m = wl.cartesian_mesh(dim, N, (3,) * dim, (0.0,) * dim, (1.0,) * dim)
    om = oracle.OracleMesh(m)
    T = 0.5 * 10.0 ** (-1.8 * (N + 1) ** 0.25)
    if N == 3:
        assert T == pytest.approx(0.5 * 10 ** (-1.8 * math.sqrt(2.0)), rel=1e-14)
    # (a) rho*p of degree N-2 per direction: no energy in the two highest shells -> alpha = 1/(1+e^s) = 1e-4 -> clipped to 0
    low = lambda *xi: 2.0 + sum(0.3 * _ortho(max(N - 2, 0), t) for t in xi)
    a = om.shock_indicator(_field(m, low), s=S_HG, alpha_min=0.0, alpha_max=1.0, smooth=False)
    assert np.allclose(a, 1e-4, rtol=1e-9)
    assert np.all(om.shock_indicator(_field(m, low), s=S_HG, alpha_min=1e-3, alpha_max=0.5, smooth=False) == 0.0)
    # (b) a L0...L0 + b L_N(xi) L0...: E = b^2/(a^2+b^2) from the top shell
    c0 = math.sqrt(0.5) ** (dim - 1)                   # the orthonormal L0 factors of the other directions
    for b in (0.01, 0.2):
        f = lambda *xi: 3.0 + b * _ortho(N, xi[0]) * c0
        a0 = 3.0 / (math.sqrt(0.5) ** dim)             # modal coefficient of the constant 3
        E = b * b / (a0 * a0 + b * b)
        expect = 1.0 / (1.0 + math.exp(-(S_HG / T) * (E - T)))
        got = om.shock_indicator(_field(m, f), s=S_HG, alpha_min=0.0, alpha_max=1.0, smooth=False)
        assert np.allclose(got, expect, rtol=1e-9)
        assert np.allclose(om.shock_indicator(_field(m, f), s=S_HG, alpha_min=0.0, alpha_max=0.5, smooth=False), min(expect, 0.5), rtol=1e-9)
    # (c) energy only in the shell N-1: the second ratio decides
    g = lambda *xi: 3.0 + 0.1 * _ortho(N - 1, xi[-1]) * c0
    E = 0.01 / (a0 * a0 + 0.01)
    got = om.shock_indicator(_field(m, g), s=S_HG, alpha_min=0.0, alpha_max=1.0, smooth=False)
    assert np.allclose(got, 1.0 / (1.0 + math.exp(-(S_HG / T) * (E - T))), rtol=1e-9)


def test_face_neighbour_maximum():
    m = wl.cartesian_mesh(2, 3, (4, 4), (0.0, 0.0), (1.0, 1.0), order="lex")
    om = oracle.OracleMesh(m)
    u = _field(m, lambda x, y: 3.0 + 0.0 * x)
    rough = _field(m, lambda x, y: 3.0 + 0.5 * _ortho(3, x) * math.sqrt(0.5))
    e = 5                                               # element (1,1) of the 4x4 lexicographic grid
    u[e] = rough[e]
    raw = om.shock_indicator(u, s=S_HG, alpha_min=1e-3, alpha_max=0.5, smooth=False)
    assert raw[e] == 0.5 and np.count_nonzero(raw) == 1
    a = om.shock_indicator(u, s=S_HG, alpha_min=1e-3, alpha_max=0.5, smooth=True)
    nb = {e - 1, e + 1, e - 4, e + 4}
    assert all(a[k] == 0.5 for k in nb | {e}) and np.count_nonzero(a) == 5
