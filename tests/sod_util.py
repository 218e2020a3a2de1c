"""Sod's shock tube as a validation problem of the shock-capturing step: set-up on a periodic
strip and the exact density profile.  The star-region values are the textbook ones of this Riemann problem
((rho, u, p) = (1, 0, 1) | (0.125, 0, 0.1), gamma = 1.4): p* = 0.30313, u* = 0.92745, rho*L = 0.42632,
rho*R = 0.26557, shock speed 1.75216; the rarefaction fan is the isentropic similarity solution.  No method arithmetic
here: both the oracle tests and the GPU tests advance the state through their own side's calls."""
import numpy as np

import workloads as wl

GAMMA = 1.4
PS, US, RSL, RSR, SS = 0.30313, 0.92745, 0.42632, 0.26557, 1.75216
SHOCK_CAPTURE = dict(s=9.21024, alpha_min=1e-3, alpha_max=0.5, smooth=True)


def sod_density(xi):
    """exact density at similarity coordinate xi = (x - x0)/t"""
    g = GAMMA
    aL = np.sqrt(g)
    aSL = aL * PS ** ((g - 1) / (2 * g))
    fan = (2 / (g + 1) - (g - 1) / ((g + 1) * aL) * xi) ** (2 / (g - 1))
    return np.where(xi < -aL, 1.0, np.where(xi < US - aSL, fan, np.where(xi < US, RSL, np.where(xi < SS, RSR, 0.125))))


def sod_strip(ne, rows=1, N=3):
    """periodic strip [0,2] x [0, rows*h]: high state on (0.5, 1.5), low state elsewhere -- Sod's problem at x = 1.5 and
    its mirror image at x = 0.5; the waves stay apart until well after t = 0.2.  Split form (eq. 10)."""
    assert ne % 4 == 0
    m = wl.cartesian_mesh(2, N, (ne, rows), (0.0, 0.0), (2.0, rows * 2.0 / ne))
    m.volume_form = 1
    xc = m.node_xyz[:, 0, :].mean(axis=1)
    hi = ((xc > 0.5) & (xc < 1.5))[:, None] * np.ones((1, m.nn), bool)
    rho, p = np.where(hi, 1.0, 0.125), np.where(hi, 1.0, 0.1)
    u0 = np.ascontiguousarray(np.stack([rho, 0 * rho, 0 * rho, p / (GAMMA - 1)], axis=1))
    return m, u0


def sod_exact_on(mesh, t):
    x = mesh.node_xyz[:, 0, :]
    return np.where(x >= 1.0, sod_density((x - 1.5) / t), sod_density((0.5 - x) / t))


def pressure(u):
    return (GAMMA - 1) * (u[:, 3] - 0.5 * (u[:, 1] ** 2 + u[:, 2] ** 2) / u[:, 0])
