"""Pins of the oracle's implicit chemistry substep (eq. 24-25): the per-node
backward-Euler Newton with a forward-difference Jacobian.  Every pin evaluates the backward-Euler equation or its
limits with the SEPARATELY pinned temperature and production-rate routines (tests/test_oracle_chem.py), not with the
Newton code."""
import numpy as np
import pytest

import oracle
import workloads as wl


def _state(k, rng):
    T = rng.uniform(3000, 8000)
    rho_s = rng.uniform(1e-4, 1e-2, 5)
    e_int = sum(rho_s[s] * k.species_thermo(s, T)["e"] for s in range(5))
    return rho_s, e_int


def _tau(k, rho_s, e_int):
    om = k.production_rates(k.temperature(rho_s, e_int), rho_s)
    return (rho_s / np.maximum(np.abs(om), 1e-300)).min()


def test_backward_euler_equation_holds_and_invariants():
    mech = wl.air5_mechanism()
    k = oracle.MechHandle(mech)
    rng = np.random.default_rng(11)
    W = np.asarray(mech.W)
    atoms_N, atoms_O = np.array([2, 0, 1, 1, 0]) / W, np.array([0, 2, 1, 0, 1]) / W   # N2, O2, NO, N, O
    for _ in range(10):
        y0, e_int = _state(k, rng)
        for factor in (0.1, 1.0, 30.0):                     # well below, at and far above the fastest depletion time
            dt = factor * _tau(k, y0, e_int)
            y, it = k.implicit_step(y0, e_int, dt)
            assert 1 <= it < 50 and np.all(y > 0)
            om = k.production_rates(k.temperature(y, e_int), y)
            res = y - y0 - dt * om                          # eq. 25 with S_Y = omega
            assert np.abs(res).max() <= 1e-11 * y0.sum()
            assert abs(y.sum() / y0.sum() - 1) < 1e-13      # total density is invariant
            assert abs((y * atoms_N).sum() / (y0 * atoms_N).sum() - 1) < 1e-12
            assert abs((y * atoms_O).sum() / (y0 * atoms_O).sum() - 1) < 1e-12


def test_limits_small_and_large_step():
    mech = wl.air5_mechanism()
    k = oracle.MechHandle(mech)
    rng = np.random.default_rng(12)
    y0, e_int = _state(k, rng)
    tau = _tau(k, y0, e_int)
    y, it = k.implicit_step(y0, e_int, 0.0)
    assert np.array_equal(y, y0) and it == 1                # dt = 0: identity after one sweep
    om0 = k.production_rates(k.temperature(y0, e_int), y0)
    e1 = np.abs((k.implicit_step(y0, e_int, 1e-3 * tau)[0] - y0) / (1e-3 * tau) - om0).max()
    e2 = np.abs((k.implicit_step(y0, e_int, 1e-4 * tau)[0] - y0) / (1e-4 * tau) - om0).max()
    assert e2 < 0.2 * e1 and e2 < 1e-3 * np.abs(om0).max()  # consistent with dY/dt = omega, first order in dt
    # a very long step lands on chemical equilibrium at fixed energy: the rates vanish against their scale
    dt = 1e6 * tau
    y, _ = k.implicit_step(y0, e_int, dt)
    om = k.production_rates(k.temperature(y, e_int), y)
    assert np.abs(om).max() * dt <= 1.01 * np.abs(y - y0).max() and np.abs(om).max() < 1e-5 * np.abs(om0).max()


def test_mesh_substep_touches_species_only():
    c = wl.make_case("c5", cells=2)
    om = oracle.OracleMesh(c.mesh)
    dt = 5.0 * om.max_dt(c.u0, 0.5)
    u, it = om.chem_implicit(c.u0, dt)
    assert 1 <= it < 50
    assert np.array_equal(u[:, 5:, :], c.u0[:, 5:, :])      # momentum and total energy rows untouched
    assert np.abs(u[:, :5, :].sum(axis=1) / c.u0[:, :5, :].sum(axis=1) - 1).max() < 1e-13
    assert np.abs(u[:, :5, :] - c.u0[:, :5, :]).max() > 0
