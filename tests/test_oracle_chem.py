"""Pins for the oracle's thermochemistry (O12).  CPU only."""
import math
from types import SimpleNamespace

import numpy as np

import oracle
import workloads as wl

RU = 8.31446261815324


def toy_mech(A=3e15, b=-1.0, Ea=6e4):
    """A2 + M <-> 2A + M (M = A2, A) and nothing else; constant cp so every thermo quantity has a closed form."""
    W = np.array([0.028, 0.014])
    nasa = np.zeros((2, 2, 7))
    nasa[0, :, 0], nasa[1, :, 0] = 3.5, 2.5
    nasa[0, :, 5], nasa[1, :, 5] = 0.0, 5.0e4  # h_f/R_u in K
    nasa[0, :, 6], nasa[1, :, 6] = 3.0, 4.0
    nu_r = np.array([[2, 0], [1, 1]], np.int32)
    nu_p = np.array([[1, 2], [0, 3]], np.int32)
    return SimpleNamespace(W=W, nasa=nasa, T_mid=1000.0, nu_r=nu_r, nu_p=nu_p,
                           A=np.array([A, 2 * A]), b=np.array([b, b]), Ea=np.array([Ea, Ea]))


def test_arrhenius_closed_forms():
    # SURVEY 8(c) O12 pins: A=3e15, b=-1, Ea=6e4 K
    k = oracle.MechHandle(toy_mech())
    A, Ea = 3e15, 6e4
    assert abs(k.k_forward(0, 6e4) / (A / (Ea * math.e)) - 1) < 1e-14
    assert abs(k.k_forward(0, 3e4) / (2 * A / (Ea * math.e ** 2)) - 1) < 1e-14
    assert abs(k.k_forward(0, 6e4) - 1.8393972058572117e10) < 1e-4
    assert abs(k.k_forward(0, 3e4) - 1.353352832366127e10) < 1e-4
    assert abs(k.k_forward(0, 6000.0) / 2.2699964881242428e7 - 1) < 1e-13


def test_equilibrium_constant_closed_form_and_third_body_independence():
    k = oracle.MechHandle(toy_mech())
    for T in (500.0, 3000.0, 9000.0):
        # constant-cp closed form: g/(R_u T) = cp/R (1 - ln T) + a6/T - a7
        gA2 = 3.5 * (1 - math.log(T)) + 0.0 / T - 3.0
        gA = 2.5 * (1 - math.log(T)) + 5.0e4 / T - 4.0
        Kc = math.exp(-(2 * gA - gA2)) * (101325.0 / (RU * T) * 1e-6)
        assert abs(k.k_equilibrium(0, T) / Kc - 1) < 1e-12
        assert abs(k.k_equilibrium(1, T) / k.k_equilibrium(0, T) - 1) < 1e-14  # independent of M


def test_nasa7_polynomial_consistency():
    mech = wl.air5_mechanism()
    k = oracle.MechHandle(mech)
    for s in range(5):
        for T in (300.0, 900.0, 2500.0, 8000.0):
            h = 1e-3 * T
            tp, tm, t0 = k.species_thermo(s, T + h), k.species_thermo(s, T - h), k.species_thermo(s, T)
            # d(h)/dT = cp ; d(s)/dT = cp/T ; cv = cp - R ; e = h - R T
            dh = (tp["h_RT"] * (T + h) - tm["h_RT"] * (T - h)) / (2 * h)
            ds = (tp["s_R"] - tm["s_R"]) / (2 * h)
            assert abs(dh - t0["cp_R"]) < 1e-6 * t0["cp_R"]
            assert abs(ds * T - t0["cp_R"]) < 1e-6 * t0["cp_R"]
            Rs = RU / mech.W[s]
            assert abs(t0["cv"] - Rs * (t0["cp_R"] - 1)) < 1e-12 * t0["cv"]
            assert abs(t0["e"] - Rs * T * (t0["h_RT"] - 1)) < 1e-9 * abs(t0["e"]) + 1e-9
        # continuity of h and s at T_mid (generator recipe) seen through the oracle's range switch
        lo, hi = k.species_thermo(s, 1000.0 - 1e-9), k.species_thermo(s, 1000.0)
        assert abs(lo["h_RT"] - hi["h_RT"]) < 1e-9 and abs(lo["s_R"] - hi["s_R"]) < 1e-9
    # formation enthalpy of N at 298.15 K as tabulated by the generator
    assert abs(k.species_thermo(3, 298.15)["h_RT"] * RU * 298.15 - 472.68e3) < 1e-6


def test_production_rates_invariants():
    mech = wl.air5_mechanism()
    k = oracle.MechHandle(mech)
    assert mech.nr == 17 and mech.ns == 5  # 3 dissociations x 5 third bodies + 2 exchanges
    atoms_N = np.array([2, 0, 1, 1, 0])
    atoms_O = np.array([0, 2, 1, 0, 1])
    # every reaction conserves atoms
    d = mech.nu_p - mech.nu_r
    assert (d @ atoms_N == 0).all() and (d @ atoms_O == 0).all()
    rng = np.random.default_rng(2)
    for _ in range(20):
        T = rng.uniform(2000, 9000)
        rho_s = rng.uniform(1e-4, 1e-2, 5)
        om = k.production_rates(T, rho_s)
        scale = np.abs(om).sum()
        assert abs(om.sum()) < 1e-13 * scale  # sum_s omega_s = 0
        assert abs((atoms_N * om / mech.W).sum()) < 1e-13 * (np.abs(om) / mech.W).sum()
        assert abs((atoms_O * om / mech.W).sum()) < 1e-13 * (np.abs(om) / mech.W).sum()


def test_detailed_balance():
    # with k_b = k_f/K_c the net rate vanishes where prod [X]^(nu''-nu') = K_c
    tm = toy_mech()
    k = oracle.MechHandle(tm)
    T = 6000.0
    Kc = k.k_equilibrium(0, T)  # mol/cm^3
    XA2 = 2.0e-6  # mol/cm^3
    XA = math.sqrt(Kc * XA2)
    rho_s = np.array([XA2, XA]) * 1e6 * tm.W
    om = k.production_rates(T, rho_s)
    # compare with the one-way (forward-only) rate scale
    fwd = k.k_forward(0, T) * XA2 * XA2 * 1e6 * tm.W[0]
    assert np.abs(om).max() < 1e-12 * fwd
    # away from equilibrium the sign follows the mass-action ratio
    om = k.production_rates(T, rho_s * np.array([1.0, 0.5]))
    assert om[1] > 0 and om[0] < 0


def test_single_reaction_rate_closed_form():
    tm = toy_mech()
    tm.nu_r, tm.nu_p = tm.nu_r[:1], tm.nu_p[:1]
    tm.A, tm.b, tm.Ea = tm.A[:1], tm.b[:1], tm.Ea[:1]
    k = oracle.MechHandle(tm)
    T, rho_s = 5000.0, np.array([0.05, 0.01])
    X = rho_s / tm.W * 1e-6
    kf = k.k_forward(0, T)
    kb = kf / k.k_equilibrium(0, T)
    R = kf * X[0] ** 2 - kb * X[0] * X[1] ** 2  # eq. 21 for A2 + A2 <-> 2A + A2
    om = k.production_rates(T, rho_s)
    assert abs(om[0] - tm.W[0] * (-1) * R * 1e6) < 1e-12 * abs(om[0])  # eq. 22
    assert abs(om[1] - tm.W[1] * (+2) * R * 1e6) < 1e-12 * abs(om[1])


def test_temperature_newton_round_trip_and_mixture_eos():
    mech = wl.air5_mechanism()
    k = oracle.MechHandle(mech)
    rng = np.random.default_rng(4)
    m = wl.cartesian_mesh(3, 1, (1, 1, 1), (0,) * 3, (1.0,) * 3)
    m.physics, m.mech = wl.REACTING_EULER, mech
    om = oracle.OracleMesh(m)
    for _ in range(20):
        T = rng.uniform(2000, 9000)
        rho_s = rng.uniform(1e-4, 1e-2, 5)
        e_int = sum(rho_s[s] * k.species_thermo(s, T)["e"] for s in range(5))
        assert abs(k.temperature(rho_s, e_int) / T - 1) < 1e-12
        vel = rng.uniform(-500, 500, 3)
        rho = rho_s.sum()
        U = np.concatenate([rho_s, rho * vel, [e_int + 0.5 * rho * vel @ vel]])
        q = om.primitives(U)
        R = sum(rho_s[s] / rho * RU / mech.W[s] for s in range(5))
        assert abs(q["T"] / T - 1) < 1e-12
        assert abs(q["p"] / (rho * R * T) - 1) < 1e-12  # p = rho R T, R = sum Y_s R_s
        cp = sum(rho_s[s] / rho * RU / mech.W[s] * k.species_thermo(s, T)["cp_R"] for s in range(5))
        assert abs(q["a"] / math.sqrt(cp / (cp - R) * R * T) - 1) < 1e-12
        assert np.allclose(q["vel"], vel, rtol=1e-14)


def test_chem_source_rows_and_mass_conservation():
    c = wl.make_case("c5", cells=2, steps=1)
    om = oracle.OracleMesh(c.mesh)
    s = om.chem_source(c.u0)
    assert np.abs(s[:, 5:, :]).max() == 0.0  # momentum and energy rows identically zero
    assert np.abs(s[:, :5, :].sum(axis=1)).max() < 1e-13 * np.abs(s).max()
    # rhs = transport + source, and total mass only moves by transport
    full = om.rhs(c.u0)
    assert np.allclose(full, om.rhs_inviscid(c.u0) + s, rtol=0, atol=1e-12 * np.abs(full).max())
    Y = c.u0[:, :5, :] / c.u0[:, :5, :].sum(axis=1, keepdims=True)
    assert np.abs(Y.sum(axis=1) - 1).max() < 1e-15 and Y.min() > 0


def test_c5_recipe_is_well_posed():
    # L chosen so the CFL step is <= 0.05 x fastest depletion time at t=0
    c = wl.make_case("c5", cells=4, steps=3)
    om = oracle.OracleMesh(c.mesh)
    dt = om.max_dt(c.u0, c.cfl)
    s = om.chem_source(c.u0)[:, :5, :]
    tau = (c.u0[:, :5, :] / np.maximum(np.abs(s), 1e-300)).min()
    assert dt <= 0.05 * tau, (dt, tau)
    u, t, min_rho, min_p = om.run(c.u0, c.steps, cfl=c.cfl)
    assert min_rho > 0 and min_p > 0 and np.isfinite(u).all()
