"""Mutants of the oracle: the oracle source with ONE named line changed, compiled into a scratch library.  The pin tests
run their checks against a mutant as well and assert that the check FAILS there -- the committed proof that a pin
would catch the plausible mistake it is meant to catch (VERDICT r1 'oracle parts with no effective pin')."""
import ctypes
import os
import subprocess
import tempfile

import oracle

_SRC = os.path.join(os.path.dirname(os.path.abspath(oracle.__file__)), "marut_oracle.cpp")

# name -> (text in oracle/marut_oracle.cpp, its replacement, what the mutant gets wrong)
MUTATIONS = {
    "mortar2d_lo_up_swapped": (
        "acc += m.Pf[s][a * n + j] * UC[(size_t)j * nvar + v];",
        "acc += m.Pf[1 - s][a * n + j] * UC[(size_t)j * nvar + v];",
        "2-D mortar: the coarse trace is interpolated to the wrong half of the coarse face"),
    "boundary_state_ignored": (
        "Ue[v] = (bk == 0) ? m.bc_state[(size_t)bc * nvar + v] : Um[v];",
        "Ue[v] = Um[v];",
        "prescribed exterior state ignored: every Dirichlet face becomes an outflow"),
    "br1_trace_not_central": (
        "double What = 0.5 * (Wm[w] + Wp[w]);",
        "double What = 0.75 * Wm[w] + 0.25 * Wp[w];",
        "BR1 interface trace is not the arithmetic mean of eq. 13"),
    "wall_trace_keeps_velocity": (
        "for (int c = 0; c < d; ++c) What[1 + c] = 0.0;",
        "for (int c = 0; c < d; ++c) What[1 + c] = Wm[1 + c];",
        "no-slip wall: the BR1 trace keeps the interior velocity instead of the wall's (zero)"),
    "adiabatic_wall_energy_flux_kept": (
        "if (bk == 3) Fw[1 + d] = 0.0;",
        "if (bk == 3) Fw[1 + d] = Fm[1 + d];",
        "adiabatic wall: the energy row of the wall's viscous flux keeps the stress work and the heat flux"),
    "ranocha_printed_energy_flux": (
        "pvn += 0.5 * (L.p * R.vel[c] + R.p * L.vel[c]) * nv[c];",
        "pvn += 0.5 * (L.p * L.vel[c] + R.p * R.vel[c]) * nv[c];",
        "pressure work {{p v}} as PAPER.md:621 prints it: not entropy conservative"),
    "br1_mortar_wrong_half": (
        "Wi += m.Pf[s][a * n + j] * WC[(size_t)j * nw + w];",
        "Wi += m.Pf[1 - s][a * n + j] * WC[(size_t)j * nw + w];",
        "BR1 gradient across a 2-D mortar: the coarse trace of W is interpolated to the wrong half"),
    "br1_mortar_no_area_factor": (
        "m.Pr_[s][i * n + a] * (2.0 * (-(What * nF[c])));",
        "m.Pr_[s][i * n + a] * (1.0 * (-(What * nF[c])));",
        "BR1 gradient across a 2-D mortar: the coarse side's projected trace misses the 2:1 area factor"),
    "viscous_mortar_gradient_wrong_half": (
        "si += m.Pf[s][a * n + j] * SC[(size_t)j * ng + k];",
        "si += m.Pf[1 - s][a * n + j] * SC[(size_t)j * ng + k];",
        "viscous flux across a 2-D mortar: the coarse gradient is interpolated to the wrong half"),
    "viscous_mortar_no_area_factor": (
        "m.Pr_[s][i * n + a] * (2.0 * (-Fs));",
        "m.Pr_[s][i * n + a] * (1.0 * (-Fs));",
        "viscous flux across a 2-D mortar: the coarse side's projected flux misses the 2:1 area factor"),
    "br1_mortar3d_wrong_subface": (
        "Wt += m.Pf[s0][a0 * n + j0] * m.Pf[s1][a1 * n + j1] * WC[(size_t)(j0 + n * j1) * nw + w];",
        "Wt += m.Pf[1 - s0][a0 * n + j0] * m.Pf[s1][a1 * n + j1] * WC[(size_t)(j0 + n * j1) * nw + w];",
        "BR1 gradient across a 3-D mortar: the coarse trace of W goes to the wrong sub-face in the first face direction"),
    "br1_mortar3d_area_factor_2": (
        "(4.0 * (-(What * nF[c])));",
        "(2.0 * (-(What * nF[c])));",
        "BR1 gradient across a 3-D mortar: the 2-D area factor"),
    "viscous_mortar3d_wrong_subface": (
        "const double pw = m.Pf[s0][a0 * n + j0] * m.Pf[s1][a1 * n + j1];",
        "const double pw = m.Pf[s0][a0 * n + j0] * m.Pf[1 - s1][a1 * n + j1];",
        "viscous flux across a 3-D mortar: coarse state and gradient go to the wrong sub-face in the second face direction"),
    "viscous_mortar3d_area_factor_2": (
        "(4.0 * (-Fc));",
        "(2.0 * (-Fc));",
        "viscous flux across a 3-D mortar: the 2-D area factor"),
}

_cache = {}


def mutant(name):
    """ctypes library of the oracle with mutation `name` applied (compiled once per test session)"""
    if name not in _cache:
        old, new, _ = MUTATIONS[name]
        src = open(_SRC).read()
        assert src.count(old) == 1, f"mutation site of {name!r} not found exactly once in the oracle source"
        d = tempfile.mkdtemp(prefix="marut_mutant_")
        cpp, so = os.path.join(d, "mutant.cpp"), os.path.join(d, "mutant.so")
        open(cpp, "w").write(src.replace(old, new))
        subprocess.run(["g++", "-O1", "-ffp-contract=off", "-fopenmp", "-std=c++17", "-shared", "-fPIC", cpp, "-o", so], check=True)
        _cache[name] = oracle._setup(ctypes.CDLL(so))
    return _cache[name]
