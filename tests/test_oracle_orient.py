"""Pins of the 3-D face-orientation handling ("face orientation tables for unstructured hexes";
PAPER.md:193; reading R20): a Cartesian mesh whose elements' local axes are rotated at random is the same
discretisation in another numbering, so the oracle's RHS must be the same physical field."""
import math

import numpy as np
import pytest

import oracle
import workloads as wl


def _meshes(N, curved, cells=3):
    lo, hi = (0.0,) * 3, (2 * math.pi,) * 3
    warp = wl.sine_warp((cells,) * 3, lo, hi, k=1) if curved else None
    m = wl.cartesian_mesh(3, N, (cells,) * 3, lo, hi, warp=warp)
    mr, node_map = wl.rotate_elements(m)
    return m, mr, node_map


def _to_new(field, node_map):
    return np.stack([field[e][:, node_map[e]] for e in range(field.shape[0])])


def test_rotated_mesh_is_geometrically_consistent():
    m, mr, node_map = _meshes(3, True)
    n = m.n
    assert mr.info["rotated"] > 10 and len(set(mr.iface[:, 4])) == 8         # every orientation code occurs
    idx = lambda i, j, k: i + n * (j + n * k)

    def face_node(f, a0, a1):
        ijk = [0, 0, 0]
        rest = [c for c in range(3) if c != f // 2]
        ijk[f // 2] = (n - 1) if f % 2 else 0
        ijk[rest[0]], ijk[rest[1]] = a0, a1
        return idx(*ijk)

    L = 2 * math.pi
    for eL, fL, eR, fR, code in mr.iface:
        for a0 in range(n):
            for a1 in range(n):
                c0, c1 = (a1, a0) if code & 4 else (a0, a1)
                b0 = n - 1 - c0 if code & 1 else c0
                b1 = n - 1 - c1 if code & 2 else c1
                d = mr.node_xyz[eL, :, face_node(fL, a0, a1)] - mr.node_xyz[eR, :, face_node(fR, b0, b1)]
                d -= L * np.round(d / L)                                         # periodic images
                assert np.abs(d).max() < 1e-12


@pytest.mark.parametrize("N,curved,phys,split", [(2, False, "euler", 0), (3, True, "euler", 0), (3, True, "euler", 1),
                                                 (2, True, "ns", 0), (4, False, "euler", 0)])
def test_rhs_is_invariant_under_rotation_of_the_local_axes(N, curved, phys, split):
    m, mr, node_map = _meshes(N, curved)
    for mesh in (m, mr):
        mesh.volume_form = split
        if phys == "ns":
            mesh.physics, mesh.mu, mesh.Pr = wl.NAVIER_STOKES, 0.02, 0.72
    u = wl.taylor_green(m, noise=1e-2)
    ur = _to_new(u, node_map)
    assert np.allclose(wl.taylor_green(mr, noise=0.0), _to_new(wl.taylor_green(m, noise=0.0), node_map), rtol=0, atol=1e-13)
    om, omr = oracle.OracleMesh(m), oracle.OracleMesh(mr)
    r, rr = om.rhs(u), omr.rhs(ur)
    assert np.abs(rr - _to_new(r, node_map)).max() <= 1e-11 * np.abs(r).max()
    assert abs(omr.max_dt(ur, 0.5) / om.max_dt(u, 0.5) - 1) < 1e-13
    if curved and phys == "euler":
        const = np.broadcast_to(np.array([1.3, 0.4, -0.2, 0.7, 3.0])[None, :, None], u.shape).copy()
        assert np.abs(omr.rhs(const)).max() < 2e-11                              # free stream on the rotated curved mesh
