"""marut_shock_indicator_noalloc (include/marut.h): the Hennemann-Gassner indicator for callers that must not allocate --
its scratch (V^-1 and the unsmoothed alpha_e) lives in one fixed device array of the library instead of the buffers
marut_shock_indicator allocates on its first call.  Checked against the existing path (bit for bit: same kernels, same
inputs) and against the tolerance of the indicator's parity test (1e-11 of the largest alpha_e, tests/test_gpu_degrees.py)
on consecutive calls that share the array: a large mesh first, then a smaller one of another degree and dimension (the
array then still holds the first call's values), then the first again.  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


def _cases():
    m1 = wl.quadtree_mesh(3, base=(32, 8), band=0.15, jitter=0.3)                 # 2-D, N = 3, mortar neighbours
    m1.bc_state = wl.shock_states(m1.gamma)
    u1 = wl.mach10_shock(m1, half_width=1.0 * m1.info["h_fine"])
    m2 = wl.cartesian_mesh(3, 4, (3, 3, 3), (0.0,) * 3, (2 * np.pi,) * 3)         # 3-D, N = 4, 27 elements
    u2 = wl.taylor_green(m2, noise=5e-2)
    return (m1, u1), (m2, u2)


def test_no_alloc_indicator_equals_the_allocating_path_on_consecutive_calls():
    import torch

    import paper_2605_26388_b200 as mb
    from paper_2605_26388_b200 import binding

    assert binding.marut_noalloc_max_elements() == 1 << 20
    (m1, u1), (m2, u2) = _cases()
    assert m1.n_elem > 20 * m2.n_elem
    g1, g2 = mb.MarutMesh(m1), mb.MarutMesh(m2)
    d1, d2 = torch.from_numpy(u1).cuda(), torch.from_numpy(u2).cuda()
    seen_positive = False
    for gm, m, u in ((g1, m1, d1), (g2, m2, d2), (g1, m1, d1), (g2, m2, d2)):     # calls in a row, one shared scratch array
        for smooth in (True, False):
            for amin, amax in ((0.0, 1.0), (1e-3, 0.5)):
                ref = torch.full((m.n_elem,), -1.0, dtype=torch.float64, device="cuda")
                out = torch.full((m.n_elem,), -2.0, dtype=torch.float64, device="cuda")
                gm.shock_indicator(u, ref, alpha_min=amin, alpha_max=amax, smooth=smooth)
                binding.marut_shock_indicator_noalloc(gm.h, u, out, alpha_min=amin, alpha_max=amax, smooth=smooth)
                torch.cuda.synchronize()
                r, o = ref.cpu().numpy(), out.cpu().numpy()
                assert np.abs(o - r).max() <= 1e-11 * max(r.max(), 1e-300), (m.n_elem, smooth, amin)
                assert np.array_equal(o, r)                                     # same kernels, same inputs
                seen_positive |= bool(r.max() > 0.1)
    assert seen_positive                                                          # the comparison is not 0 == 0
    g1.close()
    g2.close()


def test_no_alloc_indicator_against_the_oracle_after_other_calls():
    import torch

    import oracle
    import paper_2605_26388_b200 as mb
    from paper_2605_26388_b200 import binding

    (m1, u1), (m2, u2) = _cases()
    g1, g2 = mb.MarutMesh(m1), mb.MarutMesh(m2)
    a1 = torch.empty(m1.n_elem, dtype=torch.float64, device="cuda")
    a2 = torch.empty(m2.n_elem, dtype=torch.float64, device="cuda")
    binding.marut_shock_indicator_noalloc(g1.h, torch.from_numpy(u1).cuda(), a1)
    binding.marut_shock_indicator_noalloc(g2.h, torch.from_numpy(u2).cuda(), a2)
    torch.cuda.synchronize()
    for m, u0, a in ((m1, u1, a1), (m2, u2, a2)):
        ref = oracle.OracleMesh(m).shock_indicator(u0)
        assert np.abs(a.cpu().numpy() - ref).max() <= 1e-11 * max(ref.max(), 1e-300)
    g1.close()
    g2.close()


def test_no_alloc_indicator_rejects_meshes_beyond_its_scratch():
    import torch

    import paper_2605_26388_b200 as mb
    from paper_2605_26388_b200 import binding

    m = wl.cartesian_mesh(2, 1, (1025, 1024), (0.0, 0.0), (1.0, 1.0), order="lex")   # 1,049,600 elements > 2^20
    assert m.n_elem > binding.marut_noalloc_max_elements()
    gm = mb.MarutMesh(m)
    u = torch.from_numpy(wl.isentropic_vortex(m, center=(0.5, 0.5), L=1.0)).cuda()
    a = torch.empty(m.n_elem, dtype=torch.float64, device="cuda")
    with pytest.raises(mb.MarutError, match="exceed the fixed scratch"):
        binding.marut_shock_indicator_noalloc(gm.h, u, a)
    gm.shock_indicator(u, a)                                                      # the allocating path takes it
    torch.cuda.synchronize()
    assert np.isfinite(a.cpu().numpy()).all()
    gm.close()
