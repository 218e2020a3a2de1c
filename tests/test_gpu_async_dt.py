"""Device-resident time step (eq. 45): marut_max_dt_async writes the dt
marut_max_dt returns, bit for bit, and marut_ssprk_stage_dev reproduces marut_ssprk_stage bit for bit, so the step
needs no host synchronisation; the composed run is compared with the oracle as every other run is."""
import numpy as np
import pytest

import workloads as wl
from parity_util import RUN_TOL, parity_error

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,cells,split", [("c1", 8, 0), ("c1", 8, 1), ("c2", 3, 0), ("c3", 3, 0), ("c4", 32, 0), ("c5", 4, 0)])
def test_async_dt_steps(name, cells, split):
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    c = wl.make_case(name, cells=cells)
    c.mesh.volume_form = split
    om, gm = oracle.OracleMesh(c.mesh), mb.MarutMesh(c.mesh)
    u = torch.from_numpy(c.u0).cuda()
    v = u.clone()
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=u.device)
    uh = c.u0
    for _ in range(3):
        # host-synchronised step
        dt = gm.max_dt(u, c.cfl)
        gm.step(u, ua, ub, dt)
        # the same step with dt resident on the device: nothing below waits for the GPU
        gm.max_dt_async(v, c.cfl, dt_dev)
        gm.stage_dev(0, dt_dev, 0.0, v, v, ua)
        gm.stage_dev(1, dt_dev, 0.0, v, ua, ub)
        gm.stage_dev(2, dt_dev, 0.0, v, ub, v)
        torch.cuda.synchronize()
        assert dt_dev.item() == dt
        assert torch.equal(u, v)
        dth = om.max_dt(uh, c.cfl)
        assert abs(dt - dth) <= 1e-12 * dth
        uh = om.run(uh, 1, cfl=c.cfl)[0]
    assert parity_error(v.cpu().numpy(), uh).max() <= RUN_TOL
    gm.close()


@pytest.mark.parametrize("name,cells", [("c1", 8), ("c2", 3), ("c3", 3), ("c4", 32)])
def test_async_dt_ssprk54(name, cells):
    """SSP-RK54 (R19) composed from marut_rk_stage_dev: bit-identical to the host-dt composition, whose
    parity with the oracle tests/test_gpu_rk54.py establishes"""
    import torch

    import paper_2605_26388_b200 as mb

    c = wl.make_case(name, cells=cells)
    gm = mb.MarutMesh(c.mesh)
    u = torch.from_numpy(c.u0).cuda()
    v = u.clone()
    ua, ub, uc = torch.empty_like(u), torch.empty_like(u), torch.empty_like(u)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=u.device)
    for _ in range(3):
        dt = gm.max_dt(u, 1.5 * c.cfl)
        gm.ssprk54_step(u, ua, ub, uc, dt)
        gm.max_dt_async(v, 1.5 * c.cfl, dt_dev)
        gm.ssprk54_step_dev(v, ua, ub, uc, dt_dev)
        torch.cuda.synchronize()
        assert dt_dev.item() == dt
        assert torch.equal(u, v)
    assert torch.isfinite(v).all()
    gm.close()


def test_async_dt_poison_and_arguments():
    import torch

    import paper_2605_26388_b200 as mb

    c = wl.make_case("c1", cells=4)
    gm = mb.MarutMesh(c.mesh)
    u = torch.from_numpy(c.u0).cuda()
    a = torch.empty_like(u)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=u.device)
    bad = u.clone()
    bad[3, 0, 2] = -1.0                                      # negative density: the checked call reports it ...
    with pytest.raises(mb.MarutError):
        gm.max_dt(bad, 0.5)
    gm.max_dt_async(bad, 0.5, dt_dev)                        # ... the asynchronous one poisons dt
    torch.cuda.synchronize()
    assert np.isnan(dt_dev.item())
    with pytest.raises(mb.MarutError):
        gm.max_dt_async(u, -1.0, dt_dev)
    with pytest.raises(mb.MarutError):
        gm.stage_dev(3, dt_dev, 0.0, u, u, a)
    with pytest.raises(mb.MarutError):
        gm.stage_dev(0, dt_dev, 0.0, u, a, a)                # u_out aliases u_in
    with pytest.raises(mb.MarutError):
        gm.stage_dev(0, None, 0.0, u, u, a)
    with pytest.raises(mb.MarutError):
        gm.rk_stage_dev(1.0, 1.0, 1.0, dt_dev, None, u, a)    # a != 0 needs u_a
    with pytest.raises(mb.MarutError):
        gm.rk_stage_dev(0.0, 1.0, 1.0, dt_dev, None, a, a)    # u_out aliases u_in
    gm.close()


@pytest.mark.parametrize("name,cells", [("c1", 16), ("c4", 32), ("c3", 3)])
def test_step_in_cuda_graph(name, cells):
    """with dt on the device the whole step (CFL reduction + three stages) has no host dependence: captured once in a
    CUDA graph and replayed, it advances the solution exactly as the eager calls do (launch-bound small meshes,
    PAPER.md:436)"""
    import torch

    import paper_2605_26388_b200 as mb

    c = wl.make_case(name, cells=cells)
    gm = mb.MarutMesh(c.mesh)
    u = torch.from_numpy(c.u0).cuda()
    v = u.clone()
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=u.device)

    def step(w):
        gm.max_dt_async(w, c.cfl, dt_dev)
        gm.stage_dev(0, dt_dev, 0.0, w, w, ua)
        gm.stage_dev(1, dt_dev, 0.0, w, ua, ub)
        gm.stage_dev(2, dt_dev, 0.0, w, ub, w)

    nsteps = 6
    for _ in range(nsteps):
        step(u)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        step(v)
    v.copy_(torch.from_numpy(c.u0))                           # capture does not execute; start from u0 all the same
    for _ in range(nsteps):
        graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(u, v)
    # timing, informational (CUDA events on the current stream)
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    e0.record()
    for _ in range(50):
        step(u)
    e1.record()
    for _ in range(50):
        graph.replay()
    e2.record()
    torch.cuda.synchronize()
    print(f"\n{name} cells={cells}: eager {e0.elapsed_time(e1) / 50 * 1e3:.1f} us/step, graph {e1.elapsed_time(e2) / 50 * 1e3:.1f} us/step")
    del graph
    gm.close()


@pytest.mark.parametrize("name,cells,which", [("c2", 3, 2), ("c2", 3, 1), ("c1", 8, 2), ("c4", 32, 2), ("c3", 3, 0), ("c5", 4, 0)])
def test_step_with_fused_cfl_reduction(name, cells, which):
    """marut_ssprk33_step_cfl: the step equals three marut_ssprk_stage_dev calls bit for bit, and the time step it leaves
    in dt_out equals marut_max_dt_async of the new state bit for bit -- with the reduction fused into the last stage's
    kernel (line kernel, which = 2), and with the separate pass behind it (thread-per-node kernel, NS, reacting)"""
    import torch

    import paper_2605_26388_b200 as mb

    c = wl.make_case(name, cells=cells)
    gm = mb.MarutMesh(c.mesh)
    gm.debug_stage_kernel(which)
    u = torch.from_numpy(c.u0).cuda()
    v = u.clone()
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    dts = torch.zeros(2, dtype=torch.float64, device="cuda")
    dt_ref = torch.zeros(1, dtype=torch.float64, device="cuda")
    gm.max_dt_async(u, c.cfl, dts[0:1])
    for k in range(4):
        gm.max_dt_async(v, c.cfl, dt_ref)
        for s, (un, uin, uout) in enumerate(((v, v, ua), (v, ua, ub), (v, ub, v))):
            gm.stage_dev(s, dt_ref, 0.0, un, uin, uout)
        gm.ssprk33_step_cfl(u, ua, ub, c.cfl, dts[k & 1:(k & 1) + 1], dts[(k + 1) & 1:((k + 1) & 1) + 1])
        torch.cuda.synchronize()
        assert torch.equal(u, v), (name, k)
        gm.max_dt_async(v, c.cfl, dt_ref)
        torch.cuda.synchronize()
        assert dts[(k + 1) & 1].item() == dt_ref.item() and dt_ref.item() > 0, (name, k)
    with pytest.raises(mb.MarutError):
        gm.ssprk33_step_cfl(u, ua, ub, c.cfl, dts[0:1], dts[0:1])       # dt_out aliases dt_in
    gm.close()


@pytest.mark.parametrize("name,cells", [("c1", 8), ("c2", 3), ("c3", 3), ("c4", 32), ("c5", 4), ("c5", 7)])
def test_step_with_its_own_time_step(name, cells):
    """marut_ssprk33_step_dt: the step forms its CFL time step from the state it starts from (for the reacting mixture
    inside the first stage's thermochemistry pass, without a separate wave-speed pass) -- dt and the new state equal
    marut_max_dt + marut_ssprk33 step bit for bit, three steps in a row, and the run agrees with the oracle"""
    import torch

    import oracle
    import paper_2605_26388_b200 as mb

    c = wl.make_case(name, cells=cells)
    om, gm = oracle.OracleMesh(c.mesh), mb.MarutMesh(c.mesh)
    u = torch.from_numpy(c.u0).cuda()
    v = u.clone()
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=u.device)
    uh = c.u0
    launches = []
    for _ in range(3):
        dt = gm.max_dt(u, c.cfl)
        gm.step(u, ua, ub, dt)
        n0 = gm.launch_count
        gm.ssprk33_step_dt(v, ua, ub, c.cfl, dt_dev)
        launches.append(gm.launch_count - n0)
        torch.cuda.synchronize()
        assert dt_dev.item() == dt
        assert torch.equal(u, v)
        uh = om.run(uh, 1, cfl=c.cfl)[0]
    assert parity_error(v.cpu().numpy(), uh).max() <= RUN_TOL
    if name == "c5":
        assert launches[0] == 7          # 3 x (eos_kernel + stage) + dt_finalize: no wave-speed pass
    # a bad state (negative density of an ideal gas) poisons dt and the new state
    if name != "c5":
        bad = torch.from_numpy(c.u0).cuda()
        bad[0, 0, 0] = -1.0
        gm.ssprk33_step_dt(bad, ua, ub, c.cfl, dt_dev)
        torch.cuda.synchronize()
        assert np.isnan(dt_dev.item())
    with pytest.raises(mb.MarutError):
        gm.ssprk33_step_dt(v, ua, ub, 0.0, dt_dev)
    gm.close()


@pytest.mark.parametrize("name,cells,steps_fn", [("c2", 6, "cfl"), ("c4", 32, "cfl"), ("c1", 16, "cfl"), ("c5", 4, "dt")])
def test_library_steps_of_the_line_kernel_in_a_cuda_graph(name, cells, steps_fn):
    """the whole-step entry points captured in a CUDA graph with the persistent line kernel forced (its launches are
    programmatic dependents of their stream predecessor, its tiles come from tile lists on 2-D mortar meshes, and the
    fused CFL reduction is finalised by the last launch): replayed, they advance the solution exactly as the eager calls"""
    import torch

    import paper_2605_26388_b200 as mb

    c = wl.make_case(name, cells=cells)
    gm = mb.MarutMesh(c.mesh)
    if c.mesh.physics == wl.EULER:
        gm.debug_stage_kernel(2)
    u = torch.from_numpy(c.u0).cuda()
    v = u.clone()
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    d = torch.zeros(2, dtype=torch.float64, device=u.device)

    def two_steps(w):
        if steps_fn == "cfl":
            gm.ssprk33_step_cfl(w, ua, ub, c.cfl, d[0:1], d[1:2])
            gm.ssprk33_step_cfl(w, ua, ub, c.cfl, d[1:2], d[0:1])
        else:
            gm.ssprk33_step_dt(w, ua, ub, c.cfl, d[0:1])
            gm.ssprk33_step_dt(w, ua, ub, c.cfl, d[1:2])

    gm.max_dt_async(u, c.cfl, d[0:1])
    for _ in range(3):
        two_steps(u)
    torch.cuda.synchronize()
    dt_eager = d.clone()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        two_steps(v)
    v.copy_(torch.from_numpy(c.u0))
    gm.max_dt_async(v, c.cfl, d[0:1])
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(u, v) and torch.equal(d, dt_eager)
    assert torch.isfinite(d).all() and (d > 0).all()
    del graph
    gm.close()
