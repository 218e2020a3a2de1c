"""Shared helpers of the GPU parity tests: the parity metric of BASELINE.json and the two drivers."""
import numpy as np

RHS_TOL = 1e-11   # per-variable max-norm relative error on one marut_rhs   (BASELINE.json north_star)
RUN_TOL = 1e-9    # after the config's RK steps


def parity_error(gpu, cpu):
    """per variable v: max_i|gpu - cpu| / max_i|cpu|; a variable whose oracle values are all 0 is
    compared against the largest variable's scale (SURVEY 8(c) 'Parity metric')."""
    diff = np.abs(gpu - cpu).max(axis=(0, 2))
    scale = np.abs(cpu).max(axis=(0, 2))
    scale = np.where(scale > 0, scale, scale.max())
    return diff / scale


def gpu_run(gm, u0, steps, cfl, torch):
    """advance u0 by `steps` SSPRK3 steps through the C ABI, dt from marut_max_dt each step"""
    u = torch.from_numpy(np.ascontiguousarray(u0)).cuda()
    ua, ub = torch.empty_like(u), torch.empty_like(u)
    t = 0.0
    for _ in range(steps):
        dt = gm.max_dt(u, cfl)
        gm.step(u, ua, ub, dt, t)
        t += dt
    torch.cuda.synchronize()
    return u.cpu().numpy(), t
