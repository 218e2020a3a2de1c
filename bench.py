#!/usr/bin/env python
"""bench.py -- DG RHS + SSP-RK33 throughput of the CUDA path (DOF-stage updates / s, FP64) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c3|c4w|c4|c5|c1|...] [--impl reference]

A "step" is one pass of the whole hot path over the workload: the CFL reduction (marut_max_dt_async, dt stays on the
device) followed by the three fused marut_ssprk_stage launches of one SSP-RK33 step (SURVEY 8(a) rows a1..a10 as the
physics has them).  Default workload: BASELINE.json configs[1] (c2: 3-D Euler, N=4, 32^3 periodic hexes, ~20.5M DOF),
synthetic seeded inputs.  One JSON line is printed by rank 0.

Timing: W warm-up steps, then blocks of EXACTLY K steps, each block between one CUDA-event pair on the
launching stream, repeated (>= 5 times) until the timed region is >= 1 s; value / ms_per_step are the MEDIAN block
(min / max beside it); the step is replayed as a CUDA graph (--no-graph: eager launches; ms_per_step_eager is always
reported).  roofline: CUDA events around every marut_ssprk_stage call of one eager K-step block.  The default run also
measures the other configs of BASELINE.json (c1, c3, c4w, c5) with the same protocol -> "configs".

N > 1 (torchrun): the path does not shard in this build ("replicas only"): every rank
advances its own replica of the workload, no data-path collective; value = units of all ranks / max time.

--impl reference: the CPU oracle (oracle/), as it stands, on the host cores, on a bounded sample of the
same workload.  Rank 0 only.
"""
from __future__ import annotations

import argparse
import math
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "DG RHS+SSPRK3 DOF-stage updates/s (FP64)"
UNIT = "DOF-stage/s"
# bounded oracle samples: (cells per direction, target seconds)
E2E_LANES = 3
ORACLE_SAMPLE_CELLS = {"c1": None, "c2": 12, "c2s": 12, "c3": 16, "c4": 64, "c4w": 64, "c4b": 64, "c4v": 64, "c5": 8, "c2m": 8}
# c4b: per-stage Hennemann-Gassner indicator (binding defaults, R15) feeding the DG/FV blend
SHOCK_CAPTURE = dict(s=9.21024, alpha_min=1e-3, alpha_max=0.5, smooth=True)


def make_workload(name, cells=None):
    """c1..c5, c4w: the configs of BASELINE.json (workloads.make_case); c2s: c2 with the entropy-stable split-form
    volume integral; c4b: c4w as a shock-capturing run -- split form, and in
    every Runge-Kutta stage the shock indicator of the stage's input state, the blended DG/FV stage and the positivity floor;
    c2m: the Taylor-Green flow of c2 on a box with one half refined once (3-D 4:1 mortar faces, NEXT-4);
    c4v: c4w as a Navier-Stokes problem (BR1 across the 2-D mortars, NEXT-4)"""
    import workloads as wl

    if name == "c2m":
        # c2's flow on a box whose x < pi half is split once: 3-D 4:1 mortar faces (R21)
        K = cells or 24
        m = wl.octree_box_mesh(4, K=K, lo=(0.0,) * 3, hi=(2 * math.pi,) * 3)
        return wl.Case("c2m", m, wl.taylor_green(m, noise=1e-3), 20, cfl=0.4)
    if name == "c4b":
        c = wl.make_case("c4w", cells=cells)
        c.mesh.volume_form = 1
        c.name = "c4b"
        c.shock_capture = dict(SHOCK_CAPTURE)
        # shock profile one fine element wide: the indicator flags it (alpha_e reaches alpha_max along the shock); the
        # 6-element profile of c4 / c4w is resolved at N = 3 and would leave alpha_e = 0 everywhere
        c.u0 = wl.mach10_shock(c.mesh, half_width=1.0 * c.mesh.info["h_fine"])
        return c
    if name == "c4v":
        # c4w's mesh and shock as a Navier-Stokes problem: BR1 across 2-D 2:1 mortars (NEXT-4; R23)
        c = wl.make_case("c4w", cells=cells)
        c.mesh.physics, c.mesh.mu, c.mesh.Pr = wl.NAVIER_STOKES, 1e-3, 0.72
        c.name = "c4v"
        return c
    if name == "c2s":
        c = wl.make_case("c2", cells=cells)
        c.mesh.volume_form = 1
        c.name = "c2s"
        return c
    return wl.make_case(name, cells=cells)


def workload_name(case):
    m = case.mesh
    phys = {0: "Euler", 1: "Navier-Stokes (BR1)", 2: "reacting Euler, 5 species"}[m.physics]
    if getattr(m, "volume_form", 0):
        phys += " (entropy-stable split form, Ranocha flux)"
    if getattr(case, "shock_capture", None):
        phys += " + per-stage shock indicator and DG/FV sub-cell blend"
    return (f"{case.name}: {m.dim}-D {phys}, N={m.N}, {m.n_elem} elements, {m.n_elem * m.nn} nodes, "
            f"{m.n_dof} DOF, {len(m.mortar)} mortars, {len(m.bface)} boundary faces")


def algorithmic_bytes_per_dof_stage(mesh, affine=True):
    """state traffic 16 B (stage 0) + 24 B + 24 B = 64/3 B per DOF-stage; curved meshes add the
    per-node metric terms (d*d + 1 doubles per node per sweep).  Navier-Stokes is the two-sweep BR1 form the
    library implements: the gradient sweep reads u and the metrics and writes S, the stage
    sweep reads u, S, the metrics and u_n and writes u_out."""
    nv, d = mesh.n_var, mesh.dim
    met = 0.0 if affine else 8.0 * (d * d + 1) / nv
    b = 64.0 / 3.0 + met
    if mesh.physics == 1:
        grad = 8.0 * (d * (d + 1) // 2 + d) / nv   # stress tensor + heat flux from the BR1 gradient: d(d+1)/2 + d doubles per node
        b += 8.0 + met + 2.0 * grad            # second read of u, second read of the metrics, viscous tensor written + read
    return b


def single_sweep_bytes_per_dof_stage(mesh, affine=True):
    """the figure a one-sweep operator would need: context for the NS line"""
    return 64.0 / 3.0 + (0.0 if affine else 8.0 * (mesh.dim * mesh.dim + 1) / mesh.n_var)


# FP64 vector peak for the ALU-bound reacting stage: 148 SMs x 64 DFMA/clk x 2 flop x max SM clock
def fp64_peak_tflops(sm_mhz=1965.0):
    return 148 * 64 * 2 * sm_mhz * 1e6 / 1e12


# --------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """SM clock, power and clock-event reasons sampled through NVML every ~2 ms on a host thread while the
    timed region runs (an nvidia-smi subprocess is too slow to see a region of tens of milliseconds)."""

    def __init__(self, index):
        self.index, self.samples, self.stop_flag, self.thread, self.smax = index, [], False, None, None

    def start(self):
        import threading
        try:
            import pynvml as nv

            nv.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = int(vis.split(",")[self.index]) if vis and vis.split(",")[self.index].isdigit() else self.index
            h = nv.nvmlDeviceGetHandleByIndex(idx)
            self.smax = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
        except Exception:
            return

        def loop():
            while not self.stop_flag:
                try:
                    self.samples.append((nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM), nv.nvmlDeviceGetPowerUsage(h) / 1e3,
                                         nv.nvmlDeviceGetCurrentClocksEventReasons(h)))
                except Exception:
                    pass
                time.sleep(0.002)

        self.thread = threading.Thread(target=loop, daemon=True)
        self.thread.start()

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": self.smax, "reasons": [], "samples": 0}
        if self.thread is None:
            return out
        self.stop_flag = True
        self.thread.join(timeout=2)
        import pynvml as nv

        names = {nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown", nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown", nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksEventReasonHwPowerBrakeSlowdown: "hw_power_brake_slowdown"}
        if self.samples:
            sm = sorted(s[0] for s in self.samples)
            mask = 0
            for s in self.samples:
                mask |= s[2]
            out.update(sm_mhz=sm[len(sm) // 2], sm_min_mhz=sm[0], reasons=sorted(v for k, v in names.items() if mask & k),
                       samples=len(sm), power_w_max=max(s[1] for s in self.samples))
        return out


# --------------------------------------------------------------------------------------------- oracle arm
def oracle_advance(om, case, u, n):
    """n SSP-RK33 steps of the oracle, dt from its own CFL reduction; shock-capturing workloads recompute the blending
    field from the input state of every stage"""
    sc = getattr(case, "shock_capture", None)
    if not sc:
        return om.run(u, n, cfl=case.cfl)[0]
    for _ in range(n):
        dt = om.max_dt(u, case.cfl)
        un, uin = u, u
        for k in range(3):
            om.set_blend(om.shock_indicator(uin, **sc))
            uin = om.positivity_floor(om.ssprk_stage(k, dt, 0.0, un, uin))[0]
        u = uin
    return u


def oracle_sample(workload, budget_s):
    """time the CPU oracle (as it stands, never tuned) on a bounded sample of the workload: the same config at fewer
    elements per direction, as many SSP-RK33 steps (dt from its own CFL reduction) as fit the budget: two thirds of it
    on all host cores, one third on ONE core (SURVEY 8(d) 'Timing')."""
    import oracle

    cells = ORACLE_SAMPLE_CELLS[workload]
    c = make_workload(workload, cells=cells)
    om = oracle.OracleMesh(c.mesh)
    ncores = oracle.num_threads()

    def timed(budget):
        t0 = time.perf_counter()
        u = oracle_advance(om, c, c.u0, 1)          # calibration step
        t1 = time.perf_counter() - t0
        n = max(1, min(200, int(budget / max(t1, 1e-6)) - 1))
        t0 = time.perf_counter()
        oracle_advance(om, c, u, n)
        return n, time.perf_counter() - t0

    n, t = timed(budget_s * 2.0 / 3.0)
    oracle.set_num_threads(1)
    try:
        n1, t1 = timed(budget_s / 3.0)
    finally:
        oracle.set_num_threads(ncores)
    return {"case": c, "steps": n, "s_per_step": t / n, "value": c.mesh.n_dof * 3 * n / t, "value_1core": c.mesh.n_dof * 3 * n1 / t1,
            "cores": ncores,
            "sample": f"{workload} at {c.mesh.n_elem} elements ({c.mesh.n_dof} DOF), {n} SSP-RK33 steps incl. CFL reduction in "
                      f"{t:.1f} s on {ncores} cores and {n1} steps in {t1:.1f} s on 1 core, g++ -O2 -ffp-contract=off + OpenMP over elements"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import workloads as wl

    per_step_budget = 60.0 / max(1, args.steps + args.warmup)
    import oracle

    cells = ORACLE_SAMPLE_CELLS[args.workload]
    c = make_workload(args.workload, cells=cells)
    om = oracle.OracleMesh(c.mesh)
    # one "step" of this arm = `inner` SSP-RK33 steps of the sample, sized to per_step_budget
    t0 = time.perf_counter()
    u = oracle_advance(om, c, c.u0, 1)
    t1 = time.perf_counter() - t0
    inner = max(1, min(50, int(per_step_budget / max(t1, 1e-6))))
    for _ in range(args.warmup):
        u = oracle_advance(om, c, u, inner)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        u = oracle_advance(om, c, u, inner)
    t = time.perf_counter() - t0
    value = c.mesh.n_dof * 3 * inner * args.steps / t
    sample = (f"{args.workload} at {c.mesh.n_elem} elements ({c.mesh.n_dof} DOF); one bench step = {inner} SSP-RK33 steps "
              f"incl. CFL reduction; g++ -O2 -ffp-contract=off + OpenMP over elements")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(c), "full_workload": args.workload, "sampled": True},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------- N > 1
def max_over_ranks(values, world, device="cpu"):
    """element-wise MAX over the ranks of per-rank timings (the only cross-rank step of this bench: the path runs
    as independent replicas)"""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def aggregate_value(n_dof, steps, world, ms):
    """whole-job DOF-stage updates per second: every replica advances n_dof DOFs through 3 stages per step"""
    return n_dof * 3 * steps * world / (ms * 1e-3)


# --------------------------------------------------------------------------------------------- CUDA arm
def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


KERNELS = {"euler": "stage_pencil_kernel (fused Euler stage: persistent TMA-fed line kernel)",
           "euler_mortar2d": "mortar_flux2d_kernel + stage_pencil_kernel plain / mortar instantiations over tile lists (fused Euler stage, 2-D mortars)",
           "euler_node": "stage_node_kernel (fused Euler stage, thread per node)",
           "euler_mortar3d": "mortar_flux3d_kernel + stage_node_kernel (fused Euler stage, 3-D mortar instantiation)",
           "split": "stage_split_kernel (fused Euler stage, split-form volume integral)",
           "split_blend": "stage_split_kernel (fused Euler stage, split-form volume integral blended with the sub-cell FV residual)",
           "ns": "gradient_kernel + stage_phys_kernel (BR1 gradient sweep + fused NS stage)",
           "react": "eos_kernel + stage_phys_kernel (mixture temperature + fused reacting stage)"}


class Workload:
    """one workload on the current device: library handle, state buffers, and one step of the hot path (the CFL
    reduction with dt left on the device + the three fused stages) in eager form and as a replayable CUDA graph"""

    def __init__(self, name, args, torch, mb):
        import numpy as np

        self.torch, self.args, self.name = torch, args, name
        self.case = make_workload(name)
        self.mesh = self.case.mesh
        self.gm = mb.MarutMesh(self.mesh)
        self.affine = self.gm.is_affine
        self.u0_host = torch.from_numpy(np.ascontiguousarray(self.case.u0)).pin_memory()
        self.u = self.u0_host.cuda()
        self.ua, self.ub = torch.empty_like(self.u), torch.empty_like(self.u)
        # The configs are short runs (BASELINE.json: 10-20 steps; c4/c5 leave their well-posed window after ~100-190
        # steps without the paper's limiter / implicit chemistry), so the bench repeats the config:
        # every `case.steps` steps the next step starts again from the pristine u0 (its stages read u0 directly, so the
        # restart costs no extra copy and no extra traffic).
        self.u0_dev = self.u.clone()
        self.counter = 0
        self.sc = getattr(self.case, "shock_capture", None)
        self.alpha = None
        if self.sc:
            self.alpha = torch.zeros(self.mesh.n_elem, dtype=torch.float64, device=self.u.device)
            self.gm.set_blend(self.alpha)
        # dt stays on the device (marut_max_dt_async -> marut_ssprk_stage_dev: the same dt and the same stage results bit
        # for bit, tests/test_gpu_async_dt.py), so the host queues the whole step without waiting for the CFL reduction
        self.dt_dev = torch.zeros(1, dtype=torch.float64, device=self.u.device)
        self.dts = torch.zeros(2, dtype=torch.float64, device=self.u.device)   # fused step: dt ping-pong
        self.graphs = None
        # the step the graph blocks replay: marut_ssprk33_step_cfl (the next step's CFL reduction inside the last stage's
        # kernel where the stage kernel supports it) unless the workload interleaves other calls with the stages
        self.fused_step = not (self.sc or args.sync_dt or args.no_graph or args.no_fused_cfl)

    def kernel_label(self):
        m = self.mesh
        if m.physics == 1:
            return KERNELS["ns"]
        if m.physics == 2:
            return KERNELS["react"]
        if getattr(m, "volume_form", 0):
            return KERNELS["split_blend" if self.sc else "split"]
        if m.dim == 3 and len(m.mortar):
            return KERNELS["euler_mortar3d"]
        # the library runs the line kernel only on meshes whose tiles (128 / n^(d-1) elements) fill the device: 3 CTAs per SM
        lines = (m.N + 1) ** (m.dim - 1)
        ntile = -(-m.n_elem // max(1, 128 // lines))
        sms = self.torch.cuda.get_device_properties(self.u.device).multi_processor_count
        if self.affine and ntile >= 3 * sms:
            if m.dim == 2 and len(m.mortar):
                return KERNELS["euler_mortar2d"]
            return KERNELS["euler"]
        return KERNELS["euler_node"]

    def _step(self, src, ev=None):
        torch, gm, sc, stream = self.torch, self.gm, self.sc, self.torch.cuda.current_stream()
        cfl = self.case.cfl
        if self.args.sync_dt:
            dt = gm.max_dt(src, cfl)
        else:
            gm.max_dt_async(src, cfl, self.dt_dev)
        for s, (un, uin, uout) in enumerate(((src, src, self.ua), (src, self.ua, self.ub), (src, self.ub, self.u))):
            if sc:
                gm.shock_indicator(uin, self.alpha, **sc)
            if ev is not None:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
            if self.args.sync_dt:
                gm.stage(s, dt, 0.0, un, uin, uout)
            else:
                gm.stage_dev(s, self.dt_dev, 0.0, un, uin, uout)
            if ev is not None:
                e1.record(stream)
                ev.append((e0, e1))
            if sc:
                gm.positivity_floor(uout)

    def _step_cfl(self, j):
        """step j of a cycle through marut_ssprk33_step_cfl: j = 0 restarts from u0 (copy + CFL reduction), then the two
        device doubles alternate as dt_in / dt_out"""
        gm, cfl, d = self.gm, self.case.cfl, self.dts
        if self.mesh.physics == 2:
            # reacting mixture: marut_ssprk33_step_dt -- the step's own CFL reduction rides on the first stage's
            # thermochemistry pass (no separate wave-speed pass)
            if j == 0:
                self.u.copy_(self.u0_dev)
            gm.ssprk33_step_dt(self.u, self.ua, self.ub, cfl, d[0:1])
            return
        if j == 0:
            self.u.copy_(self.u0_dev)
            gm.max_dt_async(self.u, cfl, d[0:1])
            gm.ssprk33_step_cfl(self.u, self.ua, self.ub, cfl, d[0:1], d[1:2])
        elif j % 2 == 1:
            gm.ssprk33_step_cfl(self.u, self.ua, self.ub, cfl, d[1:2], d[0:1])
        else:
            gm.ssprk33_step_cfl(self.u, self.ua, self.ub, cfl, d[0:1], d[1:2])

    def step(self, ev=None, graph=False):
        j = self.counter % self.case.steps
        self.counter += 1
        if graph and self.graphs is not None:
            if self.fused_step:
                self.graphs[0 if j == 0 else (1 if j % 2 == 1 else 2)].replay()
            else:
                self.graphs[0 if j == 0 else 1].replay()
        else:
            self._step(self.u0_dev if j == 0 else self.u, ev)

    def capture(self):
        """the two variants of the step (from u0 / from u) as CUDA graphs: the library only launches on the stream it
        is given, so a step is capturable as it stands (tests/test_gpu_async_dt.py: replay equals eager bit for bit)"""
        if self.args.sync_dt or self.args.no_graph:
            return
        torch = self.torch
        gs = []
        if self.fused_step:
            for j in (0, 1, 2):
                self._step_cfl(j)                      # warm (function attributes of the fused instantiation)
            torch.cuda.synchronize()
            for j in (0, 1, 2):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    self._step_cfl(j)
                gs.append(g)
        else:
            for src in (self.u0_dev, self.u):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    self._step(src)
                gs.append(g)
        self.graphs = gs

    def block(self, K, graph, ev=None):
        """K steps bracketed by an event pair on the current stream; returns the pair"""
        torch = self.torch
        stream = torch.cuda.current_stream()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(K):
            self.step(ev, graph)
        b.record(stream)
        return a, b


def measure(w, args, barrier, world, rank, local):
    """timing protocol of one workload (SURVEY 8(d) 'Timing'): W warm-up steps; one eager block of K steps with an event
    pair around every marut_ssprk_stage call (roofline of the dominant kernel); then R >= 5 blocks of exactly K steps
    each, replayed as CUDA graphs, until the timed region is >= 1 s; the headline is the MEDIAN block."""
    import numpy as np

    torch = w.torch
    K = args.steps
    for _ in range(args.warmup):
        w.step()
    w.capture()
    for _ in range(args.warmup):
        w.step(graph=True)
    barrier()
    # eager block with per-stage events
    l0 = w.gm.launch_count
    ev = []
    a, b = w.block(K, graph=False, ev=ev)
    barrier()
    eager_ms = a.elapsed_time(b)
    launches_per_block = w.gm.launch_count - l0
    stage_ms = [x.elapsed_time(y) for x, y in ev]
    # graph blocks
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    use_graph = w.graphs is not None
    w.counter = 0                                       # the graph blocks start a cycle (restart from u0)
    blocks = []
    first = w.block(K, graph=use_graph)
    barrier()
    blocks.append(first[0].elapsed_time(first[1]))
    reps = int(min(400, max(5, math.ceil(args.min_ms / max(blocks[0], 1e-3)))))
    pairs = [w.block(K, graph=use_graph) for _ in range(reps - 1)]
    barrier()
    blocks += [x.elapsed_time(y) for x, y in pairs]
    clocks = sampler.stop() if rank == 0 else None
    if not np.isfinite(w.u.sum().item()):
        raise RuntimeError(f"{w.name}: solution became non-finite during the timed region")
    blocks_max = [max_over_ranks([t], world, device="cuda")[0] for t in blocks] if world > 1 else blocks
    med = float(np.median(blocks_max))
    return {"ms_block_median": med, "ms_blocks_min": min(blocks_max), "ms_blocks_max": max(blocks_max), "repeats": len(blocks_max),
            "timed_region_ms": float(sum(blocks_max)), "eager_ms_block": eager_ms, "stage_ms": stage_ms,
            "launches_per_block": launches_per_block, "clocks": clocks, "graph": use_graph}


def roofline_of(w, r, clocks):
    mesh, args = w.mesh, w.args
    peak, peak_src = measured_peaks()
    n_dof = mesh.n_dof
    stage_ms_avg = sum(r["stage_ms"]) / len(r["stage_ms"])
    b_alg = algorithmic_bytes_per_dof_stage(mesh, w.affine)
    achieved = b_alg * n_dof / (stage_ms_avg * 1e-3) / 1e9
    prof = {}
    tpath = os.path.join(ROOT, "profiles", "traffic.json")   # per-launch figures from the committed ncu captures
    if os.path.exists(tpath):
        try:
            prof = json.load(open(tpath))
        except Exception:
            prof = {}
    roof = {"bound": "hbm", "kernel": ("marut_ssprk_stage: " if args.sync_dt else "marut_ssprk_stage_dev: ") + w.kernel_label(),
            "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": prof.get(w.name),
            "traffic_source": "profiles/traffic.json (ncu --set full capture of the same command, committed; not measured in this run)",
            "peak_source": peak_src, "bytes_per_dof_stage": b_alg, "stage_ms_avg": stage_ms_avg,
            "stage_ms_by_stage": [sum(r["stage_ms"][k::3]) / len(r["stage_ms"][k::3]) for k in range(3)],
            "frac_of_8TBs_nominal": achieved / 8000.0}
    if 3 * n_dof * 8 < 126e6 and stage_ms_avg < 0.03:
        roof["note"] = ("the state fits L2 and a stage is one launch of a few microseconds: launch-latency bound, "
                        "neither the HBM nor the FP64 roofline applies to this size")
    if mesh.physics == 1:
        roof["single_sweep_bytes_per_dof_stage"] = single_sweep_bytes_per_dof_stage(mesh, w.affine)
        roof["frac_vs_single_sweep_bytes"] = roof["single_sweep_bytes_per_dof_stage"] * n_dof / (stage_ms_avg * 1e-3) / 1e9 / peak
    if mesh.physics == 2 or getattr(mesh, "volume_form", 0):
        # ALU-bound (chemistry / two-point volume fluxes): executed FP64 flops per stage from the committed ncu capture over the live time
        flops = prof.get(w.name + "_fp64_flops_per_stage")
        pk = fp64_peak_tflops((clocks or {}).get("sm_max_mhz") or 1965.0)
        ach = flops / (stage_ms_avg * 1e-3) / 1e12 if flops else None
        roof.update({"bound": "alu", "achieved": ach, "peak": pk, "unit": "TFLOP/s", "frac": (ach / pk) if ach else None,
                     "peak_source": "derived: 148 SMs x 64 FP64 FMA/clk x 2 x max SM clock (DESIGN.md section 7)",
                     "hbm_frac": achieved / peak})
    return roof


def measure_e2e(w, args, barrier, mb):
    """end to end through the public API with HOST buffers: every step copies its input state from pinned host memory
    (H2D), runs marut_max_dt_async + the three stages, and copies the result back (D2H).  E2E_LANES independent lanes (own
    handle, own device buffers, own stream) take the steps in turn, so the D2H of one step and the kernels of another
    overlap the H2D of the next (PCIe is full duplex; with two lanes the H2D engine idles while a lane computes); every
    step still pays both copies inside the timed region."""
    import numpy as np

    torch, mesh, sc, cfl = w.torch, w.mesh, w.sc, w.case.cfl
    lanes = []
    for k in range(E2E_LANES):
        st = torch.cuda.Stream()
        g = w.gm if k == 0 else mb.MarutMesh(mesh)
        lanes.append({"st": st, "gm": g, "u": torch.empty_like(w.u), "ua": torch.empty_like(w.u), "ub": torch.empty_like(w.u),
                      "out": torch.empty_like(w.u0_host).pin_memory(),
                      "dt": torch.zeros(1, dtype=torch.float64, device=w.u.device), "dt_out": torch.zeros(1, dtype=torch.float64).pin_memory()})
        if sc:
            lanes[k]["alpha"] = w.alpha if k == 0 else torch.zeros_like(w.alpha)
            g.set_blend(lanes[k]["alpha"])

    def e2e_step(k):
        L = lanes[k % E2E_LANES]
        with torch.cuda.stream(L["st"]):
            L["u"].copy_(w.u0_host, non_blocking=True)
            g = L["gm"]
            if args.sync_dt:
                dt = g.max_dt(L["u"], cfl)
            else:
                g.max_dt_async(L["u"], cfl, L["dt"])
            for s_, (uin, uout) in enumerate(((L["u"], L["ua"]), (L["ua"], L["ub"]), (L["ub"], L["u"]))):
                if sc:
                    g.shock_indicator(uin, L["alpha"], **sc)
                if args.sync_dt:
                    g.stage(s_, dt, 0.0, L["u"], uin, uout)
                else:
                    g.stage_dev(s_, L["dt"], 0.0, L["u"], uin, uout)
                if sc:
                    g.positivity_floor(uout)
            L["out"].copy_(L["u"], non_blocking=True)
            if not args.sync_dt:
                L["dt_out"].copy_(L["dt"], non_blocking=True)

    for k in range(2 * E2E_LANES):
        e2e_step(k)
    barrier()
    e_start, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e_start.record(lanes[0]["st"])
    for L in lanes[1:]:
        L["st"].wait_event(e_start)
    for k in range(args.steps):
        e2e_step(k)
    for L in lanes[1:]:
        lanes[0]["st"].wait_stream(L["st"])
    e_end.record(lanes[0]["st"])
    barrier()
    e2e_ms = e_start.elapsed_time(e_end)
    for L in lanes:
        if not np.isfinite(L["out"].sum().item()):
            raise RuntimeError("end-to-end result is not finite")
    for L in lanes[1:]:
        L["gm"].close()
    return e2e_ms


def run_cuda(args):
    import torch
    import torch.distributed as dist

    import paper_2605_26388_b200 as mb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def summary(w, r):
        n_dof, K = w.mesh.n_dof, args.steps
        return {"workload": workload_name(w.case), "value": aggregate_value(n_dof, K, world, r["ms_block_median"]), "unit": UNIT,
                "ms_per_step": r["ms_block_median"] / K, "ms_per_step_min": r["ms_blocks_min"] / K, "ms_per_step_max": r["ms_blocks_max"] / K,
                "ms_per_step_eager": r["eager_ms_block"] / K, "repeats": r["repeats"], "timed_region_ms": r["timed_region_ms"],
                "step_replayed_as_cuda_graph": r["graph"], "fused_cfl_step": bool(r["graph"] and w.fused_step),
                "step_call": (("marut_ssprk33_step_dt (the CFL reduction rides on the first stage's thermochemistry pass)" if w.mesh.physics == 2
                               else "marut_ssprk33_step_cfl") if (r["graph"] and w.fused_step) else "marut_max_dt_async + 3 x marut_ssprk_stage_dev"),
                "cfl": w.case.cfl, "restart_from_u0_every_steps": w.case.steps,
                "affine": bool(w.affine), "gpu_launches_per_step": r["launches_per_block"] / K,
                "roofline": roofline_of(w, r, r["clocks"]), "clocks": r["clocks"]}

    w = Workload(args.workload, args, torch, mb)
    r = measure(w, args, barrier, world, rank, local)
    e2e_ms = measure_e2e(w, args, barrier, mb)
    e2e_ms = max_over_ranks([e2e_ms], world, device="cuda")[0]
    mesh, n_dof, K = w.mesh, w.mesh.n_dof, args.steps
    main_sum = summary(w, r)
    value = main_sum["value"]
    e2e_value = aggregate_value(n_dof, K, world, e2e_ms)
    w.gm.close()
    del w
    torch.cuda.empty_cache()

    # the other configs of BASELINE.json, same protocol, device-resident figure only (N = 1, default workload only)
    others = {}
    if world == 1 and args.workload == "c2" and not args.no_configs:
        for name in ("c1", "c3", "c4w", "c5"):
            try:
                wo = Workload(name, args, torch, mb)
                ro = measure(wo, args, barrier, world, rank, local)
                others[name] = summary(wo, ro)
                wo.gm.close()
                del wo
                torch.cuda.empty_cache()
            except Exception as exc:                      # a config that cannot run is reported, never hidden
                others[name] = {"error": f"{type(exc).__name__}: {exc}"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
                "ms_per_step": main_sum["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": main_sum["workload"], "parallelism": "replicas only" if world > 1 else "1 GPU",
                           "l2": f"inputs larger than L2 ({3 * n_dof * 8 / 1e6:.0f} MB of state buffers vs 126 MB)"
                                 if 3 * n_dof * 8 > 126e6 else "state fits L2 (launch/latency-bound case; no flush)",
                           "step": ("marut_ssprk33_step_dt: three fused stage calls, the step's CFL reduction inside the first stage's "
                                    "thermochemistry pass (dt stays on the device; every restart from u0 adds a device copy)"
                                    if (main_sum["fused_cfl_step"] and main_sum["step_call"].startswith("marut_ssprk33_step_dt")) else
                                    "marut_ssprk33_step_cfl: three fused stages, the CFL reduction of the next step inside the last "
                                    "stage's kernel (dt stays on the device; every restart from u0 adds a device copy and one marut_max_dt_async)"
                                    if main_sum["fused_cfl_step"] else
                                    ("marut_max_dt" if args.sync_dt else "marut_max_dt_async (dt stays on the device)")
                                    + (" + 3 x (marut_shock_indicator + blended marut_ssprk_stage + marut_positivity_floor)"
                                       if main_sum["roofline"]["kernel"].endswith("FV residual)") else " + 3 x marut_ssprk_stage")),
                           "timing": f"median of {main_sum['repeats']} blocks of exactly {K} steps each (timed region "
                                     f"{main_sum['timed_region_ms']:.0f} ms), every block one CUDA-event pair"
                                     + (", the step replayed as a CUDA graph" if main_sum["step_replayed_as_cuda_graph"] else ", eager launches"),
                           "cfl": main_sum["cfl"], "restart_from_u0_every_steps": main_sum["restart_from_u0_every_steps"],
                           "affine": main_sum["affine"]},
                "ms_per_step_min": main_sum["ms_per_step_min"], "ms_per_step_max": main_sum["ms_per_step_max"],
                "ms_per_step_eager": main_sum["ms_per_step_eager"], "repeats": main_sum["repeats"],
                "timed_region_ms": main_sum["timed_region_ms"],
                "clocks": main_sum["clocks"],
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": n_dof * 8, "d2h_bytes_per_step": n_dof * 8 + 8,
                        "ms_per_step": e2e_ms / K,
                        "how": "pinned host buffers; %d lanes (handle + stream each) taking the steps in turn, so that the D2H and the kernels of earlier steps overlap the H2D of the next" % E2E_LANES},
                "gpu_launches": int(round(main_sum["gpu_launches_per_step"] * K)),
                "roofline": main_sum["roofline"]}
        if others:
            line["configs"] = others
        if world == 1 and not args.no_cpu_baseline:
            o = oracle_sample(args.workload, args.cpu_seconds)
            line["cpu_baseline"] = {"value": o["value"], "value_1core": o["value_1core"], "unit": UNIT, "cores": o["cores"], "kind": "oracle",
                                    "sample": o["sample"]}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="c2", choices=sorted(ORACLE_SAMPLE_CELLS))
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="budget of the cpu_baseline leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sync-dt", action="store_true", help="host-synchronised marut_max_dt every step instead of the device-resident dt")
    ap.add_argument("--no-graph", action="store_true", help="eager launches in the timed blocks instead of CUDA-graph replay")
    ap.add_argument("--no-fused-cfl", action="store_true", help="graph blocks replay marut_max_dt_async + 3 x marut_ssprk_stage_dev instead of marut_ssprk33_step_cfl")
    ap.add_argument("--no-configs", action="store_true", help="skip the other BASELINE.json configs (c1, c3, c4w, c5) of the default run")
    ap.add_argument("--min-ms", type=float, default=1000.0, help="repeat the K-step block until the timed region is at least this long")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
