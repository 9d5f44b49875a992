#!/usr/bin/env python
"""bench.py — one JSON line for the driver.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--prec f32|f64] [--k 0] [--impl reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: ONE DDM sweep = the sweep
kernel (Algorithm 1 on every subdomain: assemble b, n_wh WaveHoltz iterations of N_t-1 leapfrog steps
each, outgoing interface data, u_l) followed by the exchange kernel, on all subdomains of the config.
Metric: WaveHoltz DOF-timestep updates per second (BASELINE.json `metric`).

N > 1 (torchrun): the path shards by independent problems only ("replicas only"): every rank
sweeps its own replica of the workload, no data-path collective, weak scaling; time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "waveholtz_dof_timestep_updates_per_s"
UNIT = "DOF-steps/s"
N_WH = 5          # WaveHoltz iterations per sweep: the paper's benchmark count
SMS, FP32_LANES = 148, 128   # B200: SMs, FP32 FMA lanes per SM (FP64: half) -- B200_PROFILING.md / microarch guide


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number 1..5 (default 3)")
    ap.add_argument("--n", type=int, default=None, help="override elements per side (smaller same-shape problem)")
    ap.add_argument("--prec", default="f32", choices=["f32", "f64"])
    ap.add_argument("--k", type=int, default=0, help="DOFs per thread (0 = auto, 1 = one DOF per thread)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the secondary measurements")
    ap.add_argument("--distort", type=float, default=0.0,
                    help="> 0: the same config on general convex quads (interior vertices moved by distort*h; SURVEY F3)")
    return ap.parse_args()


def workload_name(inp, prec):
    geo = f"general convex quads (vertices distorted by {inp.meta['distort']} h)" if inp.vx is not None else "uniform quads"
    return (f"config{inp.name[3]}: {inp.nx}x{inp.ny} {geo} p={inp.p}, {inp.sx}x{inp.sy} subdomains of "
            f"{inp.nx // inp.sx}x{inp.ny // inp.sy} elements, {prec}, n_wh={N_WH}, warm start, relax 0.5")


# ---------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on the host cores
# ---------------------------------------------------------------------------------------------------
class OracleSample:
    """The oracle's DDM cycle (oracle.hz_oracle.ddm_cycle) on a bounded sample of the workload's
    subdomains.  The oracle's sparse mat-vecs and numpy vector ops are single-threaded."""

    def __init__(self, inp):
        from oracle import hz_oracle as O
        self.O = O
        if inp.vx is not None and inp.sx * inp.sy > 16:
            # general quads: the oracle assembles every element matrix in Python, so the sample is set up on the
            # lower-left 4x4 subdomains of the mesh only (same elements, same block shape, same N_t rule per element)
            ex, ey, p = inp.nx // inp.sx, inp.ny // inp.sy, inp.p
            sx, sy = min(4, inp.sx), min(4, inp.sy)
            nx, ny = sx * ex, sy * ey
            pr = O.Problem(nx, ny, p, 0, 0, 1, 1, inp.c_nodes[:ny * p + 1, :nx * p + 1], inp.omega,
                           inp.f_re[:ny * p + 1, :nx * p + 1].astype(complex), vx=inp.vx[:ny + 1, :nx + 1],
                           vy=inp.vy[:ny + 1, :nx + 1])
            self.st = O.ddm_setup(pr, sx, sy, inp.cfl_frac)   # N_t is that of the cropped mesh (fewer elements in the max)
        else:
            pr = O.Problem(inp.nx, inp.ny, inp.p, inp.x0, inp.y0, inp.x1, inp.y1, inp.c_nodes, inp.omega,
                           inp.f_re.astype(complex), vx=inp.vx, vy=inp.vy)
            self.st = O.ddm_setup(pr, inp.sx, inp.sy, inp.cfl_frac)
        self.n_sub = len(self.st.subs)
        self.dofs = self.st.subs[0].npx * self.st.subs[0].npy
        self.n_t = self.st.tab.n_t
        self.next = 0

    def run(self, count):
        """`count` subdomain cycles (round-robin over the subdomains); returns (seconds, DOF-steps)."""
        t0 = time.perf_counter()
        for _ in range(count):
            self.O.ddm_cycle(self.st, self.next % self.n_sub, N_WH, True)
            self.next += 1
        dt = time.perf_counter() - t0
        return dt, float(count) * self.dofs * N_WH * (self.n_t - 1)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2606_21695_b200.inputs import make_config
    inp = make_config(args.config, n=args.n, distort=args.distort)
    smp = OracleSample(inp)
    t, _ = smp.run(1)
    per_step = max(1, min(smp.n_sub, int(1.0 / max(t, 1e-4))))   # about 1 s of oracle work per step
    for _ in range(args.warmup):
        smp.run(per_step)
    tot_t = tot_u = 0.0
    for _ in range(args.steps):
        dt, u = smp.run(per_step)
        tot_t += dt
        tot_u += u
    val = tot_u / tot_t
    sample = f"{per_step} of {smp.n_sub} subdomain DDM cycles per step ({smp.dofs} DOF, n_wh={N_WH}, N_t={smp.n_t})"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(inp, "f64 oracle"), "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
# clocks sampled DURING the timed region
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append((time.perf_counter(), ln.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, ln in self.rows:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                clk, mxc = float(f[0]), float(f[1])
            except ValueError:
                continue
            mx = mxc
            if t0 <= ts <= t1 + 0.1:
                sm.append(clk)
                for nm, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------------
def flops_per_dof_step(p, quads=False):
    """Necessary FMAs of the assembled line-stencil formulation: 2(p+2) for A p + 5 updates.
    General quads: (p+1)^2 points per element x (2(p+1) gradient + 4 geometric factors + 2(p+1) D^T) over the
    p^2 DOFs an element adds, + 5 updates."""
    if quads:
        return 2.0 * ((p + 1) ** 2 * (4 * (p + 1) + 4) / float(p * p) + 5)
    return 2.0 * (2 * (p + 2) + 5)


def kernel_name(pinfo, quads=False):
    if quads:
        return "k_sweep_quad"
    if pinfo.cluster_size > 1:
        return "k_sweep_cl"
    if pinfo.dofs_per_thread == 1:
        return "k_sweep_dof"
    if pinfo.dofs_per_thread == -1:
        return "k_sweep_stream"
    return "k_sweep_ws" if pinfo.tile_mx == pinfo.tile_my and not os.environ.get("HZ_DISABLE_WS") else "k_sweep_tile"


def job_value(units_this_rank, ms_this_rank, world, device):
    """Whole-job throughput of `world` replicas: (sum of the units of all ranks) / (max over ranks of the
    time).  Every rank processes the same number of units (weak scaling), so the sum is world * units."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_this_rank], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    max_ms = float(t.item())
    return world * units_this_rank / (max_ms * 1e-3), max_ms


def time_sweeps(hz, torch, ctx, steps, warmup, flush, stream):
    """`steps` timed single-sweep calls (L2 flushed before each); returns device-ms lists and launch counts."""
    for _ in range(warmup):
        hz.hz_ddm_solve(ctx, 1, n_wh=N_WH, warm_start=True, relax=0.5, stream=stream)
    tot, swp, exc, launches, units = [], [], [], 0, 0.0
    for _ in range(steps):
        flush.add_(1.0)                      # write a buffer larger than L2 between timed iterations
        s = hz.hz_ddm_solve(ctx, 1, n_wh=N_WH, warm_start=True, relax=0.5, stream=stream)
        tot.append(s.total_ms)
        swp.append(s.sweep_ms_total)
        exc.append(s.exch_ms_total)
        launches += s.sweep_launches + s.exch_launches + s.other_launches
        units += s.dof_timesteps
    return tot, swp, exc, launches, units


def run_b200(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2606_21695_b200 import hz
    from paper_2606_21695_b200.inputs import make_config

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    prec = hz.HZ_F32 if args.prec == "f32" else hz.HZ_F64
    tdt = torch.float32 if prec == hz.HZ_F32 else torch.float64
    inp = make_config(args.config, n=args.n, distort=args.distort)
    quads = inp.vx is not None
    ctx, pinfo = hz.setup_from_inputs(inp, prec, args.k)
    stream = torch.cuda.current_stream().cuda_stream
    flush = torch.zeros(64 * 1024 * 1024, dtype=torch.float32, device="cuda")   # 256 MB > 126 MB L2
    nn = inp.npx * inp.npy
    u_dev = torch.zeros(2 * nn, dtype=tdt, device="cuda")
    hz.hz_ddm_solve(ctx, 2, n_wh=N_WH, reset_state=True, stream=stream)          # leave a non-trivial state

    # ---- kernel-resident timing: inputs already in HBM ----
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    t0 = time.perf_counter()
    tot, swp, exc, launches, units = time_sweeps(hz, torch, ctx, args.steps, args.warmup, flush, stream)
    barrier()
    t1 = time.perf_counter()
    clocks = sampler.stop(t0, t1) if sampler else None
    value, max_ms = job_value(units, float(sum(tot)), world, "cuda")

    # ---- end to end through the C ABI with HOST buffers: new source in, field out, every step ----
    f_host = torch.from_numpy(np.ascontiguousarray(inp.f_re)).pin_memory()
    u_host = torch.empty(2 * nn, dtype=tdt).pin_memory()
    for _ in range(2):
        hz.hz_set_source_ptr(ctx, f_host.data_ptr())
        hz.hz_ddm_solve(ctx, 1, n_wh=N_WH, u_out_ptr=u_dev.data_ptr(), stream=stream)
        u_host.copy_(u_dev)
    e2e_steps = max(3, min(args.steps, 10))
    barrier()
    te = time.perf_counter()
    e_units = 0.0
    for _ in range(e2e_steps):
        hz.hz_set_source_ptr(ctx, f_host.data_ptr())                             # H2D of f + rebuild of beta*b on device
        s = hz.hz_ddm_solve(ctx, 1, n_wh=N_WH, u_out_ptr=u_dev.data_ptr(), stream=stream)
        u_host.copy_(u_dev)                                                      # D2H of the gathered field
        e_units += s.dof_timesteps
    barrier()
    e_ms = (time.perf_counter() - te) * 1e3
    seq_value, _ = job_value(e_units, e_ms, world, "cuda")
    # the same through hz_ddm_solve_sources: one C-ABI call for the whole stream of sources, host to host, the copies
    # on private streams overlapping the sweeps (two alternating pinned inputs and outputs)
    f_pins = [f_host, (0.5 * torch.from_numpy(np.ascontiguousarray(inp.f_re))).pin_memory()]
    u_pins = [u_host, torch.empty(2 * nn, dtype=tdt).pin_memory()]
    n_src = max(e2e_steps, min(args.steps, 50))
    fp = [f_pins[i & 1].data_ptr() for i in range(n_src)]
    up = [u_pins[i & 1].data_ptr() for i in range(n_src)]
    hz.hz_ddm_solve_sources(ctx, fp[:2], up[:2], n_outer=1, n_wh=N_WH, stream=stream)       # allocation, warm-up
    barrier()
    te = time.perf_counter()
    si = hz.hz_ddm_solve_sources(ctx, fp, up, n_outer=1, n_wh=N_WH, stream=stream)
    barrier()
    p_ms = (time.perf_counter() - te) * 1e3
    e_value, _ = job_value(si.dof_timesteps, p_ms, world, "cuda")
    e2e = {"value": e_value, "unit": UNIT,
           "h2d_bytes_per_step": int(nn * 8), "d2h_bytes_per_step": int(2 * nn * u_host.element_size()),
           "steps": n_src, "what": "hz_ddm_solve_sources: per step H2D of a new source f from pinned host memory, "
                                   "rebuild of the load, 1 sweep + exchange, gather, D2H of u to pinned host memory; "
                                   "copies on private streams overlap the sweeps; wall clock around the call",
           "sequential_value": seq_value,
           "sequential_what": "hz_set_source(host f) + hz_ddm_solve(1 sweep, u_out) + D2H of u, one after the other"}

    if rank != 0:
        hz.hz_destroy(ctx)
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the sweep), live numbers ----
    sweep_ms = float(sum(swp)) / args.steps
    units_per_launch = units / args.steps
    fl = flops_per_dof_step(inp.p, quads)
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    lanes = FP32_LANES if prec == hz.HZ_F32 else FP32_LANES // 2
    peak_tf = SMS * lanes * 2 * sm_max * 1e6 / 1e12
    achieved_tf = units_per_launch * fl / (sweep_ms * 1e-3) / 1e12
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "sweep_traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as fh:
            traffic = json.load(fh).get(f"config{args.config}_{args.prec}" + ("_quads" if quads else ""))
    try:
        probe_tf = hz.hz_peak_probe(0 if prec == hz.HZ_F32 else 1, stream)
    except Exception:
        probe_tf = None
    roofline = {"bound": "alu", "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved_tf / peak_tf,
                "traffic": traffic, "kernel": kernel_name(pinfo, quads),
                "peak_source": f"derived: {SMS} SMs x {lanes} FMA lanes x 2 x {sm_max:.0f} MHz (guide unit counts, "
                               "nvidia-smi max clock); MEASURED_PEAKS.json has no CUDA-core entry",
                "peak_measured_fma_probe": probe_tf, "frac_of_probe": (achieved_tf / probe_tf) if probe_tf else None,
                "flops_per_dof_step": fl, "dof_steps_per_launch": units_per_launch, "sweep_kernel_ms": sweep_ms,
                "exchange_kernel_ms": float(sum(exc)) / args.steps}

    extras = {}
    if not args.no_extras and world == 1:
        extras = run_extras(hz, torch, args, flush, stream)
    hz.hz_destroy(ctx)

    # ---- the oracle on the host cores, bounded sample ----
    smp = OracleSample(inp)
    t_one, _ = smp.run(1)
    count = max(2, min(smp.n_sub, int(12.0 / max(t_one, 1e-4))))
    dt, u = smp.run(count)
    cpu = {"value": u / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
           "sample": f"{count} of {smp.n_sub} subdomain DDM cycles of the same workload ({smp.dofs} DOF each, n_wh={N_WH}, "
                     f"N_t={smp.n_t}), oracle/hz_oracle.py::ddm_cycle, numpy/scipy single thread"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": args.prec, "data": "synthetic",
            "config": {"workload": workload_name(inp, args.prec), "n_t": pinfo.n_t, "dofs_per_sub": pinfo.dofs_per_sub,
                       "blocks": pinfo.blocks, "threads_per_block": pinfo.threads_per_block,
                       "dofs_per_thread": pinfo.dofs_per_thread, "smem_bytes": pinfo.smem_bytes,
                       "l2": "flushed between timed steps (256 MB write)",
                       "parallelism": "replicas only (one independent problem per GPU)" if world > 1 else "1 GPU"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
            "extras": extras}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_extras(hz, torch, args, flush, stream):
    """Secondary numbers (not the headline line): the other precision on the same workload, config 2,
    and DDM time-to-solution on config 1 (fp64, tol 1e-8) -- SURVEY.md section 8(d)."""
    from paper_2606_21695_b200.inputs import make_config
    out = {}
    cases = [(args.config, "f64" if args.prec == "f32" else "f32", 0), (args.config, args.prec, 1), (2, "f32", 0), (2, "f64", 0)]
    for cfg, pr, k in cases:
        try:
            inp = make_config(cfg, n=args.n if cfg == args.config else None)
            prec = hz.HZ_F32 if pr == "f32" else hz.HZ_F64
            ctx, pinfo = hz.setup_from_inputs(inp, prec, k)
            hz.hz_ddm_solve(ctx, 2, n_wh=N_WH, reset_state=True, stream=stream)
            tot, swp, exc, _, units = time_sweeps(hz, torch, ctx, 5, 2, flush, stream)
            lanes = FP32_LANES if pr == "f32" else FP32_LANES // 2
            rate = units / (sum(swp) * 1e-3)
            out[f"config{cfg}_{pr}_k{pinfo.dofs_per_thread}"] = {
                "dof_steps_per_s_sweep_kernel": rate, "sweep_ms": sum(swp) / 5, "exchange_ms": sum(exc) / 5,
                "frac_of_derived_peak": rate * flops_per_dof_step(inp.p) / (SMS * lanes * 2 * 1965e6)}
            hz.hz_destroy(ctx)
        except Exception as e:  # an extra must never take the headline line down
            out[f"config{cfg}_{pr}_k{k}"] = {"error": str(e)}
    # DDM time-to-solution (BASELINE.json metric 1): relaxed fixed-point iteration on lambda to a global relative
    # residual (hz_residual, fp64), n_wh = 2, rho = 0.5, warm start, CUDA-graph replay between residual checks
    for cfg, pr, tol, every, nmax in ((1, "f64", 1e-8, 10, 2000), (2, "f32", 1e-4, 50, 5000), (2, "f64", 1e-4, 50, 5000)):
        key = f"config{cfg}_{pr}_time_to_solution"
        try:
            inp = make_config(cfg)
            ctx, pinfo = hz.setup_from_inputs(inp, hz.HZ_F32 if pr == "f32" else hz.HZ_F64, 0)
            hz.hz_ddm_solve(ctx, every, n_wh=2, reset_state=True, use_graph=True, stream=stream)   # graph capture, warm-up
            t0 = time.perf_counter()
            s = hz.hz_ddm_solve(ctx, nmax, n_wh=2, warm_start=True, relax=0.5, tol=tol, check_every=every,
                                reset_state=True, use_graph=True, stream=stream)
            out[key] = {"tol": tol, "sweeps": s.n_outer_done, "rel_residual": s.rel_residual, "device_ms": s.total_ms,
                        "wall_ms": (time.perf_counter() - t0) * 1e3, "n_wh": 2, "relax": 0.5, "cuda_graph": True}
            hz.hz_destroy(ctx)
        except Exception as e:
            out[key] = {"error": str(e)}
    # the same with the Krylov-accelerated outer iteration (hz_ddm_solve_gmres, restarted GMRES(50) on (lambda, u))
    for cfg, pr, tol in ((2, "f32", 1e-4), (2, "f64", 1e-4)):
        key = f"config{cfg}_{pr}_time_to_solution_gmres"
        try:
            inp = make_config(cfg)
            ctx, pinfo = hz.setup_from_inputs(inp, hz.HZ_F32 if pr == "f32" else hz.HZ_F64, 0)
            hz.hz_ddm_solve_gmres(ctx, 5, n_wh=2, restart=50, stream=stream)                      # allocation, warm-up
            t0 = time.perf_counter()
            s = hz.hz_ddm_solve_gmres(ctx, 3000, n_wh=2, relax=0.5, restart=50, tol=tol, reset_state=True, stream=stream)
            out[key] = {"tol": tol, "sweeps": s.sweeps_done, "cycles": s.cycles, "rel_residual": s.rel_residual,
                        "device_ms": s.total_ms, "wall_ms": (time.perf_counter() - t0) * 1e3, "n_wh": 2, "relax": 0.5,
                        "restart": 50}
            hz.hz_destroy(ctx)
        except Exception as e:
            out[key] = {"error": str(e)}
    # the rows SURVEY.md 8(f) marks "next": general convex quads (F3) and 3-D hexahedra (F4), sweep kernel only
    try:
        inp = make_config(3, n=args.n, distort=0.2)
        ctx, pinfo = hz.setup_from_inputs(inp, hz.HZ_F32, 0)
        hz.hz_ddm_solve(ctx, 2, n_wh=N_WH, reset_state=True, stream=stream)
        tot, swp, exc, _, units = time_sweeps(hz, torch, ctx, 3, 1, flush, stream)
        rate = units / (sum(swp) * 1e-3)
        out["config3_general_quads_f32"] = {
            "dof_steps_per_s_sweep_kernel": rate, "sweep_ms": sum(swp) / 3, "n_t": pinfo.n_t, "kernel": "k_sweep_quad",
            "frac_of_derived_peak": rate * flops_per_dof_step(inp.p, True) / (SMS * FP32_LANES * 2 * 1965e6)}
        hz.hz_destroy(ctx)
    except Exception as e:
        out["config3_general_quads_f32"] = {"error": str(e)}
    try:
        from paper_2606_21695_b200 import hz3
        from paper_2606_21695_b200.inputs import make_config_3d
        for name, n, p, s in (("hex_128cubed_p1_sub8", 128, 1, 8), ("hex_48cubed_p3_sub3", 48, 3, 3)):
            i3 = make_config_3d(n, p, s)
            c3 = hz3.hz3_mesh_setup(i3.nx, i3.ny, i3.nz, i3.box, i3.p, i3.c_nodes, i3.omega, i3.f_re)
            try:
                info3 = hz3.hz3_partition(c3, i3.sx, i3.sy, i3.sz, hz.HZ_F32)
                hz3.hz3_ddm_solve(c3, 1, n_wh=N_WH, reset_state=True, stream=stream)
                r = hz3.hz3_ddm_solve(c3, 3, n_wh=N_WH, stream=stream)
                out[name + "_f32"] = {"dof_steps_per_s_sweep_kernel": r.dof_timesteps / (r.sweep_ms_total * 1e-3),
                                      "sweep_ms": r.sweep_ms_total / 3, "n_t": info3.n_t,
                                      "nodes_per_thread": info3.nodes_per_thread, "blocks": info3.blocks}
            finally:
                hz3.hz3_destroy(c3)
    except Exception as e:
        out["hex_3d"] = {"error": str(e)}
    return out


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
