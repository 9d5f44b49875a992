#!/usr/bin/env python
"""bench.py — one JSON line for the driver, plus the measurement tables of profiles/.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--p 3] [--sub 8] [--prec f32|f64] [--k 0]
                    [--impl b200|reference] [--no-extras]
    python bench.py --sweep cfg2|cfg3|cfg4|cfg5|quads|3d|tts|minres [--scale S]     # markdown tables (profiles/*.md)

A "step" is one pass of the whole hot path over one batch of synthetic input: ONE DDM sweep = the sweep kernel
(Algorithm 1 on every subdomain: assemble b, n_wh WaveHoltz iterations of N_t-1 leapfrog steps each, outgoing
interface data, u_l) followed by the exchange kernel, on all subdomains of the config.
Metric: WaveHoltz DOF-timestep updates per second (BASELINE.json `metric`).
Default workload: the largest single-GPU configuration, config 5 (2048x2048 quads, p = 3, 38 M DOF, 65 536
subdomains of 8x8 elements), fp32; the other configs are `extras`.

N > 1 (torchrun): the path shards by independent problems only ("replicas only"): every rank sweeps its
own replica of the workload, no data-path collective, weak scaling; time = max over ranks.
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
SMS, FP32_LANES, SM_MHZ = 148, 128, 1965.0   # B200: SMs, FP32 FMA lanes per SM (FP64: half), max SM clock (guides)
E2E_SOURCES = 12  # sources of the end-to-end leg (independent of --steps)

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel: STORED figures from one
# `ncu --set full` capture each (not measured in this run); the summaries are in profiles/.
STORED_TRAFFIC = {
    "config5_p3_s8_f32": {"bytes": 1.376e9, "from": "profiles/r02_k_sweep_pack_cfg5_f32.md", "captured": "round 2"},
    "config5_p3_s8_f64": {"bytes": 2.753e9, "from": "profiles/r02_l_sweep_pack_cfg5_f64.md", "captured": "round 2"},
    "config3_p3_s8_f32": {"bytes": 62.5e6, "from": "profiles/r02_m_sweep_pack_cfg3_f32.md", "captured": "round 2"},
    "config3_p3_s8_f64": {"bytes": 137.6e6, "from": "profiles/r02_n_sweep_pack_cfg3_f64.md", "captured": "round 2"},
    "config4_p3_s32_f32": {"bytes": 238.3e6, "from": "profiles/r02_c_sweep_cw_cfg4_f32.md", "captured": "round 2"},
    "config4_p3_s32_f64": {"bytes": 501.2e6, "from": "profiles/r02_d_sweep_cw_cfg4_f64.md", "captured": "round 2"},
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config number 1..5 (default 5, the largest)")
    ap.add_argument("--n", type=int, default=None, help="override elements per side (smaller same-shape problem)")
    ap.add_argument("--p", type=int, default=None, help="degree (config 5 sweeps 1..4 at 6144/p elements per side)")
    ap.add_argument("--sub", type=int, default=None, help="elements per subdomain side (config 5 sweeps 4..64)")
    ap.add_argument("--prec", default="f32", choices=["f32", "f64"])
    ap.add_argument("--k", type=int, default=0, help="DOFs per thread (0 = auto, 1 = one DOF per thread)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the secondary measurements")
    ap.add_argument("--distort", type=float, default=0.0,
                    help="> 0: the same config on general convex quads (interior vertices moved by distort*h; SURVEY F3)")
    ap.add_argument("--sweep", default=None, choices=["cfg2", "cfg3", "cfg4", "cfg5", "quads", "3d", "tts", "minres"],
                    help="print a markdown table instead of the JSON line")
    ap.add_argument("--scale", type=int, default=1, help="--sweep cfg5/quads: shrink the mesh side by this factor")
    return ap.parse_args()


def workload_inputs(args):
    from paper_2606_21695_b200.inputs import make_config
    n = args.n
    if args.config == 5 and n is None and args.p is not None:
        n = 6144 // args.p                 # matched DOF count (BASELINE.json config 5)
    return make_config(args.config, n=n, p=args.p, sub_elems=args.sub, distort=args.distort)


def workload_name(inp, prec):
    geo = f"general convex quads (vertices distorted by {inp.meta['distort']} h)" if inp.vx is not None else "uniform quads"
    return (f"config{inp.name[3]}: {inp.nx}x{inp.ny} {geo} p={inp.p}, {inp.sx}x{inp.sy} subdomains of "
            f"{inp.nx // inp.sx}x{inp.ny // inp.sy} elements, {prec}, n_wh={N_WH}, warm start, relax 0.5")


# ---------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on ALL host cores (one process per core, each running the
# oracle's DDM cycle on its share of the subdomains)
# ---------------------------------------------------------------------------------------------------
def _oracle_window(inp, w):
    """The lower-left w x w subdomains of the workload as a problem of their own (same elements, wave speed, source
    and N_t as the full mesh: a subdomain's DDM cycle sees nothing else).  Plain arrays, picklable."""
    ex, ey, p = inp.nx // inp.sx, inp.ny // inp.sy, inp.p
    wx, wy = min(w, inp.sx), min(w, inp.sy)
    hx, hy = (inp.x1 - inp.x0) / inp.nx, (inp.y1 - inp.y0) / inp.ny
    return dict(nx=wx * ex, ny=wy * ey, p=p, x0=inp.x0, y0=inp.y0, x1=inp.x0 + wx * ex * hx, y1=inp.y0 + wy * ey * hy,
                c=inp.c_nodes[:wy * ey * p + 1, :wx * ex * p + 1].copy(), omega=inp.omega,
                f=inp.f_re[:wy * ey * p + 1, :wx * ex * p + 1].copy(), sx=wx, sy=wy, cfl=inp.cfl_frac,
                c_max=float(inp.c_nodes.max()), hx=hx, hy=hy,
                vx=None if inp.vx is None else inp.vx[:wy * ey + 1, :wx * ex + 1].copy(),
                vy=None if inp.vy is None else inp.vy[:wy * ey + 1, :wx * ex + 1].copy())


def _oracle_worker(job):
    """One host core: set the oracle up on the window, then run DDM cycles (oracle.hz_oracle.ddm_cycle) on the
    subdomains rank, rank + stride, ... for `seconds`.  -> (cycles done, seconds of cycle time, dofs, n_t)."""
    os.environ["OMP_NUM_THREADS"] = "1"
    from oracle import hz_oracle as O
    w, rank, stride, seconds = job
    pr = O.Problem(w["nx"], w["ny"], w["p"], w["x0"], w["y0"], w["x1"], w["y1"], w["c"], w["omega"],
                   w["f"].astype(complex), vx=w["vx"], vy=w["vy"])
    n_t = None if w["vx"] is not None else O.choose_nt(w["p"], w["hx"], w["hy"], w["c_max"], w["omega"], w["cfl"])
    st = O.ddm_setup(pr, w["sx"], w["sy"], w["cfl"], n_t=n_t)
    n_sub = len(st.subs)
    dofs = st.subs[0].npx * st.subs[0].npy
    done, l = 0, rank % n_sub
    t0 = time.perf_counter()
    while True:
        O.ddm_cycle(st, l, N_WH, True)
        done += 1
        l = (l + stride) % n_sub
        if time.perf_counter() - t0 >= seconds:
            break
    return done, time.perf_counter() - t0, dofs, st.tab.n_t


class OraclePool:
    """The oracle timed on the host cores of this box: os.cpu_count() processes (spawned: the parent may hold a CUDA
    context), each cycling over its share of a bounded window of the workload's subdomains."""

    def __init__(self, inp, window=16):
        import multiprocessing as mp
        from concurrent.futures import ProcessPoolExecutor
        self.cores = max(1, os.cpu_count() or 1)
        self.win = _oracle_window(inp, window)
        self.n_sub_window = self.win["sx"] * self.win["sy"]
        self.n_sub_total = inp.sx * inp.sy
        self.ex = ProcessPoolExecutor(max_workers=self.cores, mp_context=mp.get_context("spawn"))

    def run(self, seconds):
        """-> (DOF-steps/s over all cores, wall seconds, subdomain cycles done, DOF per subdomain, N_t)"""
        t0 = time.perf_counter()
        res = list(self.ex.map(_oracle_worker, [(self.win, r, self.cores, seconds) for r in range(self.cores)]))
        wall = time.perf_counter() - t0
        cycles = sum(r[0] for r in res)
        busy = max(r[1] for r in res)
        dofs, n_t = res[0][2], res[0][3]
        return cycles * dofs * N_WH * (n_t - 1) / busy, wall, cycles, dofs, n_t

    def describe(self, cycles, dofs, n_t):
        return (f"{cycles} subdomain DDM cycles (oracle/hz_oracle.py::ddm_cycle, numpy/scipy, {dofs} DOF each, n_wh={N_WH}, "
                f"N_t={n_t}) round-robin over the lower-left {self.win['sx']}x{self.win['sy']} of the workload's "
                f"{self.n_sub_total} subdomains, one process per host core")

    def close(self):
        self.ex.shutdown()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    inp = workload_inputs(args)
    pool = OraclePool(inp)
    per_step = 1.0                                   # about 1 s of oracle work on every core per step
    for _ in range(min(args.warmup, 2)):
        pool.run(0.2)
    tot_u = tot_t = 0.0
    cycles = 0
    for _ in range(args.steps):
        rate, wall, cyc, dofs, n_t = pool.run(per_step)
        tot_u += rate * wall
        tot_t += wall
        cycles += cyc
    pool.close()
    val = tot_u / tot_t
    sample = pool.describe(cycles, dofs, n_t) + f"; {args.steps} steps of about {per_step:.0f} s"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(inp, "f64 oracle"), "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": pool.cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
# clocks sampled for the whole run; the statistics use the samples taken while a timed leg ran
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.rows, self.legs, self.proc = [], [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append((time.perf_counter(), ln.strip()))

    def leg(self, name, t0, t1):
        self.legs.append((name, t0, t1))

    def stats(self, only=None):
        """Median SM clock and throttle reasons over the samples that fall inside a timed leg (`only`: leg name)."""
        sm, mx, reasons, per_leg = [], None, set(), {}
        for ts, ln in list(self.rows):
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                clk, mxc = float(f[0]), float(f[1])
            except ValueError:
                continue
            mx = mxc
            for name, t0, t1 in self.legs:
                if t0 - 0.05 <= ts <= t1 + 0.05 and (only is None or name == only):
                    sm.append(clk)
                    per_leg[name] = per_leg.get(name, 0) + 1
                    for nm, v in zip(self.NAMES, f[3:7]):
                        if v.lower().startswith("active"):
                            reasons.add(nm)
                    break
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm), "samples_per_leg": per_leg, "samples_total": len(self.rows)}

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"], "samples": 0}
        time.sleep(0.12)
        out = self.stats()
        self.proc.terminate()
        return out


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


def peak_tflops(prec_name, sm_mhz=SM_MHZ):
    lanes = FP32_LANES if prec_name == "f32" else FP32_LANES // 2
    return SMS * lanes * 2 * sm_mhz * 1e6 / 1e12


def kernel_name(pinfo, quads=False):
    return pinfo.kernel.decode()


def fma_probe(kind, stream):
    """This GPU's own FMA ceiling from the bench-only micro-benchmark library (csrc/hz_probe.cu); None if absent."""
    import ctypes as C
    path = os.path.join(ROOT, "paper_2606_21695_b200", "libhz_probe.so")
    if not os.path.exists(path):
        return None
    lib = C.CDLL(path)
    lib.hz_probe_fma.argtypes = [C.c_int, C.POINTER(C.c_double), C.c_void_p]
    r = C.c_double()
    return r.value if lib.hz_probe_fma(kind, C.byref(r), C.c_void_p(stream)) == 0 else None


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


def time_sweeps(hz, ctx, steps, warmup, flush, stream):
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


def sweep_rate(hz, inp, prec_name, k, flush, stream, steps=4, warmup=2, **flags):
    """Sweep-kernel throughput of one (config, precision, variant): dict for `extras` and the tables."""
    prec = hz.HZ_F32 if prec_name == "f32" else hz.HZ_F64
    ctx, pinfo = hz.setup_from_inputs(inp, prec, k, **flags)
    try:
        hz.hz_ddm_solve(ctx, 1, n_wh=N_WH, reset_state=True, stream=stream)
        tot, swp, exc, _, units = time_sweeps(hz, ctx, steps, warmup, flush, stream)
        rate = units / (sum(swp) * 1e-3)
        quads = inp.vx is not None
        extra = {}
        if pinfo.dofs_per_thread == 1 and not quads:
            # the one-DOF-per-thread layout fetches every operand of the line stencils from shared memory: 2(2p+1) loads and
            # 1 store per DOF-step; its roofline is the shared-memory pipe (128 B per clock and SM), north_star: "or the
            # stated L1/shared-bandwidth roofline if that binds"
            words = 4 * inp.p + 3
            smem_peak = SMS * 128.0 * SM_MHZ * 1e6
            extra = {"shared_memory_words_per_dof_step": words,
                     "frac_of_shared_memory_roofline": rate * words * (4 if prec_name == "f32" else 8) / smem_peak}
        return {**extra, "dof_steps_per_s_sweep_kernel": rate, "sweep_ms": sum(swp) / steps, "exchange_ms": sum(exc) / steps,
                "frac_of_derived_peak": rate * flops_per_dof_step(inp.p, quads) / (peak_tflops(prec_name) * 1e12),
                "kernel": kernel_name(pinfo, quads), "dofs_per_thread": pinfo.dofs_per_thread,
                "cluster_size": pinfo.cluster_size, "subs_per_block": pinfo.subs_per_block,
                "threads_per_block": pinfo.threads_per_block, "blocks": pinfo.blocks, "dofs_per_sub": pinfo.dofs_per_sub,
                "n_t": pinfo.n_t, "smem_bytes": pinfo.smem_bytes}
    finally:
        hz.hz_destroy(ctx)


def run_b200(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2606_21695_b200 import hz

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    sampler = ClockSampler(local) if rank == 0 else None       # runs for the whole process; legs are marked below
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    prec = hz.HZ_F32 if args.prec == "f32" else hz.HZ_F64
    tdt = torch.float32 if prec == hz.HZ_F32 else torch.float64
    inp = workload_inputs(args)
    quads = inp.vx is not None
    ctx, pinfo = hz.setup_from_inputs(inp, prec, args.k)
    stream = torch.cuda.current_stream().cuda_stream
    flush = torch.zeros(64 * 1024 * 1024, dtype=torch.float32, device="cuda")   # 256 MB > 126 MB L2
    nn = inp.npx * inp.npy
    hz.hz_ddm_solve(ctx, 2, n_wh=N_WH, reset_state=True, stream=stream)          # leave a non-trivial state

    # ---- kernel-resident timing: inputs already in HBM ----
    barrier()
    t0 = time.perf_counter()
    tot, swp, exc, launches, units = time_sweeps(hz, ctx, args.steps, args.warmup, flush, stream)
    barrier()
    t1 = time.perf_counter()
    if sampler:
        sampler.leg("headline", t0, t1)
    value, max_ms = job_value(units, float(sum(tot)), world, "cuda")

    # ---- end to end through the C ABI with HOST buffers: a new source in, the field out, every step ----
    u_dev = torch.zeros(2 * nn, dtype=tdt, device="cuda")
    f_np = np.ascontiguousarray(inp.f_re)
    f_pins = [torch.from_numpy(f_np).pin_memory(), (0.5 * torch.from_numpy(f_np)).pin_memory()]
    u_pins = [torch.empty(2 * nn, dtype=tdt).pin_memory(), torch.empty(2 * nn, dtype=tdt).pin_memory()]
    for _ in range(2):                                                           # warm-up of the sequential leg
        hz.hz_set_source_ptr(ctx, f_pins[0].data_ptr())
        hz.hz_ddm_solve(ctx, 1, n_wh=N_WH, u_out_ptr=u_dev.data_ptr(), stream=stream)
        u_pins[0].copy_(u_dev)
    seq_steps = 4
    barrier()
    te = time.perf_counter()
    e_units = 0.0
    for i in range(seq_steps):
        hz.hz_set_source_ptr(ctx, f_pins[i & 1].data_ptr())                      # H2D of f + rebuild of beta*b on device
        s = hz.hz_ddm_solve(ctx, 1, n_wh=N_WH, u_out_ptr=u_dev.data_ptr(), stream=stream)
        u_pins[i & 1].copy_(u_dev)                                               # D2H of the gathered field
        e_units += s.dof_timesteps
    barrier()
    t_seq1 = time.perf_counter()
    seq_value, _ = job_value(e_units, (t_seq1 - te) * 1e3, world, "cuda")
    # the same through hz_ddm_solve_sources: one C-ABI call for the whole stream of sources, host to host, the copies
    # on private streams overlapping the sweeps (two alternating pinned inputs and outputs)
    fp = [f_pins[i & 1].data_ptr() for i in range(E2E_SOURCES)]
    up = [u_pins[i & 1].data_ptr() for i in range(E2E_SOURCES)]
    hz.hz_ddm_solve_sources(ctx, fp[:2], up[:2], n_outer=1, n_wh=N_WH, stream=stream)       # allocation, warm-up
    barrier()
    tp0 = time.perf_counter()
    si = hz.hz_ddm_solve_sources(ctx, fp, up, n_outer=1, n_wh=N_WH, stream=stream)
    barrier()
    tp1 = time.perf_counter()
    if sampler:
        sampler.leg("e2e", te, tp1)
    p_ms = (tp1 - tp0) * 1e3
    e_value, p_max_ms = job_value(si.dof_timesteps, p_ms, world, "cuda")
    h2d, d2h = int(nn * 8), int(2 * nn * u_pins[0].element_size())
    e2e = {"value": e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
           "steps": E2E_SOURCES, "ms_per_step": p_max_ms / E2E_SOURCES, "frac_of_resident_value": e_value / value,
           "h2d_gb_per_s_sustained": h2d * E2E_SOURCES / (p_max_ms * 1e-3) / 1e9,
           "d2h_gb_per_s_sustained": d2h * E2E_SOURCES / (p_max_ms * 1e-3) / 1e9,
           "what": "hz_ddm_solve_sources over a fixed number of sources: per step H2D of a new source f (fp64) from pinned "
                   "host memory, rebuild of the load, 1 sweep + exchange, gather, D2H of u to pinned host memory; "
                   "copies on private streams overlap the sweeps; wall clock around the one C-ABI call",
           "sequential_value": seq_value, "sequential_steps": seq_steps,
           "sequential_what": "hz_set_source(host f) + hz_ddm_solve(1 sweep, u_out) + D2H of u, one after the other"}
    u_elem = u_pins[0].element_size()
    del f_pins, u_pins, u_dev

    if rank != 0:
        hz.hz_destroy(ctx)
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the sweep), live numbers ----
    sweep_ms = float(sum(swp)) / args.steps
    units_per_launch = units / args.steps
    fl = flops_per_dof_step(inp.p, quads)
    peak_tf = peak_tflops(args.prec)
    achieved_tf = units_per_launch * fl / (sweep_ms * 1e-3) / 1e12
    ex_sub = inp.nx // inp.sx
    tkey = f"config{args.config}_p{inp.p}_s{ex_sub}_{args.prec}" + ("_quads" if quads else "")
    stored = STORED_TRAFFIC.get(tkey)
    try:
        probe_tf = fma_probe(0 if prec == hz.HZ_F32 else 1, stream)
    except Exception:
        probe_tf = None
    op_ms = None
    try:   # the paper's normaliser: one evaluation of the global Helmholtz operator on a random vector,
           # in the arithmetic of the cycle
        v = torch.randn(2 * nn, dtype=tdt, device="cuda")
        op_ms = hz.hz_operator_time(ctx, v.data_ptr(), prec, 10, stream)
        del v
    except Exception:
        pass
    roofline = {"bound": "alu", "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved_tf / peak_tf,
                "traffic": stored["bytes"] if stored else None,
                "traffic_source": (f"STORED ncu figure ({stored['from']}, captured {stored['captured']}), not measured in "
                                   "this run") if stored else "no ncu capture of this workload is stored",
                "kernel": kernel_name(pinfo, quads),
                "peak_source": f"derived: {SMS} SMs x {FP32_LANES if prec == hz.HZ_F32 else FP32_LANES // 2} FMA lanes x 2 x "
                               f"{SM_MHZ:.0f} MHz (guide unit counts, max SM clock); MEASURED_PEAKS.json has no "
                               "CUDA-core entry",
                "peak_measured_fma_probe": probe_tf, "frac_of_probe": (achieved_tf / probe_tf) if probe_tf else None,
                "flops_per_dof_step": fl, "dof_steps_per_launch": units_per_launch, "sweep_kernel_ms": sweep_ms,
                "exchange_kernel_ms": float(sum(exc)) / args.steps,
                "operator_ms": op_ms, "operator_gb_per_s": (nn * 5 * u_elem / (op_ms * 1e-3) / 1e9) if op_ms else None,
                "operator_what": "one evaluation y = (A - i w H - w^2 M) x of the global operator in the cycle's own "
                                 "precision; bytes = x (2 words) + w^2/c^2 (1) + y (2) per node",
                "ddm_cycle_over_operator": (sweep_ms / op_ms) if op_ms else None}
    hz.hz_destroy(ctx)

    extras = {}
    if not args.no_extras and world == 1:
        extras = run_extras(hz, torch, args, flush, stream, sampler)
    del flush
    torch.cuda.empty_cache()

    # ---- the oracle on ALL host cores of this box, bounded sample of the same workload ----
    try:
        pool = OraclePool(inp)
        pool.run(0.2)                                                           # process start-up, imports, set-up
        rate, wall, cycles, dofs, n_t = pool.run(12.0 if not args.no_extras else 3.0)
        pool.close()
        cpu = {"value": rate, "unit": UNIT, "cores": pool.cores, "kind": "oracle", "seconds": wall,
               "sample": pool.describe(cycles, dofs, n_t)}
    except Exception as e:
        cpu = {"value": None, "unit": UNIT, "cores": 0, "kind": "oracle", "error": str(e)}

    clocks = sampler.stop() if sampler else None
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": args.prec, "data": "synthetic",
            "config": {"workload": workload_name(inp, args.prec), "n_t": pinfo.n_t, "dofs_per_sub": pinfo.dofs_per_sub,
                       "dofs_total": pinfo.dofs_per_sub * pinfo.blocks,
                       "blocks": pinfo.blocks, "threads_per_block": pinfo.threads_per_block,
                       "dofs_per_thread": pinfo.dofs_per_thread, "subs_per_block": pinfo.subs_per_block,
                       "cluster_size": pinfo.cluster_size, "smem_bytes": pinfo.smem_bytes,
                       "l2": "flushed between timed steps (256 MB write); the per-sweep working set also exceeds L2",
                       "parallelism": "replicas only (one independent problem per GPU)" if world > 1 else "1 GPU"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
            "extras": extras}
    print(json.dumps(_finite(line), allow_nan=False), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------------
# secondary measurements (N = 1 only): the other configs, time to solution, the comparator, F3 / F4
# ---------------------------------------------------------------------------------------------------
def time_to_solution(hz, inp, prec_name, tol, every, nmax, stream, driver="fixed_point", restart=50, n_wh=2):
    """DDM time-to-solution (BASELINE.json metric 1): global relative residual (hz_residual, fp64) to `tol`,
    n_wh = 2, rho = 0.5, warm start.  fixed_point: hz_ddm_solve with CUDA-graph replay between residual checks;
    mixed: hz_ddm_solve_mixed (fp32 sweeps on the correction, fp64 state); gmres: hz_ddm_solve_gmres on the joint state;
    gmres_lambda: hz_ddm_solve_gmres on lambda alone (cold-started sweeps of n_wh WaveHoltz iterations, rho = 1,
    basis of `restart` interface-sized vectors: no restart in practice)."""
    out = {"tol": tol, "n_wh": n_wh, "relax": 0.5, "driver": driver}
    if driver == "mixed":
        lo, _ = hz.setup_from_inputs(inp, hz.HZ_F32, 0)
        hi, _ = hz.setup_from_inputs(inp, hz.HZ_F64, 0)
        try:
            m = every
            hz.hz_ddm_solve_mixed(lo, hi, 1, m, n_wh=n_wh, reset_state=True, stream=stream)           # allocation, warm-up
            t0 = time.perf_counter()
            s = hz.hz_ddm_solve_mixed(lo, hi, max(1, nmax // m), m, n_wh=n_wh, relax=0.5, tol=tol, check_every=2,
                                      reset_state=True, stream=stream)
            out.update(sweeps=s.sweeps_lo + s.sweeps_hi, sweeps_fp32=s.sweeps_lo, sweeps_fp64=s.sweeps_hi,
                       rel_residual=s.rel_residual, device_ms=s.total_ms, wall_ms=(time.perf_counter() - t0) * 1e3,
                       m_inner=m, reached=bool(0 <= s.rel_residual <= tol))
        finally:
            hz.hz_destroy(lo)
            hz.hz_destroy(hi)
        return out
    ctx, pinfo = hz.setup_from_inputs(inp, hz.HZ_F32 if prec_name == "f32" else hz.HZ_F64, 0)
    try:
        if driver == "gmres_lambda":
            hz.hz_ddm_solve_gmres(ctx, 3, n_wh=n_wh, relax=1.0, restart=restart, lambda_only=True, stream=stream)   # allocation, warm-up
            t0 = time.perf_counter()
            s = hz.hz_ddm_solve_gmres(ctx, nmax, n_wh=n_wh, relax=1.0, restart=restart, lin_tol=0.02 * tol, reset_state=True,
                                      lambda_only=True, stream=stream)
            out.update(relax=1.0, sweeps=s.sweeps_done, waveholtz_iterations=s.sweeps_done * n_wh, cycles=s.cycles,
                       lin_residual=s.lin_residual, rel_residual=s.rel_residual, device_ms=s.total_ms,
                       wall_ms=(time.perf_counter() - t0) * 1e3, restart=restart, krylov_mb=s.krylov_bytes / 1e6,
                       reached=bool(s.rel_residual <= tol))
        elif driver == "gmres":
            hz.hz_ddm_solve_gmres(ctx, 3, n_wh=n_wh, restart=restart, stream=stream)                  # allocation, warm-up
            t0 = time.perf_counter()
            s = hz.hz_ddm_solve_gmres(ctx, nmax, n_wh=n_wh, relax=0.5, restart=restart, tol=tol, reset_state=True, stream=stream)
            out.update(sweeps=s.sweeps_done, cycles=s.cycles, rel_residual=s.rel_residual, device_ms=s.total_ms,
                       wall_ms=(time.perf_counter() - t0) * 1e3, restart=restart, reached=bool(s.rel_residual <= tol))
        else:
            hz.hz_ddm_solve(ctx, every, n_wh=n_wh, reset_state=True, use_graph=True, stream=stream)   # graph capture, warm-up
            t0 = time.perf_counter()
            s = hz.hz_ddm_solve(ctx, nmax, n_wh=n_wh, warm_start=True, relax=0.5, tol=tol, check_every=every,
                                reset_state=True, use_graph=True, stream=stream)
            out.update(sweeps=s.n_outer_done, rel_residual=s.rel_residual, device_ms=s.total_ms,
                       wall_ms=(time.perf_counter() - t0) * 1e3, cuda_graph=True, reached=bool(s.rel_residual <= tol),
                       diverged=bool(not (s.rel_residual == s.rel_residual) or s.rel_residual > 1e3))
    finally:
        hz.hz_destroy(ctx)
    return out


def paper_style_cycle(hz, torch, stream, flush, n=512, p=3, s=8, prec_name="f32"):
    """The paper's micro-benchmark: ONE DDM cycle of 5 WaveHoltz iterations applied to a random
    interface vector on a constant-coefficient square, in units of one evaluation of the global Helmholtz operator."""
    import numpy as np
    from paper_2606_21695_b200.inputs import make_config, random_lambda
    inp = make_config(1, n=n, p=p, sub_elems=s)           # config 1's medium: c = 1 everywhere
    inp.omega = 2.0 * np.pi * p * n / 10.0                # ~10 points per wavelength
    prec = hz.HZ_F32 if prec_name == "f32" else hz.HZ_F64
    ctx, info = hz.setup_from_inputs(inp, prec, 0)
    try:
        lam_c = random_lambda(np.random.default_rng(42), info.blocks, info.edge_stride)
        lam0 = torch.from_numpy(np.stack([lam_c.real, lam_c.imag], axis=2).copy()).cuda()
        ms = []
        for _ in range(5):
            hz.hz_ddm_solve(ctx, 0, reset_state=True, stream=stream)
            hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr(), stream=stream)
            flush.add_(1.0)
            ms.append(hz.hz_ddm_solve(ctx, 1, n_wh=N_WH, warm_start=False, stream=stream).sweep_ms_total)
        v = torch.randn(2 * inp.npx * inp.npy, dtype=torch.float32 if prec_name == "f32" else torch.float64, device="cuda")
        op = hz.hz_operator_time(ctx, v.data_ptr(), prec, 20, stream)
        cyc = min(ms[1:])
        return {"mesh": f"{n}x{n}, p={p}, c=1, {info.blocks} subdomains of {s}x{s} elements, {prec_name}", "n_t": info.n_t,
                "ddm_cycle_ms": cyc, "operator_ms": op, "cycle_over_operator": cyc / op,
                "mdof_per_s_per_cycle": info.blocks * info.dofs_per_sub / (cyc * 1e-3) / 1e6}
    finally:
        hz.hz_destroy(ctx)


def minres_vs_waveholtz(hz, torch, inp, prec_name, stream, max_nwh=4096):
    """WaveHoltz vs MINRES as block-level subdomain solvers (Table I) on the subdomains of `inp`
    with a seeded random interface vector: MINRES from x = 0 to the paper's tolerance (1e-6 fp32 / 1e-12 fp64) and
    the TRUE residual it reaches; WaveHoltz from u = 0 with the smallest n_wh whose true subdomain residual (same
    evaluation kernel) is at most that, in the same one-DOF-per-thread layout and in the register-blocked layout."""
    import numpy as np
    from paper_2606_21695_b200.inputs import random_lambda
    prec, tol = (hz.HZ_F32, 1e-6) if prec_name == "f32" else (hz.HZ_F64, 1e-12)
    ctx, info = hz.setup_from_inputs(inp, prec, 1)
    lam_c = random_lambda(np.random.default_rng(42), info.blocks, info.edge_stride)
    lam0 = torch.from_numpy(np.stack([lam_c.real, lam_c.imag], axis=2).copy()).cuda()   # [L][4][2][E]

    def true_res(n_wh):
        hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr(), stream=stream)
        hz.hz_ddm_solve(ctx, 1, n_wh=n_wh, warm_start=False, stream=stream)
        hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr(), stream=stream)
        return float(hz.hz_minres_cycle(ctx, info.blocks, 0.0, 0, warm_start=True, stream=stream)[2].max())

    def timed(c, n_wh):
        best = 1e30
        for _ in range(3):
            hz.hz_set_subdomain_state(c, None, lam0.data_ptr(), stream=stream)
            best = min(best, hz.hz_ddm_solve(c, 1, n_wh=n_wh, warm_start=False, stream=stream).sweep_ms_total)
        return best

    try:
        hz.hz_ddm_solve(ctx, 0, reset_state=True, stream=stream)
        hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr(), stream=stream)
        hz.hz_minres_cycle(ctx, info.blocks, tol, 100000, stream=stream)                    # warm-up
        mi, iters, res = hz.hz_minres_cycle(ctx, info.blocks, tol, 100000, stream=stream)
        target = max(tol, float(res.max()))
        lo, hi = 0, 1
        while hi <= max_nwh and true_res(hi) > target:
            lo, hi = hi, hi * 2
        while hi - lo > 1:                       # bisection on n_wh
            mid = (lo + hi) // 2
            if true_res(mid) <= target:
                hi = mid
            else:
                lo = mid
        t1 = timed(ctx, hi)
    finally:
        hz.hz_destroy(ctx)
    ctx2, info2 = hz.setup_from_inputs(inp, prec, 0)
    mk = None
    try:
        hz.hz_ddm_solve(ctx2, 0, reset_state=True, stream=stream)
        tk = timed(ctx2, hi)
        try:   # MINRES in the same register-blocked layout (k_minres_tile), where the tile is one it is compiled for
            hz.hz_ddm_solve(ctx2, 0, reset_state=True, stream=stream)
            hz.hz_set_subdomain_state(ctx2, None, lam0.data_ptr(), stream=stream)
            hz.hz_minres_cycle(ctx2, info2.blocks, tol, 100000, stream=stream)
            mk, _, resk = hz.hz_minres_cycle(ctx2, info2.blocks, tol, 100000, stream=stream)
        except hz.HzError:
            mk = None
    finally:
        hz.hz_destroy(ctx2)
    extra = {} if mk is None else {"minres_ms_register_blocked": mk.kernel_ms, "minres_iters_mean_register_blocked": mk.iters_mean,
                                   "minres_true_residual_register_blocked": float(resk.max()),
                                   "speedup_same_layout_register_blocked": mk.kernel_ms / tk}
    return {**extra, "p": inp.p, "sub_side": inp.nx // inp.sx, "dofs_per_sub": info.dofs_per_sub, "blocks": info.blocks,
            "prec": prec_name, "minres_iters_mean": mi.iters_mean, "minres_iters_max": mi.iters_max,
            "minres_true_residual": float(res.max()), "minres_ms": mi.kernel_ms, "n_wh": hi,
            "waveholtz_ms_one_dof_per_thread": t1, "waveholtz_ms_register_blocked": tk,
            "register_blocked_kernel": kernel_name(info2), "speedup_same_layout": mi.kernel_ms / t1,
            "speedup_best": mi.kernel_ms / tk}


def run_extras(hz, torch, args, flush, stream, sampler):
    from paper_2606_21695_b200.inputs import make_config
    out = {}

    def leg(key, fn):
        t0 = time.perf_counter()
        try:
            out[key] = fn()
        except Exception as e:  # an extra must never take the headline line down
            out[key] = {"error": f"{type(e).__name__}: {e}"}
        if sampler:
            sampler.leg(key, t0, time.perf_counter())

    # sweep-kernel throughput: the other precision of the headline, configs 2-4, the corners of the config-5 sweep
    # (auto variant) and the one-DOF-per-thread variant where it fits ("both threading variants")
    inputs = {}

    def get(cfg, p=None, s=None):
        key = (cfg, p, s)
        if key not in inputs:
            inputs.clear()                         # one full-size mesh in host memory at a time
            inputs[key] = make_config(cfg, n=(6144 // p if cfg == 5 and p else None), p=p, sub_elems=s)
        return inputs[key]

    cases = [(5, 3, 8, "f64", 0), (5, 3, 8, "f32", 1), (3, None, None, "f32", 0), (3, None, None, "f64", 0),
             (4, None, None, "f32", 0), (4, None, None, "f64", 0), (2, None, None, "f32", 0), (2, None, None, "f64", 0),
             (5, 1, 4, "f32", 0), (5, 1, 4, "f64", 0), (5, 1, 4, "f32", 1), (5, 1, 8, "f32", 0), (5, 2, 4, "f32", 0),
             (5, 3, 4, "f32", 0), (5, 3, 4, "f64", 0), (5, 3, 64, "f32", 0), (5, 3, 64, "f64", 0),
             (5, 4, 8, "f32", 0), (5, 4, 8, "f64", 0), (5, 4, 64, "f32", 0)]
    for cfg, p, s, pr, k in cases:
        name = f"config{cfg}" + (f"_p{p}_s{s}" if p else "") + f"_{pr}" + ("_one_dof_per_thread" if k == 1 else "")
        leg(name, lambda: sweep_rate(hz, get(cfg, p, s), pr, k, flush, stream, steps=3, warmup=1))
    inputs.clear()

    # DDM time-to-solution (BASELINE.json metric 1)
    tts = [(1, "f64", 1e-8, 10, 2000, "fixed_point"), (1, "f64", 1e-8, 10, 2000, "mixed"),
           (2, "f32", 1e-4, 50, 5000, "fixed_point"), (2, "f64", 1e-4, 50, 5000, "fixed_point"),
           (2, "f32", 1e-4, 50, 3000, "gmres"), (2, "f64", 1e-4, 50, 3000, "gmres"),
           (3, "f64", 1e-4, 50, 8000, "fixed_point"), (3, "f32", 1e-4, 25, 8000, "mixed"),
           (4, "f32", 1e-4, 50, 3000, "fixed_point"), (4, "f64", 1e-4, 50, 3000, "fixed_point")]
    for cfg, pr, tol, every, nmax, drv in tts:
        key = f"config{cfg}_{'f32_sweeps_f64_state' if drv == 'mixed' else pr}_time_to_solution" + ("" if drv != "gmres" else "_gmres")
        leg(key, lambda: time_to_solution(hz, get(cfg), pr, tol, every, nmax, stream, drv))
    # one WaveHoltz iteration per sweep (warm start): more sweeps, each half as long (n_wh in {1, 2})
    # (config 3 diverges with n_wh = 1: one WaveHoltz iteration per sweep is too loose an inner solve there; the entry
    # is kept, with a small sweep budget, so that the line shows it)
    for cfg, pr, every, nmax, drv in ((3, "f64", 50, 1000, "fixed_point"), (4, "f32", 50, 6000, "fixed_point"),
                                      (4, "f64", 50, 6000, "fixed_point")):
        key = f"config{cfg}_{'f32_sweeps_f64_state' if drv == 'mixed' else pr}_time_to_solution_n_wh_1"
        leg(key, lambda: time_to_solution(hz, get(cfg), pr, 1e-4, every, nmax, stream, drv, n_wh=1))
    # Krylov iteration on lambda alone (cold-started sweeps, interface-sized basis, no restart): config 2 to
    # the shared tolerance with 20 WaveHoltz iterations per sweep; config 3 with a bounded step count (it does not get there)
    leg("config2_f64_time_to_solution_gmres_lambda_only",
        lambda: time_to_solution(hz, get(2), "f64", 1e-4, 0, 400, stream, "gmres_lambda", restart=400, n_wh=20))
    leg("config3_f64_gmres_lambda_only_300_steps",
        lambda: time_to_solution(hz, get(3), "f64", 1e-4, 0, 300, stream, "gmres_lambda", restart=300, n_wh=16))
    inputs.clear()

    leg("paper_style_cycle_512_p3_f32", lambda: paper_style_cycle(hz, torch, stream, flush))
    # the paper's comparator on the config-5 mesh (Table I's B = 256, T = 1 corner and the 625-DOF subdomains)
    for s in (4, 8):
        for pr in ("f32", "f64"):
            leg(f"minres_vs_waveholtz_config5_p3_s{s}_{pr}",
                lambda: minres_vs_waveholtz(hz, torch, get(5, 3, s), pr, stream))
    inputs.clear()

    # the rows SURVEY.md 8(f) marks "next": general convex quads (F3) and 3-D hexahedra (F4), sweep kernel only
    leg("config3_general_quads_f32", lambda: sweep_rate(hz, make_config(3, distort=0.2), "f32", 0, flush, stream, 3, 1))

    def quad_prologue():
        """Share of the general-quad sweep that is NOT the time loop (staging of the per-element geometric factors and
        coefficients into shared memory with plain loads, b assembly, epilogue): sweep time is linear in n_wh; the
        intercept of the fit through n_wh = 1 and 5 is the prologue + epilogue (north_star (b): TMA / cp.async staging
        would only attack this share)."""
        ctx, pinfo = hz.setup_from_inputs(make_config(3, distort=0.2), hz.HZ_F32, 0)
        try:
            hz.hz_ddm_solve(ctx, 1, n_wh=N_WH, reset_state=True, stream=stream)
            t = {}
            for nwh in (1, 5):
                hz.hz_ddm_solve(ctx, 1, n_wh=nwh, stream=stream)
                t[nwh] = min(hz.hz_ddm_solve(ctx, 1, n_wh=nwh, stream=stream).sweep_ms_total for _ in range(3))
            per_it = (t[5] - t[1]) / 4.0
            fixed = t[1] - per_it
            return {"sweep_ms_n_wh_1": t[1], "sweep_ms_n_wh_5": t[5], "ms_per_waveholtz_iteration": per_it,
                    "prologue_plus_epilogue_ms": fixed, "share_of_a_5_iteration_sweep": fixed / t[5]}
        finally:
            hz.hz_destroy(ctx)
    leg("general_quads_prologue_share_f32", quad_prologue)

    def hexes():
        from paper_2606_21695_b200 import hz3
        from paper_2606_21695_b200.inputs import make_config_3d
        r3 = {}
        for name, n, p, s in (("hex_128cubed_p1_sub8", 128, 1, 8), ("hex_48cubed_p3_sub3", 48, 3, 3)):
            i3 = make_config_3d(n, p, s)
            c3 = hz3.hz3_mesh_setup(i3.nx, i3.ny, i3.nz, i3.box, i3.p, i3.c_nodes, i3.omega, i3.f_re)
            try:
                info3 = hz3.hz3_partition(c3, i3.sx, i3.sy, i3.sz, hz.HZ_F32)
                hz3.hz3_ddm_solve(c3, 1, n_wh=N_WH, reset_state=True, stream=stream)
                r = hz3.hz3_ddm_solve(c3, 3, n_wh=N_WH, stream=stream)
                rate = r.dof_timesteps / (r.sweep_ms_total * 1e-3)
                r3[name + "_f32"] = {"dof_steps_per_s_sweep_kernel": rate, "sweep_ms": r.sweep_ms_total / 3, "n_t": info3.n_t,
                                     "nodes_per_thread": info3.nodes_per_thread, "blocks": info3.blocks,
                                     "frac_of_derived_peak": rate * 2 * (3 * (p + 2) + 5) / (peak_tflops("f32") * 1e12),
                                     # the column kernel reads the x and y stencil operands from shared memory: 2(2p+1) loads
                                     # + 1 store per DOF-step against 128 B per clock and SM (its binding roofline)
                                     "frac_of_shared_memory_roofline": rate * (4 * p + 3) * 4 / (SMS * 128.0 * SM_MHZ * 1e6)}
            finally:
                hz3.hz3_destroy(c3)
        return r3
    leg("hex_3d", hexes)
    return out


# ---------------------------------------------------------------------------------------------------
# markdown tables (profiles/*.md name the `python bench.py --sweep ...` command that printed them)
# ---------------------------------------------------------------------------------------------------
def run_tables(args):
    import numpy as np
    import torch
    from paper_2606_21695_b200 import hz
    from paper_2606_21695_b200.inputs import make_config
    stream = torch.cuda.current_stream().cuda_stream
    flush = torch.zeros(64 * 1024 * 1024, dtype=torch.float32, device="cuda")
    which = args.sweep

    def rate_row(cfg, pr, k, n=None, p=None, s=None, distort=0.0, reps=3):
        inp = make_config(cfg, n=n, p=p, sub_elems=s, distort=distort)
        head = f"| {cfg} | {inp.nx} | {inp.p} | {inp.nx // inp.sx} | {pr} |"
        try:
            r = sweep_rate(hz, inp, pr, k, flush, stream, steps=reps, warmup=1)
        except hz.HzError as e:
            print(f"{head} {k or 'auto'} | — | — | — | — | — | — | — | — | — | {str(e).split(':', 1)[0]} |", flush=True)
            return
        if inp.vx is not None:
            ctx = hz.hz_mesh_setup_quads(inp.nx, inp.ny, inp.p, inp.vx, inp.vy, inp.c_nodes, inp.omega, inp.f_re)
            opp = hz.HZ_F64                       # general quads: the fp64 residual kernel is the operator kernel
        else:
            ctx = hz.hz_mesh_setup(inp.nx, inp.ny, inp.x0, inp.y0, inp.x1, inp.y1, inp.p, inp.c_nodes, inp.omega, inp.f_re)
            opp = hz.HZ_F32 if pr == "f32" else hz.HZ_F64
        v = torch.randn(2 * inp.npx * inp.npy, dtype=torch.float32 if opp == hz.HZ_F32 else torch.float64, device="cuda")
        op_ms = hz.hz_operator_time(ctx, v.data_ptr(), opp, 20, stream)
        hz.hz_destroy(ctx)
        print(f"{head} {r['kernel']} | {r['dofs_per_thread']} | {r['cluster_size']} | {r['subs_per_block']} | {r['dofs_per_sub']} | "
              f"{r['blocks']} | {r['threads_per_block']} | {r['smem_bytes']} | {r['sweep_ms']:.3f} | "
              f"{r['dof_steps_per_s_sweep_kernel']:.3e} | {r['frac_of_derived_peak']:.3f} | {op_ms:.4f} | "
              f"{r['sweep_ms'] / op_ms:.1f} |", flush=True)

    if which in ("cfg2", "cfg3", "cfg4", "cfg5", "quads"):
        print("| cfg | n | p | sub side | prec | kernel | DOF/thread | CTAs/sub | subs/block | DOF/sub | blocks | threads | smem B | "
              "sweep ms | DOF-steps/s | frac of FMA peak | operator ms (same precision) | DDM cycle / operator |")
        print("|" + "---|" * 18)
    if which in ("cfg2", "cfg3"):
        for pr in ("f32", "f64"):
            for k in (1, 0):
                rate_row(int(which[3]), pr, k)
    elif which == "cfg4":
        for pr in ("f32", "f64"):
            for k in (0, 18, 36):
                rate_row(4, pr, k, reps=2)
    elif which == "cfg5":
        for p in (1, 2, 3, 4):
            for s in (4, 8, 16, 32, 64):
                for pr in ("f32", "f64"):
                    n = 6144 // p // args.scale // s * s
                    rate_row(5, pr, 0, n=n, p=p, s=s, reps=2)
                    if (s * p + 1) ** 2 <= 1024:
                        rate_row(5, pr, 1, n=n, p=p, s=s, reps=2)       # the one-DOF-per-thread variant
    elif which == "quads":
        sc = max(args.scale, 4)
        for pr in ("f32", "f64"):
            rate_row(2, pr, 0, distort=0.2)
            rate_row(3, pr, 0, distort=0.2)
        for p in (1, 2, 3, 4):
            for s in (4, 8, 16):
                for pr in ("f32", "f64"):
                    rate_row(5, pr, 0, n=(6144 // p) // sc // s * s, p=p, s=s, reps=2, distort=0.2)
    elif which == "tts":
        print("| cfg | arithmetic | tol | driver | n_wh | sweeps | residual reached | device ms | note |")
        print("|---|---|---|---|---|---|---|---|---|")
        for cfg in (1, 2, 3, 4):
            inp = make_config(cfg)
            every = 10 if cfg == 1 else 50
            tol_hi = 1e-8 if cfg == 1 else 1e-4
            rows = [("f64", tol_hi, "fixed_point", 2), ("f32", 1e-4, "fixed_point", 2), ("f32", tol_hi, "mixed", 2),
                    ("f64", tol_hi, "fixed_point", 1), ("f32", tol_hi, "mixed", 1),
                    ("f64", tol_hi, "gmres", 2), ("f32", 1e-4, "gmres", 2),
                    ("f64", tol_hi, "gmres_lambda", {1: 40, 2: 20, 3: 16, 4: 16}[cfg])]
            for pr, tol, drv, nwh in rows:
                if drv == "gmres_lambda":
                    r = time_to_solution(hz, inp, pr, tol, 0, 1000 if cfg <= 3 else 400, stream, drv, restart=1000 if cfg <= 3 else 400, n_wh=nwh)
                else:
                    r = time_to_solution(hz, inp, pr, tol, 25 if drv == "mixed" else every, 40000 if drv != "gmres" else 4000,
                                         stream, drv, restart=50 if cfg <= 2 else 100, n_wh=nwh)
                arith = "fp32 sweeps, fp64 state" if drv == "mixed" else pr
                note = "" if r["reached"] else "NOT reached"
                if drv == "mixed":
                    note += f" {r['sweeps_fp32']} fp32 + {r['sweeps_fp64']} fp64 sweeps"
                print(f"| {cfg} | {arith} | {tol:g} | {drv} | {nwh} | {r['sweeps']} | {r['rel_residual']:.2e} | {r['device_ms']:.1f} | {note} |",
                      flush=True)
    elif which == "minres":
        print("| mesh | p | sub side | DOF/sub | blocks | prec | MINRES iters (mean / max) | MINRES true res | MINRES ms, 1 DOF/thread | "
              "MINRES ms, register-blocked | n_wh | WaveHoltz ms, 1 DOF/thread | WaveHoltz ms, register-blocked | "
              "speedup, both 1 DOF/thread | speedup, both register-blocked | speedup best vs best |")
        print("|" + "---|" * 16)
        for cfg, n, sides in ((5, 2048 // args.scale, (4, 8)), (3, 256, (4, 8, 10))):
            for s in sides:
                inp = make_config(cfg, n=n - n % s, p=3, sub_elems=s)
                for pr in ("f32", "f64"):
                    r = minres_vs_waveholtz(hz, torch, inp, pr, stream)
                    mrb = r.get("minres_ms_register_blocked")
                    best_m = min(r["minres_ms"], mrb) if mrb else r["minres_ms"]
                    best_w = min(r["waveholtz_ms_one_dof_per_thread"], r["waveholtz_ms_register_blocked"])
                    print(f"| {inp.nx}x{inp.ny} | 3 | {s} | {r['dofs_per_sub']} | {r['blocks']} | {pr} | {r['minres_iters_mean']:.0f} / "
                          f"{r['minres_iters_max']} | {r['minres_true_residual']:.1e} | {r['minres_ms']:.2f} | "
                          f"{'%.2f' % mrb if mrb else 'n/a'} | {r['n_wh']} | "
                          f"{r['waveholtz_ms_one_dof_per_thread']:.2f} | {r['waveholtz_ms_register_blocked']:.2f} "
                          f"({r['register_blocked_kernel']}) | {r['speedup_same_layout']:.1f}x | "
                          f"{'%.1fx' % r['speedup_same_layout_register_blocked'] if mrb else 'n/a'} | {best_m / best_w:.1f}x |", flush=True)
    elif which == "3d":
        from paper_2606_21695_b200 import hz3
        from paper_2606_21695_b200.inputs import make_config_3d
        print("| mesh | p | sub side | prec | nodes/thread | DOF/sub | blocks | threads | n_t | sweep ms | DOF-steps/s | frac of FMA peak | "
              "operator ms (fp64) | DDM cycle / operator |")
        print("|" + "---|" * 14)
        for n, p, s in ((128, 1, 8), (64, 1, 8), (64, 2, 4), (48, 3, 3), (48, 3, 2), (32, 4, 2)):
            for pr in ("f32", "f64"):
                for npt in (0, 1):
                    i3 = make_config_3d(n, p, s)
                    c3 = hz3.hz3_mesh_setup(i3.nx, i3.ny, i3.nz, i3.box, i3.p, i3.c_nodes, i3.omega, i3.f_re)
                    try:
                        info3 = hz3.hz3_partition(c3, i3.sx, i3.sy, i3.sz, hz.HZ_F32 if pr == "f32" else hz.HZ_F64, 0.5, npt)
                        if npt == 1 and info3.nodes_per_thread != 1:
                            continue
                        hz3.hz3_ddm_solve(c3, 1, n_wh=N_WH, reset_state=True, stream=stream)
                        r = hz3.hz3_ddm_solve(c3, 3, n_wh=N_WH, stream=stream)
                        rate = r.dof_timesteps / (r.sweep_ms_total * 1e-3)
                        v = torch.randn(2 * int(np.prod(i3.shape)), dtype=torch.float64, device="cuda")
                        op = hz3.hz3_operator_time(c3, v.data_ptr(), 10, stream)
                        print(f"| {n}^3 | {p} | {s} | {pr} | {info3.nodes_per_thread} | {info3.dofs_per_sub} | {info3.blocks} | "
                              f"{info3.threads_per_block} | {info3.n_t} | {r.sweep_ms_total / 3:.3f} | {rate:.3e} | "
                              f"{rate * 2 * (3 * (p + 2) + 5) / (peak_tflops(pr) * 1e12):.3f} | {op:.4f} | "
                              f"{r.sweep_ms_total / 3 / op:.1f} |", flush=True)
                    finally:
                        hz3.hz3_destroy(c3)


def _finite(o):
    """JSON has no NaN / Infinity: a diverged or missing number is reported as null."""
    if isinstance(o, float):
        return o if o == o and abs(o) != float("inf") else None
    if isinstance(o, dict):
        return {k: _finite(v) for k, v in o.items()}
    if isinstance(o, (list, tuple)):
        return [_finite(v) for v in o]
    return o


def main():
    args = parse_args()
    if args.sweep:
        run_tables(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
