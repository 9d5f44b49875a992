"""Sweep-kernel throughput over BASELINE.json's configs (the config-4 k sweep and the config-5
subdomain-size x degree sweep), printed as a markdown table.

    python -m paper_2606_21695_b200.sweep cfg4            # 1024^2 quads, 32x32-element subdomains, k in {auto, 18, 36}
    python -m paper_2606_21695_b200.sweep cfg5 [--scale 4]  # p in 1..4, subdomain side in {4,8,16,32,64}

`--scale S` shrinks the config-5 mesh side by S (same subdomain shapes, S^2 fewer blocks); S = 1 is the full
38 M-DOF mesh.  Rates are DOF-timestep updates per second of the sweep kernel (CUDA events inside
hz_ddm_solve), n_wh = 5, warm start; "frac" = rate x 2(2(p+2)+5) flops / (148 SMs x 128 (64) lanes x 2 x
1.965 GHz).  Entries that fit no compiled kernel (state larger than one SM's registers + shared memory)
are reported as such, not hidden.
"""
from __future__ import annotations

import argparse

import numpy as np
import torch

from . import hz
from .inputs import make_config

SMS, CLK = 148, 1.965e9


def run(cfg, prec, k, n=None, p=None, s=None, nwh=5, reps=3, distort=0.0):
    inp = make_config(cfg, n=n, p=p, sub_elems=s, distort=distort)
    name = f"| {cfg} | {inp.nx} | {inp.p} | {inp.nx // inp.sx} | {'f32' if prec == hz.HZ_F32 else 'f64'} |"
    try:
        ctx, info = hz.setup_from_inputs(inp, prec, k)
    except hz.HzError as e:
        print(f"{name} {k or 'auto'} | — | — | — | — | — | — | — | — | — | {e.args[0].split(':', 1)[0]} |", flush=True)
        return
    try:
        hz.hz_ddm_solve(ctx, 1, n_wh=nwh, reset_state=True)
        r = hz.hz_ddm_solve(ctx, reps, n_wh=nwh)
        rate = r.dof_timesteps / (r.sweep_ms_total * 1e-3)
        fl = 2 * (2 * (inp.p + 2) + 5)
        if distort > 0:   # general quads: (p+1)^2 (4(p+1)+4) FMAs per element over p^2 DOFs, + 5 updates
            fl = 2 * ((inp.p + 1) ** 2 * (4 * (inp.p + 1) + 4) / inp.p ** 2 + 5)
        peak = SMS * (128 if prec == hz.HZ_F32 else 64) * 2 * CLK
        # the paper's normaliser: one evaluation of the global operator (fp64) on a random vector
        v = torch.from_numpy(np.random.default_rng(1).standard_normal(2 * inp.npx * inp.npy)).cuda()
        op_ms = hz.hz_operator_time(ctx, v.data_ptr(), 20)
        print(f"{name} {info.dofs_per_thread} | {info.cluster_size} | {info.dofs_per_sub} | {info.blocks} | {info.threads_per_block} | "
              f"{info.smem_bytes} | {r.sweep_ms_total / reps:.3f} | {rate:.3e} | {rate * fl / peak:.3f} | {op_ms:.4f} | "
              f"{r.sweep_ms_total / reps / op_ms:.1f} |", flush=True)
    finally:
        hz.hz_destroy(ctx)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("which", choices=["cfg2", "cfg3", "cfg4", "cfg5", "quads"])
    ap.add_argument("--scale", type=int, default=4)
    a = ap.parse_args()
    print("| cfg | n | p | sub side | prec | DOF/thread | CTAs/sub | DOF/sub | blocks | threads | smem B | sweep ms | DOF-steps/s | frac of FMA peak | operator ms (fp64) | DDM cycle / operator |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    if a.which in ("cfg2", "cfg3"):
        for prec in (hz.HZ_F32, hz.HZ_F64):
            for k in (1, 9):
                run(int(a.which[3]), prec, k)
    elif a.which == "quads":   # general convex quads (distorted meshes): configs 2, 3 and a degree x side sweep
        for prec in (hz.HZ_F32, hz.HZ_F64):
            run(2, prec, 0, distort=0.2)
            run(3, prec, 0, distort=0.2)
        for p in (1, 2, 3, 4):
            for s in (4, 8, 16):
                for prec in (hz.HZ_F32, hz.HZ_F64):
                    run(5, prec, 0, n=(6144 // p) // a.scale // s * s, p=p, s=s, reps=2, distort=0.2)
    elif a.which == "cfg4":
        for prec in (hz.HZ_F32, hz.HZ_F64):
            for k in (0, 18, 36):
                run(4, prec, k, reps=2)
    else:
        for p in (1, 2, 3, 4):
            for s in (4, 8, 16, 32, 64):
                for prec in (hz.HZ_F32, hz.HZ_F64):
                    run(5, prec, 0, n=6144 // p // a.scale, p=p, s=s, reps=2)


if __name__ == "__main__":
    main()
