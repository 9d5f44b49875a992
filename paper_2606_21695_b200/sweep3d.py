"""Throughput of the 3-D sweep kernel over the block shapes of PAPER.md:265 (run under gpurun):

    python -m paper_2606_21695_b200.sweep3d
    python -m paper_2606_21695_b200.sweep3d tts      # time to solution (residual-based stop)

DOF-steps/s of the sweep kernel alone (CUDA events inside hz3_ddm_solve), n_wh = 5, warm start; frac = rate x
2(3(2p+1)+5) / FMA peak: the (2p+1)-wide band rows of the three directions + 5 updates per DOF-step, as executed by
the one-node-per-thread kernel.  The last two columns are the paper's Fig. 6 quantity: the time of one DDM cycle (5
WaveHoltz iterations on every subdomain) over the time of one evaluation of the global Helmholtz operator."""
from __future__ import annotations

import numpy as np
import torch

from . import hz, hz3
from .inputs import make_config_3d

SMS, CLK = 148, 1.965e9


def run(n, p, s, prec):
    inp = make_config_3d(n, p, s)
    ctx = hz3.hz3_mesh_setup(inp.nx, inp.ny, inp.nz, inp.box, inp.p, inp.c_nodes, inp.omega, inp.f_re)
    try:
        info = hz3.hz3_partition(ctx, inp.sx, inp.sy, inp.sz, prec)
        hz3.hz3_ddm_solve(ctx, 1, n_wh=5, reset_state=True)
        r = hz3.hz3_ddm_solve(ctx, 3, n_wh=5)
        rate = r.dof_timesteps / (r.sweep_ms_total * 1e-3)
        # the paper's normaliser: one evaluation of the global operator on a random vector
        nn = int(np.prod(inp.shape))
        v = torch.from_numpy(np.random.default_rng(1).standard_normal(2 * nn)).cuda()
        op_ms = hz3.hz3_operator_time(ctx, v.data_ptr(), 20)
        fl = 2 * (3 * (2 * p + 1) + 5)
        peak = SMS * (128 if prec == hz.HZ_F32 else 64) * 2 * CLK
        print(f"| {inp.nx}^3 | {p} | {s}^3 | {'f32' if prec == hz.HZ_F32 else 'f64'} | {info.dofs_per_sub} | {info.blocks} | "
              f"{info.threads_per_block} | {info.smem_bytes} | {info.n_t} | {r.sweep_ms_total / 3:.3f} | {rate:.3e} | "
              f"{rate * fl / peak:.3f} | {op_ms:.4f} | {r.sweep_ms_total / 3 / op_ms:.1f} |", flush=True)
    finally:
        hz3.hz3_destroy(ctx)


def tts():
    """Time to solution in 3-D: relaxed fixed-point iteration on lambda (n_wh = 2, rho = 0.5, warm start) to a global
    relative residual, checked every 50 sweeps (hz3_solve_opts.tol)."""
    print("| mesh | p | elements per subdomain | prec | subdomains | tol | sweeps | rel. residual (fp64) | device ms |")
    print("|---|---|---|---|---|---|---|---|---|")
    for n, p, s, prec, tol in ((32, 1, 8, hz.HZ_F32, 1e-4), (32, 1, 8, hz.HZ_F64, 1e-6), (24, 3, 3, hz.HZ_F32, 1e-4),
                               (24, 3, 3, hz.HZ_F64, 1e-6)):
        i3 = make_config_3d(n, p, s, ppw=10.0)
        ctx = hz3.hz3_mesh_setup(i3.nx, i3.ny, i3.nz, i3.box, i3.p, i3.c_nodes, i3.omega, i3.f_re)
        try:
            info = hz3.hz3_partition(ctx, i3.sx, i3.sy, i3.sz, prec)
            hz3.hz3_ddm_solve(ctx, 2, n_wh=2, reset_state=True)
            r = hz3.hz3_ddm_solve(ctx, 50000, n_wh=2, reset_state=True, tol=tol, check_every=50)
            print(f"| {n}^3 | {p} | {s}^3 | {'f32' if prec == hz.HZ_F32 else 'f64'} | {info.blocks} | {tol:g} | "
                  f"{r.n_outer_done} | {r.rel_residual:.2e} | {r.total_ms:.1f} |", flush=True)
        finally:
            hz3.hz3_destroy(ctx)


def main():
    import sys
    if len(sys.argv) > 1 and sys.argv[1] == "tts":
        return tts()
    print("| mesh | p | elements per subdomain | prec | DOF/sub | blocks | threads | smem B | N_t | sweep ms | DOF-steps/s | frac of FMA peak | operator ms (fp64) | DDM cycle / operator |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for n, p, s in ((128, 1, 8), (128, 1, 4), (64, 2, 4), (64, 2, 2), (48, 3, 3), (48, 3, 2), (32, 4, 2), (32, 4, 1)):
        for prec in (hz.HZ_F32, hz.HZ_F64):
            run(n, p, s, prec)


if __name__ == "__main__":
    main()
