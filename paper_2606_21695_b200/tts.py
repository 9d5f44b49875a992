"""DDM time-to-solution (BASELINE.json metric 1) of the two outer drivers, as a markdown table.

    python -m paper_2606_21695_b200.tts [--configs 1 2 3 4] [--max-sweeps 20000]

Global relative residual ||b - (A - i w H - w^2 M) u|| / ||b|| (hz_residual, fp64) to the tolerance of reading
R21 (1e-4 in both precisions; 1e-8 for config 1 in fp64), n_wh = 2, rho = 0.5, warm start.  Drivers:
hz_ddm_solve (relaxed fixed-point iteration, CUDA-graph replay between residual checks) and hz_ddm_solve_gmres
(restarted GMRES on the joint (lambda, u) state).  Times are device times of the whole call (CUDA events).
"""
from __future__ import annotations

import argparse

from . import hz
from .inputs import make_config


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="+", default=[1, 2, 3, 4])
    ap.add_argument("--max-sweeps", type=int, default=20000)
    a = ap.parse_args()
    print("| cfg | prec | tol | driver | sweeps | residual reached | device ms | note |")
    print("|---|---|---|---|---|---|---|---|")
    for cfg in a.configs:
        inp = make_config(cfg)
        cases = [("f64", 1e-8), ("f32", 1e-4)] if cfg == 1 else [("f32", 1e-4), ("f64", 1e-4)]
        for pr, tol in cases:
            prec = hz.HZ_F32 if pr == "f32" else hz.HZ_F64
            try:
                ctx, info = hz.setup_from_inputs(inp, prec, 0)
            except hz.HzError as e:
                print(f"| {cfg} | {pr} | {tol:g} | — | — | — | — | {e} |", flush=True)
                continue
            every = 10 if cfg == 1 else 50
            restart = 50 if cfg <= 2 else 100
            if info.dofs_per_thread == -1:
                note = "streamed variant (state does not fit one SM)"
                budget = min(a.max_sweeps, 400)
            else:
                note, budget = "", a.max_sweeps
            hz.hz_ddm_solve(ctx, every, n_wh=2, reset_state=True, use_graph=True)
            s = hz.hz_ddm_solve(ctx, budget, n_wh=2, relax=0.5, tol=tol, check_every=every, reset_state=True, use_graph=True)
            ok = "" if s.rel_residual <= tol else "NOT reached; "
            print(f"| {cfg} | {pr} | {tol:g} | fixed point, rho=0.5 | {s.n_outer_done} | {s.rel_residual:.2e} | {s.total_ms:.1f} | "
                  f"{ok}{note} |", flush=True)
            hz.hz_ddm_solve_gmres(ctx, 3, n_wh=2, restart=restart)
            g = hz.hz_ddm_solve_gmres(ctx, min(budget, 4000), n_wh=2, relax=0.5, restart=restart, tol=tol, reset_state=True)
            ok = "" if g.rel_residual <= tol else "NOT reached; "
            print(f"| {cfg} | {pr} | {tol:g} | GMRES({restart}) | {g.sweeps_done} | {g.rel_residual:.2e} | {g.total_ms:.1f} | "
                  f"{ok}{note} |", flush=True)
            hz.hz_destroy(ctx)


if __name__ == "__main__":
    main()
