"""WaveHoltz vs MINRES as the block-level subdomain solver (the paper's Section VII.C / Table I).

    python -m paper_2606_21695_b200.compare_minres [--n 256] [--sides 4 8] [--p 3]

For each subdomain size and precision, on the config-3 medium (random 8x8 blocks of c in [1,3], three Gaussian
sources, ~10 points per wavelength) and a seeded random interface vector lambda (the paper applies the cycle to a
random input vector), so that every subdomain has a non-trivial right-hand side:
  * MINRES on the block system (5), one DOF per thread, from x = 0 until the recurrence's relative residual is
    1e-6 (fp32) / 1e-12 (fp64) -- the paper's tolerances -- and the TRUE residual it reaches (max over subdomains);
  * WaveHoltz from u = 0 with the smallest n_wh whose true subdomain residual (same evaluation kernel) is at
    most max(tolerance, what MINRES truly reached), in the same one-DOF-per-thread layout and in the best
    register-blocked layout.
Prints a markdown table of kernel times (CUDA events) and the speedups.
"""
from __future__ import annotations

import argparse

import numpy as np
import torch

from . import hz
from .inputs import make_config, random_lambda


def waveholtz_to(ctx, info, target, lam0):
    """smallest n_wh (cold start, lambda = 0) with max subdomain residual <= target -> (n_wh, sweep ms, residual)"""
    lo, n_wh = 1, 1
    res = None
    while n_wh <= 4096:
        hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr())
        s = hz.hz_ddm_solve(ctx, 1, n_wh=n_wh, warm_start=False)
        hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr())
        _, _, r = hz.hz_minres_cycle(ctx, info.blocks, 0.0, 0, warm_start=True)
        res = r.max()
        if res <= target:
            break
        lo, n_wh = n_wh, n_wh * 2
    hi = n_wh
    while hi - lo > 1:                       # bisection on n_wh
        mid = (lo + hi) // 2
        hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr())
        hz.hz_ddm_solve(ctx, 1, n_wh=mid, warm_start=False)
        hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr())
        _, _, r = hz.hz_minres_cycle(ctx, info.blocks, 0.0, 0, warm_start=True)
        if r.max() <= target:
            hi = mid
        else:
            lo = mid
    return hi


def timed_sweep(ctx, n_wh, lam0):
    hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr())
    return hz.hz_ddm_solve(ctx, 1, n_wh=n_wh, warm_start=False).sweep_ms_total


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=256)
    ap.add_argument("--p", type=int, default=3)
    ap.add_argument("--sides", type=int, nargs="+", default=[4, 8])
    a = ap.parse_args()
    print("| p | sub side | DOF/sub | blocks | prec | MINRES iters (mean / max) | MINRES true res | MINRES ms | n_wh | "
          "WaveHoltz ms, 1 DOF/thread | WaveHoltz ms, register-blocked (k) | speedup same layout | speedup best |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for side in a.sides:
        n = a.n - a.n % side
        inp = make_config(3, n=n, p=a.p, sub_elems=side)
        for prec, tol in ((hz.HZ_F32, 1e-6), (hz.HZ_F64, 1e-12)):
            ctx, info = hz.setup_from_inputs(inp, prec, 1)
            lam_c = random_lambda(np.random.default_rng(42), info.blocks, info.edge_stride)
            lam0 = torch.from_numpy(np.stack([lam_c.real, lam_c.imag], axis=2).copy()).cuda()   # [L][4][2][E]
            hz.hz_ddm_solve(ctx, 0, reset_state=True)
            hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr())
            hz.hz_minres_cycle(ctx, info.blocks, tol, 100000)                    # warm-up
            mi, iters, res = hz.hz_minres_cycle(ctx, info.blocks, tol, 100000)
            target = max(tol, float(res.max()))
            n_wh = waveholtz_to(ctx, info, target, lam0)
            t1 = min(timed_sweep(ctx, n_wh, lam0) for _ in range(4))
            hz.hz_destroy(ctx)
            ctx, info2 = hz.setup_from_inputs(inp, prec, 0)
            tk = min(timed_sweep(ctx, n_wh, lam0) for _ in range(4))
            hz.hz_destroy(ctx)
            print(f"| {a.p} | {side} | {info.dofs_per_sub} | {info.blocks} | {'f32' if prec == hz.HZ_F32 else 'f64'} | "
                  f"{mi.iters_mean:.0f} / {mi.iters_max} | {res.max():.1e} | {mi.kernel_ms:.2f} | {n_wh} | {t1:.2f} | "
                  f"{tk:.2f} ({info2.dofs_per_thread}) | {mi.kernel_ms / t1:.1f}x | {mi.kernel_ms / tk:.1f}x |", flush=True)


if __name__ == "__main__":
    main()
