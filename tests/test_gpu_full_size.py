"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (auto variant), on
sampled outputs the oracle can compute one by one: after 2 sweeps, subdomain l's state depends only on
l and its 4 neighbours (sweep 1 of each starts from lambda = 0, u = 0), so the oracle runs the DDM
cycle (oracle.hz_oracle.ddm_cycle) on those 5 subdomains, the exchange on l's sides, and cycle 2 on l.
For config 5 (65 536 ... 2.4 M subdomains) the oracle is set up on the 3x3 window of subdomains around the
sample only (same elements, wave speed, source and N_t as the full mesh: a subdomain's cycle sees nothing else).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import hz_oracle as O  # noqa: E402
from paper_2606_21695_b200 import hz  # noqa: E402
from paper_2606_21695_b200.inputs import make_config  # noqa: E402

TOL = {hz.HZ_F64: 1e-10, hz.HZ_F32: 1e-4}


def oracle_two_sweeps_on(st, l, n_wh, relax):
    """u_l and lambda_l after 2 sweeps, touching only l and its neighbours."""
    sd = st.subs[l]
    nbs = [r for r in sd.neighbour if r >= 0]
    g, u1 = {}, {}
    for r in [l] + nbs:
        u1[r], g[r] = O.ddm_cycle(st, r, n_wh, True)           # sweep 1 (lambda = 0, u = 0)
    lam1 = [np.zeros_like(a) for a in st.lam[l]]
    for side in range(4):
        r = sd.neighbour[side]
        if r >= 0:
            lam1[side] = (1.0 - relax) * st.lam[l][side] + relax * g[r][O.OPPOSITE[side]]
    st.lam[l] = lam1
    st.u[l] = u1[l]
    u2, g2 = O.ddm_cycle(st, l, n_wh, True)                    # sweep 2 on l
    # lambda_l after the second exchange needs the neighbours' sweep-2 g: not computed; compare u_l and lambda^1
    return u1[l], lam1, u2


@pytest.mark.parametrize("cfg,prec,n_wh", [(2, hz.HZ_F64, 5), (2, hz.HZ_F32, 5), (3, hz.HZ_F32, 5), (3, hz.HZ_F64, 2),
                                           (4, hz.HZ_F32, 1), (4, hz.HZ_F64, 1)])
def test_full_size_sampled_subdomains(cfg, prec, n_wh):
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = make_config(cfg)
    relax = 0.5
    ctx, info = hz.setup_from_inputs(inp, prec, 0)
    try:
        L, N, E = info.blocks, info.dofs_per_sub, info.edge_stride
        usub = torch.zeros(L * 2 * N, dtype=torch.float64, device="cuda")
        lam = torch.zeros(L * 8 * E, dtype=torch.float64, device="cuda")
        hz.hz_ddm_solve(ctx, 1, n_wh=n_wh, warm_start=True, relax=relax, reset_state=True)
        hz.hz_get_subdomain_state(ctx, None, lam.data_ptr())
        lam1_gpu = lam.cpu().numpy().reshape(L, 4, 2, E).copy()
        hz.hz_ddm_solve(ctx, 1, n_wh=n_wh, warm_start=True, relax=relax)
        hz.hz_get_subdomain_state(ctx, usub.data_ptr(), None)
        u2_gpu = usub.cpu().numpy().reshape(L, 2, N)
    finally:
        hz.hz_destroy(ctx)
    pr = O.Problem(inp.nx, inp.ny, inp.p, inp.x0, inp.y0, inp.x1, inp.y1, inp.c_nodes, inp.omega,
                   inp.f_re.astype(complex))
    st = O.ddm_setup(pr, inp.sx, inp.sy, inp.cfl_frac)
    assert st.tab.n_t == info.n_t
    rng = np.random.default_rng(7)
    # the subdomain holding the (first) source, a corner, an edge and a random interior one
    xs, ys = inp.meta["sources"][0]
    src = min(int(ys * inp.sy), inp.sy - 1) * inp.sx + min(int(xs * inp.sx), inp.sx - 1)
    picks = {src, 0, inp.sx - 1, (inp.sy - 1) * inp.sx + inp.sx // 2}
    if cfg != 4:
        picks.add(int(rng.integers(0, L)))
    else:
        picks = {src, 0}
    tol = TOL[prec]
    scale = max(np.abs(u2_gpu).max(), 1e-300)
    for l in sorted(picks):
        u1, lam1, u2 = oracle_two_sweeps_on(st, l, n_wh, relax)
        ug = u2_gpu[l, 0] + 1j * u2_gpu[l, 1]
        # relative to the subdomain's own norm, or to the global field scale where the wave has not arrived yet
        den = max(np.linalg.norm(u2), 1e-6 * scale * np.sqrt(N))
        assert np.linalg.norm(ug - u2) / den <= tol, (cfg, l, np.linalg.norm(ug - u2) / den)
        for s in range(4):
            lg = lam1_gpu[l, s, 0, :len(lam1[s])] + 1j * lam1_gpu[l, s, 1, :len(lam1[s])]
            dl = max(np.linalg.norm(lam1[s]), 1e-6 * np.abs(lam1_gpu).max() * np.sqrt(len(lam1[s])))
            if np.linalg.norm(lam1[s]) > 0:
                assert np.linalg.norm(lg - lam1[s]) / dl <= tol, (cfg, l, s)
        # back to the initial state (lambda = 0, u = 0) for the next sample
        st.lam[l] = [np.zeros(len(a), dtype=complex) for a in lam1]
        st.u[l] = np.zeros(N, dtype=complex)


def window_problem(inp, l, n_t):
    """The oracle's DDM state of the (at most) 3x3 subdomains around subdomain l of the full problem, and l's index
    in it.  Outer sides of the window that are interfaces of the full problem only carry lambda = 0 during the two
    sweeps that are compared, exactly like a physical side with zero datum."""
    ex, ey, p = inp.nx // inp.sx, inp.ny // inp.sy, inp.p
    ix, iy = l % inp.sx, l // inp.sx
    ix0, ix1 = max(ix - 1, 0), min(ix + 1, inp.sx - 1)
    iy0, iy1 = max(iy - 1, 0), min(iy + 1, inp.sy - 1)
    hx, hy = (inp.x1 - inp.x0) / inp.nx, (inp.y1 - inp.y0) / inp.ny
    I0, I1, J0, J1 = ix0 * ex * p, (ix1 + 1) * ex * p + 1, iy0 * ey * p, (iy1 + 1) * ey * p + 1
    pr = O.Problem((ix1 - ix0 + 1) * ex, (iy1 - iy0 + 1) * ey, p, inp.x0 + ix0 * ex * hx, inp.y0 + iy0 * ey * hy,
                   inp.x0 + (ix1 + 1) * ex * hx, inp.y0 + (iy1 + 1) * ey * hy, inp.c_nodes[J0:J1, I0:I1].copy(), inp.omega,
                   inp.f_re[J0:J1, I0:I1].astype(complex))
    st = O.ddm_setup(pr, ix1 - ix0 + 1, iy1 - iy0 + 1, inp.cfl_frac, n_t=n_t)
    return st, (iy - iy0) * (ix1 - ix0 + 1) + (ix - ix0)


@pytest.mark.parametrize("p,s,prec,n_wh", [(3, 8, hz.HZ_F32, 5), (3, 8, hz.HZ_F64, 2), (1, 4, hz.HZ_F32, 2),
                                           (4, 64, hz.HZ_F32, 1), (2, 64, hz.HZ_F64, 1)])
def test_config5_full_size_sampled_subdomains(p, s, prec, n_wh):
    """Config 5 on its full 6145^2-node mesh: the headline workload of bench.py (p = 3, 8x8-element subdomains) and
    three corners of the sweep.  Also checks that a reduced mesh with `grid_blocks` gets this launch shape."""
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = make_config(5, n=6144 // p, p=p, sub_elems=s)
    relax = 0.5
    ctx, info = hz.setup_from_inputs(inp, prec, 0)
    try:
        L, N, E = info.blocks, info.dofs_per_sub, info.edge_stride
        xs, ys = inp.meta["sources"][0]
        src = min(int(ys * inp.sy), inp.sy - 1) * inp.sx + min(int(xs * inp.sx), inp.sx - 1)
        picks = sorted({src, 0, (inp.sy - 1) * inp.sx + inp.sx // 2} if s < 64 else {src})
        hz.hz_ddm_solve(ctx, 1, n_wh=n_wh, warm_start=True, relax=relax, reset_state=True)
        lam = torch.zeros(L * 8 * E, dtype=torch.float64, device="cuda")
        hz.hz_get_subdomain_state(ctx, None, lam.data_ptr())
        lam1_gpu = {l: lam.view(L, 4, 2, E)[l].cpu().numpy().copy() for l in picks}
        lam_max = float(lam.abs().max())
        del lam
        hz.hz_ddm_solve(ctx, 1, n_wh=n_wh, warm_start=True, relax=relax)
        usub = torch.zeros(L * 2 * N, dtype=torch.float64, device="cuda")
        hz.hz_get_subdomain_state(ctx, usub.data_ptr(), None)
        u2_gpu = {l: usub.view(L, 2, N)[l].cpu().numpy().copy() for l in picks}
        scale = max(float(usub.abs().max()), 1e-300)
        del usub
    finally:
        hz.hz_destroy(ctx)
    # the launch shape of the reduced-mesh parity tests (tests/test_gpu_config5_shapes.py) is this one
    small = make_config(5, n=max(3, 24 // s) * s, p=p, sub_elems=s)
    c2, i2 = hz.setup_from_inputs(small, prec, 0, grid_blocks=info.blocks)
    hz.hz_destroy(c2)
    assert i2.n_t == info.n_t
    for f in ("dofs_per_sub", "threads_per_block", "dofs_per_thread", "tile_mx", "tile_my", "cluster_size",
              "subs_per_block", "smem_bytes"):
        assert getattr(i2, f) == getattr(info, f), f
    tol = TOL[prec]
    for l in picks:
        st, lw = window_problem(inp, l, info.n_t)
        u1, lam1, u2 = oracle_two_sweeps_on(st, lw, n_wh, relax)
        ug = u2_gpu[l][0] + 1j * u2_gpu[l][1]
        den = max(np.linalg.norm(u2), 1e-6 * scale * np.sqrt(N))
        assert np.linalg.norm(ug - u2) / den <= tol, (p, s, l, np.linalg.norm(ug - u2) / den)
        for sd in range(4):
            n = len(lam1[sd])
            lg = lam1_gpu[l][sd, 0, :n] + 1j * lam1_gpu[l][sd, 1, :n]
            dl = max(np.linalg.norm(lam1[sd]), 1e-6 * lam_max * np.sqrt(n))
            if np.linalg.norm(lam1[sd]) > 0:
                assert np.linalg.norm(lg - lam1[sd]) / dl <= tol, (p, s, l, sd)
