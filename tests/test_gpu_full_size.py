"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (auto variant), on
sampled outputs the oracle can compute one by one: after 2 sweeps, subdomain l's state depends only on
l and its 4 neighbours (sweep 1 of each starts from lambda = 0, u = 0), so the oracle runs the DDM
cycle (oracle.hz_oracle.ddm_cycle) on those 5 subdomains, the exchange on l's sides, and cycle 2 on l.
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
