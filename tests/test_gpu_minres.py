"""GPU parity of the block-level MINRES comparator (hz_minres_cycle) against the oracle's MINRES on the block
system (5), and the WaveHoltz-vs-MINRES comparison at equal subdomain residual."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import hz_oracle as O  # noqa: E402
from paper_2606_21695_b200 import hz  # noqa: E402
from paper_2606_21695_b200.inputs import make_config  # noqa: E402
from test_gpu_parity import hetero_inputs, oracle_state_arrays, pack_bc, problem_from, rel  # noqa: E402


def gpu_state(ctx, info):
    usub = torch.zeros(info.blocks * 2 * info.dofs_per_sub, dtype=torch.float64, device="cuda")
    lam = torch.zeros(info.blocks * 8 * info.edge_stride, dtype=torch.float64, device="cuda")
    hz.hz_get_subdomain_state(ctx, usub.data_ptr(), lam.data_ptr())
    return (usub.cpu().numpy().reshape(info.blocks, 2, info.dofs_per_sub),
            lam.cpu().numpy().reshape(info.blocks, 4, 2, info.edge_stride))


@pytest.mark.parametrize("k", [1, 9])
@pytest.mark.parametrize("fixed_iters", [True, False])
def test_minres_cycles_match_the_oracle_fp64(fixed_iters, k):
    """Two outer iterations (so that lambda != 0 and the warm start are exercised).  With a fixed iteration
    count the iterates must agree; run to tolerance, the iteration counts must agree as well."""
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = hetero_inputs(6, 4, 3, 3, 2, seed=21, complex_f=(k == 1))   # the register-blocked partitions take a real f
    rng = np.random.default_rng(9)
    bc = [rng.standard_normal(n) + 1j * rng.standard_normal(n) for n in (inp.npy, inp.npy, inp.npx, inp.npx)]
    tol, maxit = (0.0, 40) if fixed_iters else (1e-12, 5000)
    pr = problem_from(inp, bc)
    st = O.ddm_setup(pr, inp.sx, inp.sy, inp.cfl_frac)
    its_o = [O.ddm_sweep_minres(st, tol, maxit, warm, 0.5) for warm in (False, True)]
    ctx = hz.hz_mesh_setup(inp.nx, inp.ny, inp.x0, inp.y0, inp.x1, inp.y1, inp.p, inp.c_nodes, inp.omega, inp.f_re,
                           inp.f_im, pack_bc(inp, bc))
    try:
        # k = 1: one DOF per thread; k = 9: the register-blocked layout of the WaveHoltz kernels (k_minres_tile)
        info = hz.hz_partition_ex(ctx, inp.sx, inp.sy, prec=hz.HZ_F64, dofs_per_thread=k, pack=1)
        assert info.dofs_per_thread == k
        hz.hz_ddm_solve(ctx, 0, reset_state=True)
        its_g = []
        for warm in (False, True):
            mi, iters, res = hz.hz_minres_cycle(ctx, info.blocks, tol, maxit, warm_start=warm, relax=0.5)
            its_g.append(list(iters))
        usub, lam = gpu_state(ctx, info)
    finally:
        hz.hz_destroy(ctx)
    u_o, lam_o = oracle_state_arrays(st)
    if fixed_iters:
        assert its_g == its_o == [[40] * 6, [40] * 6]
        assert rel(usub, u_o) <= 1e-9 and rel(lam, lam_o) <= 1e-9, (rel(usub, u_o), rel(lam, lam_o))
    else:
        # close to machine precision the stopping iteration depends on rounding (loss of Lanczos orthogonality)
        assert all(abs(a - b) <= max(10, b // 10) for ga, oa in zip(its_g, its_o) for a, b in zip(ga, oa)), (its_g, its_o)
        assert res.max() <= 5e-12
        assert rel(usub, u_o) <= 1e-8 and rel(lam, lam_o) <= 1e-8, (rel(usub, u_o), rel(lam, lam_o))


@pytest.mark.parametrize("p,k,prec,iters,tol", [(1, 4, hz.HZ_F64, 25, 1e-10), (1, 16, hz.HZ_F64, 25, 1e-10),
                                                (2, 4, hz.HZ_F64, 25, 1e-10), (2, 16, hz.HZ_F64, 25, 1e-10),
                                                (3, 9, hz.HZ_F64, 25, 1e-10), (4, 16, hz.HZ_F64, 25, 1e-10),
                                                (3, 1, hz.HZ_F64, 25, 1e-10),
                                                (3, 1, hz.HZ_F32, 15, 1e-4), (3, 9, hz.HZ_F32, 15, 1e-4),
                                                (1, 16, hz.HZ_F32, 15, 1e-4), (4, 16, hz.HZ_F32, 15, 1e-4)])
def test_minres_first_iterates_in_every_layout(p, k, prec, iters, tol):
    """The first N MINRES iterates (before the Lanczos recurrence has had time to amplify the different summation
    orders of the block reductions) at north_star's bars, 1e-10 in fp64 and 1e-4 in fp32, in the one-DOF-per-thread
    layout and in every register-blocked tile the comparator is compiled for; ragged tile rows / columns included."""
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = hetero_inputs(8, 8, p, 2, 2, seed=500 + 10 * p + k)
    pr = problem_from(inp)
    st = O.ddm_setup(pr, inp.sx, inp.sy, inp.cfl_frac)
    rng = np.random.default_rng(3)
    for l in range(len(st.subs)):           # a non-trivial interface vector on both sides
        st.lam[l] = [rng.standard_normal(len(a)) + 1j * rng.standard_normal(len(a)) if st.subs[l].neighbour[s] >= 0 else a
                     for s, a in enumerate(st.lam[l])]
    u0, lam0 = oracle_state_arrays(st)
    O.ddm_sweep_minres(st, 0.0, iters, False, 0.5)
    ctx = hz.hz_mesh_setup(inp.nx, inp.ny, inp.x0, inp.y0, inp.x1, inp.y1, inp.p, inp.c_nodes, inp.omega, inp.f_re)
    try:
        info = hz.hz_partition_ex(ctx, inp.sx, inp.sy, prec=prec, dofs_per_thread=k, pack=1)
        assert info.dofs_per_thread == k
        hz.hz_ddm_solve(ctx, 0, reset_state=True)
        hz.hz_set_subdomain_state(ctx, None, torch.from_numpy(lam0).cuda().data_ptr())
        mi, it_g, res = hz.hz_minres_cycle(ctx, info.blocks, 0.0, iters, warm_start=False, relax=0.5)
        assert list(it_g) == [iters] * info.blocks
        usub, lam = gpu_state(ctx, info)
    finally:
        hz.hz_destroy(ctx)
    u_o, lam_o = oracle_state_arrays(st)
    assert rel(usub, u_o) <= tol and rel(lam, lam_o) <= tol, (rel(usub, u_o), rel(lam, lam_o))


@pytest.mark.parametrize("k", [1, 9])
def test_minres_fp32_reaches_the_papers_single_precision_tolerance(k):
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = make_config(2, n=32)
    pr = problem_from(inp)
    st = O.ddm_setup(pr, inp.sx, inp.sy, inp.cfl_frac)
    O.ddm_sweep_minres(st, 1e-12, 20000, False, 0.5)
    ctx, info = hz.setup_from_inputs(inp, hz.HZ_F32, k)
    try:
        hz.hz_ddm_solve(ctx, 0, reset_state=True)
        mi, iters, res = hz.hz_minres_cycle(ctx, info.blocks, 1e-6, 20000, relax=0.5)
        usub, lam = gpu_state(ctx, info)
    finally:
        hz.hz_destroy(ctx)
    u_o, lam_o = oracle_state_arrays(st)
    # The recurrence stops at 1e-6, but in fp32 the Lanczos vectors lose orthogonality and the TRUE residual
    # stagnates one to two digits above it (measured 1.5e-5 .. 9e-5; the paper makes the same observation,
    # PAPER.md:275).  The comparator is therefore held to the true residual it can reach, not to 1e-4 parity.
    assert res.max() <= 5e-4, res.max()
    assert rel(usub, u_o) <= 1e-4 and rel(lam, lam_o) <= 1e-4, (rel(usub, u_o), rel(lam, lam_o))
    print("fp32 MINRES: true residual max", res.max(), "rel u", rel(usub, u_o), "iters", iters.max())


def test_zero_iterations_reports_the_subdomain_residual_of_waveholtz():
    """max_iters = 0, warm start: the kernel only evaluates ||rhs - K u_l|| / ||rhs||, which is how the
    WaveHoltz-vs-MINRES comparison finds the n_wh that reaches MINRES's tolerance."""
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = make_config(2, n=16)
    ctx, info = hz.setup_from_inputs(inp, hz.HZ_F64, 1)
    try:
        prev = None
        for n_wh in (2, 10, 40):
            hz.hz_ddm_solve(ctx, 1, n_wh=n_wh, warm_start=False, reset_state=True)
            # lambda was exchanged by the sweep; evaluate against the lambda the sweep used: reset it to zero
            lam0 = torch.zeros(info.blocks * 8 * info.edge_stride, dtype=torch.float64, device="cuda")
            hz.hz_set_subdomain_state(ctx, None, lam0.data_ptr())
            mi, iters, res = hz.hz_minres_cycle(ctx, info.blocks, 0.0, 0, warm_start=True)
            assert iters.max() == 0
            active = res[res > 0]
            if prev is not None:
                assert active.max() < prev
            prev = active.max()
        assert prev < 1e-6
        # oracle cross-check of the residual definition on one subdomain
        st = O.ddm_setup(problem_from(inp), inp.sx, inp.sy, inp.cfl_frac)
        l = int(np.argmax(res))
        u, g = O.ddm_cycle(st, l, 40, False)
        sd = st.subs[l]
        K, rhs = O.block_system(sd.A, sd.M, sd.H, sd.bf, st.pr.omega)
        r_o = np.linalg.norm(rhs - K @ np.concatenate([u.real, u.imag])) / np.linalg.norm(rhs)
        assert abs(res[l] - r_o) <= 1e-6 * r_o + 1e-14
    finally:
        hz.hz_destroy(ctx)
